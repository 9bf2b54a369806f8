"""Oracle of the optimal image-domain-gridding taper.

TEST INFRASTRUCTURE ONLY: importable from tests/ (and bench.py's reference legs); it imports nothing from the
product package and the product never imports it.  Arbitrary-precision arithmetic with mpmath, which is what the
paper says Table 1 was made with.

What it computes, in the paper's order and notation (section 4.3, Appendix A):
  * the effective window of a taper {a_k} for a sample shifted s pixels from the subgrid centre (Eq. 31-33,
    PAPER.md:388-404; Appendix A works in PIXEL units, x in [0, L) is the main lobe):
        f(x, s) = sum_k a_k exp(j 2 pi k s / L) sinc(x - k) exp(-j 2 pi x s / L)
  * the cost = mean over the allowed shifts |s| <= (L - beta + 1)/2 (text PAPER.md:408, A.5 PAPER.md:568; Eq. 34
    prints (L - beta - 1)/2, taken as a typo: reading R16) of the side-lobe energy
    int_{-inf}^{0} |f|^2 dx + int_{L}^{inf} |f|^2 dx = a^H R-bar a, R-bar = Q-bar (.) S-bar (A.3)
  * Q-bar from the closed form A.6 / A.7 (Ci is the standard cosine integral, the sign of A.7
    as printed is a typo), S-bar = sinc((k - l)(L - beta + 1)/L) (A.8; the last printed line
    "sin(.../N)" is the normalised sinc of the line above it)
  * the optimal taper = eigenvector of the smallest eigenvalue, epsilon = sqrt(lambda_min) (Eq. 36-37,
    PAPER.md:425-433).
Reading R16: Table 1 is reproduced -- all 38 IDG entries within 0.5 %, its printing
precision -- when the minimisation runs over the coefficients a_1 .. a_{L-1} with a_0 = 0.  That window is
symmetric about pixel L/2, the centre pixel of a subgrid (R1, R3: l_i = (i - L/2) S / L), and pixel 0, the one
pixel without a mirror partner (l = -S/2), carries no weight.  Minimising over all L coefficients instead gives
levels 0.5-14 % below the table and a window centred between pixels L/2 - 1 and L/2, which the method cannot use.

Pins (tests/test_taper_pins.py): a^H R-bar a against brute-force quadrature of Eq. 31 + Eq. 34; the PSWF column of
Table 1 (epsilon^2 = 1 - lambda_0(beta pi / 2), Eq. 26-29) from an independent Nystrom
eigen-solve, which fixes the epsilon convention; Table 1's IDG columns (tests/golden/table1_aliasing.txt).
"""
from __future__ import annotations

import mpmath as mp

DPS = 50      # decimal digits of every computation here: lambda_min reaches 2e-19 (beta = 15) next to eigenvalues ~ 1


def _h(y):
    """Ci(2 pi |y|) - ln|y| with its finite limit gamma + ln(2 pi) at y = 0 (the two singular terms of A.6 cancel)."""
    if y == 0:
        return mp.euler + mp.log(2 * mp.pi)
    return mp.ci(2 * mp.pi * abs(y)) - mp.log(abs(y))


def _G(y, d):
    """Antiderivative (vanishing at +-infinity) of sinc(y) sinc(y - d), integer d != 0: A.6 with
    sinc(y) sinc(y - d) = (-1)^d sin^2(pi y) / (pi^2 y (y - d))."""
    return mp.mpf((-1) ** d) / (2 * mp.pi ** 2 * d) * (_h(y) - _h(y - d))


def _H(y):
    """Antiderivative of sinc^2(y), odd in y, H(+-inf) = +-1/2 (the k = l entries, which A.6 leaves out)."""
    if y == 0:
        return mp.mpf(0)
    return -mp.sin(mp.pi * y) ** 2 / (mp.pi ** 2 * y) + mp.si(2 * mp.pi * y) / mp.pi


def qbar(L: int):
    """Q-bar[k][l] = int_{-inf}^{0} sinc(x-k) sinc(x-l) dx + int_{L}^{inf} ... dx (A.4; its upper
    integral runs from L and over Q(x): the printed "I" and "R(x)" are typos)."""
    with mp.workdps(DPS):
        Q = mp.zeros(L, L)
        half = mp.mpf(1) / 2
        for k in range(L):
            for l in range(k, L):
                d = l - k
                if d == 0:
                    v = (_H(mp.mpf(-k)) + half) + (half - _H(mp.mpf(L - k)))
                else:
                    v = _G(mp.mpf(-k), d) - _G(mp.mpf(L - k), d)
                Q[k, l] = Q[l, k] = v
        return Q


def sbar(L: int, beta):
    """S-bar[k][l] = mean over |s| <= (L - beta + 1)/2 of exp(j 2 pi (k - l) s / L) (A.5, A.8 PAPER.md:568-587)."""
    with mp.workdps(DPS):
        w = mp.mpf(L) - mp.mpf(beta) + 1
        S = mp.zeros(L, L)
        for k in range(L):
            for l in range(L):
                S[k, l] = mp.sincpi(mp.mpf(k - l) * w / L)
        return S


def rbar(L: int, beta, Q=None):
    """R-bar = Q-bar (.) S-bar, element-wise (A.3)."""
    with mp.workdps(DPS):
        Q = qbar(L) if Q is None else Q
        S = sbar(L, beta)
        R = mp.zeros(L, L)
        for k in range(L):
            for l in range(L):
                R[k, l] = Q[k, l] * S[k, l]
        return R


def optimal_taper(L: int, beta, Q=None):
    """-> (a[0..L-1] as mpf with a[0] = 0, unit norm, positive; epsilon).  Eq. 36-37 over the
    coefficients a_1 .. a_{L-1} (reading R16)."""
    with mp.workdps(DPS):
        R = rbar(L, beta, Q)
        sub = mp.matrix(L - 1, L - 1)
        for i in range(1, L):
            for j in range(1, L):
                sub[i - 1, j - 1] = R[i, j]
        E, V = mp.eigsy(sub)
        i_min = min(range(L - 1), key=lambda i: E[i])
        vec = [V[r, i_min] for r in range(L - 1)]
        if sum(vec) < 0:
            vec = [-v for v in vec]
        return [mp.mpf(0)] + vec, mp.sqrt(E[i_min])


def sidelobe_level(a, L: int, beta, R=None):
    """epsilon of ANY taper a[0..L-1]: sqrt(a^T R-bar a / a^T a) (Eq. 35 PAPER.md:414 over the energy of the window)."""
    with mp.workdps(DPS):
        R = rbar(L, beta) if R is None else R
        num = mp.mpf(0)
        for k in range(L):
            for l in range(L):
                num += mp.mpf(a[k]) * R[k, l] * mp.mpf(a[l])
        den = sum(mp.mpf(x) ** 2 for x in a)
        return mp.sqrt(num / den)


def pswf_epsilon(beta):
    """Classical gridding with the prolate spheroidal wave function (section 4.1): epsilon^2 = 1 - lambda_0(alpha),
    alpha = beta pi / 2 (Eq. 27-28).  lambda_0 is the largest eigenvalue of the concentration
    operator of Eq. 26 (Slepian & Pollak 1961): kernel sin(alpha (x - y)) / (pi (x - y)) on [-1, 1],
    discretised with Gauss-Legendre nodes (Nystrom), symmetrised with the square roots of the weights."""
    with mp.workdps(DPS):
        alpha = mp.mpf(beta) * mp.pi / 2
        nodes = mp.calculus.quadrature.GaussLegendre(mp.mp).calc_nodes(6, mp.mp.prec)   # 3 * 2^5 = 96 nodes (48 already agree to 6 digits)
        xs = [x for x, _ in nodes]
        ws = [w for _, w in nodes]
        n = len(xs)
        K = mp.matrix(n, n)
        for i in range(n):
            for j in range(i, n):
                d = xs[i] - xs[j]
                v = alpha / mp.pi if d == 0 else mp.sin(alpha * d) / (mp.pi * d)
                K[i, j] = K[j, i] = mp.sqrt(ws[i]) * v * mp.sqrt(ws[j])
        E = mp.eigsy(K, eigvals_only=True)
        return mp.sqrt(1 - max(E))
