"""Pins of oracle/taper_oracle.py (NEXT-2: optimal IDG taper, section 4.3 + Appendix A), all CPU.

(i)   a^H R-bar a of the closed forms (A.4-A.8) against a brute-force quadrature of the DEFINITION: the effective
      window of Eq. 31, its side-lobe energy and the mean over the shifts of Eq. 34
      -- numpy Gauss-Legendre, none of the oracle's formulas;
(ii)  the PSWF column of Table 1 from an independent Nystrom eigen-solve of Eq. 26-28: fixes what "epsilon" is;
(iii) the IDG columns of Table 1 (tests/golden/table1_aliasing.txt), all 38 entries, to the table's precision;
(iv)  invariants of the optimal window.
"""
import os

import mpmath as mp
import numpy as np
import pytest

from oracle import taper_oracle as T

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "table1_aliasing.txt")


def read_table1():
    rows = {}
    for line in open(GOLDEN):
        if line.startswith("#") or not line.strip():
            continue
        f = line.split()
        rows[float(f[0])] = [None if x == "-" else float(x) for x in f[1:]]
    return rows          # beta -> [PSWF, L=8, 16, 24, 32, 48, 64]


SIZES = (8, 16, 24, 32, 48, 64)


def _gauss_legendre(a, b, n):
    x, w = np.polynomial.legendre.leggauss(n)
    return 0.5 * (b - a) * x + 0.5 * (a + b), 0.5 * (b - a) * w


def _mainlobe_energy_mean_over_shifts(a, L, beta):
    """mean_s int_0^L |f(x, s)|^2 dx with f of Eq. 31 in the pixel units of Appendix A, by brute force."""
    a = np.asarray(a, dtype=np.float64)
    k = np.arange(L)
    half = 0.5 * (L - beta + 1)
    ss, ws = _gauss_legendre(-half, half, 48)
    total = 0.0
    for s, w_s in zip(ss, ws):
        coef = a * np.exp(2j * np.pi * k * s / L)                  # a_k z_k(s), Eq. 31 / 33
        e = 0.0
        for p in range(L):                                         # panel per pixel: sinc is smooth inside
            xs, wx = _gauss_legendre(p, p + 1, 24)
            f = (coef[None, :] * np.sinc(xs[:, None] - k[None, :])).sum(axis=1)     # |z*(x, s)| = 1
            e += float((wx * np.abs(f) ** 2).sum())
        total += w_s * e
    return total / (2 * half)


@pytest.mark.parametrize("L,beta", [(8, 3.0), (12, 5.0), (16, 4.5)])
def test_quadratic_form_equals_brute_force_quadrature_of_eq31_eq34(L, beta):
    rng = np.random.default_rng(L)
    a = rng.standard_normal(L)
    R = T.rbar(L, beta)
    closed = float(sum(mp.mpf(a[i]) * R[i, j] * mp.mpf(a[j]) for i in range(L) for j in range(L)))
    # side lobes = everything outside [0, L): total energy minus main lobe.  The integer shifts of sinc are
    # orthonormal (Shannon), so the total is sum a_k^2; checked below by quadrature over a wide range.
    brute = float(a @ a) - _mainlobe_energy_mean_over_shifts(a, L, beta)
    assert abs(closed - brute) < 1e-9 * float(a @ a)
    # a dropped term, a wrong sign or a wrong limit shows: perturbing beta changes the form
    R2 = T.rbar(L, beta + 0.5)
    other = float(sum(mp.mpf(a[i]) * R2[i, j] * mp.mpf(a[j]) for i in range(L) for j in range(L)))
    assert abs(other - brute) > 1e-4 * float(a @ a)


def test_total_energy_is_the_sum_of_squares():
    """Parseval for the sinc interpolation used above, by quadrature over |x| < 4000 (tail ~ 1/x)."""
    L = 6
    a = np.array([0.3, -1.0, 0.7, 2.0, 0.1, -0.4])
    k = np.arange(L)
    e = 0.0
    for p in range(-4000, 4000):
        xs, wx = _gauss_legendre(p, p + 1, 8)
        f = (a[None, :] * np.sinc(xs[:, None] - k[None, :])).sum(axis=1)
        e += float((wx * f ** 2).sum())
    assert abs(e - float(a @ a)) < 2e-3 * float(a @ a)


def test_pswf_column_of_table1():
    """Eq. 28: epsilon_PSWF^2 = 1 - lambda_0(beta pi / 2)."""
    table = read_table1()
    for beta in (3.0, 7.0, 11.0, 15.0):
        got = float(T.pswf_epsilon(beta))
        assert abs(got / table[beta][0] - 1.0) < 5e-3, (beta, got)


def test_idg_columns_of_table1_all_entries():
    """All 38 printed entries within 0.5 % (the table has three significant digits)."""
    table = read_table1()
    worst = 0.0
    n = 0
    for j, L in enumerate(SIZES):
        Q = T.qbar(L)
        for beta, row in table.items():
            want = row[1 + j]
            if want is None:
                continue
            _, eps = T.optimal_taper(L, beta, Q=Q)
            worst = max(worst, abs(float(eps) / want - 1.0))
            n += 1
    assert n == 38
    assert worst < 5e-3, worst


def test_unrestricted_minimum_is_not_the_table():
    """The reading matters: minimising over all L coefficients (a_0 free) lands 8-14 % below the table."""
    table = read_table1()
    with mp.workdps(T.DPS):
        lam = min(mp.eigsy(T.rbar(8, 5.0), eigvals_only=True))
        assert float(mp.sqrt(lam)) / table[5.0][1] < 0.87


def test_optimal_window_invariants():
    L, beta = 24, 6.0
    mp.mp.dps = T.DPS
    a, eps = T.optimal_taper(L, beta)
    assert a[0] == 0
    for k in range(1, L):
        assert abs(a[k] - a[L - k]) < mp.mpf(10) ** -30         # symmetric about the centre pixel L/2
        assert a[k] > 0
    assert abs(sum(x * x for x in a) - 1) < mp.mpf(10) ** -30
    assert max(range(L), key=lambda k: a[k]) == L // 2
    # it is the minimiser: its level equals epsilon, a prolate (DPSS) window of the same length is worse
    assert abs(T.sidelobe_level(a, L, beta) / eps - 1) < mp.mpf(10) ** -20
    from scipy.signal.windows import dpss
    d = dpss(L, 3.0, sym=False)
    assert float(T.sidelobe_level(list(d), L, beta)) > float(eps)
    # a wider kernel budget lowers the level
    _, eps8 = T.optimal_taper(L, 8.0)
    assert eps8 < eps
