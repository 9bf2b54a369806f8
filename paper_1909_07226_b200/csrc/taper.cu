// taper.cu -- NEXT-2 row of SURVEY.md section 8f: the optimal taper of image domain gridding (offline input of
// the hot path, not on the timed path).
//
// Section 4.3 and Appendix A: the taper {a_k} that minimises the mean, over
// the allowed sample shifts |s| <= (L - beta + 1)/2, of the side-lobe energy of the effective window (Eq. 31, 34),
//   eps^2 = a^H R a,  R = Q (.) S  (A.3),
//   Q[k][l] = int_{-inf}^{0} sinc(x-k) sinc(x-l) dx + int_{L}^{inf} sinc(x-k) sinc(x-l) dx    (A.4; closed form A.6)
//   S[k][l] = sinc((k - l)(L - beta + 1)/L)                                                  (A.8)
// is the eigenvector of R's smallest eigenvalue (Eq. 36-37).  Reading R16: the minimisation runs over
// a_1 .. a_{L-1} with a_0 = 0 -- the window is then symmetric about the subgrid's centre pixel L/2 (R1, R3) and this
// is what reproduces Table 1.
//
// One CTA, FP64.  The closed form needs Ci and Si at integer multiples of 2 pi only (the limits 0 and L are integers):
//   Si(2 pi n) = pi/2 - f(2 pi n),  Ci(2 pi n) = -g(2 pi n),
//   f(x) = int_0^inf e^{-xt}/(1 + t^2) dt,  g(x) = int_0^inf t e^{-xt}/(1 + t^2) dt   (auxiliary functions of the sine
//   and cosine integrals), evaluated by composite Gauss-Legendre quadrature of the smooth, rapidly decaying integrands.
// The eigenproblem (at most 63 x 63) is solved by cyclic Jacobi rotations in shared memory.
// FP64 resolves eps down to ~1e-7 (lambda_min ~ 1e-14 next to eigenvalues ~ 1); below that the returned window is
// still near-optimal (its level is set by the float32 rounding of the output, ~3e-8) but the returned eps is not
// reliable -- the oracle (mpmath) is the reference there.
#include "common.cuh"

namespace idg {

constexpr int kTaperMaxL = 64;
constexpr int kGL = 16;          // Gauss-Legendre points per panel
constexpr int kPanels = 16;      // panels of width 2.5 on u in [0, 40]

// nodes and weights of the kGL-point Gauss-Legendre rule on [-1, 1] (Newton iteration on P_n)
__device__ void gauss_legendre(double *x, double *w) {
  const double pi = 3.14159265358979323846;
  for (int i = 0; i < kGL; ++i) {
    double z = cos(pi * (i + 0.75) / (kGL + 0.5));
    double pp = 1.0;
    for (int it = 0; it < 100; ++it) {
      double p1 = 1.0, p2 = 0.0;
      for (int j = 1; j <= kGL; ++j) {
        const double p3 = p2;
        p2 = p1;
        p1 = ((2.0 * j - 1.0) * z * p2 - (j - 1.0) * p3) / j;
      }
      pp = kGL * (z * p1 - p2) / (z * z - 1.0);
      const double dz = p1 / pp;
      z -= dz;
      if (fabs(dz) < 1e-16) break;
    }
    x[i] = z;
    w[i] = 2.0 / ((1.0 - z * z) * pp * pp);
  }
}

// f(x) and g(x) for x = 2 pi n >= 2 pi: u = x t, f = (1/x) int_0^40 e^{-u}/(1 + u^2/x^2) du (tail < e^{-40})
__device__ void aux_fg(double x, const double *glx, const double *glw, double *f, double *g) {
  double sf = 0.0, sg = 0.0;
  const double hw = 40.0 / kPanels * 0.5;
  for (int p = 0; p < kPanels; ++p) {
    const double mid = (2 * p + 1) * hw;
    for (int i = 0; i < kGL; ++i) {
      const double u = mid + hw * glx[i];
      const double e = exp(-u) / (1.0 + (u / x) * (u / x)) * glw[i] * hw;
      sf += e;
      sg += u * e;
    }
  }
  *f = sf / x;
  *g = sg / (x * x);
}

__global__ void __launch_bounds__(64)
taper_optimal_kernel(int L, double beta, float *__restrict__ taper /*[L][L]*/, double *__restrict__ a_out /*[L]*/,
                     double *__restrict__ eps_out) {
  extern __shared__ double sm[];
  const int n = L - 1;                       // a_1 .. a_{L-1}
  double *A = sm;                            // [n][n]
  double *V = A + n * n;                     // [n][n]
  double *hh = V + n * n;                    // [L + 1]: h(m) = Ci(2 pi m) - ln m, h(0) = gamma + ln(2 pi)
  double *Hs = hh + (L + 1);                 // [L + 1]: H(m) = Si(2 pi m)/pi   (sin^2(pi m) = 0 at integers)
  double *glx = Hs + (L + 1), *glw = glx + kGL;
  __shared__ int s_imin;
  const int tid = threadIdx.x;
  const double pi = 3.14159265358979323846, two_pi = 6.283185307179586476925286766559;

  if (tid == 0) gauss_legendre(glx, glw);
  __syncthreads();
  for (int m = tid; m <= L; m += blockDim.x) {
    if (m == 0) {
      hh[0] = 0.57721566490153286061 + log(two_pi);
      Hs[0] = 0.0;
    } else {
      double f, g;
      aux_fg(two_pi * m, glx, glw, &f, &g);
      hh[m] = -g - log((double)m);
      Hs[m] = (0.5 * pi - f) / pi;
    }
  }
  __syncthreads();
  // R restricted to k, l = 1 .. L-1.  Antiderivatives of A.6: for d = l - k != 0,
  //   G(y, d) = (-1)^d / (2 pi^2 d) (h(|y|) - h(|y - d|)),  Q = G(-k, d) - G(L - k, d);
  // for d = 0, Q = (H(-k) + 1/2) + (1/2 - H(L - k)), H odd.
  const double width = (double)L - beta + 1.0;
  for (int e = tid; e < n * n; e += blockDim.x) {
    const int k = e / n + 1, l = e % n + 1;
    double q;
    if (k == l) {
      q = (0.5 - Hs[k]) + (0.5 - Hs[L - k]);
    } else {
      const int d = l - k;
      const double sgn = (d & 1) ? -1.0 : 1.0;
      const double g_lo = hh[k] - hh[abs(-k - d)];          // y = -k:     |y| = k,     |y - d| = l
      const double g_hi = hh[L - k] - hh[abs(L - k - d)];   // y = L - k:  |y| = L - k, |y - d| = L - l
      q = sgn / (2.0 * pi * pi * d) * (g_lo - g_hi);
    }
    const double arg = (double)(k - l) * width / (double)L;
    const double s = (k == l) ? 1.0 : sinpi(arg) / (pi * arg);
    A[e] = q * s;
    V[e] = (k == l) ? 1.0 : 0.0;
  }
  __syncthreads();

  // cyclic Jacobi: thread i owns row / column index i of every rotation
  for (int sweep = 0; sweep < 30; ++sweep) {
    double off = 0.0;
    if (tid < n)
      for (int j = 0; j < n; ++j)
        if (j != tid) off += A[tid * n + j] * A[tid * n + j];
    // block-wide sum of `off` through shared memory (reuse hh as scratch is not possible: still needed? no -- free now)
    __syncthreads();
    if (tid < n) glx[0] = 0.0;
    __syncthreads();
    if (tid < n) atomicAdd(&glx[0], off);
    __syncthreads();
    const double total_off = glx[0];
    __syncthreads();
    if (total_off < 1e-60) break;
    for (int p = 0; p < n - 1; ++p)
      for (int q = p + 1; q < n; ++q) {
        const double apq = A[p * n + q];
        const double app = A[p * n + p], aqq = A[q * n + q];
        double aip = 0.0, aiq = 0.0, vip = 0.0, viq = 0.0;
        if (tid < n) { aip = A[tid * n + p]; aiq = A[tid * n + q]; vip = V[tid * n + p]; viq = V[tid * n + q]; }
        __syncthreads();
        if (fabs(apq) > 1e-300) {
          const double theta = (aqq - app) / (2.0 * apq);
          const double t = (theta >= 0.0 ? 1.0 : -1.0) / (fabs(theta) + sqrt(theta * theta + 1.0));
          const double c = 1.0 / sqrt(t * t + 1.0), s = t * c;
          if (tid < n) {
            V[tid * n + p] = c * vip - s * viq;
            V[tid * n + q] = s * vip + c * viq;
            if (tid != p && tid != q) {
              const double np_ = c * aip - s * aiq, nq_ = s * aip + c * aiq;
              A[tid * n + p] = np_; A[p * n + tid] = np_;
              A[tid * n + q] = nq_; A[q * n + tid] = nq_;
            } else if (tid == p) {
              A[p * n + p] = app - t * apq;
              A[p * n + q] = 0.0; A[q * n + p] = 0.0;
            } else {
              A[q * n + q] = aqq + t * apq;
            }
          }
        }
        __syncthreads();
      }
  }
  if (tid == 0) {
    int im = 0;
    for (int i = 1; i < n; ++i)
      if (A[i * n + i] < A[im * n + im]) im = i;
    s_imin = im;
    *eps_out = sqrt(fmax(A[im * n + im], 0.0));
  }
  __syncthreads();
  // window: a_0 = 0, a_k = V[k-1][imin], scaled to peak +1 (the centre pixel L/2)
  const int im = s_imin;
  const double peak = V[(L / 2 - 1) * n + im];
  double *a = hh;                            // the tables are no longer needed
  __syncthreads();
  for (int k = tid; k < L; k += blockDim.x) a[k] = k == 0 ? 0.0 : V[(k - 1) * n + im] / peak;
  __syncthreads();
  for (int k = tid; k < L; k += blockDim.x) a_out[k] = a[k];
  for (int e = tid; e < L * L; e += blockDim.x) taper[e] = (float)(a[e / L] * a[e % L]);    // c[i][j] = a_i a_j (Eq. 30)
}

}  // namespace idg

using namespace idg;

extern "C" int idg_taper_optimal(int32_t N, double beta, float *taper_dev, double *a_host, double *epsilon_host,
                                 void *stream) {
  if (N < 4 || N > kTaperMaxL || (N & 1) || !taper_dev || !(beta >= 1.0) || !(beta < (double)N)) return IDG_ERR_INVALID_ARG;
  cudaStream_t s = (cudaStream_t)stream;
  double *out = nullptr;                     // [N] coefficients + epsilon
  IDG_CUDA_TRY(cudaMalloc(&out, sizeof(double) * (N + 1)));
  const int n = N - 1;
  const size_t smem = sizeof(double) * ((size_t)2 * n * n + 2 * (N + 1) + 2 * kGL);
  cudaError_t e = cudaFuncSetAttribute(taper_optimal_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e == cudaSuccess) {
    taper_optimal_kernel<<<1, 64, smem, s>>>(N, beta, taper_dev, out, out + N);
    count_launch();
    e = cudaGetLastError();
  }
  double host[kTaperMaxL + 1];
  if (e == cudaSuccess) e = cudaMemcpyAsync(host, out, sizeof(double) * (N + 1), cudaMemcpyDeviceToHost, s);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s);
  cudaFree(out);
  IDG_CUDA_TRY(e);
  if (a_host) for (int k = 0; k < N; ++k) a_host[k] = host[k];
  if (epsilon_host) *epsilon_host = host[N];
  return IDG_OK;
}
