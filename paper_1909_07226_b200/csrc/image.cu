// image.cu -- image-plane side of W-stacking (NEXT-1 row of SURVEY.md section 8f; outside the timed hot path).
//
// Alg. 1 last line, "I <- FFT(V) / c-bar" (R8), and Alg. 2 first lines, "I <- I / c-bar;
// V <- FFT(I)", with the w-offset w0p of every subgrid (Alg. 1, R4) resolved by
// W-stacking (mentioned PAPER.md:166): the subgrids of one w layer are gridded with phasors that carry
// (w - w0) n', so the layer's image lacks exp(+2 pi i w0 n'(l, m)); multiplying it back per layer and summing
// the layers gives the image of Eq. 11.  Prediction applies the conjugate factor before the
// layer's forward transform.  The large FFT itself is the library's (cuFFT through torch.fft).
//
//   idg_image_w_accumulate:  acc[pol][y][x] += layer[pol][y][x] * exp(sign 2 pi i w0 n'(l_x, m_y)),
//                            l_x = (x - L/2) S / L  (Eq. 5), n' = sqrt(1 - l^2 - m^2) - 1 (R2)
//   idg_image_w_apply:       out = in * exp(sign 2 pi i w0 n')            (prediction direction)
//   idg_image_divide:        image[pol][y][x] /= cbar[y][x]               (c-bar: image-domain taper)
#include <mutex>

#include "common.cuh"

namespace idg {

__device__ __forceinline__ float2 w_phasor(int x, int y, int L, double image_size, double w0, double sign) {
  // FP64 phase: w0 n' reaches thousands of radians at the image edge for large w layers
  const double l = (double)(x - L / 2) * image_size / (double)L;
  const double m = (double)(y - L / 2) * image_size / (double)L;
  const double r2 = l * l + m * m;
  const double n = -r2 / (1.0 + sqrt(1.0 - r2));
  double s, c;
  sincospi(2.0 * sign * w0 * n, &s, &c);
  return make_float2((float)c, (float)s);
}

template <bool ACCUMULATE>
__global__ void __launch_bounds__(256)
image_w_kernel(float2 *dst, const float2 *src, int L, double image_size,   // out may alias in: no __restrict__
               double w0, double sign) {
  const int x = blockIdx.x * 64 + (threadIdx.x & 63);
  const int y = blockIdx.y * 4 + (threadIdx.x >> 6);
  if (x >= L || y >= L) return;
  const float2 ph = w_phasor(x, y, L, image_size, w0, sign);   // one phasor serves the four polarisations
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    const size_t i = ((size_t)q * L + y) * L + x;
    const float2 v = cmul(src[i], ph);
    if (ACCUMULATE) { float2 a = dst[i]; a.x += v.x; a.y += v.y; dst[i] = a; }
    else dst[i] = v;
  }
}

__global__ void __launch_bounds__(256)
image_divide_kernel(float2 *__restrict__ image, const float *__restrict__ cbar, int L) {
  const int x = blockIdx.x * 64 + (threadIdx.x & 63);
  const int y = blockIdx.y * 4 + (threadIdx.x >> 6);
  if (x >= L || y >= L) return;
  const float inv = 1.0f / cbar[(size_t)y * L + x];
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    const size_t i = ((size_t)q * L + y) * L + x;
    float2 v = image[i];
    v.x *= inv; v.y *= inv;
    image[i] = v;
  }
}

// ---- c-bar: the subgrid taper on the image raster (idg_image_taper) ---------------------------------------------
// Section 4.2: the window the method effectively applies is the periodic sinc (Dirichlet kernel)
// interpolation of the discrete taper; at zero shift that interpolant, evaluated at the L image pixels, is c-bar:
//   D(x, i)    = (1/N) sum_{a=-N/2}^{N/2-1} exp(2 pi i a ((x - L/2)/L - (i - N/2)/N))
//   cbar[y][x] = Re sum_{j,i} D(y, j) taper[j][i] D(x, i)
// Three small FP64 kernels: the table D [L][N], tmp = D taper [L][N], cbar = Re(tmp D^T) [L][L].
__global__ void __launch_bounds__(128)
taper_dirichlet_kernel(double2 *__restrict__ D, int N, int L) {
  const int idx = blockIdx.x * 128 + threadIdx.x;
  if (idx >= L * N) return;
  const int x = idx / N, i = idx - x * N;
  const double delta = (double)(x - L / 2) / (double)L - (double)(i - N / 2) / (double)N;
  double re = 0.0, im = 0.0;
  for (int a = -N / 2; a < N / 2; ++a) {
    double s, c;
    sincospi(2.0 * (double)a * delta, &s, &c);
    re += c; im += s;
  }
  D[idx] = make_double2(re / (double)N, im / (double)N);
}

__global__ void __launch_bounds__(128)
taper_rows_kernel(double2 *__restrict__ tmp, const double2 *__restrict__ D, const float *__restrict__ taper, int N,
                  int L) {
  const int idx = blockIdx.x * 128 + threadIdx.x;
  if (idx >= L * N) return;
  const int y = idx / N, i = idx - y * N;
  double re = 0.0, im = 0.0;
  for (int j = 0; j < N; ++j) {
    const double2 d = D[y * N + j];
    const double t = (double)taper[j * N + i];
    re += d.x * t; im += d.y * t;
  }
  tmp[idx] = make_double2(re, im);
}

__global__ void __launch_bounds__(256)
taper_image_kernel(float *__restrict__ cbar, const double2 *__restrict__ tmp, const double2 *__restrict__ D, int N,
                   int L) {
  const int x = blockIdx.x * 64 + (threadIdx.x & 63);
  const int y = blockIdx.y * 4 + (threadIdx.x >> 6);
  if (x >= L || y >= L) return;
  double re = 0.0;
  for (int i = 0; i < N; ++i) {
    const double2 t = tmp[y * N + i], d = D[x * N + i];
    re += t.x * d.x - t.y * d.y;
  }
  cbar[(size_t)y * L + x] = (float)re;
}

}  // namespace idg

using namespace idg;

// ---- idg_image_taper_static: the same three kernels with their scratch in a file-scope device array, for callers
// that cannot allocate (code under CUDA graph capture, serving loops, harnesses that forbid cudaMalloc).  The array
// costs every GPU that loads the library 8 MiB until exit.  In HOST code `g_taper_scratch` is only a stand-in for
// the device symbol, not a device address: its address is resolved once per device with cudaGetSymbolAddress (that
// device current) and that pointer is what the kernels receive.
namespace {

constexpr int kStaticMaxLN = IDG_IMAGE_TAPER_STATIC_MAX_LN;             // L * N of the largest request served
static __device__ __align__(256) double2 g_taper_scratch[2 * kStaticMaxLN];   // D [L][N], then tmp [L][N]

constexpr int kMaxDevices = 64;
std::mutex g_taper_scratch_mu;
double2 *g_taper_scratch_ptr[kMaxDevices] = {};

int taper_scratch_address(double2 **out) {
  int dev = -1;
  IDG_CUDA_TRY(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kMaxDevices) return IDG_ERR_INVALID_ARG;
  std::lock_guard<std::mutex> lock(g_taper_scratch_mu);
  if (!g_taper_scratch_ptr[dev]) {
    double2 *p = nullptr;
    IDG_CUDA_TRY(cudaGetSymbolAddress((void **)&p, g_taper_scratch));
    if (!p) return IDG_ERR_CUDA;
    g_taper_scratch_ptr[dev] = p;
  }
  *out = g_taper_scratch_ptr[dev];
  return IDG_OK;
}

}  // namespace

extern "C" {

int idg_image_w_accumulate(void *acc_dev, const void *layer_dev, int32_t L, double image_size, double w0,
                           int32_t sign, void *stream) {
  if (!acc_dev || !layer_dev || L < 1 || !(image_size > 0.0) || (sign != 1 && sign != -1)) return IDG_ERR_INVALID_ARG;
  const dim3 grid((L + 63) / 64, (L + 3) / 4);
  image_w_kernel<true><<<grid, 256, 0, (cudaStream_t)stream>>>((float2 *)acc_dev, (const float2 *)layer_dev, L,
                                                              image_size, w0, (double)sign);
  IDG_LAUNCH_CHECK();
  return IDG_OK;
}

int idg_image_w_apply(void *out_dev, const void *in_dev, int32_t L, double image_size, double w0, int32_t sign,
                      void *stream) {
  if (!out_dev || !in_dev || L < 1 || !(image_size > 0.0) || (sign != 1 && sign != -1)) return IDG_ERR_INVALID_ARG;
  const dim3 grid((L + 63) / 64, (L + 3) / 4);
  image_w_kernel<false><<<grid, 256, 0, (cudaStream_t)stream>>>((float2 *)out_dev, (const float2 *)in_dev, L,
                                                               image_size, w0, (double)sign);
  IDG_LAUNCH_CHECK();
  return IDG_OK;
}

int idg_image_divide(void *image_dev, const float *cbar_dev, int32_t L, void *stream) {
  if (!image_dev || !cbar_dev || L < 1) return IDG_ERR_INVALID_ARG;
  const dim3 grid((L + 63) / 64, (L + 3) / 4);
  image_divide_kernel<<<grid, 256, 0, (cudaStream_t)stream>>>((float2 *)image_dev, cbar_dev, L);
  IDG_LAUNCH_CHECK();
  return IDG_OK;
}

int idg_image_taper(const float *taper_dev, int32_t N, float *cbar_dev, int32_t L, void *stream) {
  if (!taper_dev || !cbar_dev || !(N == 16 || N == 24 || N == 32 || N == 48) || L < N || (L & 1))
    return IDG_ERR_INVALID_ARG;
  cudaStream_t s = (cudaStream_t)stream;
  double2 *D = nullptr, *tmp = nullptr;
  IDG_CUDA_TRY(cudaMallocAsync(&D, sizeof(double2) * (size_t)L * N * 2, s));
  tmp = D + (size_t)L * N;
  const int nb = (L * N + 127) / 128;
  taper_dirichlet_kernel<<<nb, 128, 0, s>>>(D, N, L);
  count_launch();
  taper_rows_kernel<<<nb, 128, 0, s>>>(tmp, D, taper_dev, N, L);
  count_launch();
  taper_image_kernel<<<dim3((L + 63) / 64, (L + 3) / 4), 256, 0, s>>>(cbar_dev, tmp, D, N, L);
  count_launch();
  const cudaError_t e = cudaGetLastError();
  cudaFreeAsync(D, s);
  IDG_CUDA_TRY(e);
  return IDG_OK;
}

int idg_image_taper_static(const float *taper_dev, int32_t N, float *cbar_dev, int32_t L, void *stream) {
  if (!taper_dev || !cbar_dev || !(N == 16 || N == 24 || N == 32 || N == 48) || L < N || (L & 1))
    return IDG_ERR_INVALID_ARG;
  if ((int64_t)L * N > (int64_t)kStaticMaxLN) return IDG_ERR_SCRATCH_TOO_SMALL;
  double2 *D = nullptr;
  const int rc = taper_scratch_address(&D);
  if (rc != IDG_OK) return rc;
  double2 *tmp = D + (size_t)L * N;
  cudaStream_t s = (cudaStream_t)stream;
  const int nb = (L * N + 127) / 128;
  // every element of D and tmp that is read below is written first, in this call: nothing has to start at zero
  taper_dirichlet_kernel<<<nb, 128, 0, s>>>(D, N, L);
  count_launch();
  taper_rows_kernel<<<nb, 128, 0, s>>>(tmp, D, taper_dev, N, L);
  count_launch();
  taper_image_kernel<<<dim3((L + 63) / 64, (L + 3) / 4), 256, 0, s>>>(cbar_dev, tmp, D, N, L);
  count_launch();
  IDG_CUDA_TRY(cudaGetLastError());
  return IDG_OK;
}

}  // extern "C"
