// mixbench.cu -- the bare instruction mix of the gridder / degridder inner loop, timed on the device.
//
// SURVEY.md section 8(d) asks for the op-count roofline to be reported next to the MEASURED peak of the
// 17 FMA : 1 FMUL : 2 MUFU mix.  This kernel runs exactly what one (visibility, pixel) pair costs in
// gridder_kernel (Eq. 25) -- 1 FFMA (phase) + sin.approx / cos.approx (1 FMUL + 2 MUFU) +
// 16 FMA as 8 FFMA2 with a (pair, broadcast scalar, accumulator pair) operand pattern -- on registers only: no
// shared or global memory in the loop, the same CTA shape and residency as the N = 32 gridder (256 threads x 4
// pixels, 2 CTAs per SM).  What it reaches is the practical ceiling of the FP32 path on this chip; bench.py
// prints it beside the derived lane-op peak.
#include "common.cuh"

namespace idg {

// VARIANT 0: operands as in gridder_kernel -- the visibility pairs come from shared memory (LDS.128 at a
//            warp-uniform address) and sit in vector registers; 8 FFMA2 per pair.
// VARIANT 1: the visibility pairs are kernel parameters, which ptxas keeps in UNIFORM registers (FFMA2 with a UR
//            pair operand): the ceiling if the warp-uniform operand did not cost register-file reads.  Not reachable
//            for real data from CUDA C: ptxas moves REDUX / shared-memory values back to vector registers.
// VARIANT 2: 16 scalar FFMA per pair instead of 8 FFMA2 (visibilities from shared memory).
template <int VARIANT>
__global__ void __launch_bounds__(256, 2)
mix_kernel(float4 *__restrict__ out, const float4 *__restrict__ in, int iters, float kd, float4 pr, float4 pi) {
  constexpr int PPT = 4;
  __shared__ float4 s_vis[512];
  for (int i = threadIdx.x; i < 512; i += 256) s_vis[i] = in[i];
  __syncthreads();
  float2 re01[PPT], re23[PPT], im01[PPT], im23[PPT];
  float ph[PPT], pidx[PPT];
#pragma unroll
  for (int k = 0; k < PPT; ++k) {
    re01[k] = re23[k] = im01[k] = im23[k] = make_float2(0.f, 0.f);
    ph[k] = 1e-3f * (float)(threadIdx.x + 256 * k);
    pidx[k] = 1e-4f * (float)(threadIdx.x * PPT + k + 1);
  }
#pragma unroll 4
  for (int i = 0; i < iters; ++i) {
    const float4 vr = VARIANT == 1 ? pr : s_vis[2 * (i & 255)];
    const float4 vi = VARIANT == 1 ? pi : s_vis[2 * (i & 255) + 1];
    const float2 vr01 = make_float2(vr.x, vr.y), vr23 = make_float2(vr.z, vr.w);
    const float2 vi01 = make_float2(vi.x, vi.y), vi23 = make_float2(vi.z, vi.w);
#pragma unroll
    for (int k = 0; k < PPT; ++k) {
      ph[k] = fmaf(pidx[k], kd, ph[k]);
      float s, co;
      __sincosf(ph[k], &s, &co);
      const float ns = -s;
      if (VARIANT == 2) {
        re01[k].x = fmaf(vr.x, co, re01[k].x); re01[k].x = fmaf(vi.x, ns, re01[k].x);
        re01[k].y = fmaf(vr.y, co, re01[k].y); re01[k].y = fmaf(vi.y, ns, re01[k].y);
        re23[k].x = fmaf(vr.z, co, re23[k].x); re23[k].x = fmaf(vi.z, ns, re23[k].x);
        re23[k].y = fmaf(vr.w, co, re23[k].y); re23[k].y = fmaf(vi.w, ns, re23[k].y);
        im01[k].x = fmaf(vr.x, s, im01[k].x);  im01[k].x = fmaf(vi.x, co, im01[k].x);
        im01[k].y = fmaf(vr.y, s, im01[k].y);  im01[k].y = fmaf(vi.y, co, im01[k].y);
        im23[k].x = fmaf(vr.z, s, im23[k].x);  im23[k].x = fmaf(vi.z, co, im23[k].x);
        im23[k].y = fmaf(vr.w, s, im23[k].y);  im23[k].y = fmaf(vi.w, co, im23[k].y);
      } else {
        re01[k] = ffma2(vr01, make_float2(co, co), re01[k]); re01[k] = ffma2(vi01, make_float2(ns, ns), re01[k]);
        re23[k] = ffma2(vr23, make_float2(co, co), re23[k]); re23[k] = ffma2(vi23, make_float2(ns, ns), re23[k]);
        im01[k] = ffma2(vr01, make_float2(s, s), im01[k]);   im01[k] = ffma2(vi01, make_float2(co, co), im01[k]);
        im23[k] = ffma2(vr23, make_float2(s, s), im23[k]);   im23[k] = ffma2(vi23, make_float2(co, co), im23[k]);
      }
    }
  }
  float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
  for (int k = 0; k < PPT; ++k) {
    acc.x += re01[k].x + re01[k].y; acc.y += re23[k].x + re23[k].y;
    acc.z += im01[k].x + im01[k].y; acc.w += im23[k].x + im23[k].y;
  }
  out[(size_t)blockIdx.x * 256 + threadIdx.x] = acc;     // results consumed
}

}  // namespace idg

using namespace idg;

extern "C" int idg_bench_instruction_mix(int32_t iters, int32_t variant, double *tflop_equiv_per_s, void *stream) {
  if (iters < 1 || variant < 0 || variant > 2 || !tflop_equiv_per_s) return IDG_ERR_INVALID_ARG;
  cudaStream_t s = (cudaStream_t)stream;
  int dev = 0, n_sm = 0;
  IDG_CUDA_TRY(cudaGetDevice(&dev));
  IDG_CUDA_TRY(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
  const int blocks = n_sm * 2 * 4;                        // four waves of the resident set
  float4 *out = nullptr;
  IDG_CUDA_TRY(cudaMalloc(&out, sizeof(float4) * (256 * (size_t)blocks + 512)));
  float4 *in = out + 256 * (size_t)blocks;
  cudaError_t e = cudaMemsetAsync(in, 0x3c, sizeof(float4) * 512, s);     // small finite floats
  cudaEvent_t a = nullptr, b = nullptr;
  cudaEventCreate(&a); cudaEventCreate(&b);
  const float4 vr = make_float4(0.3f, -0.2f, 0.1f, 0.25f), vi = make_float4(-0.15f, 0.35f, 0.05f, -0.3f);
  float best = 0.f;
  for (int rep = 0; rep < 4 && e == cudaSuccess; ++rep) {   // first repetition warms up; best of the rest
    cudaEventRecord(a, s);
    if (variant == 0) mix_kernel<0><<<blocks, 256, 0, s>>>(out, in, iters, 1.7e-3f, vr, vi);
    else if (variant == 1) mix_kernel<1><<<blocks, 256, 0, s>>>(out, in, iters, 1.7e-3f, vr, vi);
    else mix_kernel<2><<<blocks, 256, 0, s>>>(out, in, iters, 1.7e-3f, vr, vi);
    count_launch();
    cudaEventRecord(b, s);
    e = cudaEventSynchronize(b);
    float ms = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, a, b);
    if (rep > 0 && e == cudaSuccess && (best == 0.f || ms < best)) best = ms;
  }
  if (e == cudaSuccess) e = cudaGetLastError();
  cudaEventDestroy(a); cudaEventDestroy(b); cudaFree(out);
  IDG_CUDA_TRY(e);
  // 18 FP32 lane-ops = 36 FLOP-equivalents per (iteration, pixel); 4 pixels per thread
  const double pairs = (double)blocks * 256.0 * 4.0 * (double)iters;
  *tflop_equiv_per_s = 36.0 * pairs / ((double)best * 1e-3) / 1e12;
  return IDG_OK;
}
