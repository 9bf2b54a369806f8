// mmabench.cu -- measurement aid for the tensor-core kernels (gridder_tc.cu, degridder_tc.cu): the issue rate of
// tcgen05.mma.cta_group::1.kind::f16, M = 128, K = 16, A operand in tensor memory, B operand in shared memory, FP32
// accumulators, as those kernels use it.  One elected thread per CTA issues `n_mma` MMAs back to back (loop unrolled
// by 8, uniform operands, four A tiles and one accumulator) and commits them to an mbarrier; the CTA reports the
// cycles (clock64) between the first issue and the completion.  `ctas_per_sm` CTAs of 128 threads and 128
// tensor-memory columns are launched per SM (1..4), so that the rate of an SM is seen, not that of one instruction
// stream.  Operand values are zero: the probe measures time, the kernels' parity tests check the arithmetic.
#include <vector>

#include "common.cuh"

namespace idg {

namespace {

__device__ __forceinline__ uint32_t mb_smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

template <int NN>
__global__ void __launch_bounds__(128) mma_rate_kernel(int n_mma, long long *cycles) {
  constexpr int COLS = NN <= 64 ? 128 : (NN == 128 ? 256 : 512);     // accumulator (NN columns) + four A tiles (32)
  __shared__ __align__(1024) unsigned char s_b[NN * 32];              // one B tile [NN n][16 k] fp16, K-major, no swizzle
  __shared__ uint32_t s_tmem;
  __shared__ uint64_t bar;
  const int tid = threadIdx.x, warp = tid >> 5;
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(mb_smem_u32(&s_tmem)), "n"(COLS));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  if (tid == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(mb_smem_u32(&bar)));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  for (int e = tid; e < NN * 32 / 4; e += 128) reinterpret_cast<uint32_t *>(s_b)[e] = 0u;
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t tb = s_tmem;
  for (int c = 0; c < COLS; c += 8) {                                 // zero the allocation: accumulator and A tiles
    const uint32_t ta = tb + ((uint32_t)(warp * 32) << 16) + c;
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%1,%1,%1,%1,%1,%1,%1};" ::"r"(ta), "r"(0u) : "memory");
  }
  asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  constexpr uint32_t kDesc = (1u << 4) | ((uint32_t)(NN >> 3) << 17) | ((128u >> 4) << 24);
  const long long t0 = clock64();
  if (warp == 0) {
    const uint64_t desc = (uint64_t)((mb_smem_u32(s_b) & 0x3FFFF) >> 4) | ((uint64_t)(128 >> 4) << 16) |
                          ((uint64_t)(256 >> 4) << 32) | ((uint64_t)1 << 46);
    uint32_t leader = 0;
    asm volatile("{ .reg .pred p; elect.sync _|p, 0xffffffff; selp.u32 %0, 1, 0, p; }" : "=r"(leader));
    if (leader) {
      for (int i = 0; i < n_mma; i += 8) {
#pragma unroll
        for (int j = 0; j < 8; ++j)
          asm volatile("{ .reg .pred p; setp.ne.b32 p, %4, 0; tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p; }"
                       ::"r"(tb), "r"(tb + (uint32_t)NN + (uint32_t)(j & 3) * 8u), "l"(desc), "r"(kDesc), "r"(1u) : "memory");
      }
      asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.b64 [%0];" ::"r"(mb_smem_u32(&bar)) : "memory");
    }
    __syncwarp();
    uint32_t ok = 0;
    for (int spins = 0; spins < (1 << 28) && !ok; ++spins)
      asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0; selp.u32 %0, 1, 0, p; }"
                   : "=r"(ok) : "r"(mb_smem_u32(&bar)) : "memory");
  }
  __syncthreads();
  const long long t1 = clock64();
  if (tid == 0) cycles[blockIdx.x] = t1 - t0;
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tb), "n"(COLS));
}

}  // namespace

}  // namespace idg

using namespace idg;

extern "C" int idg_bench_mma_rate(int32_t n, int32_t ctas_per_sm, int32_t n_mma, double *cycles_per_mma_per_sm,
                                  void *stream) {
  if (!(n == 16 || n == 64 || n == 128 || n == 256) || ctas_per_sm < 1 || n_mma < 8 || (n_mma & 7) ||
      !cycles_per_mma_per_sm)
    return IDG_ERR_INVALID_ARG;
  const int max_ctas = n <= 64 ? 4 : (n == 128 ? 2 : 1);              // tensor-memory columns: 512 per SM
  if (ctas_per_sm > max_ctas) return IDG_ERR_INVALID_ARG;
  cudaStream_t s = (cudaStream_t)stream;
  int dev = 0, n_sm = 0;
  IDG_CUDA_TRY(cudaGetDevice(&dev));
  IDG_CUDA_TRY(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
  const int blocks = n_sm * ctas_per_sm;
  long long *cyc = nullptr;
  IDG_CUDA_TRY(cudaMalloc(&cyc, sizeof(long long) * (size_t)blocks));
  std::vector<long long> host((size_t)blocks, 0);
  cudaError_t e = cudaSuccess;
  for (int rep = 0; rep < 2 && e == cudaSuccess; ++rep) {             // the first launch warms up
    if (n == 16) mma_rate_kernel<16><<<blocks, 128, 0, s>>>(n_mma, cyc);
    else if (n == 64) mma_rate_kernel<64><<<blocks, 128, 0, s>>>(n_mma, cyc);
    else if (n == 128) mma_rate_kernel<128><<<blocks, 128, 0, s>>>(n_mma, cyc);
    else mma_rate_kernel<256><<<blocks, 128, 0, s>>>(n_mma, cyc);
    count_launch();
    e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaMemcpyAsync(host.data(), cyc, sizeof(long long) * (size_t)blocks, cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
  }
  cudaFree(cyc);
  IDG_CUDA_TRY(e);
  double mean = 0.0;
  for (long long c : host) mean += (double)c / (double)blocks;
  // every CTA issued n_mma MMAs in `mean` cycles while ctas_per_sm - 1 others on its SM did the same
  *cycles_per_mma_per_sm = mean / (double)n_mma / (double)ctas_per_sm;
  return IDG_OK;
}
