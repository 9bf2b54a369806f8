// subgrid_fft.cu -- rows a2 / a5: batched centred 2-D FFT of every subgrid plane, in place.
//
// "V_p <- FFT(I_p)" and "I_p <- IFFT(V_p)"; reading R6:
//   out[b][a] = (1/N^2) sum_{j,i} in[j][i] exp(sign 2 pi i ((a-N/2)(i-N/2) + (b-N/2)(j-N/2))/N)
// sign = -1 forward, +1 inverse, scale 1/N^2 both ways.  For N = 0 mod 4 (all four sizes) the
// centred transform is the plain one with checkerboard signs on input and output:
//   out[a] = (-1)^a FFT((-1)^i in[i]).
//
// One CTA per subgrid, one thread per (plane, row): the 32 KB subgrid is brought into shared
// memory with coalesced 16-byte loads, each thread transforms one row entirely in registers,
// rows go back to shared memory (pitch N+1 complex: conflict free both ways), each thread then
// transforms one column and stores it straight to HBM (consecutive threads -> consecutive x).
// Traffic: one read and one write of the subgrid, 64 N^2 bytes.
#include <algorithm>

#include <cuda.h>     // CUtensorMap (types only; the encoder is fetched through cudaGetDriverEntryPoint)

#include "common.cuh"
#include "fft_codelets.cuh"

namespace idg {

// ---- TMA plumbing (sm_100a): mbarrier + cp.async.bulk.tensor ------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
  uint32_t ok = 0;
  for (int spins = 0; spins < (1 << 24); ++spins) {      // bounded: a transfer that never lands traps, it does not hang
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n" : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    if (ok) return;
  }
  __trap();
}
__device__ __forceinline__ void tma_load_3d(void *dst, const CUtensorMap *map, int c0, int c1, int c2, uint64_t *bar) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
      ::"r"(smem_u32(dst)), "l"(reinterpret_cast<uint64_t>(map)), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar))
      : "memory");
}

// GATHER (rows a4 + a5 fused, idg_splitter_ifft): the input is not read from the subgrid array but gathered from
// the grid window of the subgrid, V_p[pol][b][a] = grid[pol][y0+b][x0+a], so the splitter's copy
// -- one write and one read of every subgrid -- never goes through HBM.  The arithmetic is the same: results are
// bit-identical to idg_splitter followed by idg_subgrid_fft(+1).
template <int N, bool INV, bool GATHER = false>
__global__ void __launch_bounds__(4 * N)
subgrid_fft_kernel(float2 *__restrict__ subgrids, const idg_subgrid_meta *__restrict__ meta = nullptr,
                   const float2 *__restrict__ grid = nullptr, int32_t L = 0) {
  constexpr int PITCH = N + 1;
  extern __shared__ float2 sm[];  // [4][N][PITCH]
  const int tid = threadIdx.x;
  float2 *sg = subgrids + (size_t)blockIdx.x * 4 * N * N;

  if (GATHER) {
    const int x0 = meta[blockIdx.x].x0, y0 = meta[blockIdx.x].y0;
    // window rows start on 16-byte boundaries (x0 and L even, and the caller's grid itself 16-byte aligned -- the
    // header asks only for 8): two pixels per load
    if (((x0 | L) & 1) == 0 && (reinterpret_cast<uintptr_t>(grid) & 15u) == 0) {
#pragma unroll 8
      for (int i = tid; i < 2 * N * N; i += 4 * N) {
        const int e = 2 * i;
        const int row = e / N, col = e - row * N;   // row runs over plane*N + y
        const int q = row / N, y = row - q * N;
        const float4 v = __ldg(reinterpret_cast<const float4 *>(&grid[((size_t)q * L + (y0 + y)) * L + (x0 + col)]));
        sm[row * PITCH + col] = make_float2(v.x, v.y);
        sm[row * PITCH + col + 1] = make_float2(v.z, v.w);
      }
    } else {
#pragma unroll 8
      for (int e = tid; e < 4 * N * N; e += 4 * N) {
        const int row = e / N, col = e - row * N;
        const int q = row / N, y = row - q * N;
        sm[row * PITCH + col] = __ldg(&grid[((size_t)q * L + (y0 + y)) * L + (x0 + col)]);
      }
    }
  } else {
  const float4 *in4 = reinterpret_cast<const float4 *>(sg);
#pragma unroll 4
  for (int i = tid; i < 2 * N * N; i += 4 * N) {
    const float4 v = in4[i];
    const int e = 2 * i;            // complex index in [4][N][N]
    const int row = e / N, col = e - row * N;   // row runs over plane*N + y
    sm[row * PITCH + col] = make_float2(v.x, v.y);
    sm[row * PITCH + col + 1] = make_float2(v.z, v.w);
  }
  }
  __syncthreads();

  float2 x[N];
  {  // row pass: thread = (plane, y)
    float2 *rowp = sm + tid * PITCH;
#pragma unroll
    for (int c = 0; c < N; ++c) {
      const float2 v = rowp[c];
      x[c] = (c & 1) ? make_float2(-v.x, -v.y) : v;
    }
    fft::Fft<N, INV>::run(x);
#pragma unroll
    for (int c = 0; c < N; ++c) rowp[c] = (c & 1) ? make_float2(-x[c].x, -x[c].y) : x[c];
  }
  __syncthreads();
  {  // column pass: thread = (plane, x)
    const int q = tid / N, c = tid - q * N;
    const float2 *colp = sm + q * N * PITCH + c;
#pragma unroll
    for (int r = 0; r < N; ++r) {
      const float2 v = colp[r * PITCH];
      x[r] = (r & 1) ? make_float2(-v.x, -v.y) : v;
    }
    fft::Fft<N, INV>::run(x);
    constexpr float scale = 1.0f / (float)(N * N);
    float2 *outp = sg + q * N * N + c;
#pragma unroll
    for (int r = 0; r < N; ++r) {
      const float sgn = (r & 1) ? -scale : scale;
      outp[r * N] = make_float2(x[r].x * sgn, x[r].y * sgn);
    }
  }
}

// Rows a4 + a5 fused, Blackwell data movement (idg_splitter_ifft for N = 16, 32, 48): a persistent CTA walks the
// subgrids; one elected thread fetches the whole [4][N][N] grid window of a subgrid with cp.async.bulk.tensor (TMA,
// 3-D tensor map over the grid seen as float32 [4][L][2L], box 32 floats x N rows x 4 planes = 16 complex pixels of
// every row: N/16 boxes per subgrid) into shared memory behind an mbarrier, two subgrids in flight, so
// the window of subgrid p+1 arrives while the FFT of subgrid p runs and no thread spends registers or issue slots on
// the gather.  The box rows are 128 bytes, written with the 128-byte swizzle (16-byte chunk index XOR row index
// mod 8): the row pass reads and writes its row with LDS.128 / STS.128 and the column pass reads with LDS.64, both
// conflict free in the unpadded layout.  The tensor copy wants the global address of a box 16-byte aligned (measured:
// an odd x0, 8 bytes off, faults), so for odd x0 the boxes start one pixel to the left and the last pixel of every
// row comes from one plain load per thread.  Same arithmetic as subgrid_fft_kernel<N, true, true>: bit-identical.
template <int N, int kTmaStages>
__global__ void __launch_bounds__(4 * N)
splitter_ifft_tma_kernel(const __grid_constant__ CUtensorMap tmap, const idg_subgrid_meta *__restrict__ meta,
                         const float2 *__restrict__ grid, int L, float2 *__restrict__ subgrids, int P) {
  constexpr int NB = N / 16;                    // boxes (16 complex pixels wide) per subgrid row
  constexpr int BOX_BYTES = 4 * N * 128;        // one box: 4 planes x N rows x 128 bytes
  constexpr int BUF_BYTES = NB * BOX_BYTES;     // = 32 N^2: one subgrid
  extern __shared__ unsigned char smem_dyn[];
  __shared__ uint64_t mbar[kTmaStages];
  // 1024-byte alignment for the 128-byte swizzle, by pointer arithmetic on the shared array (keeps LDS / STS)
  unsigned char *base = smem_dyn + ((1024u - (smem_u32(smem_dyn) & 1023u)) & 1023u);
  const int tid = threadIdx.x;

  auto issue = [&](int p, int stage) {           // thread 0 only
    const int x0 = meta[p].x0, y0 = meta[p].y0;
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // earlier generic-proxy accesses of the buffer first
    mbar_expect_tx(&mbar[stage], BUF_BYTES);
#pragma unroll
    for (int h = 0; h < NB; ++h)
      tma_load_3d(base + stage * BUF_BYTES + h * BOX_BYTES, &tmap, 2 * (x0 & ~1) + 32 * h, y0, 0, &mbar[stage]);
  };

  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < kTmaStages; ++s) mbar_init(&mbar[s], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < kTmaStages - 1; ++s)
      if (blockIdx.x + s * gridDim.x < P) issue(blockIdx.x + s * gridDim.x, s);
  }

  int it = 0;
  for (int p = blockIdx.x; p < P; p += gridDim.x, ++it) {
    const int stage = it % kTmaStages;
    // the buffer of iteration it + kTmaStages - 1 was last read in iteration it - 1 (barrier at its end)
    if (tid == 0) {
      const int pn = p + (kTmaStages - 1) * gridDim.x;
      if (pn < P) issue(pn, (it + kTmaStages - 1) % kTmaStages);
    }
    // odd x0: the boxes hold the pixels x0 - 1 .. x0 + N - 2 of every row; the last pixel is fetched here
    const int x0 = meta[p].x0;
    const bool odd = (x0 & 1) != 0;
    float2 last = make_float2(0.f, 0.f);
    if (odd) {
      const int q = tid / N, y = tid - q * N;
      last = __ldg(&grid[((size_t)q * L + (meta[p].y0 + y)) * L + (x0 + N - 1)]);
    }
    mbar_wait(&mbar[stage], (it / kTmaStages) & 1);
    unsigned char *buf = base + stage * BUF_BYTES;

    float2 x[N];
    {  // row pass: thread = (plane, y) = box row R
      unsigned char *rowp = buf + tid * 128;
      const int sw = tid & 7;
      if (!odd) {
#pragma unroll
        for (int h = 0; h < NB; ++h)
#pragma unroll
          for (int j = 0; j < 8; ++j) {
            const float4 v = *reinterpret_cast<const float4 *>(rowp + h * BOX_BYTES + ((j ^ sw) << 4));
            x[h * 16 + 2 * j] = make_float2(v.x, v.y);
            x[h * 16 + 2 * j + 1] = make_float2(-v.z, -v.w);      // checkerboard sign of the centred transform
          }
      } else {
#pragma unroll
        for (int h = 0; h < NB; ++h)
#pragma unroll
          for (int j = 0; j < 8; ++j) {
            const float4 v = *reinterpret_cast<const float4 *>(rowp + h * BOX_BYTES + ((j ^ sw) << 4));
            if (h * 16 + 2 * j >= 1) x[h * 16 + 2 * j - 1] = make_float2(-v.x, -v.y);   // box position b holds pixel b - 1
            x[h * 16 + 2 * j] = make_float2(v.z, v.w);
          }
        x[N - 1] = make_float2(-last.x, -last.y);
      }
      fft::Fft<N, true>::run(x);
#pragma unroll
      for (int h = 0; h < NB; ++h)
#pragma unroll
        for (int j = 0; j < 8; ++j) {
          const float2 a = x[h * 16 + 2 * j], b = x[h * 16 + 2 * j + 1];
          *reinterpret_cast<float4 *>(rowp + h * BOX_BYTES + ((j ^ sw) << 4)) = make_float4(a.x, a.y, -b.x, -b.y);
        }
    }
    __syncthreads();
    {  // column pass: thread = (plane, x)
      const int q = tid / N, c = tid - q * N;
      const int h = c >> 4, xin = c & 15;
      const unsigned char *colp = buf + h * BOX_BYTES + q * N * 128 + ((xin & 1) << 3);
#pragma unroll
      for (int r = 0; r < N; ++r) {
        const float2 v = *reinterpret_cast<const float2 *>(colp + r * 128 + (((xin >> 1) ^ (r & 7)) << 4));
        x[r] = (r & 1) ? make_float2(-v.x, -v.y) : v;
      }
      fft::Fft<N, true>::run(x);
      constexpr float scale = 1.0f / (float)(N * N);
      float2 *outp = subgrids + (size_t)p * 4 * N * N + q * N * N + c;
#pragma unroll
      for (int r = 0; r < N; ++r) {
        const float sgn = (r & 1) ? -scale : scale;
        outp[r * N] = make_float2(x[r].x * sgn, x[r].y * sgn);
      }
    }
    __syncthreads();
  }
}

// The same, one WARP per unit of work and no CTA-wide barrier (N = 16, 32, where 32 rows = 32 / N planes fill a warp):
// warp w of the grid walks the items (subgrid, group of 32 / N planes); it owns kStages buffers of 32 box rows and
// their mbarriers, lane 0 issues the tensor copies of the item kStages - 1 ahead, the lanes transform their row,
// exchange through the warp's own buffer (__syncwarp) and transform their column.  A warp that waits for its data
// stalls nobody else.
template <int N, int kStages, int kWarps>
__global__ void __launch_bounds__(32 * kWarps)
splitter_ifft_tma_warp_kernel(const __grid_constant__ CUtensorMap tmap, const idg_subgrid_meta *__restrict__ meta,
                              const float2 *__restrict__ grid, int L, float2 *__restrict__ subgrids, int64_t n_items) {
  static_assert(N == 16 || N == 32, "a warp must hold whole planes");
  constexpr int NB = N / 16, PL = 32 / N, GROUPS = 4 / PL;   // boxes per row, planes per item, items per subgrid
  constexpr int BOX_BYTES = 32 * 128;                        // 32 box rows of 128 bytes
  constexpr int ITEM_BYTES = NB * BOX_BYTES;
  extern __shared__ unsigned char smem_dyn[];
  __shared__ uint64_t mbar[kWarps * kStages];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  unsigned char *base = smem_dyn + ((1024u - (smem_u32(smem_dyn) & 1023u)) & 1023u) + warp * (kStages * ITEM_BYTES);
  uint64_t *bar = mbar + warp * kStages;

  auto issue = [&](int64_t item, int stage) {    // lane 0 only
    const int p = (int)(item / GROUPS), q0 = (int)(item % GROUPS) * PL;
    const int x0 = meta[p].x0, y0 = meta[p].y0;
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    mbar_expect_tx(&bar[stage], ITEM_BYTES);
#pragma unroll
    for (int h = 0; h < NB; ++h)
      tma_load_3d(base + stage * ITEM_BYTES + h * BOX_BYTES, &tmap, 2 * (x0 & ~1) + 32 * h, y0, q0, &bar[stage]);
  };

  if (lane == 0) {
#pragma unroll
    for (int s = 0; s < kStages; ++s) mbar_init(&bar[s], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncwarp();
  const int64_t first = (int64_t)blockIdx.x * kWarps + warp, stride = (int64_t)gridDim.x * kWarps;
  if (lane == 0) {
#pragma unroll
    for (int s = 0; s < kStages - 1; ++s)
      if (first + s * stride < n_items) issue(first + s * stride, s);
  }
  const int pl = lane / N, yy = lane - pl * N;      // row pass: lane = (plane in item, y); column pass: (plane, x)
  int it = 0;
  for (int64_t item = first; item < n_items; item += stride, ++it) {
    const int stage = it % kStages;
    if (lane == 0) {
      const int64_t nxt = item + (kStages - 1) * stride;
      if (nxt < n_items) issue(nxt, (it + kStages - 1) % kStages);
    }
    const int p = (int)(item / GROUPS), q = (int)(item % GROUPS) * PL + pl;
    const int x0 = meta[p].x0;
    const bool odd = (x0 & 1) != 0;
    float2 last = make_float2(0.f, 0.f);
    if (odd) last = __ldg(&grid[((size_t)q * L + (meta[p].y0 + yy)) * L + (x0 + N - 1)]);
    mbar_wait(&bar[stage], (it / kStages) & 1);
    unsigned char *buf = base + stage * ITEM_BYTES;

    float2 x[N];
    {
      unsigned char *rowp = buf + lane * 128;
      const int sw = lane & 7;
      if (!odd) {
#pragma unroll
        for (int h = 0; h < NB; ++h)
#pragma unroll
          for (int j = 0; j < 8; ++j) {
            const float4 v = *reinterpret_cast<const float4 *>(rowp + h * BOX_BYTES + ((j ^ sw) << 4));
            x[h * 16 + 2 * j] = make_float2(v.x, v.y);
            x[h * 16 + 2 * j + 1] = make_float2(-v.z, -v.w);
          }
      } else {
#pragma unroll
        for (int h = 0; h < NB; ++h)
#pragma unroll
          for (int j = 0; j < 8; ++j) {
            const float4 v = *reinterpret_cast<const float4 *>(rowp + h * BOX_BYTES + ((j ^ sw) << 4));
            if (h * 16 + 2 * j >= 1) x[h * 16 + 2 * j - 1] = make_float2(-v.x, -v.y);
            x[h * 16 + 2 * j] = make_float2(v.z, v.w);
          }
        x[N - 1] = make_float2(-last.x, -last.y);
      }
      fft::Fft<N, true>::run(x);
#pragma unroll
      for (int h = 0; h < NB; ++h)
#pragma unroll
        for (int j = 0; j < 8; ++j) {
          const float2 a = x[h * 16 + 2 * j], b = x[h * 16 + 2 * j + 1];
          *reinterpret_cast<float4 *>(rowp + h * BOX_BYTES + ((j ^ sw) << 4)) = make_float4(a.x, a.y, -b.x, -b.y);
        }
    }
    __syncwarp();
    {
      const int c = yy, h = c >> 4, xin = c & 15;
      const unsigned char *colp = buf + h * BOX_BYTES + pl * N * 128 + ((xin & 1) << 3);
#pragma unroll
      for (int r = 0; r < N; ++r) {
        const float2 v = *reinterpret_cast<const float2 *>(colp + r * 128 + (((xin >> 1) ^ (r & 7)) << 4));
        x[r] = (r & 1) ? make_float2(-v.x, -v.y) : v;
      }
      fft::Fft<N, true>::run(x);
      constexpr float scale = 1.0f / (float)(N * N);
      float2 *outp = subgrids + (size_t)p * 4 * N * N + q * N * N + c;
#pragma unroll
      for (int r = 0; r < N; ++r) {
        const float sgn = (r & 1) ? -scale : scale;
        outp[r * N] = make_float2(x[r].x * sgn, x[r].y * sgn);
      }
    }
    __syncwarp();
  }
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn tensor_map_encoder() {
  static EncodeTiledFn fn = [] {
    void *p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess ||
        q != cudaDriverEntryPointSuccess)
      p = nullptr;
    return (EncodeTiledFn)p;
  }();
  return fn;
}

static bool encode_grid_map(CUtensorMap *map, const float2 *grid, int64_t L, int N, int planes) {
  EncodeTiledFn enc = tensor_map_encoder();
  if (!enc || (reinterpret_cast<uintptr_t>(grid) & 15u) != 0) return false;
  const cuuint64_t gdim[3] = {(cuuint64_t)(2 * L), (cuuint64_t)L, 4};
  const cuuint64_t gstride[2] = {(cuuint64_t)(8 * L), (cuuint64_t)(8 * L * L)};
  const cuuint32_t box[3] = {32, (cuuint32_t)N, (cuuint32_t)planes};
  const cuuint32_t estr[3] = {1, 1, 1};
  return enc(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<float2 *>(grid), gdim, gstride, box, estr,
             CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
             CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

template <int N, int kStages, int kWarps>
static int launch_gather_tma_warp(const idg_plan *plan, const float2 *grid, float2 *subgrids, cudaStream_t stream,
                                  int64_t p0, int64_t np, bool *done) {
  *done = false;
  const int64_t L = plan->prm.grid_size;
  CUtensorMap map;
  if (!encode_grid_map(&map, grid, L, N, 32 / N)) return IDG_OK;
  auto kern = splitter_ifft_tma_warp_kernel<N, kStages, kWarps>;
  constexpr size_t smem = (size_t)kWarps * kStages * (N / 16) * 4096 + 1024;
  IDG_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  int dev = 0, n_sm = 0, per_sm = 0;
  IDG_CUDA_TRY(cudaGetDevice(&dev));
  IDG_CUDA_TRY(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
  IDG_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, 32 * kWarps, smem));
  if (per_sm < 1) return IDG_OK;
  const int64_t n_items = np * (4 / (32 / N));
  const int64_t blocks = std::min<int64_t>((n_items + kWarps - 1) / kWarps, (int64_t)n_sm * per_sm);
  kern<<<(unsigned)blocks, 32 * kWarps, smem, stream>>>(map, plan->meta_dev + p0, grid, (int)L,
                                                        subgrids + (size_t)p0 * 4 * N * N, n_items);
  IDG_LAUNCH_CHECK();
  *done = true;
  return IDG_OK;
}

// returns IDG_OK and sets *done = true when the TMA kernel was launched; *done = false -> the caller takes the
// LDG gather (grid not 16-byte aligned, or N = 24 whose rows are not a whole number of 128-byte boxes)
template <int N, int kTmaStages>
static int launch_gather_tma(const idg_plan *plan, const float2 *grid, float2 *subgrids, cudaStream_t stream,
                             int64_t p0, int64_t np, bool *done) {
  *done = false;
  const int64_t L = plan->prm.grid_size;
  EncodeTiledFn enc = tensor_map_encoder();
  if (!enc || (reinterpret_cast<uintptr_t>(grid) & 15u) != 0 || np > 0x7fffffff) return IDG_OK;
  CUtensorMap map;
  const cuuint64_t gdim[3] = {(cuuint64_t)(2 * L), (cuuint64_t)L, 4};
  const cuuint64_t gstride[2] = {(cuuint64_t)(8 * L), (cuuint64_t)(8 * L * L)};
  const cuuint32_t box[3] = {32, (cuuint32_t)N, 4};
  const cuuint32_t estr[3] = {1, 1, 1};
  if (enc(&map, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<float2 *>(grid), gdim, gstride, box, estr,
          CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
          CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
    return IDG_OK;
  constexpr size_t smem = (size_t)kTmaStages * 32 * N * N + 1024;
  IDG_CUDA_TRY(cudaFuncSetAttribute(splitter_ifft_tma_kernel<N, kTmaStages>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  int dev = 0, n_sm = 0, per_sm = 0;
  IDG_CUDA_TRY(cudaGetDevice(&dev));
  IDG_CUDA_TRY(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
  IDG_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, splitter_ifft_tma_kernel<N, kTmaStages>, 4 * N, smem));
  if (per_sm < 1) return IDG_OK;
  const int64_t blocks = std::min<int64_t>(np, (int64_t)n_sm * per_sm);
  splitter_ifft_tma_kernel<N, kTmaStages><<<(unsigned)blocks, 4 * N, smem, stream>>>(
      map, plan->meta_dev + p0, grid, (int)L, subgrids + (size_t)p0 * 4 * N * N, (int)np);
  IDG_LAUNCH_CHECK();
  *done = true;
  return IDG_OK;
}

template <int N>
static int launch_n(const idg_plan *plan, float2 *subgrids, int direction, cudaStream_t stream, int64_t p0,
                    int64_t np) {
  subgrids += (size_t)p0 * 4 * N * N;
  constexpr size_t smem = sizeof(float2) * 4 * N * (N + 1);
  if (direction < 0) {
    IDG_CUDA_TRY(cudaFuncSetAttribute(subgrid_fft_kernel<N, false>,
                                      cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    subgrid_fft_kernel<N, false><<<(unsigned)np, 4 * N, smem, stream>>>(subgrids);
  } else {
    IDG_CUDA_TRY(cudaFuncSetAttribute(subgrid_fft_kernel<N, true>,
                                      cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    subgrid_fft_kernel<N, true><<<(unsigned)np, 4 * N, smem, stream>>>(subgrids);
  }
  IDG_LAUNCH_CHECK();
  return IDG_OK;
}

template <int N>
static int launch_gather_n(const idg_plan *plan, const float2 *grid, float2 *subgrids, cudaStream_t stream,
                           int64_t p0, int64_t np) {
  constexpr size_t smem = sizeof(float2) * 4 * N * (N + 1);
  IDG_CUDA_TRY(cudaFuncSetAttribute(subgrid_fft_kernel<N, true, true>,
                                    cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  subgrid_fft_kernel<N, true, true><<<(unsigned)np, 4 * N, smem, stream>>>(
      subgrids + (size_t)p0 * 4 * N * N, plan->meta_dev + p0, grid, plan->prm.grid_size);
  IDG_LAUNCH_CHECK();
  return IDG_OK;
}

int launch_splitter_ifft(const idg_plan *plan, const float2 *grid, float2 *subgrids, cudaStream_t stream,
                         int64_t p0, int64_t np) {
  if (np < 0) np = plan->P - p0;
  if (np <= 0) return IDG_OK;
  bool done = false;
  int rc = IDG_OK;
  switch (plan->prm.subgrid_size) {       // TMA gather where a subgrid row is a whole number of 128-byte boxes
    // N = 16, 32: one warp per 32 box rows, two buffers per warp, four warps per CTA (measured best of 1-3 stages x
    // 2-14 warps on the SKA-like plan: 1.91 ms against 2.11 ms for the CTA-per-subgrid form and 2.32 ms for the LDG gather)
    case 16: rc = launch_gather_tma_warp<16, 2, 4>(plan, grid, subgrids, stream, p0, np, &done); break;
    case 32: rc = launch_gather_tma_warp<32, 2, 4>(plan, grid, subgrids, stream, p0, np, &done); break;
    case 48: rc = launch_gather_tma<48, 2>(plan, grid, subgrids, stream, p0, np, &done); break;
    default: break;
  }
  if (rc != IDG_OK || done) return rc;
  switch (plan->prm.subgrid_size) {
    case 16: return launch_gather_n<16>(plan, grid, subgrids, stream, p0, np);
    case 24: return launch_gather_n<24>(plan, grid, subgrids, stream, p0, np);
    case 32: return launch_gather_n<32>(plan, grid, subgrids, stream, p0, np);
    case 48: return launch_gather_n<48>(plan, grid, subgrids, stream, p0, np);
    default: return IDG_ERR_UNSUPPORTED_SUBGRID_SIZE;
  }
}

int launch_subgrid_fft(const idg_plan *plan, float2 *subgrids, int direction, cudaStream_t stream, int64_t p0,
                       int64_t np) {
  if (np < 0) np = plan->P - p0;
  if (np <= 0) return IDG_OK;
  switch (plan->prm.subgrid_size) {
    case 16: return launch_n<16>(plan, subgrids, direction, stream, p0, np);
    case 24: return launch_n<24>(plan, subgrids, direction, stream, p0, np);
    case 32: return launch_n<32>(plan, subgrids, direction, stream, p0, np);
    case 48: return launch_n<48>(plan, subgrids, direction, stream, p0, np);
    default: return IDG_ERR_UNSUPPORTED_SUBGRID_SIZE;
  }
}

}  // namespace idg
