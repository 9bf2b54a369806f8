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
#include "common.cuh"
#include "fft_codelets.cuh"

namespace idg {

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
