// adder.cu -- rows a3 / a4: adder and splitter (HBM bound).
//
// Adder (Eq. 24; Alg. 1; R7):
//   grid[pol][y0+b][x0+a] += V_p[pol][b][a], no phase factor, no shift.
// Splitter (Alg. 2): V_p[pol][b][a] = grid[pol][y0+b][x0+a].
//
// Subgrids overlap ("subgrids may overlap"), heavily near the uv origin.  Instead
// of one atomic per subgrid pixel, the plan buckets the subgrids by the 32 x 32 grid tiles they
// touch (stable in the subgrid index).  One work item = one tile and up to kAdderChunk of its
// subgrids: the CTA gathers their overlapping parts into registers in plan order and adds the
// tile to the grid once, with one vector reduction (red.global.add.v2.f32) per pixel.  Every
// subgrid element is read exactly once; the grid sees one reduction per (work item, pixel)
// instead of one per (subgrid, pixel).  Long lists (the uv core) are split over several work
// items so no CTA becomes the tail.
#include <algorithm>

#include "common.cuh"

namespace idg {

__device__ __forceinline__ void red_add_f32x2(float2 *addr, float2 v) {
  asm volatile("red.global.add.v2.f32 [%0], {%1, %2};" ::"l"(addr), "f"(v.x), "f"(v.y) : "memory");
}

template <int N>
__global__ void __launch_bounds__(256)
adder_kernel(const AdderItem *__restrict__ items, const int32_t *__restrict__ list,
             const idg_subgrid_meta *__restrict__ meta, const float2 *__restrict__ subgrids,
             float2 *__restrict__ grid, int32_t L) {
  constexpr int TS = kAdderTile, ROWS = TS / 8;
  const AdderItem it = items[blockIdx.x];
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
  const int gx = it.tile_x + tx;
  float2 acc[ROWS][4];
#pragma unroll
  for (int k = 0; k < ROWS; ++k)
#pragma unroll
    for (int q = 0; q < 4; ++q) acc[k][q] = make_float2(0.f, 0.f);

  for (int e = it.begin; e < it.end; ++e) {
    const int32_t s = __ldg(&list[e]);
    const int sx = gx - __ldg(&meta[s].x0);
    const int sy0 = it.tile_y + ty - __ldg(&meta[s].y0);
    if (sx < 0 || sx >= N) continue;
    const float2 *sg = subgrids + (size_t)s * 4 * N * N + sx;
#pragma unroll
    for (int k = 0; k < ROWS; ++k) {
      const int sy = sy0 + 8 * k;
      if (sy >= 0 && sy < N) {
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          const float2 v = __ldg(&sg[(q * N + sy) * N]);
          acc[k][q].x += v.x; acc[k][q].y += v.y;
        }
      }
    }
  }
  if (gx < L) {
#pragma unroll
    for (int k = 0; k < ROWS; ++k) {
      const int gy = it.tile_y + ty + 8 * k;
      if (gy < L) {
#pragma unroll
        for (int q = 0; q < 4; ++q)
          red_add_f32x2(&grid[((size_t)q * L + gy) * L + gx], acc[k][q]);
      }
    }
  }
}

template <int N>
__global__ void __launch_bounds__(256)
splitter_kernel(const idg_subgrid_meta *__restrict__ meta, const float2 *__restrict__ grid,
                float2 *__restrict__ subgrids, int32_t L) {
  const int x0 = meta[blockIdx.x].x0, y0 = meta[blockIdx.x].y0;
  float2 *sg = subgrids + (size_t)blockIdx.x * 4 * N * N;
#pragma unroll 4
  for (int e = threadIdx.x; e < 4 * N * N; e += 256) {
    const int q = e / (N * N), r = e - q * N * N;
    const int y = r / N, x = r - y * N;
    sg[e] = __ldg(&grid[((size_t)q * L + (y0 + y)) * L + (x0 + x)]);
  }
}

int launch_adder(const idg_plan *plan, const float2 *subgrids, float2 *grid, cudaStream_t stream) {
  if (plan->n_adder_items == 0) return IDG_OK;
  const unsigned nb = (unsigned)plan->n_adder_items;
  const int32_t L = plan->prm.grid_size;
#define IDG_ADD(N_) adder_kernel<N_><<<nb, 256, 0, stream>>>(plan->adder_items_dev, plan->adder_list_dev, plan->meta_dev, subgrids, grid, L)
  switch (plan->prm.subgrid_size) {
    case 16: IDG_ADD(16); break;
    case 24: IDG_ADD(24); break;
    case 32: IDG_ADD(32); break;
    case 48: IDG_ADD(48); break;
    default: return IDG_ERR_UNSUPPORTED_SUBGRID_SIZE;
  }
#undef IDG_ADD
  IDG_CUDA_TRY(cudaGetLastError());
  return IDG_OK;
}

int launch_splitter(const idg_plan *plan, const float2 *grid, float2 *subgrids,
                    cudaStream_t stream) {
  if (plan->P == 0) return IDG_OK;
  const unsigned nb = (unsigned)plan->P;
  const int32_t L = plan->prm.grid_size;
#define IDG_SPL(N_) splitter_kernel<N_><<<nb, 256, 0, stream>>>(plan->meta_dev, grid, subgrids, L)
  switch (plan->prm.subgrid_size) {
    case 16: IDG_SPL(16); break;
    case 24: IDG_SPL(24); break;
    case 32: IDG_SPL(32); break;
    case 48: IDG_SPL(48); break;
    default: return IDG_ERR_UNSUPPORTED_SUBGRID_SIZE;
  }
#undef IDG_SPL
  IDG_CUDA_TRY(cudaGetLastError());
  return IDG_OK;
}

}  // namespace idg
