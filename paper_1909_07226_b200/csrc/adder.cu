// adder.cu -- rows a3 / a4: adder and splitter (HBM bound).
//
// Adder (Eq. 24; Alg. 1; R7):
//   grid[pol][y0+b][x0+a] += V_p[pol][b][a], no phase factor, no shift.
// Splitter (Alg. 2): V_p[pol][b][a] = grid[pol][y0+b][x0+a].
//
// Subgrids overlap ("subgrids may overlap"), heavily near the uv origin.  Instead
// of one atomic per subgrid pixel, the plan buckets the subgrids by grid tiles: a subgrid belongs
// to the 128-pixel tile COLUMN its x0 falls in and to every 8-row band it overlaps (stable in the
// subgrid index).  One work item = one tile and up to kAdderChunk of its subgrids: the CTA sums
// their rows into a shared-memory accumulator of 8 rows x (128 + N) pixels -- wide enough for a
// subgrid that starts in the last column of the tile -- in plan order and adds it to the grid
// once, with one vector reduction (red.global.add.v2.f32) per touched pixel.  Every subgrid row
// is read exactly once and WHOLE (256 contiguous, aligned bytes at N = 32: no sector or DRAM
// burst is fetched twice, which rows split between two tile columns cost the first version); the
// grid sees one reduction per (work item, pixel) instead of one per (subgrid, pixel); the N
// columns two neighbouring tiles share receive reductions from both.  Long lists (the uv core)
// are split over several work items so no CTA becomes the tail.
#include <algorithm>

#include "common.cuh"

namespace idg {

__device__ __forceinline__ void red_add_f32x2(float2 *addr, float2 v) {
  asm volatile("red.global.add.v2.f32 [%0], {%1, %2};" ::"l"(addr), "f"(v.x), "f"(v.y) : "memory");
}

template <int N, int NPOL>
__global__ void __launch_bounds__(256)
adder_kernel(const AdderItem *__restrict__ items, const int4 *__restrict__ list,
             const idg_subgrid_meta *__restrict__ meta, const float2 *__restrict__ subgrids,
             float2 *__restrict__ grid, int32_t L) {
  // The tile accumulator lives in shared memory, [pol][row][x].  Warp w owns polarisation w % NPOL and
  // the rows w / NPOL + (8 / NPOL) k of the tile: every (pol, row) slot has exactly one writer, so the
  // accumulation needs neither atomics nor barriers, and a warp always reads whole subgrid rows
  // (N consecutive float2: 256 B at N = 32), one lane per pixel.
  constexpr int TX = kAdderTileX + N, TY = kAdderTileY, RSTEP = 8 / NPOL, ROWS = TY / RSTEP;
  constexpr int PASSES = (N + 31) / 32;            // N = 48: a row takes two passes of 32 lanes
  __shared__ float2 tile[NPOL][TY][TX];            // 128 + N columns: x0 - tile_x <= 127, so x0 - tile_x + N - 1 < TX
  const AdderItem it = items[blockIdx.x];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int q = warp % NPOL, r0 = warp / NPOL;
  const int xw = it.x_hi - it.x_lo;                // only the columns this item's subgrids cover
  for (int i = threadIdx.x; i < NPOL * TY * xw; i += 256) tile[i / (TY * xw)][(i / xw) % TY][it.x_lo + i % xw] = make_float2(0.f, 0.f);
  __syncthreads();

  for (int e0 = it.begin; e0 < it.end; e0 += 2) {   // two subgrids per trip: twice the loads in flight
    float2 v[2][ROWS][PASSES];
    int tx0[2];
    bool ok[2][ROWS];
#pragma unroll
    for (int j = 0; j < 2; ++j) {
      const bool have = e0 + j < it.end;
      const int4 ent = have ? __ldg(&list[e0 + j]) : make_int4(0, 0, 0, 0);
      tx0[j] = ent.y;
      const int sy0 = r0 - ent.z;
      const float2 *sg = subgrids + ((size_t)ent.x * NPOL + q) * N * N;
#pragma unroll
      for (int k = 0; k < ROWS; ++k) {
        const int sy = sy0 + RSTEP * k;
        ok[j][k] = have && sy >= 0 && sy < N;
#pragma unroll
        for (int p = 0; p < PASSES; ++p) {
          const int sx = lane + 32 * p;
          v[j][k][p] = (ok[j][k] && sx < N) ? __ldg(&sg[sy * N + sx]) : make_float2(0.f, 0.f);
        }
      }
    }
#pragma unroll
    for (int j = 0; j < 2; ++j)
#pragma unroll
      for (int k = 0; k < ROWS; ++k)
        if (ok[j][k]) {
#pragma unroll
          for (int p = 0; p < PASSES; ++p) {
            const int sx = lane + 32 * p, x = tx0[j] + sx;
            if (sx < N) {
              float2 a = tile[q][r0 + RSTEP * k][x];
              a.x += v[j][k][p].x; a.y += v[j][k][p].y;
              tile[q][r0 + RSTEP * k][x] = a;
            }
          }
        }
  }
  __syncthreads();
  // one vector reduction per touched pixel of the tile (untouched ones hold exact zeros and are skipped)
  for (int i = threadIdx.x; i < NPOL * TY * xw; i += 256) {
    const int x = it.x_lo + i % xw, r = (i / xw) % TY, qq = i / (TY * xw);
    const float2 a = tile[qq][r][x];
    const int gx = it.tile_x + x, gy = it.tile_y + r;
    if ((a.x != 0.f || a.y != 0.f) && gx < L && gy < L) red_add_f32x2(&grid[((size_t)qq * L + gy) * L + gx], a);
  }
}

template <int N, int NPOL>
__global__ void __launch_bounds__(256)
splitter_kernel(const idg_subgrid_meta *__restrict__ meta, const float2 *__restrict__ grid,
                float2 *__restrict__ subgrids, int32_t L) {
  const int x0 = meta[blockIdx.x].x0, y0 = meta[blockIdx.x].y0;
  float2 *sg = subgrids + (size_t)blockIdx.x * NPOL * N * N;
#pragma unroll 4
  for (int e = threadIdx.x; e < NPOL * N * N; e += 256) {
    const int q = e / (N * N), r = e - q * N * N;
    const int y = r / N, x = r - y * N;
    sg[e] = __ldg(&grid[((size_t)q * L + (y0 + y)) * L + (x0 + x)]);
  }
}

int launch_adder(const idg_plan *plan, const float2 *subgrids, float2 *grid, cudaStream_t stream, int n_pol) {
  if (plan->n_adder_items == 0) return IDG_OK;
  const unsigned nb = (unsigned)plan->n_adder_items;
  const int32_t L = plan->prm.grid_size;
#define IDG_ADD(N_)                                                                                          \
  if (n_pol == 1) adder_kernel<N_, 1><<<nb, 256, 0, stream>>>(plan->adder_items_dev, plan->adder_list_dev, plan->meta_dev, subgrids, grid, L); \
  else adder_kernel<N_, 4><<<nb, 256, 0, stream>>>(plan->adder_items_dev, plan->adder_list_dev, plan->meta_dev, subgrids, grid, L)
  switch (plan->prm.subgrid_size) {
    case 16: IDG_ADD(16); break;
    case 24: IDG_ADD(24); break;
    case 32: IDG_ADD(32); break;
    case 48: IDG_ADD(48); break;
    default: return IDG_ERR_UNSUPPORTED_SUBGRID_SIZE;
  }
#undef IDG_ADD
  IDG_LAUNCH_CHECK();
  return IDG_OK;
}

int launch_splitter(const idg_plan *plan, const float2 *grid, float2 *subgrids,
                    cudaStream_t stream, int64_t p0, int64_t np, int n_pol) {
  if (np < 0) np = plan->P - p0;
  if (np <= 0) return IDG_OK;
  const unsigned nb = (unsigned)np;
  subgrids += (size_t)p0 * n_pol * plan->prm.subgrid_size * plan->prm.subgrid_size;
  const int32_t L = plan->prm.grid_size;
#define IDG_SPL(N_)                                                                          \
  if (n_pol == 1) splitter_kernel<N_, 1><<<nb, 256, 0, stream>>>(plan->meta_dev + p0, grid, subgrids, L); \
  else splitter_kernel<N_, 4><<<nb, 256, 0, stream>>>(plan->meta_dev + p0, grid, subgrids, L)
  switch (plan->prm.subgrid_size) {
    case 16: IDG_SPL(16); break;
    case 24: IDG_SPL(24); break;
    case 32: IDG_SPL(32); break;
    case 48: IDG_SPL(48); break;
    default: return IDG_ERR_UNSUPPORTED_SUBGRID_SIZE;
  }
#undef IDG_SPL
  IDG_LAUNCH_CHECK();
  return IDG_OK;
}

}  // namespace idg
