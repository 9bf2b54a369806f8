// common.cuh -- internal declarations of libidg_b200 (CUDA, sm_100a only).
// Product code: shares nothing with oracle/.  See include/idg_b200.h for the boundary.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <new>
#include <vector>

#include "../../include/idg_b200.h"

namespace idg {

constexpr double kSpeedOfLight = 299792458.0;
constexpr int kAdderTileX = 96;  // adder work item: the subgrids whose x0 lies in a 128-pixel column, one 8-row
constexpr int kAdderTileY = 8;       // band of the grid at a time (accumulator 8 rows x (128 + N) pixels)
constexpr int kAdderChunk = 64;      // max subgrids accumulated by one work item

struct AdderItem {                    // one unit of adder work: a grid tile and a slice of its list
  int32_t tile_x, tile_y;             // tile origin on the grid (pixels)
  int32_t begin, end;                 // range in adder_list
  int32_t x_lo, x_hi;                 // accumulator columns its subgrids cover (zeroed / flushed range), 0 .. 128 + N
};

}  // namespace idg

struct idg_plan {
  idg_plan_params prm{};
  int32_t B = 0, T = 0, C = 0, n_stations = 0;
  int64_t P = 0, n_planned = 0, n_skipped = 0;
  int32_t max_n_time = 0, max_n_chan = 0, min_n_chan = 0;
  int32_t n_slots_needed = 0;         // A-term slots the metadata indexes (last slot + 1)
  bool planner_made = false;          // metadata from run_planner: sorted by baseline, every sample covered once or skipped
  bool sorted_by_baseline = false;    // baselines non-decreasing in metadata order (the *_host calls chunk by baseline)
  float dg_waste[4] = {0.f, 0.f, 0.f, 0.f};   // degridder: idle channel slots if threads own 1, 2, 4, 8 channels
  float uniform_dkd = 0.f;            // 2 pi df / c0 when the channels are equally spaced, else 0 (scalar.cu)
  std::vector<idg_subgrid_meta> meta_host;
  idg_subgrid_meta *meta_dev = nullptr;
  double *freqs_dev = nullptr;        // [C] Hz
  float4 *lmn_dev = nullptr;          // [N*N] (l, m, n', 0) per subgrid pixel (R1, R2), rounded from FP64
  float2 *subgrids_dev = nullptr;     // [P][4][N][N]
  // adder: subgrids bucketed by the grid tiles they overlap (stable in p -> fixed order)
  int4 *adder_list_dev = nullptr;     // {subgrid index, x0 - tile_x, y0 - tile_y, 0}, grouped by tile
  idg::AdderItem *adder_items_dev = nullptr;
  int64_t n_adder_items = 0;
  // staging for the *_host entry points
  float *h_uvw_dev = nullptr;
  float2 *h_vis_dev = nullptr, *h_aterms_dev = nullptr, *h_grid_dev = nullptr;
  float *h_taper_dev = nullptr;
  int64_t h_aterm_slots = 0;
  // copy/compute overlap of the *_host entry points: a copy stream and per-chunk events (created on first use)
  cudaStream_t h_copy_stream = nullptr;
  static constexpr int kHostChunks = 24;
  cudaEvent_t h_ev_in[kHostChunks + 2] = {};    // chunk uploads, then [kHostChunks] = small inputs, [+1] = grid
  cudaEvent_t h_ev_out[kHostChunks + 1] = {};   // chunk results ready on the compute stream, [kHostChunks] = start
};

namespace idg {

void set_last_cuda_error(cudaError_t e);

#define IDG_CUDA_TRY(expr)                                   \
  do {                                                       \
    cudaError_t _e = (expr);                                 \
    if (_e != cudaSuccess) {                                 \
      idg::set_last_cuda_error(_e);                          \
      return _e == cudaErrorMemoryAllocation ? IDG_ERR_OUT_OF_MEMORY : IDG_ERR_CUDA; \
    }                                                        \
  } while (0)

// kernels launched by this library since it was loaded (idg_kernel_launches); every launch site checks with
// IDG_LAUNCH_CHECK, which counts it
void count_launch();
#define IDG_LAUNCH_CHECK()             \
  do {                                 \
    idg::count_launch();               \
    IDG_CUDA_TRY(cudaGetLastError()); \
  } while (0)

// extern "C" bodies: nothing may throw across the C boundary (std::vector growth inside the library)
#define IDG_API_TRY try {
#define IDG_API_CATCH                                         \
  }                                                           \
  catch (const std::bad_alloc &) { return IDG_ERR_OUT_OF_MEMORY; } \
  catch (...) { return IDG_ERR_INVALID_ARG; }

inline bool aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

// planner (plan.cu)
int run_planner(const idg_plan_params &prm, const float *uvw_dev, const double *freqs_host,
                const int32_t *baselines_host, int32_t B, int32_t T, int32_t C,
                std::vector<idg_subgrid_meta> &meta_out, idg_subgrid_meta **meta_dev_out,
                int64_t *planned, int64_t *skipped, cudaStream_t stream);

// stage launchers (one .cu each); all asynchronous on `stream`
// p0 / np select the subgrids [p0, p0 + np) of the plan (np < 0: all); `subgrids` is always the base of the
// full [P][4][N][N] array.  The host-buffer entry points use ranges to overlap copies with compute.
int launch_gridder(const idg_plan *plan, const float *uvw, const float2 *vis, const float2 *aterms,
                   const float *taper, float2 *subgrids, cudaStream_t stream, int64_t p0 = 0, int64_t np = -1);
// tensor-core gridder (gridder_tc.cu): N = 32, per-block A-terms, >= 8 channels per block
bool gridder_tc_eligible(const idg_plan *plan);
int launch_gridder_tc(const idg_plan *plan, const float *uvw, const float2 *vis, const float2 *aterms,
                      const float *taper, float2 *subgrids, cudaStream_t stream, int64_t p0, int64_t np);
// tensor-core degridder (degridder_tc.cu): N = 32, per-block A-terms, mean block >= 384 visibilities
bool degridder_tc_eligible(const idg_plan *plan);
int launch_degridder_tc(const idg_plan *plan, const float *uvw, const float2 *subgrids, const float2 *aterms,
                        const float *taper, float2 *vis_out, cudaStream_t stream, int64_t p0, int64_t np);
int launch_degridder(const idg_plan *plan, const float *uvw, const float2 *subgrids,
                     const float2 *aterms, const float *taper, float2 *vis_out,
                     cudaStream_t stream, int64_t p0 = 0, int64_t np = -1);
int launch_subgrid_fft(const idg_plan *plan, float2 *subgrids, int direction, cudaStream_t stream,
                       int64_t p0 = 0, int64_t np = -1);
int launch_adder(const idg_plan *plan, const float2 *subgrids, float2 *grid, cudaStream_t stream, int n_pol = 4);
int launch_splitter_ifft(const idg_plan *plan, const float2 *grid, float2 *subgrids, cudaStream_t stream,
                         int64_t p0 = 0, int64_t np = -1);
int launch_splitter(const idg_plan *plan, const float2 *grid, float2 *subgrids,
                    cudaStream_t stream, int64_t p0 = 0, int64_t np = -1, int n_pol = 4);
// scalar variant (NEXT-3, scalar.cu): vis [B][T][C], gains [slots][stations][N][N], subgrids [P][N][N]
int launch_gridder_scalar(const idg_plan *plan, const float *uvw, const float2 *vis, const float2 *gains,
                          const float *taper, float2 *subgrids, cudaStream_t stream);
int launch_degridder_scalar(const idg_plan *plan, const float *uvw, const float2 *subgrids, const float2 *gains,
                            const float *taper, float2 *vis_out, cudaStream_t stream);

// packed FP32 FMA (sm_100 FFMA2): d = a * b + c on both halves
__device__ __forceinline__ float2 ffma2(float2 a, float2 b, float2 c) {
  unsigned long long ra, rb, rc, rd;
  ra = *reinterpret_cast<unsigned long long *>(&a);
  rb = *reinterpret_cast<unsigned long long *>(&b);
  rc = *reinterpret_cast<unsigned long long *>(&c);
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(rd) : "l"(ra), "l"(rb), "l"(rc));
  return *reinterpret_cast<float2 *>(&rd);
}

__device__ __forceinline__ float2 fmul2(float2 a, float2 b) {
  unsigned long long ra, rb, rd;
  ra = *reinterpret_cast<unsigned long long *>(&a);
  rb = *reinterpret_cast<unsigned long long *>(&b);
  asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(rd) : "l"(ra), "l"(rb));
  return *reinterpret_cast<float2 *>(&rd);
}

// acc += v * (c + i s) for a complex accumulator, as two FFMA2
__device__ __forceinline__ void cmac(float2 &acc, float2 v, float c, float s) {
  acc = ffma2(make_float2(v.x, v.x), make_float2(c, s), acc);
  acc = ffma2(make_float2(v.y, v.y), make_float2(-s, c), acc);
}

__device__ __forceinline__ float2 cmul(float2 a, float2 b) {
  return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
__device__ __forceinline__ float2 cmul_conj_a(float2 a, float2 b) {  // conj(a) * b
  return make_float2(a.x * b.x + a.y * b.y, a.x * b.y - a.y * b.x);
}
__device__ __forceinline__ float2 cmul_conj_b(float2 a, float2 b) {  // a * conj(b)
  return make_float2(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y);
}
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }

}  // namespace idg
