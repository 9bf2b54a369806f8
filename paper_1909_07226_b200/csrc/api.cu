// api.cu -- the C ABI of include/idg_b200.h: argument checks, plan ownership, stage sequencing.
#include <algorithm>
#include <atomic>
#include <cmath>
#include <climits>
#include <cstring>
#include <new>

#include "common.cuh"

namespace idg {

static thread_local int g_last_cuda_error = 0;
void set_last_cuda_error(cudaError_t e) { g_last_cuda_error = (int)e; }
static std::atomic<long long> g_kernel_launches{0};
void count_launch() { g_kernel_launches.fetch_add(1, std::memory_order_relaxed); }

static bool supported_size(int n) { return n == 16 || n == 24 || n == 32 || n == 48; }
static bool is_pow2(int n) { return n > 0 && (n & (n - 1)) == 0; }

static int check_params(const idg_plan_params *p) {
  if (!p) return IDG_ERR_INVALID_ARG;
  if (!supported_size(p->subgrid_size)) return IDG_ERR_UNSUPPORTED_SUBGRID_SIZE;
  if (p->grid_size < p->subgrid_size || (p->grid_size & 1)) return IDG_ERR_INVALID_ARG;
  if (p->kernel_size <= 0 || p->kernel_size >= p->subgrid_size) return IDG_ERR_INVALID_ARG;
  if (p->max_timesteps < 1 || p->aterm_interval < 1) return IDG_ERR_INVALID_ARG;
  if (!is_pow2(p->max_channels) || p->max_channels > 256) return IDG_ERR_INVALID_ARG;
  if (p->reserved != 0 || (p->flags & ~(IDG_PLAN_FORCE_BLOCKS | IDG_PLAN_SPAN_ATERMS | IDG_PLAN_FP32_GRIDDER))) return IDG_ERR_INVALID_ARG;
  if (!(p->image_size > 0.0) || !(p->image_size < 1.4) || !(p->w_step >= 0.0)) return IDG_ERR_INVALID_ARG;
  return IDG_OK;
}

// Bucket the subgrids by grid tiles (stable counting sort in p): tile column = the 128-pixel column x0 falls in,
// tile rows = every 8-row band the subgrid overlaps; cut every tile's list into work items of at most kAdderChunk
// subgrids.
static int build_adder_lists(idg_plan *pl, cudaStream_t stream) {
  const int N = pl->prm.subgrid_size, L = pl->prm.grid_size, TX = kAdderTileX, TY = kAdderTileY;
  const int ntx = (L + TX - 1) / TX, nty = (L + TY - 1) / TY;
  std::vector<int64_t> offs((size_t)ntx * nty + 1, 0);
  for (const auto &m : pl->meta_host)
    for (int ty = m.y0 / TY; ty <= (m.y0 + N - 1) / TY; ++ty) ++offs[(size_t)ty * ntx + m.x0 / TX + 1];
  for (size_t i = 1; i < offs.size(); ++i) offs[i] += offs[i - 1];
  const int64_t total = offs.back();
  if (total > (int64_t)INT32_MAX) return IDG_ERR_INVALID_ARG;   // AdderItem ranges are int32
  std::vector<int32_t> list((size_t)total);
  std::vector<int64_t> cur(offs.begin(), offs.end() - 1);
  for (int64_t p = 0; p < pl->P; ++p) {
    const auto &m = pl->meta_host[(size_t)p];
    for (int ty = m.y0 / TY; ty <= (m.y0 + N - 1) / TY; ++ty)
      list[(size_t)cur[(size_t)ty * ntx + m.x0 / TX]++] = (int32_t)p;
  }
  // work items of at most `chunk` subgrids: kAdderChunk when there is plenty of work, shorter lists on small
  // plans so that the items still fill the GPU (a few per resident CTA slot)
  const int64_t chunk = std::max<int64_t>(8, std::min<int64_t>(kAdderChunk, total / 4096));
  std::vector<AdderItem> items;
  for (int ty = 0; ty < nty; ++ty)
    for (int tx = 0; tx < ntx; ++tx) {
      const int64_t b = offs[(size_t)ty * ntx + tx], e = offs[(size_t)ty * ntx + tx + 1];
      for (int64_t s = b; s < e; s += chunk) {
        const int64_t se = std::min<int64_t>(e, s + chunk);
        int lo = TX + N, hi = 0;          // accumulator columns this item's subgrids cover (of 128 + N)
        for (int64_t i = s; i < se; ++i) {
          const int x0 = pl->meta_host[(size_t)list[(size_t)i]].x0 - tx * TX;
          lo = std::min(lo, x0);
          hi = std::max(hi, x0 + N);
        }
        items.push_back(AdderItem{tx * TX, ty * TY, (int32_t)s, (int32_t)se, lo, hi});
      }
    }
  pl->n_adder_items = (int64_t)items.size();
  if (total > 0) {
    // the list entry carries the subgrid's offset relative to its tile: one load per entry in the kernel
    std::vector<int4> packed((size_t)total);
    for (int ty = 0; ty < nty; ++ty)
      for (int tx = 0; tx < ntx; ++tx)
        for (int64_t i = offs[(size_t)ty * ntx + tx]; i < offs[(size_t)ty * ntx + tx + 1]; ++i) {
          const auto &m = pl->meta_host[(size_t)list[(size_t)i]];
          packed[(size_t)i] = make_int4(list[(size_t)i], m.x0 - tx * TX, m.y0 - ty * TY, 0);
        }
    IDG_CUDA_TRY(cudaMalloc(&pl->adder_list_dev, sizeof(int4) * (size_t)total));
    IDG_CUDA_TRY(cudaMalloc(&pl->adder_items_dev, sizeof(AdderItem) * items.size()));
    IDG_CUDA_TRY(cudaMemcpyAsync(pl->adder_list_dev, packed.data(), sizeof(int4) * (size_t)total,
                                 cudaMemcpyHostToDevice, stream));
    IDG_CUDA_TRY(cudaMemcpyAsync(pl->adder_items_dev, items.data(), sizeof(AdderItem) * items.size(),
                                 cudaMemcpyHostToDevice, stream));
    IDG_CUDA_TRY(cudaStreamSynchronize(stream));  // the host vectors go out of scope
  }
  return IDG_OK;
}

// Everything a plan owns besides the metadata: frequencies, scratch, adder lists.
static int finish_plan(idg_plan *pl, const double *freqs_host, cudaStream_t stream) {
  const int N = pl->prm.subgrid_size;
  pl->P = (int64_t)pl->meta_host.size();
  pl->max_n_time = 0; pl->max_n_chan = 0; pl->min_n_chan = pl->meta_host.empty() ? 0 : INT32_MAX; pl->n_slots_needed = 0;
  pl->sorted_by_baseline = true;
  const bool span = (pl->prm.flags & IDG_PLAN_SPAN_ATERMS) != 0;
  int32_t prev_b = 0;
  for (const auto &m : pl->meta_host) {
    pl->max_n_time = std::max(pl->max_n_time, m.n_time);
    pl->max_n_chan = std::max(pl->max_n_chan, m.n_chan);
    pl->min_n_chan = std::min(pl->min_n_chan, m.n_chan);
    const int32_t last = span ? (m.time_begin + m.n_time - 1) / pl->prm.aterm_interval : m.aterm_slot;
    pl->n_slots_needed = std::max(pl->n_slots_needed, last + 1);
    if (m.baseline < prev_b) pl->sorted_by_baseline = false;
    prev_b = m.baseline;
  }
  // fraction of idle channel slots in the degridder if every thread owns cpt = 1, 2, 4, 8 channels of a timestep
  for (int k = 0; k < 4; ++k) {
    const int cpt = 1 << k;
    double used = 0.0, slots = 0.0;
    for (const auto &m : pl->meta_host) {
      used += (double)m.n_time * m.n_chan;
      slots += (double)m.n_time * ((m.n_chan + cpt - 1) / cpt) * cpt;
    }
    pl->dg_waste[k] = slots > 0.0 ? (float)(1.0 - used / slots) : 0.f;
  }
  pl->uniform_dkd = 0.f;
  if (pl->C >= 2) {
    const double df = freqs_host[1] - freqs_host[0];
    bool uniform = df != 0.0;
    for (int32_t c = 1; c + 1 < pl->C; ++c)
      uniform = uniform && std::fabs((freqs_host[c + 1] - freqs_host[c]) - df) <= 1e-9 * std::fabs(df);
    if (uniform) pl->uniform_dkd = (float)(6.283185307179586476925286766559 * df / kSpeedOfLight);
  }
  IDG_CUDA_TRY(cudaMalloc(&pl->freqs_dev, sizeof(double) * pl->C));
  IDG_CUDA_TRY(cudaMemcpyAsync(pl->freqs_dev, freqs_host, sizeof(double) * pl->C,
                               cudaMemcpyHostToDevice, stream));
  IDG_CUDA_TRY(cudaStreamSynchronize(stream));
  {
    // pixel direction cosines (R1: l_x = (x - N/2) S/N; R2: n' = sqrt(1 - l^2 - m^2) - 1 in its cancellation-free
    // form), the same for every subgrid of the plan
    std::vector<float4> lmn((size_t)N * N);
    for (int32_t y = 0; y < N; ++y)
      for (int32_t x = 0; x < N; ++x) {
        const double l = (double)(x - N / 2) * pl->prm.image_size / (double)N;
        const double m = (double)(y - N / 2) * pl->prm.image_size / (double)N;
        const double r2 = l * l + m * m;
        lmn[(size_t)y * N + x] = make_float4((float)l, (float)m, (float)(-r2 / (1.0 + std::sqrt(1.0 - r2))), 0.f);
      }
    IDG_CUDA_TRY(cudaMalloc(&pl->lmn_dev, sizeof(float4) * lmn.size()));
    IDG_CUDA_TRY(cudaMemcpyAsync(pl->lmn_dev, lmn.data(), sizeof(float4) * lmn.size(), cudaMemcpyHostToDevice, stream));
    IDG_CUDA_TRY(cudaStreamSynchronize(stream));
  }
  if (pl->P > 0)
    IDG_CUDA_TRY(cudaMalloc(&pl->subgrids_dev, sizeof(float2) * 4 * N * N * (size_t)pl->P));
  return build_adder_lists(pl, stream);
}

}  // namespace idg

using namespace idg;

extern "C" {

const char *idg_strerror(int code) {
  switch (code) {
    case IDG_OK: return "ok";
    case IDG_ERR_INVALID_ARG: return "invalid argument";
    case IDG_ERR_OUT_OF_MEMORY: return "out of memory";
    case IDG_ERR_CUDA: return "CUDA error (see idg_last_cuda_error)";
    case IDG_ERR_PLAN_MISMATCH: return "metadata does not match the plan parameters or array shapes";
    case IDG_ERR_UNSUPPORTED_SUBGRID_SIZE: return "subgrid size must be 16, 24, 32 or 48";
    case IDG_ERR_SCRATCH_TOO_SMALL: return "request exceeds the fixed scratch of the no-allocation (*_static) entry point";
    default: return "unknown error code";
  }
}

int idg_last_cuda_error(void) { return g_last_cuda_error; }

long long idg_kernel_launches(void) { return idg::g_kernel_launches.load(std::memory_order_relaxed); }

void idg_plan_destroy(idg_plan *pl) {
  if (!pl) return;
  cudaFree(pl->meta_dev); cudaFree(pl->freqs_dev); cudaFree(pl->lmn_dev); cudaFree(pl->subgrids_dev);
  cudaFree(pl->adder_list_dev); cudaFree(pl->adder_items_dev);
  cudaFree(pl->h_uvw_dev); cudaFree(pl->h_vis_dev); cudaFree(pl->h_aterms_dev);
  cudaFree(pl->h_grid_dev); cudaFree(pl->h_taper_dev);
  if (pl->h_copy_stream) cudaStreamDestroy(pl->h_copy_stream);
  for (auto e : pl->h_ev_in) if (e) cudaEventDestroy(e);
  for (auto e : pl->h_ev_out) if (e) cudaEventDestroy(e);
  delete pl;
}

int idg_plan_create(idg_plan **out, const idg_plan_params *prm, const float *uvw_dev,
                    const double *freqs_host, const int32_t *baselines_host, int32_t B, int32_t T,
                    int32_t C, int32_t n_stations, void *cuda_stream) {
  IDG_API_TRY
  if (out) *out = nullptr;
  if (!out || !uvw_dev || !freqs_host || !baselines_host || B < 1 || T < 1 || C < 1 || n_stations < 1)
    return IDG_ERR_INVALID_ARG;
  int rc = check_params(prm);
  if (rc != IDG_OK) return rc;
  for (int32_t b = 0; b < B; ++b)
    if (baselines_host[2 * b] < 0 || baselines_host[2 * b] >= n_stations ||
        baselines_host[2 * b + 1] < 0 || baselines_host[2 * b + 1] >= n_stations)
      return IDG_ERR_INVALID_ARG;
  idg_plan *pl = new (std::nothrow) idg_plan();
  if (!pl) return IDG_ERR_OUT_OF_MEMORY;
  pl->prm = *prm; pl->B = B; pl->T = T; pl->C = C; pl->n_stations = n_stations;
  pl->planner_made = true;
  cudaStream_t stream = (cudaStream_t)cuda_stream;
  try {
    rc = run_planner(*prm, uvw_dev, freqs_host, baselines_host, B, T, C, pl->meta_host, &pl->meta_dev,
                     &pl->n_planned, &pl->n_skipped, stream);
  } catch (const std::bad_alloc &) { rc = IDG_ERR_OUT_OF_MEMORY; }
  if (rc == IDG_OK) {
    try { rc = finish_plan(pl, freqs_host, stream); } catch (const std::bad_alloc &) { rc = IDG_ERR_OUT_OF_MEMORY; }
  }
  if (rc != IDG_OK) { idg_plan_destroy(pl); return rc; }
  *out = pl;
  return IDG_OK;
  IDG_API_CATCH
}

int idg_plan_from_metadata(idg_plan **out, const idg_plan_params *prm,
                           const idg_subgrid_meta *meta_host, int64_t P, const double *freqs_host,
                           int32_t B, int32_t T, int32_t C, int32_t n_stations, void *cuda_stream) {
  IDG_API_TRY
  if (out) *out = nullptr;
  if (!out || (!meta_host && P > 0) || P < 0 || !freqs_host || B < 1 || T < 1 || C < 1 || n_stations < 1)
    return IDG_ERR_INVALID_ARG;
  int rc = check_params(prm);
  if (rc != IDG_OK) return rc;
  const int N = prm->subgrid_size, L = prm->grid_size;
  int64_t planned = 0;
  for (int64_t p = 0; p < P; ++p) {
    const idg_subgrid_meta &m = meta_host[p];
    // ranges in int64: time_begin + n_time may not wrap past the <= T check
    bool ok = m.baseline >= 0 && m.baseline < B && m.station1 >= 0 && m.station1 < n_stations &&
              m.station2 >= 0 && m.station2 < n_stations && m.time_begin >= 0 && m.n_time >= 1 &&
              (int64_t)m.time_begin + m.n_time <= T && m.chan_begin >= 0 && m.n_chan >= 1 &&
              m.n_chan <= 256 && (int64_t)m.chan_begin + m.n_chan <= C && m.aterm_slot >= 0 &&
              m.x0 >= 0 && m.y0 >= 0 && (int64_t)m.x0 + N <= L && (int64_t)m.y0 + N <= L;
    // with IDG_PLAN_SPAN_ATERMS the kernels walk the slots from aterm_slot on: it must be the first timestep's
    if (ok && (prm->flags & IDG_PLAN_SPAN_ATERMS)) ok = m.aterm_slot == m.time_begin / prm->aterm_interval;
    if (!ok) return IDG_ERR_PLAN_MISMATCH;
    planned += (int64_t)m.n_time * m.n_chan;
  }
  idg_plan *pl = new (std::nothrow) idg_plan();
  if (!pl) return IDG_ERR_OUT_OF_MEMORY;
  pl->prm = *prm; pl->B = B; pl->T = T; pl->C = C; pl->n_stations = n_stations;
  try { pl->meta_host.assign(meta_host, meta_host + P); } catch (const std::bad_alloc &) { delete pl; return IDG_ERR_OUT_OF_MEMORY; }
  pl->n_planned = planned;
  pl->n_skipped = (int64_t)B * T * C - planned;
  cudaStream_t stream = (cudaStream_t)cuda_stream;
  rc = IDG_OK;
  if (P > 0) {
    cudaError_t e = cudaMalloc(&pl->meta_dev, sizeof(idg_subgrid_meta) * (size_t)P);
    if (e == cudaSuccess)
      e = cudaMemcpyAsync(pl->meta_dev, meta_host, sizeof(idg_subgrid_meta) * (size_t)P,
                          cudaMemcpyHostToDevice, stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(stream);
    if (e != cudaSuccess) { set_last_cuda_error(e); rc = IDG_ERR_CUDA; }
  }
  if (rc == IDG_OK) {
    try { rc = finish_plan(pl, freqs_host, stream); } catch (const std::bad_alloc &) { rc = IDG_ERR_OUT_OF_MEMORY; }
  }
  if (rc != IDG_OK) { idg_plan_destroy(pl); return rc; }
  *out = pl;
  return IDG_OK;
  IDG_API_CATCH
}

int idg_plan_size(const idg_plan *pl, int64_t *n_subgrids, int64_t *n_planned_vis,
                  int64_t *n_skipped_vis) {
  if (!pl) return IDG_ERR_INVALID_ARG;
  if (n_subgrids) *n_subgrids = pl->P;
  if (n_planned_vis) *n_planned_vis = pl->n_planned;
  if (n_skipped_vis) *n_skipped_vis = pl->n_skipped;
  return IDG_OK;
}

int idg_plan_metadata(const idg_plan *pl, idg_subgrid_meta *out_host, int64_t capacity) {
  if (!pl || (!out_host && pl->P > 0) || capacity < pl->P) return IDG_ERR_INVALID_ARG;
  if (pl->P > 0) std::memcpy(out_host, pl->meta_host.data(), sizeof(idg_subgrid_meta) * (size_t)pl->P);
  return IDG_OK;
}

int idg_plan_subgrids(const idg_plan *pl, void **subgrids_dev) {
  if (!pl || !subgrids_dev) return IDG_ERR_INVALID_ARG;
  *subgrids_dev = pl->subgrids_dev;
  return IDG_OK;
}

int idg_plan_aterm_slots(const idg_plan *pl, int32_t *n_slots) {
  if (!pl || !n_slots) return IDG_ERR_INVALID_ARG;
  *n_slots = pl->n_slots_needed;
  return IDG_OK;
}

int idg_plan_uses_tensor_cores(const idg_plan *pl, int32_t *flag) {
  if (!pl || !flag) return IDG_ERR_INVALID_ARG;
  *flag = (gridder_tc_eligible(pl) ? 1 : 0) | (degridder_tc_eligible(pl) ? 2 : 0);
  return IDG_OK;
}

int idg_plan_w_offset(const idg_plan *pl, int32_t w_index, double *w0) {
  if (!pl || !w0) return IDG_ERR_INVALID_ARG;
  *w0 = pl->prm.w_step > 0.0 ? ((double)w_index + 0.5) * pl->prm.w_step : 0.0;   // R4
  return IDG_OK;
}

}  // extern "C"
