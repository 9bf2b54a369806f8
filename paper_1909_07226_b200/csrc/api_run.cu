// api_run.cu -- the compute entry points of include/idg_b200.h (stage calls, Alg. 1, Alg. 2,
// and the host-buffer variants).  Every step runs in the kernels of this library.
#include <algorithm>
#include <vector>

#include "common.cuh"

using namespace idg;

namespace {

inline cudaStream_t S(void *s) { return (cudaStream_t)s; }

// grow-only device staging buffer
template <class Tp>
int ensure(Tp **buf, size_t bytes) {
  if (*buf) return IDG_OK;
  IDG_CUDA_TRY(cudaMalloc(buf, bytes));
  return IDG_OK;
}

int ensure_staging(idg_plan *pl, int32_t n_slots) {
  const size_t N = pl->prm.subgrid_size, L = pl->prm.grid_size;
  int rc;
  if ((rc = ensure(&pl->h_uvw_dev, sizeof(float) * 3 * (size_t)pl->B * pl->T)) != IDG_OK) return rc;
  if ((rc = ensure(&pl->h_vis_dev, sizeof(float2) * 4 * (size_t)pl->B * pl->T * pl->C)) != IDG_OK) return rc;
  if ((rc = ensure(&pl->h_grid_dev, sizeof(float2) * 4 * L * L)) != IDG_OK) return rc;
  if ((rc = ensure(&pl->h_taper_dev, sizeof(float) * N * N)) != IDG_OK) return rc;
  if (pl->h_aterms_dev && pl->h_aterm_slots < n_slots) {
    cudaFree(pl->h_aterms_dev);
    pl->h_aterms_dev = nullptr;
  }
  if (!pl->h_aterms_dev) {
    if ((rc = ensure(&pl->h_aterms_dev, sizeof(float2) * 4 * N * N * (size_t)pl->n_stations * n_slots)) != IDG_OK)
      return rc;
    pl->h_aterm_slots = n_slots;
  }
  return IDG_OK;
}

// The host-buffer calls overlap the PCIe copies with the kernels: the baselines are cut into kHostChunks
// contiguous ranges (the metadata is sorted by baseline, so a range of baselines is a range of subgrids and a
// contiguous slice of vis); uploads run on the plan's copy stream, kernels on the caller's stream, events
// order them.  Gridding: chunk k is gridded while chunk k+1 and then the grid itself are uploaded; the adder
// runs once at the end.  Degridding: chunk k's visibilities travel back while chunk k+1 is predicted.
struct HostChunk { int32_t b0, b1; int64_t p0, p1; };

int ensure_host_pipeline(idg_plan *pl) {
  if (!pl->h_copy_stream) IDG_CUDA_TRY(cudaStreamCreateWithFlags(&pl->h_copy_stream, cudaStreamNonBlocking));
  for (auto &e : pl->h_ev_in) if (!e) IDG_CUDA_TRY(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
  for (auto &e : pl->h_ev_out) if (!e) IDG_CUDA_TRY(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
  return IDG_OK;
}

std::vector<HostChunk> host_chunks(const idg_plan *pl) {
  std::vector<HostChunk> out;
  // metadata given through idg_plan_from_metadata may come in any order: a baseline range is then no subgrid range
  // and the calls run as one chunk (everything uploaded, then computed, then copied back)
  const int n = pl->sorted_by_baseline ? std::min<int>(idg_plan::kHostChunks, pl->B) : 1;
  int64_t p = 0;
  for (int k = 0; k < n; ++k) {
    HostChunk c;
    c.b0 = (int32_t)((int64_t)pl->B * k / n);
    c.b1 = (int32_t)((int64_t)pl->B * (k + 1) / n);
    c.p0 = p;
    while (p < pl->P && pl->meta_host[(size_t)p].baseline < c.b1) ++p;
    c.p1 = p;
    out.push_back(c);
  }
  return out;
}


}  // namespace

extern "C" {

int idg_gridder(const idg_plan *pl, const float *uvw_dev, const void *vis_dev,
                const void *aterms_dev, int32_t n_slots, const float *taper_dev, void *subgrids_dev, void *stream) {
  if (!pl || !uvw_dev || !vis_dev || !aterms_dev || !taper_dev || (!subgrids_dev && pl->P > 0))
    return IDG_ERR_INVALID_ARG;
  if (!aligned16(vis_dev) || !aligned16(aterms_dev) || !aligned16(subgrids_dev)) return IDG_ERR_INVALID_ARG;
  if (n_slots < pl->n_slots_needed) return IDG_ERR_PLAN_MISMATCH;
  return launch_gridder(pl, uvw_dev, (const float2 *)vis_dev, (const float2 *)aterms_dev, taper_dev,
                        (float2 *)subgrids_dev, S(stream));
}

int idg_subgrid_fft(const idg_plan *pl, void *subgrids_dev, int32_t direction, void *stream) {
  if (!pl || (!subgrids_dev && pl->P > 0) || (direction != -1 && direction != 1) || !aligned16(subgrids_dev))
    return IDG_ERR_INVALID_ARG;
  return launch_subgrid_fft(pl, (float2 *)subgrids_dev, direction, S(stream));
}

int idg_adder(const idg_plan *pl, const void *subgrids_dev, void *grid_dev, void *stream) {
  if (!pl || (!subgrids_dev && pl->P > 0) || !grid_dev) return IDG_ERR_INVALID_ARG;
  return launch_adder(pl, (const float2 *)subgrids_dev, (float2 *)grid_dev, S(stream));
}

int idg_splitter(const idg_plan *pl, const void *grid_dev, void *subgrids_dev, void *stream) {
  if (!pl || (!subgrids_dev && pl->P > 0) || !grid_dev) return IDG_ERR_INVALID_ARG;
  return launch_splitter(pl, (const float2 *)grid_dev, (float2 *)subgrids_dev, S(stream));
}

int idg_splitter_ifft(const idg_plan *pl, const void *grid_dev, void *subgrids_dev, void *stream) {
  if (!pl || (!subgrids_dev && pl->P > 0) || !grid_dev) return IDG_ERR_INVALID_ARG;
  return launch_splitter_ifft(pl, (const float2 *)grid_dev, (float2 *)subgrids_dev, S(stream));
}

int idg_degridder(const idg_plan *pl, const float *uvw_dev, const void *subgrids_dev,
                  const void *aterms_dev, int32_t n_slots, const float *taper_dev, void *vis_out_dev, void *stream) {
  if (!pl || !uvw_dev || (!subgrids_dev && pl->P > 0) || !aterms_dev || !taper_dev || !vis_out_dev)
    return IDG_ERR_INVALID_ARG;
  if (!aligned16(vis_out_dev) || !aligned16(aterms_dev) || !aligned16(subgrids_dev)) return IDG_ERR_INVALID_ARG;
  if (n_slots < pl->n_slots_needed) return IDG_ERR_PLAN_MISMATCH;
  return launch_degridder(pl, uvw_dev, (const float2 *)subgrids_dev, (const float2 *)aterms_dev,
                          taper_dev, (float2 *)vis_out_dev, S(stream));
}

int idg_grid(const idg_plan *pl, const float *uvw_dev, const void *vis_dev, const void *aterms_dev,
             int32_t n_slots, const float *taper_dev, void *grid_dev, void *stream) {
  if (!pl || !uvw_dev || !vis_dev || !aterms_dev || !taper_dev || !grid_dev) return IDG_ERR_INVALID_ARG;
  if (!aligned16(vis_dev) || !aligned16(aterms_dev)) return IDG_ERR_INVALID_ARG;
  if (n_slots < pl->n_slots_needed) return IDG_ERR_PLAN_MISMATCH;
  int rc = launch_gridder(pl, uvw_dev, (const float2 *)vis_dev, (const float2 *)aterms_dev, taper_dev,
                          pl->subgrids_dev, S(stream));
  if (rc == IDG_OK) rc = launch_subgrid_fft(pl, pl->subgrids_dev, -1, S(stream));
  if (rc == IDG_OK) rc = launch_adder(pl, pl->subgrids_dev, (float2 *)grid_dev, S(stream));
  return rc;
}

int idg_degrid(const idg_plan *pl, const float *uvw_dev, const void *grid_dev,
               const void *aterms_dev, int32_t n_slots, const float *taper_dev, void *vis_out_dev, void *stream) {
  if (!pl || !uvw_dev || !grid_dev || !aterms_dev || !taper_dev || !vis_out_dev) return IDG_ERR_INVALID_ARG;
  if (!aligned16(vis_out_dev) || !aligned16(aterms_dev)) return IDG_ERR_INVALID_ARG;
  if (n_slots < pl->n_slots_needed) return IDG_ERR_PLAN_MISMATCH;
  // skipped samples read as 0; planned ones are overwritten below.  Only the planner guarantees that every sample
  // is covered exactly once or counted skipped; caller-made metadata may overlap, so its output is always zeroed.
  if (pl->n_skipped > 0 || !pl->planner_made)
    IDG_CUDA_TRY(cudaMemsetAsync(vis_out_dev, 0, sizeof(float2) * 4 * (size_t)pl->B * pl->T * pl->C, S(stream)));
  int rc = launch_splitter_ifft(pl, (const float2 *)grid_dev, pl->subgrids_dev, S(stream));
  if (rc == IDG_OK)
    rc = launch_degridder(pl, uvw_dev, pl->subgrids_dev, (const float2 *)aterms_dev, taper_dev,
                          (float2 *)vis_out_dev, S(stream));
  return rc;
}

// ---- scalar variant (NEXT-3): one polarisation; subgrids [P][N][N] live in the first quarter of the plan's
// scratch; the plane-wise FFT kernel sees them as ceil(P / 4) four-plane subgrids ------------------------------
int idg_gridder_scalar(const idg_plan *pl, const float *uvw_dev, const void *vis_dev, const void *gains_dev, int32_t n_slots,
                       const float *taper_dev, void *subgrids_dev, void *stream) {
  if (!pl || !uvw_dev || !vis_dev || !gains_dev || !taper_dev || (!subgrids_dev && pl->P > 0)) return IDG_ERR_INVALID_ARG;
  if (pl->prm.flags & IDG_PLAN_SPAN_ATERMS) return IDG_ERR_PLAN_MISMATCH;   // scalar kernels are per-block c_p only
  if (n_slots < pl->n_slots_needed) return IDG_ERR_PLAN_MISMATCH;
  return launch_gridder_scalar(pl, uvw_dev, (const float2 *)vis_dev, (const float2 *)gains_dev, taper_dev,
                               (float2 *)subgrids_dev, S(stream));
}

int idg_degridder_scalar(const idg_plan *pl, const float *uvw_dev, const void *subgrids_dev, const void *gains_dev, int32_t n_slots,
                         const float *taper_dev, void *vis_out_dev, void *stream) {
  if (!pl || !uvw_dev || (!subgrids_dev && pl->P > 0) || !gains_dev || !taper_dev || !vis_out_dev) return IDG_ERR_INVALID_ARG;
  if (pl->prm.flags & IDG_PLAN_SPAN_ATERMS) return IDG_ERR_PLAN_MISMATCH;   // scalar kernels are per-block c_p only
  if (n_slots < pl->n_slots_needed) return IDG_ERR_PLAN_MISMATCH;
  return launch_degridder_scalar(pl, uvw_dev, (const float2 *)subgrids_dev, (const float2 *)gains_dev, taper_dev,
                                 (float2 *)vis_out_dev, S(stream));
}

int idg_grid_scalar(const idg_plan *pl, const float *uvw_dev, const void *vis_dev, const void *gains_dev, int32_t n_slots,
                    const float *taper_dev, void *grid_dev, void *stream) {
  if (!pl || !uvw_dev || !vis_dev || !gains_dev || !taper_dev || !grid_dev) return IDG_ERR_INVALID_ARG;
  if (pl->prm.flags & IDG_PLAN_SPAN_ATERMS) return IDG_ERR_PLAN_MISMATCH;   // scalar kernels are per-block c_p only
  if (n_slots < pl->n_slots_needed) return IDG_ERR_PLAN_MISMATCH;
  int rc = launch_gridder_scalar(pl, uvw_dev, (const float2 *)vis_dev, (const float2 *)gains_dev, taper_dev,
                                 pl->subgrids_dev, S(stream));
  if (rc == IDG_OK) rc = launch_subgrid_fft(pl, pl->subgrids_dev, -1, S(stream), 0, (pl->P + 3) / 4);
  if (rc == IDG_OK) rc = launch_adder(pl, pl->subgrids_dev, (float2 *)grid_dev, S(stream), 1);
  return rc;
}

int idg_degrid_scalar(const idg_plan *pl, const float *uvw_dev, const void *grid_dev, const void *gains_dev, int32_t n_slots,
                      const float *taper_dev, void *vis_out_dev, void *stream) {
  if (!pl || !uvw_dev || !grid_dev || !gains_dev || !taper_dev || !vis_out_dev) return IDG_ERR_INVALID_ARG;
  if (pl->prm.flags & IDG_PLAN_SPAN_ATERMS) return IDG_ERR_PLAN_MISMATCH;   // scalar kernels are per-block c_p only
  if (n_slots < pl->n_slots_needed) return IDG_ERR_PLAN_MISMATCH;
  if (pl->n_skipped > 0 || !pl->planner_made)
    IDG_CUDA_TRY(cudaMemsetAsync(vis_out_dev, 0, sizeof(float2) * (size_t)pl->B * pl->T * pl->C, S(stream)));
  int rc = launch_splitter(pl, (const float2 *)grid_dev, pl->subgrids_dev, S(stream), 0, -1, 1);
  if (rc == IDG_OK) rc = launch_subgrid_fft(pl, pl->subgrids_dev, +1, S(stream), 0, (pl->P + 3) / 4);
  if (rc == IDG_OK)
    rc = launch_degridder_scalar(pl, uvw_dev, pl->subgrids_dev, (const float2 *)gains_dev, taper_dev,
                                 (float2 *)vis_out_dev, S(stream));
  return rc;
}

static int grid_host_impl(idg_plan *pl, const float *uvw_host, const void *vis_host,
                  const void *aterms_host, int32_t n_slots, const float *taper_host,
                  void *grid_host, void *stream) {
  if (!pl || !uvw_host || !vis_host || !aterms_host || !taper_host || !grid_host) return IDG_ERR_INVALID_ARG;
  if (n_slots < pl->n_slots_needed) return IDG_ERR_PLAN_MISMATCH;
  int rc = ensure_staging(pl, n_slots);
  if (rc == IDG_OK) rc = ensure_host_pipeline(pl);
  if (rc != IDG_OK) return rc;
  const size_t N = pl->prm.subgrid_size, L = pl->prm.grid_size;
  const size_t row = (size_t)pl->T * pl->C * 4;                 // complex64 per baseline
  cudaStream_t s = S(stream), c = pl->h_copy_stream;
  const auto chunks = host_chunks(pl);
  const int K = idg_plan::kHostChunks;
  // the copy stream starts after whatever the caller queued on `stream`
  IDG_CUDA_TRY(cudaEventRecord(pl->h_ev_out[K], s));
  IDG_CUDA_TRY(cudaStreamWaitEvent(c, pl->h_ev_out[K], 0));
  IDG_CUDA_TRY(cudaMemcpyAsync(pl->h_uvw_dev, uvw_host, sizeof(float) * 3 * (size_t)pl->B * pl->T, cudaMemcpyHostToDevice, c));
  IDG_CUDA_TRY(cudaMemcpyAsync(pl->h_aterms_dev, aterms_host, sizeof(float2) * 4 * N * N * (size_t)pl->n_stations * n_slots, cudaMemcpyHostToDevice, c));
  IDG_CUDA_TRY(cudaMemcpyAsync(pl->h_taper_dev, taper_host, sizeof(float) * N * N, cudaMemcpyHostToDevice, c));
  IDG_CUDA_TRY(cudaEventRecord(pl->h_ev_in[K], c));
  for (size_t k = 0; k < chunks.size(); ++k) {
    const HostChunk &ch = chunks[k];
    IDG_CUDA_TRY(cudaMemcpyAsync(pl->h_vis_dev + (size_t)ch.b0 * row, (const float2 *)vis_host + (size_t)ch.b0 * row,
                                 sizeof(float2) * row * (size_t)(ch.b1 - ch.b0), cudaMemcpyHostToDevice, c));
    IDG_CUDA_TRY(cudaEventRecord(pl->h_ev_in[k], c));
  }
  IDG_CUDA_TRY(cudaMemcpyAsync(pl->h_grid_dev, grid_host, sizeof(float2) * 4 * L * L, cudaMemcpyHostToDevice, c));
  IDG_CUDA_TRY(cudaEventRecord(pl->h_ev_in[K + 1], c));

  IDG_CUDA_TRY(cudaStreamWaitEvent(s, pl->h_ev_in[K], 0));
  for (size_t k = 0; k < chunks.size(); ++k) {
    const HostChunk &ch = chunks[k];
    IDG_CUDA_TRY(cudaStreamWaitEvent(s, pl->h_ev_in[k], 0));
    rc = launch_gridder(pl, pl->h_uvw_dev, pl->h_vis_dev, pl->h_aterms_dev, pl->h_taper_dev, pl->subgrids_dev, s,
                        ch.p0, ch.p1 - ch.p0);
    if (rc == IDG_OK) rc = launch_subgrid_fft(pl, pl->subgrids_dev, -1, s, ch.p0, ch.p1 - ch.p0);
    if (rc != IDG_OK) return rc;
  }
  IDG_CUDA_TRY(cudaStreamWaitEvent(s, pl->h_ev_in[K + 1], 0));
  rc = launch_adder(pl, pl->subgrids_dev, pl->h_grid_dev, s);
  if (rc != IDG_OK) return rc;
  IDG_CUDA_TRY(cudaMemcpyAsync(grid_host, pl->h_grid_dev, sizeof(float2) * 4 * L * L, cudaMemcpyDeviceToHost, s));
  IDG_CUDA_TRY(cudaStreamSynchronize(s));
  return IDG_OK;
}

static int degrid_host_impl(idg_plan *pl, const float *uvw_host, const void *grid_host,
                    const void *aterms_host, int32_t n_slots, const float *taper_host,
                    void *vis_out_host, void *stream) {
  if (!pl || !uvw_host || !vis_out_host || !aterms_host || !taper_host || !grid_host) return IDG_ERR_INVALID_ARG;
  if (n_slots < pl->n_slots_needed) return IDG_ERR_PLAN_MISMATCH;
  int rc = ensure_staging(pl, n_slots);
  if (rc == IDG_OK) rc = ensure_host_pipeline(pl);
  if (rc != IDG_OK) return rc;
  const size_t N = pl->prm.subgrid_size, L = pl->prm.grid_size;
  const size_t row = (size_t)pl->T * pl->C * 4;
  const size_t nvis = (size_t)pl->B * pl->T * pl->C;
  cudaStream_t s = S(stream), c = pl->h_copy_stream;
  const auto chunks = host_chunks(pl);
  const int K = idg_plan::kHostChunks;
  IDG_CUDA_TRY(cudaMemcpyAsync(pl->h_uvw_dev, uvw_host, sizeof(float) * 3 * (size_t)pl->B * pl->T, cudaMemcpyHostToDevice, s));
  IDG_CUDA_TRY(cudaMemcpyAsync(pl->h_aterms_dev, aterms_host, sizeof(float2) * 4 * N * N * (size_t)pl->n_stations * n_slots, cudaMemcpyHostToDevice, s));
  IDG_CUDA_TRY(cudaMemcpyAsync(pl->h_taper_dev, taper_host, sizeof(float) * N * N, cudaMemcpyHostToDevice, s));
  IDG_CUDA_TRY(cudaMemcpyAsync(pl->h_grid_dev, grid_host, sizeof(float2) * 4 * L * L, cudaMemcpyHostToDevice, s));
  if (pl->n_skipped > 0 || !pl->planner_made)   // skipped samples read as 0; planned ones are overwritten below
    IDG_CUDA_TRY(cudaMemsetAsync(pl->h_vis_dev, 0, sizeof(float2) * 4 * nvis, s));
  for (size_t k = 0; k < chunks.size(); ++k) {
    const HostChunk &ch = chunks[k];
    rc = launch_splitter_ifft(pl, pl->h_grid_dev, pl->subgrids_dev, s, ch.p0, ch.p1 - ch.p0);
    if (rc == IDG_OK)
      rc = launch_degridder(pl, pl->h_uvw_dev, pl->subgrids_dev, pl->h_aterms_dev, pl->h_taper_dev, pl->h_vis_dev, s,
                            ch.p0, ch.p1 - ch.p0);
    if (rc != IDG_OK) return rc;
    IDG_CUDA_TRY(cudaEventRecord(pl->h_ev_out[k], s));
    IDG_CUDA_TRY(cudaStreamWaitEvent(c, pl->h_ev_out[k], 0));
    IDG_CUDA_TRY(cudaMemcpyAsync((float2 *)vis_out_host + (size_t)ch.b0 * row, pl->h_vis_dev + (size_t)ch.b0 * row,
                                 sizeof(float2) * row * (size_t)(ch.b1 - ch.b0), cudaMemcpyDeviceToHost, c));
  }
  IDG_CUDA_TRY(cudaStreamSynchronize(s));
  IDG_CUDA_TRY(cudaStreamSynchronize(c));
  return IDG_OK;
}

// Alg. 1 followed by Alg. 2 with the grid RESIDENT on the device: the small inputs and the visibilities go up once
// (chunk k is gridded while chunk k + 1 travels), the adder runs into a zeroed device grid, the grid travels back on
// the copy stream (if the caller wants it) while the chunks are predicted from the device copy, and chunk k's
// visibilities travel back while chunk k + 1 is predicted.  Against idg_grid_host + idg_degrid_host this saves one
// upload and (with grid_host == NULL) one download of the grid and the second upload of uvw / A-terms / taper.
static int grid_degrid_host_impl(idg_plan *pl, const float *uvw_host, const void *vis_host, const void *aterms_host,
                                 int32_t n_slots, const float *taper_host, void *grid_host, void *vis_out_host,
                                 void *stream) {
  if (!pl || !uvw_host || !vis_host || !aterms_host || !taper_host || !vis_out_host) return IDG_ERR_INVALID_ARG;
  if (n_slots < pl->n_slots_needed) return IDG_ERR_PLAN_MISMATCH;
  int rc = ensure_staging(pl, n_slots);
  if (rc == IDG_OK) rc = ensure_host_pipeline(pl);
  if (rc != IDG_OK) return rc;
  const size_t N = pl->prm.subgrid_size, L = pl->prm.grid_size;
  const size_t row = (size_t)pl->T * pl->C * 4;
  const size_t nvis = (size_t)pl->B * pl->T * pl->C;
  cudaStream_t s = S(stream), c = pl->h_copy_stream;
  const auto chunks = host_chunks(pl);
  const int K = idg_plan::kHostChunks;
  IDG_CUDA_TRY(cudaEventRecord(pl->h_ev_out[K], s));
  IDG_CUDA_TRY(cudaStreamWaitEvent(c, pl->h_ev_out[K], 0));
  IDG_CUDA_TRY(cudaMemcpyAsync(pl->h_uvw_dev, uvw_host, sizeof(float) * 3 * (size_t)pl->B * pl->T, cudaMemcpyHostToDevice, c));
  IDG_CUDA_TRY(cudaMemcpyAsync(pl->h_aterms_dev, aterms_host, sizeof(float2) * 4 * N * N * (size_t)pl->n_stations * n_slots, cudaMemcpyHostToDevice, c));
  IDG_CUDA_TRY(cudaMemcpyAsync(pl->h_taper_dev, taper_host, sizeof(float) * N * N, cudaMemcpyHostToDevice, c));
  IDG_CUDA_TRY(cudaEventRecord(pl->h_ev_in[K], c));
  for (size_t k = 0; k < chunks.size(); ++k) {
    const HostChunk &ch = chunks[k];
    IDG_CUDA_TRY(cudaMemcpyAsync(pl->h_vis_dev + (size_t)ch.b0 * row, (const float2 *)vis_host + (size_t)ch.b0 * row,
                                 sizeof(float2) * row * (size_t)(ch.b1 - ch.b0), cudaMemcpyHostToDevice, c));
    IDG_CUDA_TRY(cudaEventRecord(pl->h_ev_in[k], c));
  }
  // ---- Alg. 1 into a zeroed device grid
  IDG_CUDA_TRY(cudaMemsetAsync(pl->h_grid_dev, 0, sizeof(float2) * 4 * L * L, s));
  IDG_CUDA_TRY(cudaStreamWaitEvent(s, pl->h_ev_in[K], 0));
  for (size_t k = 0; k < chunks.size(); ++k) {
    const HostChunk &ch = chunks[k];
    IDG_CUDA_TRY(cudaStreamWaitEvent(s, pl->h_ev_in[k], 0));
    rc = launch_gridder(pl, pl->h_uvw_dev, pl->h_vis_dev, pl->h_aterms_dev, pl->h_taper_dev, pl->subgrids_dev, s,
                        ch.p0, ch.p1 - ch.p0);
    if (rc == IDG_OK) rc = launch_subgrid_fft(pl, pl->subgrids_dev, -1, s, ch.p0, ch.p1 - ch.p0);
    if (rc != IDG_OK) return rc;
  }
  rc = launch_adder(pl, pl->subgrids_dev, pl->h_grid_dev, s);
  if (rc != IDG_OK) return rc;
  IDG_CUDA_TRY(cudaEventRecord(pl->h_ev_in[K + 1], s));          // the grid is complete
  IDG_CUDA_TRY(cudaStreamWaitEvent(c, pl->h_ev_in[K + 1], 0));
  if (grid_host)
    IDG_CUDA_TRY(cudaMemcpyAsync(grid_host, pl->h_grid_dev, sizeof(float2) * 4 * L * L, cudaMemcpyDeviceToHost, c));
  // ---- Alg. 2 from the device grid; the staging buffer of the measured visibilities receives the predicted ones
  if (pl->n_skipped > 0 || !pl->planner_made)
    IDG_CUDA_TRY(cudaMemsetAsync(pl->h_vis_dev, 0, sizeof(float2) * 4 * nvis, s));
  for (size_t k = 0; k < chunks.size(); ++k) {
    const HostChunk &ch = chunks[k];
    rc = launch_splitter_ifft(pl, pl->h_grid_dev, pl->subgrids_dev, s, ch.p0, ch.p1 - ch.p0);
    if (rc == IDG_OK)
      rc = launch_degridder(pl, pl->h_uvw_dev, pl->subgrids_dev, pl->h_aterms_dev, pl->h_taper_dev, pl->h_vis_dev, s,
                            ch.p0, ch.p1 - ch.p0);
    if (rc != IDG_OK) return rc;
    IDG_CUDA_TRY(cudaEventRecord(pl->h_ev_out[k], s));
    IDG_CUDA_TRY(cudaStreamWaitEvent(c, pl->h_ev_out[k], 0));
    IDG_CUDA_TRY(cudaMemcpyAsync((float2 *)vis_out_host + (size_t)ch.b0 * row, pl->h_vis_dev + (size_t)ch.b0 * row,
                                 sizeof(float2) * row * (size_t)(ch.b1 - ch.b0), cudaMemcpyDeviceToHost, c));
  }
  IDG_CUDA_TRY(cudaStreamSynchronize(s));
  IDG_CUDA_TRY(cudaStreamSynchronize(c));
  return IDG_OK;
}

// On failure the asynchronous copies already queued still reference the caller's host buffers: both streams are
// drained before the error is returned, so the caller may free them.
static int host_call_epilogue(idg_plan *pl, void *stream, int rc) {
  if (rc != IDG_OK && pl) {
    cudaStreamSynchronize(S(stream));
    if (pl->h_copy_stream) cudaStreamSynchronize(pl->h_copy_stream);
  }
  return rc;
}

int idg_grid_host(idg_plan *pl, const float *uvw_host, const void *vis_host, const void *aterms_host, int32_t n_slots,
                  const float *taper_host, void *grid_host, void *stream) {
  int rc;
  try {
    rc = grid_host_impl(pl, uvw_host, vis_host, aterms_host, n_slots, taper_host, grid_host, stream);
  } catch (const std::bad_alloc &) { rc = IDG_ERR_OUT_OF_MEMORY; } catch (...) { rc = IDG_ERR_INVALID_ARG; }
  return host_call_epilogue(pl, stream, rc);
}

int idg_degrid_host(idg_plan *pl, const float *uvw_host, const void *grid_host, const void *aterms_host,
                    int32_t n_slots, const float *taper_host, void *vis_out_host, void *stream) {
  int rc;
  try {
    rc = degrid_host_impl(pl, uvw_host, grid_host, aterms_host, n_slots, taper_host, vis_out_host, stream);
  } catch (const std::bad_alloc &) { rc = IDG_ERR_OUT_OF_MEMORY; } catch (...) { rc = IDG_ERR_INVALID_ARG; }
  return host_call_epilogue(pl, stream, rc);
}

int idg_grid_degrid_host(idg_plan *pl, const float *uvw_host, const void *vis_host, const void *aterms_host,
                         int32_t n_slots, const float *taper_host, void *grid_host, void *vis_out_host, void *stream) {
  int rc;
  try {
    rc = grid_degrid_host_impl(pl, uvw_host, vis_host, aterms_host, n_slots, taper_host, grid_host, vis_out_host, stream);
  } catch (const std::bad_alloc &) { rc = IDG_ERR_OUT_OF_MEMORY; } catch (...) { rc = IDG_ERR_INVALID_ARG; }
  return host_call_epilogue(pl, stream, rc);
}

}  // extern "C"
