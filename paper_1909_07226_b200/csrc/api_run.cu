// api_run.cu -- the compute entry points of include/idg_b200.h (stage calls, Alg. 1, Alg. 2,
// and the host-buffer variants).  Every step runs in the kernels of this library.
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

int needed_slots(const idg_plan *pl) {
  int s = 0;
  for (const auto &m : pl->meta_host) s = m.aterm_slot + 1 > s ? m.aterm_slot + 1 : s;
  return s;
}

}  // namespace

extern "C" {

int idg_gridder(const idg_plan *pl, const float *uvw_dev, const void *vis_dev,
                const void *aterms_dev, const float *taper_dev, void *subgrids_dev, void *stream) {
  if (!pl || !uvw_dev || !vis_dev || !aterms_dev || !taper_dev || (!subgrids_dev && pl->P > 0))
    return IDG_ERR_INVALID_ARG;
  return launch_gridder(pl, uvw_dev, (const float2 *)vis_dev, (const float2 *)aterms_dev, taper_dev,
                        (float2 *)subgrids_dev, S(stream));
}

int idg_subgrid_fft(const idg_plan *pl, void *subgrids_dev, int32_t direction, void *stream) {
  if (!pl || (!subgrids_dev && pl->P > 0) || (direction != -1 && direction != 1))
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

int idg_degridder(const idg_plan *pl, const float *uvw_dev, const void *subgrids_dev,
                  const void *aterms_dev, const float *taper_dev, void *vis_out_dev, void *stream) {
  if (!pl || !uvw_dev || (!subgrids_dev && pl->P > 0) || !aterms_dev || !taper_dev || !vis_out_dev)
    return IDG_ERR_INVALID_ARG;
  return launch_degridder(pl, uvw_dev, (const float2 *)subgrids_dev, (const float2 *)aterms_dev,
                          taper_dev, (float2 *)vis_out_dev, S(stream));
}

int idg_grid(const idg_plan *pl, const float *uvw_dev, const void *vis_dev, const void *aterms_dev,
             const float *taper_dev, void *grid_dev, void *stream) {
  if (!pl || !uvw_dev || !vis_dev || !aterms_dev || !taper_dev || !grid_dev) return IDG_ERR_INVALID_ARG;
  int rc = launch_gridder(pl, uvw_dev, (const float2 *)vis_dev, (const float2 *)aterms_dev, taper_dev,
                          pl->subgrids_dev, S(stream));
  if (rc == IDG_OK) rc = launch_subgrid_fft(pl, pl->subgrids_dev, -1, S(stream));
  if (rc == IDG_OK) rc = launch_adder(pl, pl->subgrids_dev, (float2 *)grid_dev, S(stream));
  return rc;
}

int idg_degrid(const idg_plan *pl, const float *uvw_dev, const void *grid_dev,
               const void *aterms_dev, const float *taper_dev, void *vis_out_dev, void *stream) {
  if (!pl || !uvw_dev || !grid_dev || !aterms_dev || !taper_dev || !vis_out_dev) return IDG_ERR_INVALID_ARG;
  if (pl->n_skipped > 0)  // skipped samples read as 0; planned ones are overwritten below
    IDG_CUDA_TRY(cudaMemsetAsync(vis_out_dev, 0, sizeof(float2) * 4 * (size_t)pl->B * pl->T * pl->C, S(stream)));
  int rc = launch_splitter(pl, (const float2 *)grid_dev, pl->subgrids_dev, S(stream));
  if (rc == IDG_OK) rc = launch_subgrid_fft(pl, pl->subgrids_dev, +1, S(stream));
  if (rc == IDG_OK)
    rc = launch_degridder(pl, uvw_dev, pl->subgrids_dev, (const float2 *)aterms_dev, taper_dev,
                          (float2 *)vis_out_dev, S(stream));
  return rc;
}

int idg_grid_host(idg_plan *pl, const float *uvw_host, const void *vis_host,
                  const void *aterms_host, int32_t n_slots, const float *taper_host,
                  void *grid_host, void *stream) {
  if (!pl || !uvw_host || !vis_host || !aterms_host || !taper_host || !grid_host) return IDG_ERR_INVALID_ARG;
  if (n_slots < needed_slots(pl)) return IDG_ERR_PLAN_MISMATCH;
  int rc = ensure_staging(pl, n_slots);
  if (rc != IDG_OK) return rc;
  const size_t N = pl->prm.subgrid_size, L = pl->prm.grid_size;
  const size_t nvis = (size_t)pl->B * pl->T * pl->C;
  cudaStream_t s = S(stream);
  IDG_CUDA_TRY(cudaMemcpyAsync(pl->h_uvw_dev, uvw_host, sizeof(float) * 3 * (size_t)pl->B * pl->T, cudaMemcpyHostToDevice, s));
  IDG_CUDA_TRY(cudaMemcpyAsync(pl->h_vis_dev, vis_host, sizeof(float2) * 4 * nvis, cudaMemcpyHostToDevice, s));
  IDG_CUDA_TRY(cudaMemcpyAsync(pl->h_aterms_dev, aterms_host, sizeof(float2) * 4 * N * N * (size_t)pl->n_stations * n_slots, cudaMemcpyHostToDevice, s));
  IDG_CUDA_TRY(cudaMemcpyAsync(pl->h_taper_dev, taper_host, sizeof(float) * N * N, cudaMemcpyHostToDevice, s));
  IDG_CUDA_TRY(cudaMemcpyAsync(pl->h_grid_dev, grid_host, sizeof(float2) * 4 * L * L, cudaMemcpyHostToDevice, s));
  rc = idg_grid(pl, pl->h_uvw_dev, pl->h_vis_dev, pl->h_aterms_dev, pl->h_taper_dev, pl->h_grid_dev, stream);
  if (rc != IDG_OK) return rc;
  IDG_CUDA_TRY(cudaMemcpyAsync(grid_host, pl->h_grid_dev, sizeof(float2) * 4 * L * L, cudaMemcpyDeviceToHost, s));
  IDG_CUDA_TRY(cudaStreamSynchronize(s));
  return IDG_OK;
}

int idg_degrid_host(idg_plan *pl, const float *uvw_host, const void *grid_host,
                    const void *aterms_host, int32_t n_slots, const float *taper_host,
                    void *vis_out_host, void *stream) {
  if (!pl || !uvw_host || !vis_out_host || !aterms_host || !taper_host || !grid_host) return IDG_ERR_INVALID_ARG;
  if (n_slots < needed_slots(pl)) return IDG_ERR_PLAN_MISMATCH;
  int rc = ensure_staging(pl, n_slots);
  if (rc != IDG_OK) return rc;
  const size_t N = pl->prm.subgrid_size, L = pl->prm.grid_size;
  const size_t nvis = (size_t)pl->B * pl->T * pl->C;
  cudaStream_t s = S(stream);
  IDG_CUDA_TRY(cudaMemcpyAsync(pl->h_uvw_dev, uvw_host, sizeof(float) * 3 * (size_t)pl->B * pl->T, cudaMemcpyHostToDevice, s));
  IDG_CUDA_TRY(cudaMemcpyAsync(pl->h_aterms_dev, aterms_host, sizeof(float2) * 4 * N * N * (size_t)pl->n_stations * n_slots, cudaMemcpyHostToDevice, s));
  IDG_CUDA_TRY(cudaMemcpyAsync(pl->h_taper_dev, taper_host, sizeof(float) * N * N, cudaMemcpyHostToDevice, s));
  IDG_CUDA_TRY(cudaMemcpyAsync(pl->h_grid_dev, grid_host, sizeof(float2) * 4 * L * L, cudaMemcpyHostToDevice, s));
  if (pl->n_skipped == 0 && pl->P == 0)
    IDG_CUDA_TRY(cudaMemsetAsync(pl->h_vis_dev, 0, sizeof(float2) * 4 * nvis, s));
  rc = idg_degrid(pl, pl->h_uvw_dev, pl->h_grid_dev, pl->h_aterms_dev, pl->h_taper_dev, pl->h_vis_dev, stream);
  if (rc != IDG_OK) return rc;
  IDG_CUDA_TRY(cudaMemcpyAsync(vis_out_host, pl->h_vis_dev, sizeof(float2) * 4 * nvis, cudaMemcpyDeviceToHost, s));
  IDG_CUDA_TRY(cudaStreamSynchronize(s));
  return IDG_OK;
}

}  // extern "C"
