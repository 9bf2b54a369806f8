// plan.cu -- the IDG planner on the GPU (row a0).
//
// Section 3.2 of the paper (Fig. 2) asks for a partition of the
// visibilities into blocks of one baseline x a run of timesteps x a run of channels whose uv
// samples fit a "tight box" of L_p x L_p pixels; it gives no algorithm.  The rule implemented
// here is the greedy walk written out in DESIGN.md (readings R10-R12): per baseline, channel
// groups of max_channels halved until one timestep fits the pixel budget N - kernel_size, then
// timesteps appended while the box of the two end channels stays inside the budget, the A-term
// slot (R5) and the w layer (R4) do not change and max_timesteps is not reached.
//
// One thread walks one baseline (the walk is sequential in time by construction); pass 1 counts,
// the host scans the B counts, pass 2 emits at the scanned offsets, so the metadata order is
// (baseline, channel group, time).  All floating point is double with explicit round-to-nearest
// intrinsics (__dmul_rn, __dadd_rn, ...), which nvcc never contracts into FMAs: the metadata is
// a pure function of the inputs and reproducible bit for bit.
#include "common.cuh"

namespace idg {

struct PlanConst {
  int32_t B, T, C, N, L, max_timesteps, max_channels, aterm_interval, force, span;
  double budget, w_step;
};

template <bool EMIT>
__device__ void walk_baseline(const PlanConst pc, const float *__restrict__ uvw_b,
                              const double *__restrict__ freqs, const double *__restrict__ scale,
                              int32_t b, int32_t st1, int32_t st2, idg_subgrid_meta *out,
                              int64_t *count_out, int64_t *planned_out, int64_t *skipped_out) {
  const double inv_c0 = 1.0 / kSpeedOfLight;
  int64_t count = 0, planned = 0, skipped = 0;
  int32_t c0 = 0;
  while (c0 < pc.C) {
    int32_t n = pc.max_channels;
    while (n > pc.C - c0) n = n / 2;
    if (!pc.force) {
      while (n > 1) {
        const double ds = __dsub_rn(scale[c0 + n - 1], scale[c0]);
        double mx = 0.0;
        for (int32_t t = 0; t < pc.T; ++t) {
          const double du = fabs(__dmul_rn((double)uvw_b[3 * t + 0], ds));
          const double dv = fabs(__dmul_rn((double)uvw_b[3 * t + 1], ds));
          if (du > mx) mx = du;
          if (dv > mx) mx = dv;
        }
        if (mx > pc.budget) n = n / 2; else break;
      }
    }
    const double s_lo = scale[c0], s_hi = scale[c0 + n - 1];
    const double k_mid = __dmul_rn(__dmul_rn(0.5, __dadd_rn(freqs[c0], freqs[c0 + n - 1])), inv_c0);
    int32_t t0 = 0;
    while (t0 < pc.T) {
      int32_t t1 = t0;
      double umin = 0, umax = 0, vmin = 0, vmax = 0;
      int32_t wi0 = 0;
      while (t1 < pc.T && t1 - t0 < pc.max_timesteps &&
             (pc.span || t1 / pc.aterm_interval == t0 / pc.aterm_interval)) {
        int32_t wi = 0;
        if (pc.w_step > 0.0)
          wi = (int32_t)floor(__ddiv_rn(__dmul_rn((double)uvw_b[3 * t1 + 2], k_mid), pc.w_step));
        if (t1 == t0) wi0 = wi; else if (wi != wi0) break;
        const double u = (double)uvw_b[3 * t1 + 0], v = (double)uvw_b[3 * t1 + 1];
        const double ua = __dmul_rn(u, s_lo), ub = __dmul_rn(u, s_hi);
        const double va = __dmul_rn(v, s_lo), vb = __dmul_rn(v, s_hi);
        double numin, numax, nvmin, nvmax;
        if (t1 == t0) {
          numin = fmin(ua, ub); numax = fmax(ua, ub); nvmin = fmin(va, vb); nvmax = fmax(va, vb);
        } else {
          numin = fmin(umin, fmin(ua, ub)); numax = fmax(umax, fmax(ua, ub));
          nvmin = fmin(vmin, fmin(va, vb)); nvmax = fmax(vmax, fmax(va, vb));
          if (!pc.force && (__dsub_rn(numax, numin) > pc.budget || __dsub_rn(nvmax, nvmin) > pc.budget))
            break;
        }
        umin = numin; umax = numax; vmin = nvmin; vmax = nvmax;
        ++t1;
      }
      const int32_t xc = (int32_t)floor(__dadd_rn(__dmul_rn(0.5, __dadd_rn(umin, umax)), 0.5));
      const int32_t yc = (int32_t)floor(__dadd_rn(__dmul_rn(0.5, __dadd_rn(vmin, vmax)), 0.5));
      const int32_t x0 = xc + pc.L / 2 - pc.N / 2, y0 = yc + pc.L / 2 - pc.N / 2;
      const int64_t nvis = (int64_t)(t1 - t0) * n;
      if (x0 >= 0 && y0 >= 0 && x0 + pc.N <= pc.L && y0 + pc.N <= pc.L) {
        if (EMIT) {
          idg_subgrid_meta m;
          m.baseline = b; m.station1 = st1; m.station2 = st2;
          m.time_begin = t0; m.n_time = t1 - t0; m.chan_begin = c0; m.n_chan = n;
          m.aterm_slot = t0 / pc.aterm_interval; m.x0 = x0; m.y0 = y0; m.w_index = wi0;
          m.reserved = 0;
          out[count] = m;
        }
        ++count; planned += nvis;
      } else {
        skipped += nvis;
      }
      t0 = t1;
    }
    c0 += n;
  }
  if (!EMIT) { *count_out = count; *planned_out = planned; *skipped_out = skipped; }
}

template <bool EMIT>
__global__ void plan_kernel(const PlanConst pc, const float *__restrict__ uvw,
                            const double *__restrict__ freqs, const double *__restrict__ scale,
                            const int32_t *__restrict__ baselines, int64_t *counts /*[3][B]*/,
                            const int64_t *__restrict__ offsets, idg_subgrid_meta *meta) {
  const int32_t b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= pc.B) return;
  const float *uvw_b = uvw + (size_t)b * pc.T * 3;
  if (EMIT)
    walk_baseline<true>(pc, uvw_b, freqs, scale, b, baselines[2 * b], baselines[2 * b + 1],
                        meta + offsets[b], nullptr, nullptr, nullptr);
  else
    walk_baseline<false>(pc, uvw_b, freqs, scale, b, 0, 0, nullptr, counts + b, counts + pc.B + b,
                         counts + 2 * (size_t)pc.B + b);
}

int run_planner(const idg_plan_params &prm, const float *uvw_dev, const double *freqs_host,
                const int32_t *baselines_host, int32_t B, int32_t T, int32_t C,
                std::vector<idg_subgrid_meta> &meta_out, idg_subgrid_meta **meta_dev_out,
                int64_t *planned, int64_t *skipped, cudaStream_t stream) {
  PlanConst pc;
  pc.B = B; pc.T = T; pc.C = C; pc.N = prm.subgrid_size; pc.L = prm.grid_size;
  pc.max_timesteps = prm.max_timesteps; pc.max_channels = prm.max_channels;
  pc.aterm_interval = prm.aterm_interval; pc.force = (prm.flags & IDG_PLAN_FORCE_BLOCKS) != 0;
  pc.span = (prm.flags & IDG_PLAN_SPAN_ATERMS) != 0;
  pc.budget = (double)(prm.subgrid_size - prm.kernel_size);
  pc.w_step = prm.w_step;
  // pixel scale per channel: (f / c0) * S, two roundings in this order (host, no contraction:
  // the translation unit is compiled with -ffp-contract=off)
  std::vector<double> scale(C);
  const double inv_c0 = 1.0 / kSpeedOfLight;
  for (int32_t c = 0; c < C; ++c) {
    volatile double k = freqs_host[c] * inv_c0;
    scale[c] = k * prm.image_size;
  }
  double *freqs_dev = nullptr, *scale_dev = nullptr;
  int32_t *bl_dev = nullptr;
  int64_t *counts_dev = nullptr, *offsets_dev = nullptr;
  idg_subgrid_meta *meta_dev = nullptr;
  int rc = IDG_OK;
  auto cleanup = [&]() {
    cudaFree(freqs_dev); cudaFree(scale_dev); cudaFree(bl_dev); cudaFree(counts_dev);
    cudaFree(offsets_dev);
  };
#define PLAN_TRY(expr)                                                        \
  do {                                                                        \
    cudaError_t _e = (expr);                                                  \
    if (_e != cudaSuccess) {                                                  \
      set_last_cuda_error(_e);                                                \
      rc = _e == cudaErrorMemoryAllocation ? IDG_ERR_OUT_OF_MEMORY : IDG_ERR_CUDA; \
      cleanup(); cudaFree(meta_dev);                                          \
      return rc;                                                              \
    }                                                                         \
  } while (0)
  PLAN_TRY(cudaMalloc(&freqs_dev, sizeof(double) * C));
  PLAN_TRY(cudaMalloc(&scale_dev, sizeof(double) * C));
  PLAN_TRY(cudaMalloc(&bl_dev, sizeof(int32_t) * 2 * (size_t)B));
  PLAN_TRY(cudaMalloc(&counts_dev, sizeof(int64_t) * 3 * (size_t)B));
  PLAN_TRY(cudaMalloc(&offsets_dev, sizeof(int64_t) * (size_t)B));
  PLAN_TRY(cudaMemcpyAsync(freqs_dev, freqs_host, sizeof(double) * C, cudaMemcpyHostToDevice, stream));
  PLAN_TRY(cudaMemcpyAsync(scale_dev, scale.data(), sizeof(double) * C, cudaMemcpyHostToDevice, stream));
  PLAN_TRY(cudaMemcpyAsync(bl_dev, baselines_host, sizeof(int32_t) * 2 * (size_t)B,
                           cudaMemcpyHostToDevice, stream));
  const int threads = 32;  // small blocks: B is a few thousand, spread the walks over all SMs
  const int blocks = (B + threads - 1) / threads;
  plan_kernel<false><<<blocks, threads, 0, stream>>>(pc, uvw_dev, freqs_dev, scale_dev, bl_dev,
                                                     counts_dev, nullptr, nullptr);
  count_launch();
  PLAN_TRY(cudaGetLastError());
  std::vector<int64_t> counts(3 * (size_t)B);
  PLAN_TRY(cudaMemcpyAsync(counts.data(), counts_dev, sizeof(int64_t) * 3 * (size_t)B,
                           cudaMemcpyDeviceToHost, stream));
  PLAN_TRY(cudaStreamSynchronize(stream));
  std::vector<int64_t> offsets(B);
  int64_t P = 0, pl = 0, sk = 0;
  for (int32_t b = 0; b < B; ++b) {
    offsets[b] = P; P += counts[b]; pl += counts[(size_t)B + b]; sk += counts[2 * (size_t)B + b];
  }
  meta_out.resize((size_t)P);
  if (P > 0) {
    PLAN_TRY(cudaMalloc(&meta_dev, sizeof(idg_subgrid_meta) * (size_t)P));
    PLAN_TRY(cudaMemcpyAsync(offsets_dev, offsets.data(), sizeof(int64_t) * (size_t)B,
                             cudaMemcpyHostToDevice, stream));
    plan_kernel<true><<<blocks, threads, 0, stream>>>(pc, uvw_dev, freqs_dev, scale_dev, bl_dev,
                                                      nullptr, offsets_dev, meta_dev);
    count_launch();
    PLAN_TRY(cudaGetLastError());
    PLAN_TRY(cudaMemcpyAsync(meta_out.data(), meta_dev, sizeof(idg_subgrid_meta) * (size_t)P,
                             cudaMemcpyDeviceToHost, stream));
    PLAN_TRY(cudaStreamSynchronize(stream));
  }
#undef PLAN_TRY
  cleanup();
  *meta_dev_out = meta_dev;
  *planned = pl;
  *skipped = sk;
  return IDG_OK;
}

}  // namespace idg
