// scalar.cu -- NEXT-3 row: the scalar (one polarisation, Stokes-I-like) variant of the
// gridder and degridder.  The paper derives the method for scalar visibilities first (Eq. 1-25, PAPER.md:51-235;
// the 2x2 form is a substitution) and quotes a "Stokes I only" timing for the classical gridder
// (PAPER.md:481).  With complex gains g (Eq. 2):
//   gridder   Sg[y][x] = taper[y][x] conj(g1[y][x]) (sum_k Y_k exp(+i phase_k(x, y))) g2[y][x]
//   degridder Y_k = sum_xy g1 (taper Ip) conj(g2) exp(-i phase_k(x, y))
// which is the XX plane of the 4-polarisation path when the Jones matrices are g times the identity -- that
// identity is what the tests use, so the 4-polarisation oracle pins this variant too.
//
// Per (visibility, pixel): 1 FFMA + 1 FMUL + 2 MUFU + 4 FFMA -- the XU (MUFU) pipe, 16 lanes/clk/SM, is the
// bound here (2.27 GVis/s at N = 32), not the FP32 lanes.  Layouts: vis [B][T][C] complex64, gains
// [slots][stations][N][N] complex64, subgrids [P][N][N] complex64.  Phase arithmetic as in gridder.cu.
#include "common.cuh"

namespace idg {

constexpr int kSVisBatch = 512;   // scalar visibilities staged per batch (8 B each)
constexpr int kSMaxChan = 256;

template <int N, int NT, int PPT, int MINB, int R>
__global__ void __launch_bounds__(NT, MINB)
gridder_scalar_kernel(const idg_subgrid_meta *__restrict__ meta, const float *__restrict__ uvw,
                      const double *__restrict__ freqs, const float2 *__restrict__ vis,
                      const float2 *__restrict__ gains, const float *__restrict__ taper,
                      float2 *__restrict__ subgrids, int32_t T, int32_t C, int32_t n_stations, int32_t L,
                      double image_size, double w_step, float dkd) {
  static_assert(NT * PPT == N * N, "pixels must tile the CTA exactly");
  __shared__ float2 s_vis[kSVisBatch];
  __shared__ float4 s_t[kSVisBatch * 2];
  __shared__ float s_kd[kSMaxChan];
  const int tid = threadIdx.x;
  const idg_subgrid_meta m = meta[blockIdx.x];
  const int n_chan = m.n_chan, n_time = m.n_time;
  const double two_pi = 6.283185307179586476925286766559;
  const double inv_c0 = 1.0 / kSpeedOfLight;
  const double u0 = (double)(m.x0 + N / 2 - L / 2) / image_size;
  const double v0 = (double)(m.y0 + N / 2 - L / 2) / image_size;
  const double w0 = w_step > 0.0 ? ((double)m.w_index + 0.5) * w_step : 0.0;
  const double k_mid = 0.5 * (freqs[m.chan_begin] + freqs[m.chan_begin + n_chan - 1]) * inv_c0;
  for (int c = tid; c < n_chan; c += NT)
    s_kd[c] = (float)(two_pi * (freqs[m.chan_begin + c] * inv_c0 - k_mid));
  float pl[PPT], pm[PPT], pn[PPT];
#pragma unroll
  for (int k = 0; k < PPT; ++k) {
    const int pix = tid + k * NT;
    const int y = pix / N, x = pix - y * N;
    const double l = (double)(x - N / 2) * image_size / (double)N;
    const double mm = (double)(y - N / 2) * image_size / (double)N;
    const double r2 = l * l + mm * mm;
    pl[k] = (float)l; pm[k] = (float)mm; pn[k] = (float)(-r2 / (1.0 + sqrt(1.0 - r2)));
  }
  float2 acc[PPT];
#pragma unroll
  for (int k = 0; k < PPT; ++k) acc[k] = make_float2(0.f, 0.f);

  const int tb_max = n_chan >= kSVisBatch ? 1 : kSVisBatch / n_chan;
  const float *uvw_b = uvw + (size_t)m.baseline * T * 3;
  for (int t0 = 0; t0 < n_time; t0 += tb_max) {
    const int tb = min(tb_max, n_time - t0);
    for (int c_lo = 0; c_lo < n_chan; c_lo += kSVisBatch) {
      const int nc = min(kSVisBatch, n_chan - c_lo);
      __syncthreads();
      for (int i = tid; i < tb * nc; i += NT) {
        const int tl = i / nc, r = i - tl * nc;
        s_vis[i] = __ldg(&vis[((size_t)m.baseline * T + (m.time_begin + t0 + tl)) * C + (m.chan_begin + c_lo + r)]);
      }
      for (int tl = tid; tl < tb; tl += NT) {
        const float *p = uvw_b + (size_t)(m.time_begin + t0 + tl) * 3;
        const float u = p[0], v = p[1], w = p[2];
        s_t[2 * tl] = make_float4(u, v, w, 0.f);
        s_t[2 * tl + 1] = make_float4((float)(two_pi * ((double)u * k_mid - u0)),
                                      (float)(two_pi * ((double)v * k_mid - v0)),
                                      (float)(two_pi * ((double)w * k_mid - w0)), 0.f);
      }
      __syncthreads();
      for (int tl = 0; tl < tb; ++tl) {
        const float4 tu = s_t[2 * tl], tbs = s_t[2 * tl + 1];
        float pidx[PPT], base[PPT];
#pragma unroll
        for (int k = 0; k < PPT; ++k) {
          pidx[k] = fmaf(tu.x, pl[k], fmaf(tu.y, pm[k], tu.z * pn[k]));
          base[k] = fmaf(tbs.x, pl[k], fmaf(tbs.y, pm[k], tbs.z * pn[k]));
        }
        const float2 *vp = s_vis + (size_t)tl * nc;
        if (R == 1) {
#pragma unroll 4
          for (int c = 0; c < nc; ++c) {
            const float kd = s_kd[c_lo + c];
            const float2 v = vp[c];
#pragma unroll
            for (int k = 0; k < PPT; ++k) {
              float s, co;
              __sincosf(fmaf(pidx[k], kd, base[k]), &s, &co);
              acc[k].x = fmaf(v.x, co, acc[k].x); acc[k].x = fmaf(-v.y, s, acc[k].x);
              acc[k].y = fmaf(v.x, s, acc[k].y);  acc[k].y = fmaf(v.y, co, acc[k].y);
            }
          }
        } else {
          // per-channel phase recurrence (uniform channel spacing): sin/cos on every R-th channel, one complex
          // rotation by exp(i pidx dkd) for the channels in between -- trades MUFU for FP32 FMAs
          float cr[PPT], sr[PPT];
#pragma unroll
          for (int k = 0; k < PPT; ++k) __sincosf(pidx[k] * dkd, &sr[k], &cr[k]);
          for (int c0 = 0; c0 < nc; c0 += R) {
            const float kd = s_kd[c_lo + c0];
            float co[PPT], sn[PPT];
#pragma unroll
            for (int k = 0; k < PPT; ++k) __sincosf(fmaf(pidx[k], kd, base[k]), &sn[k], &co[k]);
#pragma unroll
            for (int j = 0; j < R; ++j) {
              if (c0 + j < nc) {
                const float2 v = vp[c0 + j];
#pragma unroll
                for (int k = 0; k < PPT; ++k) {
                  acc[k].x = fmaf(v.x, co[k], acc[k].x); acc[k].x = fmaf(-v.y, sn[k], acc[k].x);
                  acc[k].y = fmaf(v.x, sn[k], acc[k].y); acc[k].y = fmaf(v.y, co[k], acc[k].y);
                  if (j + 1 < R) {
                    const float c2 = fmaf(co[k], cr[k], -sn[k] * sr[k]);
                    sn[k] = fmaf(sn[k], cr[k], co[k] * sr[k]);
                    co[k] = c2;
                  }
                }
              }
            }
          }
        }
      }
    }
  }
  const size_t g1_off = ((size_t)m.aterm_slot * n_stations + m.station1) * (N * N);
  const size_t g2_off = ((size_t)m.aterm_slot * n_stations + m.station2) * (N * N);
  float2 *out = subgrids + (size_t)blockIdx.x * N * N;
#pragma unroll
  for (int k = 0; k < PPT; ++k) {
    const int pix = tid + k * NT;
    const float2 g1 = __ldg(&gains[g1_off + pix]), g2 = __ldg(&gains[g2_off + pix]);
    const float tp = __ldg(&taper[pix]);
    const float2 r = cmul(cmul_conj_a(g1, acc[k]), g2);
    out[pix] = make_float2(tp * r.x, tp * r.y);
  }
}

template <int N, int NT, int CPT, int R>
__global__ void __launch_bounds__(NT)
degridder_scalar_kernel(const idg_subgrid_meta *__restrict__ meta, const float *__restrict__ uvw,
                        const double *__restrict__ freqs, const float2 *__restrict__ subgrids,
                        const float2 *__restrict__ gains, const float *__restrict__ taper,
                        float2 *__restrict__ vis_out, int32_t T, int32_t C, int32_t n_stations, int32_t L,
                        double image_size, double w_step, float dkd) {
  constexpr int NPIX = N * N;
  constexpr int CH = NPIX < 1024 ? NPIX : 1024;
  __shared__ float2 s_pix[CH];
  __shared__ float4 s_lmn[CH];
  const int tid = threadIdx.x;
  const idg_subgrid_meta m = meta[blockIdx.x];
  const int n_chan = m.n_chan, n_time = m.n_time;
  const double two_pi = 6.283185307179586476925286766559;
  const double inv_c0 = 1.0 / kSpeedOfLight;
  const double u0 = (double)(m.x0 + N / 2 - L / 2) / image_size;
  const double v0 = (double)(m.y0 + N / 2 - L / 2) / image_size;
  const double w0 = w_step > 0.0 ? ((double)m.w_index + 0.5) * w_step : 0.0;
  const double k_mid = 0.5 * (freqs[m.chan_begin] + freqs[m.chan_begin + n_chan - 1]) * inv_c0;
  const int groups = (n_chan + CPT - 1) / CPT;
  const int n_items = n_time * groups;
  const size_t g1_off = ((size_t)m.aterm_slot * n_stations + m.station1) * NPIX;
  const size_t g2_off = ((size_t)m.aterm_slot * n_stations + m.station2) * NPIX;
  const float2 *sg = subgrids + (size_t)blockIdx.x * NPIX;

  for (int item0 = 0; item0 < n_items; item0 += NT) {
    const int item = item0 + tid;
    const bool active = item < n_items;
    const int tl = active ? item / groups : 0;
    const int cg = active ? (item - tl * groups) * CPT : 0;
    const float *p = uvw + ((size_t)m.baseline * T + (m.time_begin + tl)) * 3;
    const float u = p[0], v = p[1], w = p[2];
    const float bu = (float)(two_pi * ((double)u * k_mid - u0));
    const float bv = (float)(two_pi * ((double)v * k_mid - v0));
    const float bw = (float)(two_pi * ((double)w * k_mid - w0));
    float kd[CPT];
#pragma unroll
    for (int c = 0; c < CPT; ++c)
      kd[c] = (float)(two_pi * (freqs[m.chan_begin + min(cg + c, n_chan - 1)] * inv_c0 - k_mid));
    float2 acc[CPT];
#pragma unroll
    for (int c = 0; c < CPT; ++c) acc[c] = make_float2(0.f, 0.f);
    for (int pix0 = 0; pix0 < NPIX; pix0 += CH) {
      const int npx = min(CH, NPIX - pix0);
      __syncthreads();
      for (int i = tid; i < npx; i += NT) {
        const int pix = pix0 + i;
        const int y = pix / N, x = pix - y * N;
        const double l = (double)(x - N / 2) * image_size / (double)N;
        const double mm = (double)(y - N / 2) * image_size / (double)N;
        const double r2 = l * l + mm * mm;
        s_lmn[i] = make_float4((float)l, (float)mm, (float)(-r2 / (1.0 + sqrt(1.0 - r2))), 0.f);
        const float tp = __ldg(&taper[pix]);
        float2 q = __ldg(&sg[pix]);
        q.x *= tp; q.y *= tp;
        s_pix[i] = cmul_conj_b(cmul(__ldg(&gains[g1_off + pix]), q), __ldg(&gains[g2_off + pix]));
      }
      __syncthreads();
      if (active) {
#pragma unroll 2
        for (int i = 0; i < npx; ++i) {
          const float4 c3 = s_lmn[i];
          const float2 q = s_pix[i];
          const float pidx = fmaf(u, c3.x, fmaf(v, c3.y, w * c3.z));
          const float base = fmaf(bu, c3.x, fmaf(bv, c3.y, bw * c3.z));
          if (R == 1) {
#pragma unroll
            for (int c = 0; c < CPT; ++c) {
              float s, co;
              __sincosf(fmaf(pidx, kd[c], base), &s, &co);
              acc[c].x = fmaf(q.x, co, acc[c].x); acc[c].x = fmaf(q.y, s, acc[c].x);
              acc[c].y = fmaf(q.y, co, acc[c].y); acc[c].y = fmaf(-q.x, s, acc[c].y);
            }
          } else {
            float sr, cr;
            __sincosf(pidx * dkd, &sr, &cr);
#pragma unroll
            for (int c0 = 0; c0 < CPT; c0 += R) {
              float s, co;
              __sincosf(fmaf(pidx, kd[c0], base), &s, &co);
#pragma unroll
              for (int j = 0; j < R && c0 + j < CPT; ++j) {
                const int c = c0 + j;
                acc[c].x = fmaf(q.x, co, acc[c].x); acc[c].x = fmaf(q.y, s, acc[c].x);
                acc[c].y = fmaf(q.y, co, acc[c].y); acc[c].y = fmaf(-q.x, s, acc[c].y);
                const float c2 = fmaf(co, cr, -s * sr);
                s = fmaf(s, cr, co * sr);
                co = c2;
              }
            }
          }
        }
      }
    }
    if (active) {
      float2 *o = vis_out + ((size_t)m.baseline * T + (m.time_begin + tl)) * C + m.chan_begin + cg;
#pragma unroll
      for (int c = 0; c < CPT; ++c)
        if (cg + c < n_chan) o[c] = acc[c];
    }
  }
}

// channel spacing 2 pi df / c0 if the plan's channels are equally spaced (then the recurrence is exact up to
// rounding), else 0: the kernels then evaluate sin/cos for every channel
static float uniform_dkd(const idg_plan *plan) { return plan->uniform_dkd; }

template <int N, int NT, int PPT, int MINB>
static int launch_gs(const idg_plan *plan, const float *uvw, const float2 *vis, const float2 *gains,
                     const float *taper, float2 *subgrids, cudaStream_t stream) {
  const float dkd = uniform_dkd(plan);
  if (dkd != 0.f && plan->max_n_chan >= 4)
    gridder_scalar_kernel<N, NT, PPT, MINB, 4><<<(unsigned)plan->P, NT, 0, stream>>>(
        plan->meta_dev, uvw, plan->freqs_dev, vis, gains, taper, subgrids, plan->T, plan->C, plan->n_stations,
        plan->prm.grid_size, plan->prm.image_size, plan->prm.w_step, dkd);
  else
    gridder_scalar_kernel<N, NT, PPT, MINB, 1><<<(unsigned)plan->P, NT, 0, stream>>>(
        plan->meta_dev, uvw, plan->freqs_dev, vis, gains, taper, subgrids, plan->T, plan->C, plan->n_stations,
        plan->prm.grid_size, plan->prm.image_size, plan->prm.w_step, 0.f);
  IDG_LAUNCH_CHECK();
  return IDG_OK;
}

int launch_gridder_scalar(const idg_plan *plan, const float *uvw, const float2 *vis, const float2 *gains,
                          const float *taper, float2 *subgrids, cudaStream_t stream) {
  if (plan->P == 0) return IDG_OK;
  switch (plan->prm.subgrid_size) {
    case 16: return launch_gs<16, 64, 4, 6>(plan, uvw, vis, gains, taper, subgrids, stream);
    case 24: return launch_gs<24, 96, 6, 4>(plan, uvw, vis, gains, taper, subgrids, stream);
    case 32: return launch_gs<32, 128, 8, 4>(plan, uvw, vis, gains, taper, subgrids, stream);
    case 48: return launch_gs<48, 288, 8, 1>(plan, uvw, vis, gains, taper, subgrids, stream);
    default: return IDG_ERR_UNSUPPORTED_SUBGRID_SIZE;
  }
}

template <int N>
static int launch_ds(const idg_plan *plan, const float *uvw, const float2 *subgrids, const float2 *gains,
                     const float *taper, float2 *vis_out, cudaStream_t stream) {
  const int mc = plan->max_n_chan;
  const int cpt = mc >= 8 ? 8 : (mc >= 4 ? 4 : (mc >= 2 ? 2 : 1));
  const float dkd = uniform_dkd(plan);
#define IDG_DS(CPT_, R_)                                                                                  \
  degridder_scalar_kernel<N, 128, CPT_, R_><<<(unsigned)plan->P, 128, 0, stream>>>(                       \
      plan->meta_dev, uvw, plan->freqs_dev, subgrids, gains, taper, vis_out, plan->T, plan->C,            \
      plan->n_stations, plan->prm.grid_size, plan->prm.image_size, plan->prm.w_step, dkd)
  if (cpt == 8 && dkd != 0.f) IDG_DS(8, 4); else if (cpt == 4 && dkd != 0.f) IDG_DS(4, 4);
  else if (cpt == 8) IDG_DS(8, 1); else if (cpt == 4) IDG_DS(4, 1); else if (cpt == 2) IDG_DS(2, 1); else IDG_DS(1, 1);
#undef IDG_DS
  IDG_LAUNCH_CHECK();
  return IDG_OK;
}

int launch_degridder_scalar(const idg_plan *plan, const float *uvw, const float2 *subgrids, const float2 *gains,
                            const float *taper, float2 *vis_out, cudaStream_t stream) {
  if (plan->P == 0) return IDG_OK;
  switch (plan->prm.subgrid_size) {
    case 16: return launch_ds<16>(plan, uvw, subgrids, gains, taper, vis_out, stream);
    case 24: return launch_ds<24>(plan, uvw, subgrids, gains, taper, vis_out, stream);
    case 32: return launch_ds<32>(plan, uvw, subgrids, gains, taper, vis_out, stream);
    case 48: return launch_ds<48>(plan, uvw, subgrids, gains, taper, vis_out, stream);
    default: return IDG_ERR_UNSUPPORTED_SUBGRID_SIZE;
  }
}

}  // namespace idg
