// gridder.cu -- row a1: subgrid images by direct evaluation.
//
// Eq. 25, Alg. 1 inner loops, polarised form of section
// 3.4, one c_p per block:
//   P[y][x]  = sum_{t,c} Y[b][t][c] exp(+2 pi i (du l_x + dv m_y + dw n'_xy)),   du = u_t f_c/c0 - u0 ...
//   Sg[y][x] = taper[y][x] A1[y][x]^H P[y][x] A2[y][x]                            (R5)
//
// B200 design (not the paper's; the paper gives none): one CTA per subgrid, every thread keeps
// PPT pixels x 4 polarisations of complex accumulators in registers for the whole block, the
// visibilities of a batch of timesteps are staged once in shared memory and broadcast to all
// threads.  FP32 everywhere on the pixel x visibility product; the cancellation-prone part of
// the phase is taken out per TIMESTEP in FP64 (cost ~ K, not K N^2):
//   phase(t,c,pix) = pidx(t,pix) * kd_c + base(t,pix)
//   pidx = u_t l + v_t m + w_t n'            (metres x direction cosine, FP32)
//   base = bu l + bv m + bw n',  bu = 2 pi (u_t k_mid - u0)  (FP64 -> FP32), k_mid = block centre
//   kd_c = 2 pi (k_c - k_mid)                (FP64 -> FP32)
// so that per (visibility, pixel) the work is 1 FMA (phase) + sin/cos.approx (1 FMUL + 2 MUFU) +
// 16 FMA issued as 8 packed FFMA2.
//
// Operand layout of the FFMA2s (measured, profiles/r01_*): the visibilities are re-packed at
// staging time into polarisation PAIRS, (re XX, re XY, re YX, re YY) and (im ...), so that one
// FFMA2 is  (acc_pol0, acc_pol1) += (v_pol0, v_pol1) * broadcast(cos or sin)  -- the scalar
// broadcast and the operand negation are free FFMA2 operand modifiers, which removes the
// FADD/MOV shuffles a (re, im)-paired accumulator needs.  The accumulators are therefore
// re[pol pair], im[pol pair] per pixel.
#include "common.cuh"

namespace idg {

constexpr int kMaxChan = 256;    // max channels per subgrid

__device__ __forceinline__ float2 bc2(float a) { return make_float2(a, a); }
__device__ __forceinline__ float2 lo2(float4 v) { return make_float2(v.x, v.y); }
__device__ __forceinline__ float2 hi2(float4 v) { return make_float2(v.z, v.w); }

template <int N, int NT, int PPT, int MINB, int VB, int TB, bool SPAN, bool ONECHAN, int SPL = 1>
__global__ void __launch_bounds__(NT, MINB)
gridder_kernel(const idg_subgrid_meta *__restrict__ meta, const float *__restrict__ uvw,
               const double *__restrict__ freqs, const float4 *__restrict__ lmn, const float4 *__restrict__ vis,
               const float4 *__restrict__ aterms, const float *__restrict__ taper,
               float2 *__restrict__ subgrids, int32_t T, int32_t C, int32_t n_stations,
               int32_t L, double image_size, double w_step, int32_t aterm_interval) {
  constexpr int vis_batch = VB, time_batch = TB;
  // SPL CTAs share one subgrid (blockIdx.y = which part of its pixels): at N = 48 two 192-thread CTAs per subgrid
  // run two to an SM, so that one's staging phase and epilogue hide behind the other's visibility loop
  static_assert(NT * PPT * SPL == N * N, "pixels must tile the CTAs exactly");
  const int pix_base = SPL > 1 ? blockIdx.y * (NT * PPT) : 0;
  extern __shared__ float4 g_smem[];
  float4 *s_vis = g_smem;                  // [vis_batch][2]: (re XX, re XY, re YX, re YY), (im ...)
  float4 *s_t = s_vis + vis_batch * 2;     // [time_batch][2]: (u, v, w, -), (bu, bv, bw, -)
  float4 *s_lmn = s_t + time_batch * 2;    // [NT*PPT]: (l, m, n', -) per pixel of this CTA
  float *s_kd = reinterpret_cast<float *>(s_lmn + NT * PPT);   // [kMaxChan]

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

  // pixel direction cosines (l, m, n') from the plan's table (R1: l_x = (x - N/2) S/N; R2: n' = sqrt(1-l^2-m^2) - 1),
  // kept in shared memory: they are needed once per timestep only, not in the channel loop.  The N = 24 instances
  // measured 3-4 % slower with the table load than with the FP64 evaluation and keep the latter (same values).
#pragma unroll
  for (int k = 0; k < PPT; ++k) {
    const int pix = pix_base + tid + k * NT;
    if (N != 24) {
      s_lmn[tid + k * NT] = __ldg(&lmn[pix]);
    } else {
      const int y = pix / N, x = pix - y * N;
      const double l = (double)(x - N / 2) * image_size / (double)N;
      const double mm = (double)(y - N / 2) * image_size / (double)N;
      const double r2 = l * l + mm * mm;
      s_lmn[tid + k * NT] = make_float4((float)l, (float)mm, (float)(-r2 / (1.0 + sqrt(1.0 - r2))), 0.f);
    }
  }

  float2 re01[PPT], re23[PPT], im01[PPT], im23[PPT];
#pragma unroll
  for (int k = 0; k < PPT; ++k) re01[k] = re23[k] = im01[k] = im23[k] = make_float2(0.f, 0.f);

  // taper * A1^H * P * A2 per pixel with the Jones matrices of one A-term slot, written pol-planar.  With
  // IDG_PLAN_SPAN_ATERMS (NEXT-4, per-sample c_pk: section 3.4) the accumulators are flushed
  // whenever the slot of the timestep changes, so the subgrid is the sum of the per-slot corrected parts.
  auto flush = [&](int slot, bool accumulate) {
    const size_t a1_off = ((size_t)slot * n_stations + m.station1) * (N * N);
    const size_t a2_off = ((size_t)slot * n_stations + m.station2) * (N * N);
    float2 *out = subgrids + (size_t)blockIdx.x * 4 * N * N;
#pragma unroll
    for (int k = 0; k < PPT; ++k) {
      const int pix = pix_base + tid + k * NT;
      const float4 a01 = __ldg(&aterms[(a1_off + pix) * 2]), a23 = __ldg(&aterms[(a1_off + pix) * 2 + 1]);
      const float4 b01 = __ldg(&aterms[(a2_off + pix) * 2]), b23 = __ldg(&aterms[(a2_off + pix) * 2 + 1]);
      const float tp = __ldg(&taper[pix]);
      const float2 a0 = make_float2(a01.x, a01.y), a1 = make_float2(a01.z, a01.w);
      const float2 a2 = make_float2(a23.x, a23.y), a3 = make_float2(a23.z, a23.w);
      const float2 b0 = make_float2(b01.x, b01.y), b1 = make_float2(b01.z, b01.w);
      const float2 b2 = make_float2(b23.x, b23.y), b3 = make_float2(b23.z, b23.w);
      const float2 p0 = make_float2(re01[k].x, im01[k].x), p1 = make_float2(re01[k].y, im01[k].y);
      const float2 p2 = make_float2(re23[k].x, im23[k].x), p3 = make_float2(re23[k].y, im23[k].y);
      const float2 t00 = cadd(cmul_conj_a(a0, p0), cmul_conj_a(a2, p2));
      const float2 t01 = cadd(cmul_conj_a(a0, p1), cmul_conj_a(a2, p3));
      const float2 t10 = cadd(cmul_conj_a(a1, p0), cmul_conj_a(a3, p2));
      const float2 t11 = cadd(cmul_conj_a(a1, p1), cmul_conj_a(a3, p3));
      float2 r[4] = {cadd(cmul(t00, b0), cmul(t01, b2)), cadd(cmul(t00, b1), cmul(t01, b3)),
                     cadd(cmul(t10, b0), cmul(t11, b2)), cadd(cmul(t10, b1), cmul(t11, b3))};
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        float2 v = make_float2(tp * r[q].x, tp * r[q].y);
        if (SPAN && accumulate) { const float2 o = out[q * N * N + pix]; v.x += o.x; v.y += o.y; }
        out[q * N * N + pix] = v;
      }
      if (SPAN) re01[k] = re23[k] = im01[k] = im23[k] = make_float2(0.f, 0.f);
    }
  };
  int cur_slot = m.aterm_slot;
  bool flushed = false;

  const int tb_max = n_chan >= vis_batch ? 1 : min(vis_batch / n_chan, time_batch);  // timesteps per batch
  const float *uvw_b = uvw + (size_t)m.baseline * T * 3;

  for (int t0 = 0; t0 < n_time; t0 += tb_max) {
    const int tb = min(tb_max, n_time - t0);
    for (int c_lo = 0; c_lo < n_chan; c_lo += vis_batch) {   // only loops when n_chan > batch
      const int nc = min(vis_batch, n_chan - c_lo);
      __syncthreads();
      // stage visibilities [tb][nc], re-packed into polarisation pairs, and the per-timestep terms
      for (int i = tid; i < tb * nc; i += NT) {
        const int tl = i / nc, r = i - tl * nc;
        const size_t g = (((size_t)m.baseline * T + (m.time_begin + t0 + tl)) * C +
                          (m.chan_begin + c_lo + r)) * 2;
        const float4 a = __ldg(&vis[g]), b = __ldg(&vis[g + 1]);
        s_vis[2 * i] = make_float4(a.x, a.z, b.x, b.z);
        s_vis[2 * i + 1] = make_float4(a.y, a.w, b.y, b.w);
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

      if (ONECHAN) {
        // plans with one channel per subgrid: k_mid is that channel, kd = 0 exactly and the phase is `base` alone;
        // the timesteps take the place of the channel loop (3 FMA + sin/cos + 16 FMA per pair, no per-timestep set-up)
        float ql[PPT], qm[PPT], qn[PPT];
#pragma unroll
        for (int k = 0; k < PPT; ++k) { const float4 q = s_lmn[tid + k * NT]; ql[k] = q.x; qm[k] = q.y; qn[k] = q.z; }
#pragma unroll 4
        for (int tl = 0; tl < tb; ++tl) {
          const float4 tbs = s_t[2 * tl + 1];
          const float4 vr = s_vis[2 * tl], vi = s_vis[2 * tl + 1];
#pragma unroll
          for (int k = 0; k < PPT; ++k) {
            float s, co;
            __sincosf(fmaf(tbs.x, ql[k], fmaf(tbs.y, qm[k], tbs.z * qn[k])), &s, &co);
            const float ns = -s;
            re01[k] = ffma2(lo2(vr), bc2(co), re01[k]); re01[k] = ffma2(lo2(vi), bc2(ns), re01[k]);
            re23[k] = ffma2(hi2(vr), bc2(co), re23[k]); re23[k] = ffma2(hi2(vi), bc2(ns), re23[k]);
            im01[k] = ffma2(lo2(vr), bc2(s), im01[k]);  im01[k] = ffma2(lo2(vi), bc2(co), im01[k]);
            im23[k] = ffma2(hi2(vr), bc2(s), im23[k]);  im23[k] = ffma2(hi2(vi), bc2(co), im23[k]);
          }
        }
      } else
      for (int tl = 0; tl < tb; ++tl) {
        if (SPAN) {
          const int slot = (m.time_begin + t0 + tl) / aterm_interval;
          if (slot != cur_slot) { flush(cur_slot, flushed); flushed = true; cur_slot = slot; }
        }
        const float4 tu = s_t[2 * tl], tbs = s_t[2 * tl + 1];
        float pidx[PPT], base[PPT];
#pragma unroll
        for (int k = 0; k < PPT; ++k) {
          const float4 q = s_lmn[tid + k * NT];
          pidx[k] = fmaf(tu.x, q.x, fmaf(tu.y, q.y, tu.z * q.z));
          base[k] = fmaf(tbs.x, q.x, fmaf(tbs.y, q.y, tbs.z * q.z));
        }
        const float4 *vp = s_vis + (size_t)tl * nc * 2;
        const float *kdp = s_kd + c_lo;
#pragma unroll 4
        for (int c = 0; c < nc; ++c) {
          const float kd = kdp[c];
          const float4 vr = vp[2 * c], vi = vp[2 * c + 1];
#pragma unroll
          for (int k = 0; k < PPT; ++k) {
            float s, co;
            __sincosf(fmaf(pidx[k], kd, base[k]), &s, &co);
            const float ns = -s;
            // (re + i im) += (vr + i vi)(co + i s)
            re01[k] = ffma2(lo2(vr), bc2(co), re01[k]); re01[k] = ffma2(lo2(vi), bc2(ns), re01[k]);
            re23[k] = ffma2(hi2(vr), bc2(co), re23[k]); re23[k] = ffma2(hi2(vi), bc2(ns), re23[k]);
            im01[k] = ffma2(lo2(vr), bc2(s), im01[k]);  im01[k] = ffma2(lo2(vi), bc2(co), im01[k]);
            im23[k] = ffma2(hi2(vr), bc2(s), im23[k]);  im23[k] = ffma2(hi2(vi), bc2(co), im23[k]);
          }
        }
      }
    }
  }

  flush(cur_slot, flushed);
}

// VB visibilities and TB timesteps are staged per batch.  Every batch costs the CTA two barriers, at which its
// faster warps idle; larger batches measured +2.5 % (N = 32, 48) and up to +10 % (N = 24, blocks of 2048-4096
// visibilities) over 256-visibility batches.  Single-channel plans keep 256 timesteps per batch.
template <int N, int NT, int PPT, int MINB, int VB, int TB, int SPL = 1>
static int launch_n(const idg_plan *plan, const float *uvw, const float2 *vis, const float2 *aterms,
                    const float *taper, float2 *subgrids, cudaStream_t stream, int64_t p0, int64_t np) {
  const bool span = (plan->prm.flags & IDG_PLAN_SPAN_ATERMS) != 0;
  // single-channel plans without the span flag take the ONECHAN instance
  const bool one = !span && plan->max_n_chan == 1;
  constexpr size_t smem_one = sizeof(float4) * (256 * 4 + NT * PPT) + sizeof(float) * kMaxChan;
  constexpr size_t smem_any = sizeof(float4) * ((size_t)VB * 2 + (size_t)TB * 2 + NT * PPT) + sizeof(float) * kMaxChan;
  const size_t smem = one ? smem_one : smem_any;
  auto kern = span ? gridder_kernel<N, NT, PPT, MINB, VB, TB, true, false, SPL>
                   : (one ? gridder_kernel<N, NT, PPT, MINB, 256, 256, false, true, SPL>
                          : gridder_kernel<N, NT, PPT, MINB, VB, TB, false, false, SPL>);
  IDG_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  kern<<<dim3((unsigned)np, SPL), NT, smem, stream>>>(
      plan->meta_dev + p0, uvw, plan->freqs_dev, plan->lmn_dev, reinterpret_cast<const float4 *>(vis),
      reinterpret_cast<const float4 *>(aterms), taper, subgrids + (size_t)p0 * 4 * N * N, plan->T, plan->C,
      plan->n_stations, plan->prm.grid_size, plan->prm.image_size, plan->prm.w_step, plan->prm.aterm_interval);
  IDG_LAUNCH_CHECK();
  return IDG_OK;
}

int launch_gridder(const idg_plan *plan, const float *uvw, const float2 *vis, const float2 *aterms,
                   const float *taper, float2 *subgrids, cudaStream_t stream, int64_t p0, int64_t np) {
  if (np < 0) np = plan->P - p0;
  if (np <= 0) return IDG_OK;
  // N = 32, per-block A-terms, at least 8 channels per block: the contraction runs on the tensor cores (gridder_tc.cu;
  // measured 3-8 % faster than the FFMA2 kernel below on the SKA-like / LOFAR-like plans, same parity)
  if (gridder_tc_eligible(plan)) return launch_gridder_tc(plan, uvw, vis, aterms, taper, subgrids, stream, p0, np);
  switch (plan->prm.subgrid_size) {
    case 16: return launch_n<16, 64, 4, 8, 512, 128>(plan, uvw, vis, aterms, taper, subgrids, stream, p0, np);
    case 24:
      // 96-thread CTAs lose ~8 % once a block takes more than four batches (the three warps of a CTA drift apart
      // between barriers); blocks that long go to 64 threads x 9 pixels, which does not show the effect
      if (plan->P > 0 && plan->n_planned / plan->P > 4096)
        return launch_n<24, 64, 9, 6, 512, 128>(plan, uvw, vis, aterms, taper, subgrids, stream, p0, np);
      return launch_n<24, 96, 6, 5, 1024, 64>(plan, uvw, vis, aterms, taper, subgrids, stream, p0, np);
    case 32: return launch_n<32, 256, 4, 2, 512, 512>(plan, uvw, vis, aterms, taper, subgrids, stream, p0, np);
    case 48:
      // blocks of up to ~1000 visibilities: two 192-thread CTAs per subgrid, two to an SM (one CTA of 384 threads leaves
      // its staging phase and epilogue exposed: 1 channel 0.60 -> 0.65, A-term interval 8 0.64 -> 0.70; long blocks
      // measured 1-14 % slower that way and keep the single CTA)
      if (plan->P > 0 && plan->n_planned / plan->P <= 1024)
        return launch_n<48, 192, 6, 2, 1024, 512, 2>(plan, uvw, vis, aterms, taper, subgrids, stream, p0, np);
      return launch_n<48, 384, 6, 1, 2048, 512>(plan, uvw, vis, aterms, taper, subgrids, stream, p0, np);
    default: return IDG_ERR_UNSUPPORTED_SUBGRID_SIZE;
  }
}

}  // namespace idg
