// degridder.cu -- row a6: predict the visibilities of every block from its subgrid image.
//
// Alg. 2 inner loops (R9: I[i,j] there is I_p[i,j]), polarised form
// (PAPER.md:249), exact adjoint of the gridder:
//   Dg[y][x]   = A1[y][x] (taper[y][x] Ip[y][x]) A2[y][x]^H                      (R5)
//   Y[b][t][c] = sum_{y,x} Dg[y][x] exp(-2 pi i (du l_x + dv m_y + dw n'_xy))
//
// B200 design: one CTA per subgrid.  The reduction axis is the pixels, so here the THREADS own
// visibilities (one timestep x CPT consecutive channels each, complex accumulators in
// registers) and the corrected pixels Dg plus their (l, m, n') are staged in shared memory in
// chunks and broadcast to every thread: no cross-thread reduction at all.  Phase split as in the
// gridder (per-timestep FP64 part, FP32 per pixel x channel).
#include "common.cuh"

namespace idg {

constexpr int kPixChunk = 1024;  // pixels staged per chunk: 48 B each

__device__ __forceinline__ float2 dbc2(float a) { return make_float2(a, a); }
__device__ __forceinline__ float2 dlo2(float4 v) { return make_float2(v.x, v.y); }
__device__ __forceinline__ float2 dhi2(float4 v) { return make_float2(v.z, v.w); }

// FILT selects the subgrids a launch works on (plans that mix channel-group sizes are degridded in two launches):
// 0 all, 1 only those with n_chan a multiple of 8, 2 only the others.
template <int N, int NT, int CPT, bool SPAN, bool SPLIT, bool ONECHAN = false, int FILT = 0>
__global__ void __launch_bounds__(NT, NT == 128 ? 4 : (NT == 64 ? 8 : (NT == 32 ? 16 : 2)))
degridder_kernel(const idg_subgrid_meta *__restrict__ meta, const float *__restrict__ uvw,
                 const double *__restrict__ freqs, const float4 *__restrict__ lmn,
                 const float2 *__restrict__ subgrids,
                 const float4 *__restrict__ aterms, const float *__restrict__ taper,
                 float4 *__restrict__ vis_out, int32_t T, int32_t C, int32_t n_stations, int32_t L,
                 double image_size, double w_step, int32_t aterm_interval) {
  constexpr int NPIX = N * N;
  constexpr int CH = NPIX < kPixChunk ? NPIX : kPixChunk;
  // corrected pixels, packed in polarisation pairs like the gridder's visibilities:
  // (re XX, re XY, re YX, re YY), (im ...) -- one FFMA2 updates two polarisations
  __shared__ float4 s_pix[CH * 2];
  __shared__ float4 s_lmn[CH];       // l, m, n', unused
  static_assert(CH * 8 >= NT * 8, "the SPLIT reduction reuses the pixel staging area, [NT][8] floats");

  const int tid = threadIdx.x;
  const idg_subgrid_meta m = meta[blockIdx.x];
  const int n_chan = m.n_chan, n_time = m.n_time;
  if (FILT == 1 && (n_chan & 7) != 0) return;
  if (FILT == 2 && (n_chan & 7) == 0) return;
  const double two_pi = 6.283185307179586476925286766559;
  const double inv_c0 = 1.0 / kSpeedOfLight;
  const double u0 = (double)(m.x0 + N / 2 - L / 2) / image_size;
  const double v0 = (double)(m.y0 + N / 2 - L / 2) / image_size;
  const double w0 = w_step > 0.0 ? ((double)m.w_index + 0.5) * w_step : 0.0;
  const double k_mid = 0.5 * (freqs[m.chan_begin] + freqs[m.chan_begin + n_chan - 1]) * inv_c0;

  // ONECHAN (single-channel plans): a thread owns CPT consecutive TIMESTEPS of the one channel instead of CPT
  // channels of one timestep, so that the three shared-memory reads per pixel still serve CPT visibilities
  const int groups = ONECHAN ? 1 : (n_chan + CPT - 1) / CPT;       // channel groups per timestep
  const int n_items = ONECHAN ? (n_time + CPT - 1) / CPT : n_time * groups;
  // IDG_PLAN_SPAN_ATERMS (NEXT-4, per-sample c_pk: Alg. 2): the block is walked slot by slot; the
  // corrected pixels are staged with the slot's Jones matrices and only the threads whose timestep lies in
  // that slot accumulate.  Without the flag there is one slot, m.aterm_slot.
  const int slot_first = m.aterm_slot;
  const int slot_last = SPAN ? (m.time_begin + n_time - 1) / aterm_interval : slot_first;
  const float2 *sg = subgrids + (size_t)blockIdx.x * 4 * NPIX;

  // SPLIT (plans whose largest block fills at most half the CTA, e.g. A-terms refreshed every few timesteps): the
  // threads are arranged as G groups x n_items; group g sums the pixels g, g + G, ... and the partial sums are
  // reduced through shared memory at the end, so that short blocks still use the whole CTA.
  const int G = SPLIT ? max(1, min(8, NT / max(n_items, 1))) : 1;
  const int grp = SPLIT ? tid / max(n_items, 1) : 0;
  for (int item0 = 0; item0 < n_items; item0 += NT) {
    const int item = SPLIT ? tid - grp * n_items : item0 + tid;
    const bool active = SPLIT ? grp < G : item < n_items;
    const int tl = active ? (ONECHAN ? item * CPT : item / groups) : 0;
    const int cg = (active && !ONECHAN) ? (item - tl * groups) * CPT : 0;
    const float *p = uvw + ((size_t)m.baseline * T + (m.time_begin + tl)) * 3;
    const float u = p[0], v = p[1], w = p[2];
    const float bu = (float)(two_pi * ((double)u * k_mid - u0));
    const float bv = (float)(two_pi * ((double)v * k_mid - v0));
    const float bw = (float)(two_pi * ((double)w * k_mid - w0));
    float kd[CPT];
    constexpr int NB = ONECHAN ? CPT : 1;           // ONECHAN: the phase coefficients of each of the CPT timesteps
    float bus[NB], bvs[NB], bws[NB];
#pragma unroll
    for (int c = 0; c < CPT; ++c) {
      if (ONECHAN) {
        const float *pc = uvw + ((size_t)m.baseline * T + (m.time_begin + min(tl + c, n_time - 1))) * 3;
        bus[c] = (float)(two_pi * ((double)pc[0] * k_mid - u0));
        bvs[c] = (float)(two_pi * ((double)pc[1] * k_mid - v0));
        bws[c] = (float)(two_pi * ((double)pc[2] * k_mid - w0));
        kd[c] = 0.f;
      } else {
        const int cc = min(cg + c, n_chan - 1);
        kd[c] = (float)(two_pi * (freqs[m.chan_begin + cc] * inv_c0 - k_mid));
      }
    }
    float2 re01[CPT], re23[CPT], im01[CPT], im23[CPT];
#pragma unroll
    for (int c = 0; c < CPT; ++c) re01[c] = re23[c] = im01[c] = im23[c] = make_float2(0.f, 0.f);

    const int my_slot = SPAN ? (m.time_begin + tl) / aterm_interval : slot_first;
    const int n_slots = SPAN ? slot_last - slot_first + 1 : 1;      // compile-time 1 without the flag
    for (int si = 0; si < n_slots; ++si) {
    const int slot = slot_first + si;
    const size_t a1_off = ((size_t)slot * n_stations + m.station1) * NPIX;
    const size_t a2_off = ((size_t)slot * n_stations + m.station2) * NPIX;
    for (int pix0 = 0; pix0 < NPIX; pix0 += CH) {
      const int npx = min(CH, NPIX - pix0);
      __syncthreads();
      // stage Dg = A1 (taper Ip) A2^H and the pixel coordinates for this chunk
      for (int i = tid; i < npx; i += NT) {
        const int pix = pix0 + i;
        if ((CPT >= 8 || SPLIT || ONECHAN) && !(N == 16 && NT == 256)) {
          s_lmn[i] = __ldg(&lmn[pix]);       // the plan's table (always for short blocks: their staging phase counts)
        } else {
          // measured: with 1-4 channels per thread (and in the N = 16, 256-thread instance) the kernel is 2-4 % faster
          // when the staging phase computes the direction cosines (same values as the table: R1, R2 in FP64,
          // rounded once) instead of loading them
          const int y = pix / N, x = pix - y * N;
          const double l = (double)(x - N / 2) * image_size / (double)N;
          const double mm = (double)(y - N / 2) * image_size / (double)N;
          const double r2 = l * l + mm * mm;
          s_lmn[i] = make_float4((float)l, (float)mm, (float)(-r2 / (1.0 + sqrt(1.0 - r2))), 0.f);
        }
        const float tp = __ldg(&taper[pix]);
        float2 p0 = __ldg(&sg[0 * NPIX + pix]), p1 = __ldg(&sg[1 * NPIX + pix]);
        float2 p2 = __ldg(&sg[2 * NPIX + pix]), p3 = __ldg(&sg[3 * NPIX + pix]);
        p0.x *= tp; p0.y *= tp; p1.x *= tp; p1.y *= tp;
        p2.x *= tp; p2.y *= tp; p3.x *= tp; p3.y *= tp;
        const float4 a01 = __ldg(&aterms[(a1_off + pix) * 2]), a23 = __ldg(&aterms[(a1_off + pix) * 2 + 1]);
        const float4 b01 = __ldg(&aterms[(a2_off + pix) * 2]), b23 = __ldg(&aterms[(a2_off + pix) * 2 + 1]);
        const float2 a0 = make_float2(a01.x, a01.y), a1 = make_float2(a01.z, a01.w);
        const float2 a2 = make_float2(a23.x, a23.y), a3 = make_float2(a23.z, a23.w);
        const float2 b0 = make_float2(b01.x, b01.y), b1 = make_float2(b01.z, b01.w);
        const float2 b2 = make_float2(b23.x, b23.y), b3 = make_float2(b23.z, b23.w);
        // T = A1 P
        const float2 t00 = cadd(cmul(a0, p0), cmul(a1, p2)), t01 = cadd(cmul(a0, p1), cmul(a1, p3));
        const float2 t10 = cadd(cmul(a2, p0), cmul(a3, p2)), t11 = cadd(cmul(a2, p1), cmul(a3, p3));
        // R = T A2^H: (A2^H)[i][j] = conj(A2[j][i])
        const float2 r0 = cadd(cmul_conj_b(t00, b0), cmul_conj_b(t01, b1));
        const float2 r1 = cadd(cmul_conj_b(t00, b2), cmul_conj_b(t01, b3));
        const float2 r2q = cadd(cmul_conj_b(t10, b0), cmul_conj_b(t11, b1));
        const float2 r3 = cadd(cmul_conj_b(t10, b2), cmul_conj_b(t11, b3));
        s_pix[2 * i] = make_float4(r0.x, r1.x, r2q.x, r3.x);
        s_pix[2 * i + 1] = make_float4(r0.y, r1.y, r2q.y, r3.y);
      }
      __syncthreads();
      if (active && (!SPAN || my_slot == slot)) {
#pragma unroll(CPT >= 8 ? 1 : 2)
        for (int i = grp; i < npx; i += G) {
          const float4 c3 = s_lmn[i];
          const float4 qr = s_pix[2 * i], qi = s_pix[2 * i + 1];
          // single-channel plans: kd = 0 exactly, the phase is `base` alone
          const float pidx = ONECHAN ? 0.f : fmaf(u, c3.x, fmaf(v, c3.y, w * c3.z));
          const float base = ONECHAN ? 0.f : fmaf(bu, c3.x, fmaf(bv, c3.y, bw * c3.z));
#pragma unroll
          for (int c = 0; c < CPT; ++c) {
            float s, co;
            __sincosf(ONECHAN ? fmaf(bus[ONECHAN ? c : 0], c3.x, fmaf(bvs[ONECHAN ? c : 0], c3.y, bws[ONECHAN ? c : 0] * c3.z))
                              : fmaf(pidx, kd[c], base), &s, &co);
            const float ns = -s;
            // (re + i im) += (qr + i qi)(co - i s): the conjugate phasor of the gridder
            re01[c] = ffma2(dlo2(qr), dbc2(co), re01[c]); re01[c] = ffma2(dlo2(qi), dbc2(s), re01[c]);
            re23[c] = ffma2(dhi2(qr), dbc2(co), re23[c]); re23[c] = ffma2(dhi2(qi), dbc2(s), re23[c]);
            im01[c] = ffma2(dlo2(qi), dbc2(co), im01[c]); im01[c] = ffma2(dlo2(qr), dbc2(ns), im01[c]);
            im23[c] = ffma2(dhi2(qi), dbc2(co), im23[c]); im23[c] = ffma2(dhi2(qr), dbc2(ns), im23[c]);
          }
        }
      }
    }
    }
    if (SPLIT && G > 1) {
      // partial sums of the pixel groups through the pixel staging area
      constexpr int SPR = (CH / NT) >= CPT ? CPT : (CH / NT);      // channel slots that fit per round
      static_assert(SPR >= 1, "the staging area must hold one slot per thread");
      float *red = reinterpret_cast<float *>(s_pix);
      if (SPR == CPT) {
        // N >= 32: all slots at once, [G - 1][n_items][CPT][8].  (A bank-conflict-free [slot][component][thread]
        // layout measured 1 % SLOWER on the SKA-like plan: the phase is a few hundred cycles of a 120 k-cycle CTA and
        // the change moved the register allocation of the main loop.)
        __syncthreads();
        if (active && grp > 0) {
          float *r = red + ((size_t)(grp - 1) * n_items + item) * (CPT * 8);
#pragma unroll
          for (int c = 0; c < CPT; ++c) {
            r[8 * c + 0] = re01[c].x; r[8 * c + 1] = re01[c].y; r[8 * c + 2] = re23[c].x; r[8 * c + 3] = re23[c].y;
            r[8 * c + 4] = im01[c].x; r[8 * c + 5] = im01[c].y; r[8 * c + 6] = im23[c].x; r[8 * c + 7] = im23[c].y;
          }
        }
        __syncthreads();
        if (active && grp == 0) {
          for (int g = 1; g < G; ++g) {
            const float *r = red + ((size_t)(g - 1) * n_items + item) * (CPT * 8);
#pragma unroll
            for (int c = 0; c < CPT; ++c) {
              re01[c].x += r[8 * c + 0]; re01[c].y += r[8 * c + 1]; re23[c].x += r[8 * c + 2]; re23[c].y += r[8 * c + 3];
              im01[c].x += r[8 * c + 4]; im01[c].y += r[8 * c + 5]; im23[c].x += r[8 * c + 6]; im23[c].y += r[8 * c + 7];
            }
          }
        }
      } else {
        // N < 32: rounds of SPR slots, [slot][component][thread] (consecutive threads, consecutive banks)
#pragma unroll
        for (int c0 = 0; c0 < CPT; c0 += SPR) {
          __syncthreads();
          if (active && grp > 0) {
#pragma unroll
            for (int c = c0; c < c0 + SPR && c < CPT; ++c) {
              float *rc = red + (size_t)(c - c0) * 8 * NT + tid;            // tid = grp * n_items + item
              rc[0 * NT] = re01[c].x; rc[1 * NT] = re01[c].y; rc[2 * NT] = re23[c].x; rc[3 * NT] = re23[c].y;
              rc[4 * NT] = im01[c].x; rc[5 * NT] = im01[c].y; rc[6 * NT] = im23[c].x; rc[7 * NT] = im23[c].y;
            }
          }
          __syncthreads();
          if (active && grp == 0) {
            for (int g = 1; g < G; ++g) {
#pragma unroll
              for (int c = c0; c < c0 + SPR && c < CPT; ++c) {
                const float *rc = red + (size_t)(c - c0) * 8 * NT + g * n_items + item;
                re01[c].x += rc[0 * NT]; re01[c].y += rc[1 * NT]; re23[c].x += rc[2 * NT]; re23[c].y += rc[3 * NT];
                im01[c].x += rc[4 * NT]; im01[c].y += rc[5 * NT]; im23[c].x += rc[6 * NT]; im23[c].y += rc[7 * NT];
              }
            }
          }
        }
      }
    }
    if (active && grp == 0) {
      float4 *o = vis_out + (((size_t)m.baseline * T + (m.time_begin + tl)) * C + m.chan_begin + cg) * 2;
#pragma unroll
      for (int c = 0; c < CPT; ++c) {
        if (ONECHAN ? tl + c < n_time : cg + c < n_chan) {
          float4 *oc = ONECHAN ? o + (size_t)c * C * 2 : o + 2 * c;      // next timestep / next channel
          oc[0] = make_float4(re01[c].x, im01[c].x, re01[c].y, im01[c].y);
          oc[1] = make_float4(re23[c].x, im23[c].x, re23[c].y, im23[c].y);
        }
      }
    }
  }
}

template <int N, int NT, int CPT, bool SPLIT = false, bool ONE = false>
static int launch_k(const idg_plan *plan, const float *uvw, const float2 *subgrids,
                    const float2 *aterms, const float *taper, float2 *vis_out, cudaStream_t stream,
                    int64_t p0, int64_t np) {
  const bool span = (plan->prm.flags & IDG_PLAN_SPAN_ATERMS) != 0;
  auto kern = span ? degridder_kernel<N, NT, CPT, true, SPLIT>
                   : (ONE ? degridder_kernel<N, NT, CPT, false, SPLIT, ONE>
                          : degridder_kernel<N, NT, CPT, false, SPLIT>);
  kern<<<(unsigned)np, NT, 0, stream>>>(
      plan->meta_dev + p0, uvw, plan->freqs_dev, plan->lmn_dev, subgrids + (size_t)p0 * 4 * N * N,
      reinterpret_cast<const float4 *>(aterms),
      taper, reinterpret_cast<float4 *>(vis_out), plan->T, plan->C, plan->n_stations,
      plan->prm.grid_size, plan->prm.image_size, plan->prm.w_step, plan->prm.aterm_interval);
  IDG_LAUNCH_CHECK();
  return IDG_OK;
}

// one of the two launches of a plan that mixes channel-group sizes (FILT 1: 8 channels per thread on the subgrids
// whose channel count is a multiple of 8; FILT 2: 4 per thread on the rest)
template <int N, int NT, int CPT, int FILT>
static int launch_filtered(const idg_plan *plan, const float *uvw, const float2 *subgrids,
                           const float2 *aterms, const float *taper, float2 *vis_out, cudaStream_t stream,
                           int64_t p0, int64_t np) {
  degridder_kernel<N, NT, CPT, false, false, false, FILT><<<(unsigned)np, NT, 0, stream>>>(
      plan->meta_dev + p0, uvw, plan->freqs_dev, plan->lmn_dev, subgrids + (size_t)p0 * 4 * N * N,
      reinterpret_cast<const float4 *>(aterms),
      taper, reinterpret_cast<float4 *>(vis_out), plan->T, plan->C, plan->n_stations,
      plan->prm.grid_size, plan->prm.image_size, plan->prm.w_step, plan->prm.aterm_interval);
  IDG_LAUNCH_CHECK();
  return IDG_OK;
}

template <int N>
static int launch_n(const idg_plan *plan, const float *uvw, const float2 *subgrids,
                    const float2 *aterms, const float *taper, float2 *vis_out, cudaStream_t stream,
                    int64_t p0, int64_t np) {
  // threads own (timestep, CPT channels); pick CPT and the CTA size from the plan's largest block
  const int mc = plan->max_n_chan;
  // single-channel plans: kd = 0 and the phase is `base` alone; threads own four consecutive timesteps (the pixel
  // reads from shared memory are shared by the four), the pixels are split over thread groups when the block is short
  if (mc == 1 && (plan->prm.flags & IDG_PLAN_SPAN_ATERMS) == 0) {
    if (plan->max_n_time < 8)
      return launch_k<N, 128, 1, true, true>(plan, uvw, subgrids, aterms, taper, vis_out, stream, p0, np);
    const int items4 = (plan->max_n_time + 3) / 4;
    // N = 16: a block of up to 32 items is one warp's work; single-warp CTAs (16 per SM, no idle threads, barriers
    // that cost nothing) measured 0.63 of the roofline against 0.58 for 128 threads in four pixel groups
    if constexpr (N == 16)
      if (items4 <= 32) return launch_k<N, 32, 4, false, true>(plan, uvw, subgrids, aterms, taper, vis_out, stream, p0, np);
    if constexpr (N == 24)      // two warps, two pixel groups: 0.61 against 0.60 (128 threads) and 0.55 (one warp)
      if (items4 <= 32) return launch_k<N, 64, 4, true, true>(plan, uvw, subgrids, aterms, taper, vis_out, stream, p0, np);
    if (items4 <= 64) return launch_k<N, 128, 4, true, true>(plan, uvw, subgrids, aterms, taper, vis_out, stream, p0, np);
    if (items4 <= 128) return launch_k<N, 128, 4, false, true>(plan, uvw, subgrids, aterms, taper, vis_out, stream, p0, np);
    return launch_k<N, 256, 4, false, true>(plan, uvw, subgrids, aterms, taper, vis_out, stream, p0, np);
  }
  // more channels per thread amortise the per-pixel shared-memory reads and phase set-up, as long as the
  // largest block still fills a 128-thread CTA
  int cpt = mc >= 4 ? 4 : (mc >= 2 ? 2 : 1);
  const int items8 = plan->max_n_time * ((mc + 7) / 8);
  // 8 channels per thread when that still fills a 128-thread CTA, or (N >= 32) half of one: then two thread groups
  // share the pixels (SPLIT below)
  if (mc >= 8 && (items8 >= 128 || (N >= 24 && items8 >= 16 && items8 <= 64) || (N >= 32 && items8 >= 32 && items8 <= 64))) cpt = 8;
  // plans that mix channel-group sizes (a 20-channel band cut into 16 + 4) and would idle more than 5 % of the
  // 8-channel slots: two launches, 8 channels per thread on the subgrids that fill them, 4 on the rest
  if (cpt == 8 && items8 >= 128 && plan->dg_waste[3] > 0.05f && plan->dg_waste[2] <= 0.05f &&
      (plan->prm.flags & IDG_PLAN_SPAN_ATERMS) == 0) {
    int rc = items8 <= 128 ? launch_filtered<N, 128, 8, 1>(plan, uvw, subgrids, aterms, taper, vis_out, stream, p0, np)
                           : launch_filtered<N, 256, 8, 1>(plan, uvw, subgrids, aterms, taper, vis_out, stream, p0, np);
    if (rc != IDG_OK) return rc;
    return plan->max_n_time <= 128
               ? launch_filtered<N, 128, 4, 2>(plan, uvw, subgrids, aterms, taper, vis_out, stream, p0, np)
               : launch_filtered<N, 256, 4, 2>(plan, uvw, subgrids, aterms, taper, vis_out, stream, p0, np);
  }
  // otherwise: do not idle more than 5 % of the slots
  while (cpt > 1 && plan->dg_waste[cpt == 8 ? 3 : (cpt == 4 ? 2 : 1)] > 0.05f) cpt /= 2;
  const int items = plan->max_n_time * ((mc + cpt - 1) / cpt);
  const bool small = items <= 128;
  if (items <= 64 && cpt == 8)
    return launch_k<N, 128, 8, true>(plan, uvw, subgrids, aterms, taper, vis_out, stream, p0, np);
  if constexpr (N == 16)      // single-warp CTAs for blocks of at most 32 (timestep, 4 channels) items, as above
    if (items <= 32 && cpt == 4) return launch_k<N, 32, 4>(plan, uvw, subgrids, aterms, taper, vis_out, stream, p0, np);
  if (items <= 64 && cpt <= 4 && N >= 24) {   // short blocks: split the pixels over thread groups (measured: no gain at N = 16)
    if (cpt == 4) return launch_k<N, 128, 4, true>(plan, uvw, subgrids, aterms, taper, vis_out, stream, p0, np);
    if (cpt == 2) return launch_k<N, 128, 2, true>(plan, uvw, subgrids, aterms, taper, vis_out, stream, p0, np);
    return launch_k<N, 128, 1, true>(plan, uvw, subgrids, aterms, taper, vis_out, stream, p0, np);
  }
#define IDG_DG(CPT_)                                                                         \
  return small ? launch_k<N, 128, CPT_>(plan, uvw, subgrids, aterms, taper, vis_out, stream, p0, np) \
               : launch_k<N, 256, CPT_>(plan, uvw, subgrids, aterms, taper, vis_out, stream, p0, np)
  if (cpt == 8) { IDG_DG(8); }
  if (cpt == 4) { IDG_DG(4); }
  if (cpt == 2) { IDG_DG(2); }
  IDG_DG(1);
#undef IDG_DG
}

int launch_degridder(const idg_plan *plan, const float *uvw, const float2 *subgrids,
                     const float2 *aterms, const float *taper, float2 *vis_out,
                     cudaStream_t stream, int64_t p0, int64_t np) {
  if (np < 0) np = plan->P - p0;
  if (np <= 0) return IDG_OK;
  if (degridder_tc_eligible(plan)) return launch_degridder_tc(plan, uvw, subgrids, aterms, taper, vis_out, stream, p0, np);
  switch (plan->prm.subgrid_size) {
    case 16: return launch_n<16>(plan, uvw, subgrids, aterms, taper, vis_out, stream, p0, np);
    case 24: return launch_n<24>(plan, uvw, subgrids, aterms, taper, vis_out, stream, p0, np);
    case 32: return launch_n<32>(plan, uvw, subgrids, aterms, taper, vis_out, stream, p0, np);
    case 48: return launch_n<48>(plan, uvw, subgrids, aterms, taper, vis_out, stream, p0, np);
    default: return IDG_ERR_UNSUPPORTED_SUBGRID_SIZE;
  }
}

}  // namespace idg
