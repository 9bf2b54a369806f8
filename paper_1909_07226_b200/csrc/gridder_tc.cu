// gridder_tc.cu -- row a1 on the 5th-generation tensor cores (N = 32): the subgrid image as a dense contraction.
//
// Eq. 25 is  S[pixel][comp] = sum_k Phi[pixel][k] Y[k][comp]  with the phasor matrix
// Phi[pixel][k] = exp(+i phase(pixel, k)) generated on the fly and the 8 real components (re / im of the four
// polarisations) of the visibilities as columns: a real GEMM with M = 1024 pixels, N = 8, K = 2 K_p (cos and sin
// rows).  The FP32 path spends 16 of its 18 lane-ops per (visibility, pixel) on exactly this product; here it runs
// as tcgen05.mma.kind::f16 with FP32 accumulators in tensor memory, and the CUDA cores only generate phasors.
//
// Precision: north_star wants 1e-4 relative L2 against float64, an 11-bit operand alone gives ~2e-4.  Both
// operands are therefore split into two halves, x = hi + lo with hi = fp16(x), lo = fp16(x - hi) (22 bits):
//   K rows per visibility:    cos_hi, sin_hi, cos_lo, sin_lo                       (A operand, from tensor memory)
//   N columns:                8 components of Y_hi, then 8 components of Y_lo      (B operand, from shared memory;
//                             the lo x lo products are dropped: Y_lo meets zeros in the cos_lo / sin_lo rows)
// so one M128 x N16 x K16 MMA covers 128 pixels x 4 visibilities, and the result is D[:, j] + D[:, 8 + j].  The
// visibilities of a block are scaled by a power of two so that their largest component sits near 2^14 (fp16 range).
//
// Structure of a CTA (HALF a subgrid: 4 pixel tiles of 128, blockIdx.y picks the half; 288 threads at 72 registers and
// 128 tensor-memory columns -- 64 of accumulators + ONE slot of 64 -- so that THREE CTAs share an SM: the generator
// warps are latency-bound, and 24 of them per SM with a single slot beat 16 with a ring of three by 8 %): warps 0-7
// generate -- thread
// (warpgroup g, lane L) owns the pixels (2 g + k) 128 + L, k = 0, 1, i.e. row L of two of the four tiles; per ring slot
// of 8 visibilities (8 channels of one timestep) it evaluates the phase of the first channel (FP64/FP32 split of
// gridder.cu) and sin/cos.approx, obtains the other seven phasors by one complex rotation each when the channels are
// equally spaced (ROT; both pixels of the thread in one packed f32x2 multiply + FMA pair), splits every phasor into
// fp16 hi + lo (hi = cvt.f16x2(x); the residual hi - x with one mixed-precision add per component, sub.f32.f16 = FHADD,
// its sign folded into the B tile; lo = cvt.f16x2 of that), and writes its rows of the A tiles straight from registers
// into the slot (tcgen05.st), then arrives on the slot's "full" mbarrier.  The terms of the NEXT slot (per-timestep
// dot products, rotation and anchor sin/cos) are computed in stages between this slot's rotations and the slot's
// "empty" barrier is tested at the start of the step, so that no shared-memory, MUFU or mbarrier latency sits between
// two steps of a warp.  Warp 8 issues: it waits for the slot, issues the 8 MMAs of the slot (2 batches of 4
// visibilities x 4 pixel tiles, each batch reading its 512-byte B tile from shared memory) and commits them to the
// slot's "empty" mbarrier.  The accumulators D[4 tiles][128 x 16] stay in tensor memory for the whole block; the
// epilogue reads them back (tcgen05.ld), applies taper and A-terms and stores.  The M128 x N16 x K16 MMA with A in
// tensor memory runs at its floor of M N / 256 = 8-9 cycles (measured), a tenth of the tensor pipe: the kernel is
// bound by the generator warps (6 issue slots per (visibility, pixel) + ~70 per slot and warp of hand-over), which
// issued on ~60 % of the cycles with 16 generator warps per SM (two CTAs of 256 columns).  Measurements and variants: profiles/r02_experiments.md
// section 7.
#include <cuda_fp16.h>

#include "common.cuh"

namespace idg {

namespace tc {

constexpr int N = 32, NPIX = N * N;
constexpr int SPL = 2;                                      // CTAs per subgrid (blockIdx.y = which half of the pixels)
constexpr int TILES = NPIX / 128 / SPL;                     // 4 pixel tiles of 128 (MMA M) per CTA
constexpr int GEN_THREADS = 256, NT = GEN_THREADS + 32;     // 8 generator warps + the issuing warp
constexpr int PPT = TILES * 128 / GEN_THREADS;              // 2 pixels per generator thread
constexpr int VS = 128;                                     // visibilities per staging batch (32 B tiles of 512 bytes)
constexpr int KB = 2;                                       // MMA batches (of 4 visibilities) per ring slot
constexpr int COLS_D = TILES * 16;                          // accumulator columns: 64
constexpr int COLS_SLOT = TILES * 8 * KB;                   // A columns per ring slot: [tile][batch][K16 fp16 = 8 x 32-bit]
constexpr int kSmemB = 2 * (VS / 4) * 512, kSmemT = 2 * (VS / 4) * 2 * 16, kSmemKd = VS * 4;
constexpr int kSmem = kSmemB + kSmemT + kSmemKd;

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *b, uint32_t c) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(c));
}
__device__ __forceinline__ void mbar_arrive(uint64_t *b) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(b)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *b, uint32_t parity) {
  uint32_t ok = 0;
  for (int spins = 0; spins < (1 << 26); ++spins) {        // bounded: a lost arrival traps instead of hanging the GPU
    asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                 : "=r"(ok) : "r"(smem_u32(b)), "r"(parity) : "memory");
    if (ok) return;
  }
  __trap();
}
__device__ __forceinline__ void mbar_wait_addr(uint32_t addr, uint32_t parity) {
  uint32_t ok = 0;
  for (int spins = 0; spins < (1 << 26); ++spins) {
    asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3; selp.u32 %0, 1, 0, p; }"
                 : "=r"(ok) : "r"(addr), "r"(parity), "r"(500u) : "memory");      // parked up to 500 ns between polls
    if (ok) return;
  }
  __trap();
}
// the issuing warp is idle most of the time: let the hardware park it between polls instead of spinning on issue slots
__device__ __forceinline__ void mbar_wait_parked(uint64_t *b, uint32_t parity) {
  uint32_t ok = 0;
  for (int spins = 0; spins < (1 << 22); ++spins) {
    asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3; selp.u32 %0, 1, 0, p; }"
                 : "=r"(ok) : "r"(smem_u32(b)), "r"(parity), "r"(400u) : "memory");
    if (ok) return;
  }
  __trap();
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

// instruction descriptor: D = F32, A = B = F16, both K-major, N = 16, M = 128 (cute::UMMA::InstrDescriptor bit layout)
constexpr uint32_t kIdesc = (1u << 4) | (0u << 7) | (0u << 10) | ((16u >> 3) << 17) | ((128u >> 4) << 24);

// shared-memory matrix descriptor of one B tile [16 n][16 k] fp16, K-major, no swizzle: core matrices of 8 rows x
// 16 bytes; the two K chunks 128 bytes apart (leading byte offset), the two row groups 256 bytes apart (stride)
__device__ __forceinline__ uint64_t b_desc(uint32_t smem_addr) {
  return (uint64_t)((smem_addr & 0x3FFFF) >> 4) | ((uint64_t)(128 >> 4) << 16) | ((uint64_t)(256 >> 4) << 32) |
         ((uint64_t)1 << 46);
}

}  // namespace tc

using namespace tc;

// ROT: equally spaced channels -- the first channel of every group of 8 gets sin/cos.approx, the other seven come
// from one complex rotation by exp(i pidx dkd) each (4 FP32 ops instead of 1 FMA + 1 FMUL + 2 MUFU; seven
// rotations add ~1e-6 of phase error), which takes the kernel off the MUFU bound.
template <int RING, bool ROT>
__global__ void __launch_bounds__(tc::NT, 4)
gridder_tc_kernel(const idg_subgrid_meta *__restrict__ meta, const float *__restrict__ uvw,
                  const double *__restrict__ freqs, const float4 *__restrict__ lmn, const float4 *__restrict__ vis,
                  const float4 *__restrict__ aterms, const float *__restrict__ taper, float2 *__restrict__ subgrids,
                  int32_t T, int32_t C, int32_t n_stations, int32_t L, double image_size, double w_step, float dkd) {
  constexpr int TMEM_COLS = 128;
  static_assert(COLS_D + RING * COLS_SLOT <= TMEM_COLS, "ring does not fit the tensor-memory allocation");
  extern __shared__ __align__(128) unsigned char smem_dyn[];
  unsigned char *s_b = smem_dyn;                                          // [2][VS / 4][512]: B tiles, two staging buffers
  float4 *s_t = reinterpret_cast<float4 *>(smem_dyn + kSmemB);            // [2][VS / 4][2]: per timestep (u, v, w), (bu, bv, bw)
  float *s_kd = reinterpret_cast<float *>(smem_dyn + kSmemB + kSmemT);    // [VS]: kd per channel of the block, zero padded
  __shared__ uint64_t bar_empty[RING], bar_done;
  __shared__ uint32_t s_tmem, s_maxbits;

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const idg_subgrid_meta m = meta[blockIdx.x];
  const int pix_base = blockIdx.y * (TILES * 128);
  const int n_chan = m.n_chan, n_time = m.n_time;
  const int ncp = (n_chan + 4 * KB - 1) / (4 * KB) * (4 * KB);   // channels padded to whole ring slots
  const int tb_max = max(1, VS / ncp);               // timesteps per staging batch
  const int spt = ncp / (4 * KB);                    // ring slots per timestep

  if (warp == 8) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&s_tmem)), "n"(TMEM_COLS));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  if (tid == 0) {
    for (int s = 0; s < RING; ++s) mbar_init(&bar_empty[s], 1);
    mbar_init(&bar_done, 1);
    s_maxbits = 0;
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = s_tmem;

  // largest visibility component of the block -> power-of-two scale into the fp16 range
  {
    float mx = 0.f;
    for (int i = tid; i < n_time * n_chan; i += NT) {
      const int tl = i / n_chan, c = i - tl * n_chan;
      const size_t g = (((size_t)m.baseline * T + (m.time_begin + tl)) * C + (m.chan_begin + c)) * 2;
      const float4 a = __ldg(&vis[g]), b = __ldg(&vis[g + 1]);
      mx = fmaxf(mx, fmaxf(fmaxf(fabsf(a.x), fabsf(a.y)), fmaxf(fabsf(a.z), fabsf(a.w))));
      mx = fmaxf(mx, fmaxf(fmaxf(fabsf(b.x), fabsf(b.y)), fmaxf(fabsf(b.z), fabsf(b.w))));
    }
    if (isfinite(mx)) atomicMax(&s_maxbits, __float_as_uint(mx));     // non-negative floats order like their bits
  }
  __syncthreads();
  const float vmax = __uint_as_float(s_maxbits);
  int e = 0;
  if (vmax > 0.f) frexpf(vmax, &e);                   // vmax = f 2^e, f in [0.5, 1)
  const float scale = ldexpf(1.0f, 14 - e), inv_scale = ldexpf(1.0f, e - 14);

  const double two_pi = 6.283185307179586476925286766559;
  const double inv_c0 = 1.0 / kSpeedOfLight;
  const double u0 = (double)(m.x0 + N / 2 - L / 2) / image_size;
  const double v0 = (double)(m.y0 + N / 2 - L / 2) / image_size;
  const double w0 = w_step > 0.0 ? ((double)m.w_index + 0.5) * w_step : 0.0;
  const double k_mid = 0.5 * (freqs[m.chan_begin] + freqs[m.chan_begin + n_chan - 1]) * inv_c0;
  const float *uvw_b = uvw + (size_t)m.baseline * T * 3;

  for (int c = tid; c < VS; c += NT)
    s_kd[c] = c < n_chan ? (float)(two_pi * (freqs[m.chan_begin + c] * inv_c0 - k_mid)) : 0.f;

  const int g = (warp >> 2) & 1, Lrow = tid & 127;               // generator: warpgroup, row of the 128-pixel tiles
  const uint32_t lane_base = (uint32_t)((warp & 3) * 32) << 16;

  if (warp < 8) {
    // ===================================== generators =====================================
    float ql[PPT], qm[PPT], qn[PPT];
#pragma unroll
    for (int k = 0; k < PPT; ++k) {
      const float4 q = __ldg(&lmn[pix_base + (PPT * g + k) * 128 + Lrow]);
      ql[k] = q.x; qm[k] = q.y; qn[k] = q.z;
    }
    uint32_t slot = 0, round = 0;                              // ring slot of the next step; times the ring went round
    uint32_t empty_base = smem_u32(&bar_empty[0]);
    asm volatile("" : "+r"(empty_base));                       // kept in a register (not rematerialised per slot)
    for (int t0 = 0, sb = 0; t0 < n_time; t0 += tb_max, ++sb) {
      const int tb = min(tb_max, n_time - t0), buf = sb & 1;
      unsigned char *bt = s_b + buf * (kSmemB / 2);
      float4 *st = s_t + buf * (VS / 4) * 2;
      // ---- stage: B tiles of tb x ncp visibilities (scaled, split, zero padded) and the per-timestep terms
      for (int i = tid; i < tb * ncp; i += GEN_THREADS) {
        const int tl = i / ncp, c = i - tl * ncp;
        float4 a = make_float4(0.f, 0.f, 0.f, 0.f), b = a;
        if (c < n_chan) {
          const size_t gi = (((size_t)m.baseline * T + (m.time_begin + t0 + tl)) * C + (m.chan_begin + c)) * 2;
          a = __ldg(&vis[gi]); b = __ldg(&vis[gi + 1]);
        }
        const float vr[4] = {a.x * scale, a.z * scale, b.x * scale, b.z * scale};
        const float vi[4] = {a.y * scale, a.w * scale, b.y * scale, b.w * scale};
        unsigned char *tile = bt + (i >> 2) * 512 + ((i & 3) >> 1) * 128 + (i & 1) * 8;   // K = 4 (i & 3) + q
#pragma unroll
        for (int p = 0; p < 4; ++p) {
          const __half rh = __float2half_rn(vr[p]), ih = __float2half_rn(vi[p]);
          const __half rl = __float2half_rn(vr[p] - __half2float(rh)), il = __float2half_rn(vi[p] - __half2float(ih));
          const __half nih = __hneg(ih), nil = __hneg(il), z = __float2half_rn(0.f);
          // rows n = p (re), 4 + p (im), 8 + p (re, lo), 12 + p (im, lo); K order cos_hi, sin_hi, cos_lo, sin_lo
          const __half2 re_a = __halves2half2(rh, nih), im_a = __halves2half2(ih, rh);
          const __half2 rel = __halves2half2(rl, nil), iml = __halves2half2(il, rl), zz = __halves2half2(z, z);
          // the cos_lo / sin_lo rows of A hold hi - x = -lo: their B coefficients are negated
          const __half2 re_n = __hneg2(re_a), im_n = __hneg2(im_a);
          *reinterpret_cast<uint2 *>(tile + (p) * 16) = make_uint2(*reinterpret_cast<const uint32_t *>(&re_a), *reinterpret_cast<const uint32_t *>(&re_n));
          *reinterpret_cast<uint2 *>(tile + (4 + p) * 16) = make_uint2(*reinterpret_cast<const uint32_t *>(&im_a), *reinterpret_cast<const uint32_t *>(&im_n));
          *reinterpret_cast<uint2 *>(tile + 256 + (p) * 16) = make_uint2(*reinterpret_cast<const uint32_t *>(&rel), *reinterpret_cast<const uint32_t *>(&zz));
          *reinterpret_cast<uint2 *>(tile + 256 + (4 + p) * 16) = make_uint2(*reinterpret_cast<const uint32_t *>(&iml), *reinterpret_cast<const uint32_t *>(&zz));
        }
      }
      for (int tl = tid; tl < tb; tl += GEN_THREADS) {
        const float *p = uvw_b + (size_t)(m.time_begin + t0 + tl) * 3;
        const float u = p[0], v = p[1], w = p[2];
        st[2 * tl] = make_float4(u, v, w, 0.f);
        st[2 * tl + 1] = make_float4((float)(two_pi * ((double)u * k_mid - u0)), (float)(two_pi * ((double)v * k_mid - v0)),
                                     (float)(two_pi * ((double)w * k_mid - w0)), 0.f);
      }
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");     // the MMAs read the B tiles through the async proxy
      asm volatile("bar.sync 1, 256;" ::: "memory");                   // generators only
      // ---- generate: per timestep, per ring slot of 4 KB channels.  Software-pipelined: the per-timestep terms and
      // the anchor sin/cos of the NEXT slot are started before this slot's rotations, and the slot's "empty" barrier
      // is tested early, so that none of those latencies sits between two slots of a warp.
      float npidx[PPT], nbase[PPT], ncr[PPT], nsr[PPT], nco[PPT], nsi[PPT];
      auto prep_time = [&](int tl) {
        const float4 tu = st[2 * tl], tbs = st[2 * tl + 1];
#pragma unroll
        for (int k = 0; k < PPT; ++k) {
          npidx[k] = fmaf(tu.x, ql[k], fmaf(tu.y, qm[k], tu.z * qn[k]));
          nbase[k] = fmaf(tbs.x, ql[k], fmaf(tbs.y, qm[k], tbs.z * qn[k]));
          if (ROT) __sincosf(npidx[k] * dkd, &nsr[k], &ncr[k]);
        }
      };
      auto prep_anchor = [&](int cs) {
        const float kd = s_kd[cs * (4 * KB)];
#pragma unroll
        for (int k = 0; k < PPT; ++k) __sincosf(fmaf(npidx[k], kd, nbase[k]), &nsi[k], &nco[k]);
      };
      prep_time(0);
      prep_anchor(0);
      for (int tl = 0; tl < tb; ++tl) {
        for (int cs = 0; cs < spt; ++cs) {
          float pidx[PPT], base[PPT], cr[PPT], sr[PPT], co[PPT], si[PPT];
#pragma unroll
          for (int k = 0; k < PPT; ++k) {
            pidx[k] = npidx[k]; base[k] = nbase[k]; cr[k] = ncr[k]; sr[k] = nsr[k]; co[k] = nco[k]; si[k] = nsi[k];
          }
          const uint32_t empty_addr = empty_base + 8u * slot;
          uint32_t slot_free = 1;
          if (round > 0)                                                  // non-blocking; consumed before the stores
            asm volatile("{ .reg .pred p; mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                         : "=r"(slot_free) : "r"(empty_addr), "r"((round - 1) & 1u) : "memory");
          // next slot: (tl, cs + 1) or (tl + 1, 0); its terms are computed in stages between this slot's rotations
          const bool new_time = cs + 1 == spt;
          const int ncs = new_time ? 0 : cs + 1, ntl = min(tl + (new_time ? 1 : 0), tb - 1);
          float4 tu, tbs;
          float nkd;
          uint32_t areg[PPT][8 * KB];
#pragma unroll
          for (int j = 0; j < 4 * KB; ++j) {
            if (j == 0) { tu = st[2 * ntl]; tbs = st[2 * ntl + 1]; nkd = s_kd[ncs * (4 * KB)]; }
            if (j == 2 && new_time) {
#pragma unroll
              for (int k = 0; k < PPT; ++k) {
                npidx[k] = fmaf(tu.x, ql[k], fmaf(tu.y, qm[k], tu.z * qn[k]));
                nbase[k] = fmaf(tbs.x, ql[k], fmaf(tbs.y, qm[k], tbs.z * qn[k]));
              }
            }
            if (j == 3 && new_time && ROT) {
#pragma unroll
              for (int k = 0; k < PPT; ++k) __sincosf(npidx[k] * dkd, &nsr[k], &ncr[k]);
            }
            if (j == 4) {
#pragma unroll
              for (int k = 0; k < PPT; ++k) __sincosf(fmaf(npidx[k], nkd, nbase[k]), &nsi[k], &nco[k]);
            }
            if (ROT && j > 0) {                                           // (co, si) *= (cr + i sr), both pixels packed
              static_assert(PPT == 2, "packed rotation over the thread's two pixels");
              const float2 C = make_float2(co[0], co[1]), S = make_float2(si[0], si[1]);
              const float2 CR = make_float2(cr[0], cr[1]), SR = make_float2(sr[0], sr[1]);
              const float2 C2 = ffma2(C, CR, fmul2(S, make_float2(-sr[0], -sr[1])));
              const float2 S2 = ffma2(S, CR, fmul2(C, SR));
              co[0] = C2.x; co[1] = C2.y; si[0] = S2.x; si[1] = S2.y;
            }
#pragma unroll
            for (int k = 0; k < PPT; ++k) {
              if (!ROT && j > 0) __sincosf(fmaf(pidx[k], s_kd[cs * (4 * KB) + j], base[k]), &si[k], &co[k]);
              const __half2 h = __floats2half2_rn(co[k], si[k]);          // low half = cos (even K), high = sin
              const uint32_t hb = *reinterpret_cast<const uint32_t *>(&h);
              float dc, ds;                                               // hi - x in one mixed-precision add each (FHADD)
              asm("{ .reg .f16 lo, hi; mov.b32 {lo, hi}, %2; sub.rn.f32.f16 %0, lo, %3; sub.rn.f32.f16 %1, hi, %4; }"
                  : "=f"(dc), "=f"(ds) : "r"(hb), "f"(co[k]), "f"(si[k]));
              const __half2 l = __floats2half2_rn(dc, ds);                // = -(x - hi): the sign sits in the B tile
              areg[k][2 * j] = hb;
              areg[k][2 * j + 1] = *reinterpret_cast<const uint32_t *>(&l);
            }
            if ((j & 3) == 3) {                                           // 4 visibilities done: one MMA batch of rows
              if (j == 3) {
                if (!slot_free) mbar_wait_addr(empty_addr, (round - 1) & 1u);
                tc_fence_after();
              }
#pragma unroll
              for (int k = 0; k < PPT; ++k) {
                const int r0 = 2 * (j - 3);
                const uint32_t ta = tmem + lane_base + (uint32_t)(COLS_D + (PPT * g + k) * (8 * KB) + r0) + slot * (uint32_t)COLS_SLOT;
                asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};"
                             ::"r"(ta), "r"(areg[k][r0]), "r"(areg[k][r0 + 1]), "r"(areg[k][r0 + 2]), "r"(areg[k][r0 + 3]),
                               "r"(areg[k][r0 + 4]), "r"(areg[k][r0 + 5]), "r"(areg[k][r0 + 6]), "r"(areg[k][r0 + 7]) : "memory");
              }
            }
          }
          asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
          tc_fence_before();
          // hand-over on a named barrier: the generators only arrive, the issuing warp sleeps in bar.sync until all
          // eight have (an mbarrier here cost the issuer ~170 instructions of polling per slot, 9 % of the kernel's)
          static_assert(RING == 1, "one named barrier: a slot's phase ends before its next arrivals (empty barrier)");
          asm volatile("bar.arrive 2, %0;" ::"n"(NT) : "memory");
          if (++slot == RING) { slot = 0; ++round; }
        }
      }
    }
  } else {
    // ===================================== issuer (warp 8, convergent; one elected lane issues) ====================
    uint32_t leader = 0;
    asm volatile("{ .reg .pred p; elect.sync _|p, 0xffffffff; selp.u32 %0, 1, 0, p; }" : "=r"(leader));
    int gs = 0;
    for (int t0 = 0, sb = 0; t0 < n_time; t0 += tb_max, ++sb) {
      const int tb = min(tb_max, n_time - t0);
      const uint32_t bt = smem_u32(s_b + (sb & 1) * (kSmemB / 2));
      for (int si = 0; si < tb * spt; ++si, ++gs) {
        const int slot = gs % RING;
        asm volatile("bar.sync 2, %0;" ::"n"(NT) : "memory");
        tc_fence_after();
        if (leader) {
          const uint32_t a0 = tmem + (uint32_t)(COLS_D + slot * COLS_SLOT);
#pragma unroll
          for (int kb = 0; kb < KB; ++kb) {
            const uint64_t bd = b_desc(bt + (si * KB + kb) * 512);
            const uint32_t acc = (gs > 0 || kb > 0) ? 1u : 0u;
#pragma unroll
            for (int tile = 0; tile < TILES; ++tile)
              asm volatile("{ .reg .pred p; setp.ne.b32 p, %4, 0; tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p; }"
                           ::"r"(tmem + tile * 16), "r"(a0 + tile * (8 * KB) + kb * 8), "l"(bd), "r"(kIdesc), "r"(acc) : "memory");
          }
          asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.b64 [%0];" ::"r"(smem_u32(&bar_empty[slot])) : "memory");
        }
        __syncwarp();
      }
    }
    if (leader) asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.b64 [%0];" ::"r"(smem_u32(&bar_done)) : "memory");
    __syncwarp();
  }

  // ===================================== epilogue (generators) =====================================
  if (warp < 8) {
    mbar_wait(&bar_done, 0);
    tc_fence_after();
    const size_t a1_off = ((size_t)m.aterm_slot * n_stations + m.station1) * NPIX;
    const size_t a2_off = ((size_t)m.aterm_slot * n_stations + m.station2) * NPIX;
    float2 *out = subgrids + (size_t)blockIdx.x * 4 * NPIX;
#pragma unroll
    for (int k = 0; k < PPT; ++k) {
      const int pix = pix_base + (PPT * g + k) * 128 + Lrow;
      uint32_t r[16];
      asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                   : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
                     "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
                   : "r"(tmem + lane_base + (uint32_t)((PPT * g + k) * 16)));
      asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
      float re[4], im[4];
#pragma unroll
      for (int p = 0; p < 4; ++p) {
        re[p] = (__uint_as_float(r[p]) + __uint_as_float(r[8 + p])) * inv_scale;
        im[p] = (__uint_as_float(r[4 + p]) + __uint_as_float(r[12 + p])) * inv_scale;
      }
      // taper * A1^H * P * A2 per pixel (R5), written pol-planar: as in gridder_kernel
      const float4 a01 = __ldg(&aterms[(a1_off + pix) * 2]), a23 = __ldg(&aterms[(a1_off + pix) * 2 + 1]);
      const float4 b01 = __ldg(&aterms[(a2_off + pix) * 2]), b23 = __ldg(&aterms[(a2_off + pix) * 2 + 1]);
      const float tp = __ldg(&taper[pix]);
      const float2 a0 = make_float2(a01.x, a01.y), a1 = make_float2(a01.z, a01.w);
      const float2 a2 = make_float2(a23.x, a23.y), a3 = make_float2(a23.z, a23.w);
      const float2 b0 = make_float2(b01.x, b01.y), b1 = make_float2(b01.z, b01.w);
      const float2 b2 = make_float2(b23.x, b23.y), b3 = make_float2(b23.z, b23.w);
      const float2 p0 = make_float2(re[0], im[0]), p1 = make_float2(re[1], im[1]);
      const float2 p2 = make_float2(re[2], im[2]), p3 = make_float2(re[3], im[3]);
      const float2 t00 = cadd(cmul_conj_a(a0, p0), cmul_conj_a(a2, p2));
      const float2 t01 = cadd(cmul_conj_a(a0, p1), cmul_conj_a(a2, p3));
      const float2 t10 = cadd(cmul_conj_a(a1, p0), cmul_conj_a(a3, p2));
      const float2 t11 = cadd(cmul_conj_a(a1, p1), cmul_conj_a(a3, p3));
      const float2 rr[4] = {cadd(cmul(t00, b0), cmul(t01, b2)), cadd(cmul(t00, b1), cmul(t01, b3)),
                            cadd(cmul(t10, b0), cmul(t11, b2)), cadd(cmul(t10, b1), cmul(t11, b3))};
#pragma unroll
      for (int q = 0; q < 4; ++q) out[q * NPIX + pix] = make_float2(tp * rr[q].x, tp * rr[q].y);
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 8) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(TMEM_COLS));
}

// The tensor-core gridder serves per-block A-terms at N = 32 when every block has 8 to 128 channels (a ring slot is 8
// channels of one timestep; a staging batch of 128 visibilities holds at least one timestep); everything else takes
// gridder_kernel.
bool gridder_tc_eligible(const idg_plan *plan) {
  // sweep (N = 32, 16 channels, fraction of the FP32 lane-op roofline, this kernel / the FFMA2 kernel) by block length:
  // 128 visibilities 0.79 / 0.71; 256: 0.86 / 0.73; 512: 0.90 / 0.75; 2048: 0.93 / 0.75; 8192 at 64 channels: 0.97 / 0.76.
  // Shorter blocks are not measured (the fixed cost per CTA -- allocation, block maximum, fill, drain, epilogue -- grows)
  return plan->prm.subgrid_size == 32 && !(plan->prm.flags & (IDG_PLAN_SPAN_ATERMS | IDG_PLAN_FP32_GRIDDER)) &&
         plan->min_n_chan >= 8 &&
         plan->max_n_chan <= tc::VS &&                  // a staging batch holds at least one timestep of the block
         plan->P > 0 && plan->n_planned / plan->P >= 128;
}

int launch_gridder_tc(const idg_plan *plan, const float *uvw, const float2 *vis, const float2 *aterms,
                      const float *taper, float2 *subgrids, cudaStream_t stream, int64_t p0, int64_t np) {
  constexpr int RING = 1;
  const bool rot = plan->uniform_dkd != 0.f;
  auto kern = rot ? gridder_tc_kernel<RING, true> : gridder_tc_kernel<RING, false>;
  IDG_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmem));
  IDG_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
  kern<<<dim3((unsigned)np, tc::SPL), tc::NT, kSmem, stream>>>(
      plan->meta_dev + p0, uvw, plan->freqs_dev, plan->lmn_dev, reinterpret_cast<const float4 *>(vis),
      reinterpret_cast<const float4 *>(aterms), taper, subgrids + (size_t)p0 * 4 * tc::NPIX, plan->T, plan->C,
      plan->n_stations, plan->prm.grid_size, plan->prm.image_size, plan->prm.w_step, plan->uniform_dkd);
  IDG_LAUNCH_CHECK();
  return IDG_OK;
}

}  // namespace idg
