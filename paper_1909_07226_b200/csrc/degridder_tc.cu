// degridder_tc.cu -- row a6 on the 5th-generation tensor cores (N = 32): the prediction as a dense contraction.
//
// Alg. 2 inner loops are  Y[k][comp] = sum_pixel conj(Phi[pixel][k]) Dg[pixel][comp]  with the
// phasor matrix of the gridder and the 8 real components of the corrected pixels Dg = A1 (taper Ip) A2^H (R5): a real
// GEMM with M = the block's visibilities, N = 8, K = 2 x 1024 (cos and sin rows per pixel).  The FP32 kernel
// (degridder.cu) spends 16 of its 18 lane-ops per (visibility, pixel) on that product and is bound by the FMA pipe;
// here it runs as tcgen05.mma.kind::f16 with FP32 accumulators in tensor memory and the CUDA cores only generate
// phasors.  Operands are split x = hi + lo in fp16 exactly as in gridder_tc.cu (22 bits; lo x lo dropped):
//   K rows per pixel:   cos_hi, sin_hi, hi - cos, hi - sin                     (A operand, tensor memory)
//   N columns:          8 components against Dg_hi, then 8 against Dg_lo        (B operand, shared memory)
// The pixels of a subgrid are scaled by a power of two so that their largest component sits near 2^14.
//
// Orientation: the contraction index is the pixel, so here the THREADS own visibilities: a group of 128 threads
// (4 warps = the 128 lanes of tensor memory) owns a tile of 128 visibilities of the block; a thread evaluates its
// visibility's phase a (x - 16) + b (y - 16) + W n' (a = 2 pi (u k_c - u0) S/N etc., FP64 once per tile; two FMAs per
// pixel, n' from a shared-memory table) for 16 pixels of a row at a time, takes sin/cos.approx, splits, and writes its
// row of four A tiles (16 pixels = 4 x K16) with two tcgen05.st.x16.  The B operand -- 512 bytes per 4 pixels, 128 KB
// for a subgrid -- is staged in shared memory for HALF a subgrid at a time (64 KB), so that two CTAs of four groups
// (512 threads, 64 registers, 256 tensor-memory columns) share an SM: a round of four visibility tiles stages both
// halves and keeps its accumulators D[128 x 16] in tensor memory across them; blocks of more than 512 visibilities
// take several rounds.  One warp of the group (they take turns) waits for the other three on a named barrier, issues
// the slot's four MMAs and commits them to the group's "empty" mbarrier, which the group tests before its next store.
// Blocks with fewer than four tiles split the pixels of a tile over several groups; the partial sums meet in shared
// memory.  Unlike the gridder there is no rotation recurrence (neighbouring pixels do not differ by a constant phase:
// n' is not affine), so every phasor costs two MUFU operations: the kernel is bound by the XU pipe and by the 32 warps
// per SM that 64 registers allow.  Measurements and variants: profiles/r02_experiments.md section 8.
#include <cuda_fp16.h>

#include "common.cuh"

namespace idg {

namespace dtc {

constexpr int N = 32, NPIX = N * N;
constexpr int GROUPS = 4, NT = GROUPS * 128;                 // 4 groups of 128 threads (one visibility tile each)
constexpr int COLS_GROUP = 48;                               // tensor-memory columns per group: D (16) + one A slot (32)
constexpr int TMEM_COLS = 256;                               // 4 x 48 rounded up to a power of two: two CTAs per SM
constexpr int HALF = NPIX / 2;                               // pixels whose B tiles are resident at a time
constexpr int SLOTS_H = HALF / 16;                           // 32 slots of 16 pixels (4 K16 blocks) per half
constexpr int kSmemB = (HALF / 4) * 512;                     // 65536: B tiles of one half, [K block][512]
constexpr int kSmemN = NPIX * 4;                             // n' per pixel
constexpr int kSmemRed = GROUPS * 8 * 128 * 4;               // partial sums, [group][component][lane]
constexpr int kSmem = kSmemB + kSmemN + kSmemRed;

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *b, uint32_t c) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(c));
}
__device__ __forceinline__ uint32_t mbar_test(uint32_t addr, uint32_t parity) {
  uint32_t ok;
  asm volatile("{ .reg .pred p; mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
               : "=r"(ok) : "r"(addr), "r"(parity) : "memory");
  return ok;
}
__device__ __forceinline__ void mbar_wait(uint32_t addr, uint32_t parity) {
  uint32_t ok = 0;
  for (int spins = 0; spins < (1 << 26); ++spins) {          // bounded: a lost arrival traps instead of hanging the GPU
    asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                 : "=r"(ok) : "r"(addr), "r"(parity) : "memory");
    if (ok) return;
  }
  __trap();
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

// instruction descriptor: D = F32, A = B = F16, both K-major, N = 16, M = 128
constexpr uint32_t kIdesc = (1u << 4) | ((16u >> 3) << 17) | ((128u >> 4) << 24);
// shared-memory descriptor of one B tile [16 n][16 k] fp16, K-major, no swizzle (as in gridder_tc.cu)
__device__ __forceinline__ uint64_t b_desc(uint32_t smem_addr) {
  return (uint64_t)((smem_addr & 0x3FFFF) >> 4) | ((uint64_t)(128 >> 4) << 16) | ((uint64_t)(256 >> 4) << 32) |
         ((uint64_t)1 << 46);
}

}  // namespace dtc

using namespace dtc;


// corrected pixel Dg = A1 (taper Ip) A2^H (R5), as degridder_kernel: (re, im) of XX, XY, YX, YY
__device__ __forceinline__ void corrected_pixel(const float2 *__restrict__ sg, const float4 *__restrict__ aterms,
                                                const float *__restrict__ taper, size_t a1_off, size_t a2_off, int pix,
                                                float (&pr)[4], float (&pi)[4]) {
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
  const float2 t00 = cadd(cmul(a0, p0), cmul(a1, p2)), t01 = cadd(cmul(a0, p1), cmul(a1, p3));
  const float2 t10 = cadd(cmul(a2, p0), cmul(a3, p2)), t11 = cadd(cmul(a2, p1), cmul(a3, p3));
  const float2 r0 = cadd(cmul_conj_b(t00, b0), cmul_conj_b(t01, b1));
  const float2 r1 = cadd(cmul_conj_b(t00, b2), cmul_conj_b(t01, b3));
  const float2 r2 = cadd(cmul_conj_b(t10, b0), cmul_conj_b(t11, b1));
  const float2 r3 = cadd(cmul_conj_b(t10, b2), cmul_conj_b(t11, b3));
  pr[0] = r0.x; pr[1] = r1.x; pr[2] = r2.x; pr[3] = r3.x;
  pi[0] = r0.y; pi[1] = r1.y; pi[2] = r2.y; pi[3] = r3.y;
}

__global__ void __launch_bounds__(dtc::NT, 2)
degridder_tc_kernel(const idg_subgrid_meta *__restrict__ meta, const float *__restrict__ uvw,
                    const double *__restrict__ freqs, const float4 *__restrict__ lmn,
                    const float2 *__restrict__ subgrids, const float4 *__restrict__ aterms,
                    const float *__restrict__ taper, float4 *__restrict__ vis_out, int32_t T, int32_t C,
                    int32_t n_stations, int32_t L, double image_size, double w_step) {
  extern __shared__ __align__(128) unsigned char smem_dyn[];
  unsigned char *s_b = smem_dyn;
  float *s_n = reinterpret_cast<float *>(smem_dyn + kSmemB);
  float *s_red = reinterpret_cast<float *>(smem_dyn + kSmemB + kSmemN);
  __shared__ uint64_t bar_empty[GROUPS];
  __shared__ uint32_t s_tmem, s_maxbits;

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int g = warp >> 2, wg = warp & 3, lrow = tid & 127;
  const idg_subgrid_meta m = meta[blockIdx.x];
  const int n_chan = m.n_chan, n_time = m.n_time;
  const float2 *sg = subgrids + (size_t)blockIdx.x * 4 * NPIX;
  const size_t a1_off = ((size_t)m.aterm_slot * n_stations + m.station1) * NPIX;
  const size_t a2_off = ((size_t)m.aterm_slot * n_stations + m.station2) * NPIX;

  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&s_tmem)), "n"(TMEM_COLS));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  if (tid == 0) {
    for (int s = 0; s < GROUPS; ++s) mbar_init(&bar_empty[s], 1);
    s_maxbits = 0;
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = s_tmem;

  // ---- largest component of the corrected subgrid -> one power-of-two scale into the fp16 range for both halves
  {
    float mx = 0.f;
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      float pr[4], pi[4];
      const int pix = h * HALF + tid;
      corrected_pixel(sg, aterms, taper, a1_off, a2_off, pix, pr, pi);
#pragma unroll
      for (int j = 0; j < 4; ++j) mx = fmaxf(mx, fmaxf(fabsf(pr[j]), fabsf(pi[j])));
      s_n[pix] = __ldg(&lmn[pix]).z;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    if (lane == 0 && isfinite(mx)) atomicMax(&s_maxbits, __float_as_uint(mx));    // non-negative floats order like their bits
  }
  __syncthreads();
  const float vmax = __uint_as_float(s_maxbits);
  int e = 0;
  if (vmax > 0.f) frexpf(vmax, &e);
  const float scale = ldexpf(1.0f, 14 - e), inv_scale = ldexpf(1.0f, e - 14);

  const int nv = n_time * n_chan, nt = (nv + 127) / 128;
  int parts = 1;
  while (parts < GROUPS && nt * parts * 2 <= GROUPS) parts *= 2;     // 1 tile: 4 parts of the pixels, 2 tiles: 2, else 1
  const int n_units = nt * parts, spp = SLOTS_H / parts;             // slots per part and half (a multiple of 4: whole rows)
  const double two_pi = 6.283185307179586476925286766559;
  const double inv_c0 = 1.0 / kSpeedOfLight;
  const double u0 = (double)(m.x0 + N / 2 - L / 2) / image_size;
  const double v0 = (double)(m.y0 + N / 2 - L / 2) / image_size;
  const double w0 = w_step > 0.0 ? ((double)m.w_index + 0.5) * w_step : 0.0;
  const float dl = (float)(image_size / (double)N);                  // l_x = (x - N/2) dl, m_y = (y - N/2) dl (R1)
  const uint32_t lane_base = (uint32_t)(wg * 32) << 16;
  const uint32_t col_d = tmem + (uint32_t)(g * COLS_GROUP), col_a = col_d + 16;
  uint32_t empty_addr = smem_u32(&bar_empty[g]);
  asm volatile("" : "+r"(empty_addr));
  uint32_t cnt = 0;                                                  // slots this group has handed over so far
  // per-thread constants of the slot loop, opaque to the compiler so that it keeps them in registers instead of
  // re-deriving them from %tid and the shared-memory window in every slot (64 registers per thread)
  uint32_t sttm_addr = col_a + lane_base, barid = 1u + (uint32_t)g, wgq = (uint32_t)wg;
  asm volatile("" : "+r"(sttm_addr), "+r"(barid), "+r"(wgq));

  for (int ub = 0; ub < n_units; ub += GROUPS) {
    const int unit = ub + g;
    const bool has = unit < n_units;
    const int tile = has ? unit / parts : 0, part = has ? unit - tile * parts : 0;
    const int vi = tile * 128 + lrow;
    const bool act = has && vi < nv;
    const int vc = min(vi, nv - 1);
    const int tl = vc / n_chan, ch = vc - tl * n_chan;
    float a = 0.f, bv = 0.f, W = 0.f;
    if (has) {
      const float *p = uvw + ((size_t)m.baseline * T + (m.time_begin + tl)) * 3;
      const double kc = freqs[m.chan_begin + ch] * inv_c0;
      a = (float)(two_pi * ((double)p[0] * kc - u0)) * dl;           // phase = a (x - N/2) + bv (y - N/2) + W n'
      bv = (float)(two_pi * ((double)p[1] * kc - v0)) * dl;
      W = (float)(two_pi * ((double)p[2] * kc - w0));
    }
    for (int half = 0; half < 2; ++half) {
      // ---- stage the B tiles of this half: thread = pixel; K = 4 q + (cos_hi, sin_hi, hi - cos, hi - sin), q = pixel & 3
      __syncthreads();                                               // every group's MMAs on the previous tiles are complete
      {
        float pr[4], pi[4];
        corrected_pixel(sg, aterms, taper, a1_off, a2_off, half * HALF + tid, pr, pi);
        unsigned char *bt = s_b + (tid >> 2) * 512 + ((tid & 3) >> 1) * 128 + (tid & 1) * 8;
        const __half z = __float2half_rn(0.f);
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          const float vr = pr[j] * scale, vim = pi[j] * scale;
          const __half rh = __float2half_rn(vr), ih = __float2half_rn(vim);
          const __half rl = __float2half_rn(vr - __half2float(rh)), il = __float2half_rn(vim - __half2float(ih));
          // Y_re = sum cos Dg_re + sin Dg_im, Y_im = sum cos Dg_im - sin Dg_re; the "hi - x" rows carry the opposite sign
          const __half2 re_a = __halves2half2(rh, ih), re_n = __hneg2(re_a);
          const __half2 im_a = __halves2half2(ih, __hneg(rh)), im_n = __hneg2(im_a);
          const __half2 re_l = __halves2half2(rl, il), im_l = __halves2half2(il, __hneg(rl)), zz = __halves2half2(z, z);
          *reinterpret_cast<uint2 *>(bt + j * 16) = make_uint2(*reinterpret_cast<const uint32_t *>(&re_a), *reinterpret_cast<const uint32_t *>(&re_n));
          *reinterpret_cast<uint2 *>(bt + (4 + j) * 16) = make_uint2(*reinterpret_cast<const uint32_t *>(&im_a), *reinterpret_cast<const uint32_t *>(&im_n));
          *reinterpret_cast<uint2 *>(bt + 256 + j * 16) = make_uint2(*reinterpret_cast<const uint32_t *>(&re_l), *reinterpret_cast<const uint32_t *>(&zz));
          *reinterpret_cast<uint2 *>(bt + 256 + (4 + j) * 16) = make_uint2(*reinterpret_cast<const uint32_t *>(&im_l), *reinterpret_cast<const uint32_t *>(&zz));
        }
      }
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // the MMAs read the B tiles through the async proxy
      __syncthreads();
      if (!has) continue;
      // ---- rows of 32 pixels = 2 slots of 16; local slot ls = part spp + 2 r + j of this half
      uint32_t n_addr = smem_u32(s_n) + (uint32_t)(half * HALF + part * spp * 16) * 4u;
      uint32_t b_addr = smem_u32(s_b) + (uint32_t)(part * spp) * 2048u;
      float brow = bv * (float)(half * (N / 2) + ((part * spp) >> 1) - N / 2);
      for (int r = 0; r < spp; r += 2) {
#pragma unroll
        for (int j = 0; j < 2; ++j) {
          uint32_t slot_free = 1;
          if (cnt > 0) slot_free = mbar_test(empty_addr, (cnt - 1) & 1u);    // non-blocking; consumed before the store
#pragma unroll
          for (int hq = 0; hq < 2; ++hq) {
            float nn[8];
            asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(nn[0]), "=f"(nn[1]), "=f"(nn[2]), "=f"(nn[3])
                         : "r"(n_addr + (uint32_t)(j * 16 + hq * 8) * 4u));
            asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(nn[4]), "=f"(nn[5]), "=f"(nn[6]), "=f"(nn[7])
                         : "r"(n_addr + (uint32_t)(j * 16 + hq * 8 + 4) * 4u));
            uint32_t areg[16];
#pragma unroll
            for (int q = 0; q < 8; ++q) {
              float si, co;
              __sincosf(fmaf(W, nn[q], fmaf(a, (float)(j * 16 + hq * 8 + q - N / 2), brow)), &si, &co);
              const __half2 h = __floats2half2_rn(co, si);            // low half = cos (even K), high = sin
              const uint32_t hb = *reinterpret_cast<const uint32_t *>(&h);
              float dc, ds;                                           // hi - x in one mixed-precision add each (FHADD)
              asm("{ .reg .f16 lo, hi; mov.b32 {lo, hi}, %2; sub.rn.f32.f16 %0, lo, %3; sub.rn.f32.f16 %1, hi, %4; }"
                  : "=f"(dc), "=f"(ds) : "r"(hb), "f"(co), "f"(si));
              const __half2 l = __floats2half2_rn(dc, ds);
              areg[2 * q] = hb;
              areg[2 * q + 1] = *reinterpret_cast<const uint32_t *>(&l);
            }
            if (hq == 0) {
              if (!slot_free) mbar_wait(empty_addr, (cnt - 1) & 1u);
              tc_fence_after();
            }
            asm volatile("tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};"
                         ::"r"(sttm_addr + (uint32_t)(hq * 16)), "r"(areg[0]), "r"(areg[1]), "r"(areg[2]), "r"(areg[3]), "r"(areg[4]),
                           "r"(areg[5]), "r"(areg[6]), "r"(areg[7]), "r"(areg[8]), "r"(areg[9]), "r"(areg[10]),
                           "r"(areg[11]), "r"(areg[12]), "r"(areg[13]), "r"(areg[14]), "r"(areg[15]) : "memory");
          }
          asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
          tc_fence_before();
          // hand-over inside the group: the warps take turns to wait for the other three and issue the slot's MMAs
          if ((cnt & 3u) != wgq) {
            asm volatile("bar.arrive %0, 128;" ::"r"(barid) : "memory");
          } else {
            asm volatile("bar.sync %0, 128;" ::"r"(barid) : "memory");
            tc_fence_after();
            uint32_t leader = 0;
            asm volatile("{ .reg .pred p; elect.sync _|p, 0xffffffff; selp.u32 %0, 1, 0, p; }" : "=r"(leader));
            if (leader) {
              const uint32_t bt = b_addr + (uint32_t)j * 2048u;
#pragma unroll
              for (int kb = 0; kb < 4; ++kb) {
                const uint32_t acc = (kb > 0 || half > 0 || r > 0 || j > 0) ? 1u : 0u;
                asm volatile("{ .reg .pred p; setp.ne.b32 p, %4, 0; tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p; }"
                             ::"r"(col_d), "r"(col_a + kb * 8), "l"(b_desc(bt + kb * 512)), "r"(kIdesc), "r"(acc) : "memory");
              }
              asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.b64 [%0];" ::"r"(empty_addr) : "memory");
            }
            __syncwarp();
          }
          ++cnt;
        }
        n_addr += 128u;
        b_addr += 4096u;
        brow += bv;
      }
      // the half's last commit covers every MMA of it: after this wait the B tiles may be replaced
      mbar_wait(empty_addr, (cnt - 1) & 1u);
      tc_fence_after();
    }
    float y[8];
    if (has) {
      uint32_t r[16];
      asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                   : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
                     "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
                   : "r"(col_d + lane_base));
      asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
      tc_fence_before();                                             // the next unit's first MMA overwrites D
#pragma unroll
      for (int j = 0; j < 8; ++j) y[j] = (__uint_as_float(r[j]) + __uint_as_float(r[8 + j])) * inv_scale;
    }
    if (parts > 1) {                                                 // uniform over the CTA: the parts of a tile meet
      if (has && part > 0) {
#pragma unroll
        for (int j = 0; j < 8; ++j) s_red[(g * 8 + j) * 128 + lrow] = y[j];
      }
      __syncthreads();
      if (has && part == 0) {
        for (int q = 1; q < parts; ++q)
#pragma unroll
          for (int j = 0; j < 8; ++j) y[j] += s_red[((g + q) * 8 + j) * 128 + lrow];
      }
    }
    if (act && part == 0) {
      float4 *o = vis_out + (((size_t)m.baseline * T + (m.time_begin + tl)) * C + m.chan_begin + ch) * 2;
      o[0] = make_float4(y[0], y[4], y[1], y[5]);                    // (re, im) of XX, XY
      o[1] = make_float4(y[2], y[6], y[3], y[7]);                    // YX, YY
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(TMEM_COLS));
}

// N = 32, one A-term slot per block; any channel count (threads own visibilities).  Short blocks pay the fixed cost
// per subgrid (staging the B tiles twice, pipeline fill, the reduction over pixel parts) and leave lanes of their
// 128-visibility tiles idle.  Sweep (N = 32, fraction of the FP32 roofline, this kernel / the FFMA2 kernel) by block
// length: 128 visibilities 0.55 / 0.64; 256: 0.68 / 0.69; 512: 0.81 / 0.71 (16 channels) and 0.81 / 0.69 (4 channels);
// 2048: 0.82 / 0.73; 8192: 0.82 / 0.72.
bool degridder_tc_eligible(const idg_plan *plan) {
  return plan->prm.subgrid_size == 32 && !(plan->prm.flags & (IDG_PLAN_SPAN_ATERMS | IDG_PLAN_FP32_GRIDDER)) &&
         plan->P > 0 && plan->n_planned / plan->P >= 384;
}

int launch_degridder_tc(const idg_plan *plan, const float *uvw, const float2 *subgrids, const float2 *aterms,
                        const float *taper, float2 *vis_out, cudaStream_t stream, int64_t p0, int64_t np) {
  IDG_CUDA_TRY(cudaFuncSetAttribute(degridder_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmem));
  degridder_tc_kernel<<<(unsigned)np, dtc::NT, kSmem, stream>>>(
      plan->meta_dev + p0, uvw, plan->freqs_dev, plan->lmn_dev, subgrids + (size_t)p0 * 4 * dtc::NPIX,
      reinterpret_cast<const float4 *>(aterms), taper, reinterpret_cast<float4 *>(vis_out), plan->T, plan->C,
      plan->n_stations, plan->prm.grid_size, plan->prm.image_size, plan->prm.w_step);
  IDG_LAUNCH_CHECK();
  return IDG_OK;
}

}  // namespace idg
