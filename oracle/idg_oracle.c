/*
 * idg_oracle.c -- float64 CPU oracle for the Image Domain Gridding hot path.
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call this file.  It shares
 * no code, header, table or helper with the CUDA product under
 * paper_1909_07226_b200/; the two are written independently from the paper.
 *
 * What it is: Algorithm 1 and Algorithm 2 of
 * van der Tol, Veenboer & Offringa, "Image Domain Gridding" (arXiv 1909.07226), step by
 * step in the paper's order, in double precision on inputs upcast from the same
 * float32 / complex64 arrays the GPU receives.  IDG approximates the direct imaging
 * equation (Eq. 11) / the discrete measurement equation (Eq. 6,
 * PAPER.md:84), so the oracle is the algorithm, not the direct sum.  Where the
 * paper's text is garbled or silent the reading of DESIGN.md section "Readings"
 * (R1..R15) is taken; each function names the reading it uses.
 *
 * Plain loops, no blocking, no fusion, no reordering.  The only parallelism is an
 * OpenMP "for" over independent subgrids.  Build: gcc -O2 -ffp-contract=off -fopenmp
 * (no FMA contraction, so the planner's doubles are reproducible bit for bit).
 *
 * Pins (tests/test_oracle_pins.py, all "-m 'not gpu'"):
 *   oracle_plan            P5 plan invariants (exact cover, box bounds, one slot / w layer)
 *   oracle_gridder + oracle_subgrid_fft + oracle_adder
 *                          P1 lattice identity vs brute-force Eq. 11 (round-off),
 *                          P4 off-lattice agreement with Eq. 11 (taper side-lobe level)
 *   oracle_subgrid_fft     numpy.fft with fftshift/ifftshift (library special case)
 *   oracle_splitter + oracle_subgrid_fft + oracle_degridder
 *                          P2 point-source closed form; L = N equals Eq. 6 for any image
 *   both directions        P3 adjoint identity <G v, x> = <v, G^H x> (1e-10)
 * No function here is "parity unpinned".  (Throughput is unpinned by the paper for
 * this hardware: only the GeForce 840M figure exists.)
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_C0 299792458.0
#define ORACLE_FORCE_BLOCKS 1
#define ORACLE_SPAN_ATERMS 2 /* NEXT-4: a block may span A-term slots; c_pk then varies inside the k-sum */
static const double ORACLE_TWO_PI = 6.283185307179586476925286766559;

/* Same binary layout as the boundary's structs (the layout is the contract, the
 * declaration is repeated here on purpose: no shared header). */
typedef struct {
  int32_t grid_size, subgrid_size, kernel_size, max_timesteps, max_channels, aterm_interval,
      flags, reserved;
  double image_size, w_step;
} oracle_params;

typedef struct {
  int32_t baseline, station1, station2, time_begin, n_time, chan_begin, n_chan, aterm_slot, x0,
      y0, w_index, reserved;
} oracle_meta;

typedef double complex cplx;

int oracle_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

/* ---------------------------------------------------------------------------------------
 * Partitioning (section 3.2, Fig. 2).  The paper gives no
 * algorithm ("a tight box per subset"), reading R10/R11/R12: greedy walk over the
 * timesteps of one baseline and one channel group; a block ends when the uv bounding box
 * of its samples (in grid pixels) would exceed N - kernel_size, when it reaches
 * max_timesteps, when the A-term slot changes (R5: one c_p per block) or
 * when the w layer changes (R4).  Channel groups start at max_channels (a power of two)
 * and are halved until they fit the channels left and a single timestep fits the box.
 * Returns the number of subgrids; writes at most `capacity` of them to `out` (may be
 * NULL to count).  All arithmetic in double, one rounding per operation.
 * ------------------------------------------------------------------------------------- */
int64_t oracle_plan(const oracle_params *prm, const float *uvw /*[B][T][3]*/,
                    const double *freqs /*[C]*/, const int32_t *baselines /*[B][2]*/, int32_t B,
                    int32_t T, int32_t C, oracle_meta *out, int64_t capacity,
                    int64_t *n_planned_vis, int64_t *n_skipped_vis) {
  const int32_t N = prm->subgrid_size, L = prm->grid_size;
  const int force = (prm->flags & ORACLE_FORCE_BLOCKS) != 0;
  const int span = (prm->flags & ORACLE_SPAN_ATERMS) != 0;
  const double budget = (double)(N - prm->kernel_size);
  double *scale = (double *)malloc(sizeof(double) * (size_t)C);
  for (int32_t c = 0; c < C; ++c) scale[c] = (freqs[c] * (1.0 / ORACLE_C0)) * prm->image_size;
  int64_t count = 0, planned = 0, skipped = 0;
  for (int32_t b = 0; b < B; ++b) {
    const float *uvw_b = uvw + (size_t)b * T * 3;
    int32_t c0 = 0;
    while (c0 < C) {
      int32_t n = prm->max_channels;          /* a power of two (R11) */
      while (n > C - c0) n = n / 2;           /* halve until the group fits the band ... */
      if (!force) {
        while (n > 1) {                       /* ... and the box of a single timestep */
          const double ds = scale[c0 + n - 1] - scale[c0];
          double mx = 0.0;
          for (int32_t t = 0; t < T; ++t) {
            const double du = fabs((double)uvw_b[3 * t + 0] * ds);
            const double dv = fabs((double)uvw_b[3 * t + 1] * ds);
            if (du > mx) mx = du;
            if (dv > mx) mx = dv;
          }
          if (mx > budget) n = n / 2; else break;
        }
      }
      const double s_lo = scale[c0], s_hi = scale[c0 + n - 1];
      const double k_mid = (0.5 * (freqs[c0] + freqs[c0 + n - 1])) * (1.0 / ORACLE_C0);
      int32_t t0 = 0;
      while (t0 < T) {
        int32_t t1 = t0;
        double umin = 0, umax = 0, vmin = 0, vmax = 0;
        int32_t wi0 = 0;
        while (t1 < T && t1 - t0 < prm->max_timesteps &&
               (span || t1 / prm->aterm_interval == t0 / prm->aterm_interval)) {
          int32_t wi = 0;
          if (prm->w_step > 0.0)
            wi = (int32_t)floor(((double)uvw_b[3 * t1 + 2] * k_mid) / prm->w_step);
          if (t1 == t0) wi0 = wi; else if (wi != wi0) break;
          const double u = (double)uvw_b[3 * t1 + 0], v = (double)uvw_b[3 * t1 + 1];
          const double ua = u * s_lo, ub = u * s_hi, va = v * s_lo, vb = v * s_hi;
          double numin, numax, nvmin, nvmax;
          if (t1 == t0) {
            numin = fmin(ua, ub); numax = fmax(ua, ub); nvmin = fmin(va, vb); nvmax = fmax(va, vb);
          } else {
            numin = fmin(umin, fmin(ua, ub)); numax = fmax(umax, fmax(ua, ub));
            nvmin = fmin(vmin, fmin(va, vb)); nvmax = fmax(vmax, fmax(va, vb));
            if (!force && (numax - numin > budget || nvmax - nvmin > budget)) break;
          }
          umin = numin; umax = numax; vmin = nvmin; vmax = nvmax;
          ++t1;
        }
        /* centre pixel = box midpoint rounded half up (R12); corner = centre - N/2 (R3) */
        const int32_t xc = (int32_t)floor(0.5 * (umin + umax) + 0.5);
        const int32_t yc = (int32_t)floor(0.5 * (vmin + vmax) + 0.5);
        const int32_t x0 = xc + L / 2 - N / 2, y0 = yc + L / 2 - N / 2;
        const int64_t nvis = (int64_t)(t1 - t0) * n;
        if (x0 >= 0 && y0 >= 0 && x0 + N <= L && y0 + N <= L) {
          if (out && count < capacity) {
            oracle_meta m;
            m.baseline = b; m.station1 = baselines[2 * b]; m.station2 = baselines[2 * b + 1];
            m.time_begin = t0; m.n_time = t1 - t0; m.chan_begin = c0; m.n_chan = n;
            m.aterm_slot = t0 / prm->aterm_interval; m.x0 = x0; m.y0 = y0; m.w_index = wi0;
            m.reserved = 0;
            out[count] = m;
          }
          ++count; planned += nvis;
        } else {
          skipped += nvis;   /* subgrid would leave the grid: skipped and counted */
        }
        t0 = t1;
      }
      c0 += n;
    }
  }
  free(scale);
  if (n_planned_vis) *n_planned_vis = planned;
  if (n_skipped_vis) *n_skipped_vis = skipped;
  return count;
}

/* Pixel direction cosines of the N x N subgrid image (R1: Eq. 5 PAPER.md:77 applied to
 * the subgrid, l_i = (i - N/2) S/N, same in both directions) and n' = sqrt(1-l^2-m^2) - 1
 * (R2), evaluated as -r^2/(1+sqrt(1-r^2)) to keep all digits. */
static double pix_l(int32_t i, int32_t N, double S) { return (double)(i - N / 2) * S / (double)N; }
static double pix_n(double l, double m) {
  const double r2 = l * l + m * m;
  return -r2 / (1.0 + sqrt(1.0 - r2));
}

/* Subgrid centre in wavelengths (R3: centre pixel = corner + N/2, the DC pixel of the
 * centred DFT; grid cell = 1/S) and w offset (R4). */
static void subgrid_offsets(const oracle_params *prm, const oracle_meta *m, double *u0,
                            double *v0, double *w0) {
  const int32_t N = prm->subgrid_size, L = prm->grid_size;
  *u0 = (double)(m->x0 + N / 2 - L / 2) / prm->image_size;
  *v0 = (double)(m->y0 + N / 2 - L / 2) / prm->image_size;
  *w0 = prm->w_step > 0.0 ? ((double)m->w_index + 0.5) * prm->w_step : 0.0;
}

/* 2x2 products, row-major [xx xy yx yy] */
static void mat_mul(const cplx a[4], const cplx b[4], cplx r[4]) {
  r[0] = a[0] * b[0] + a[1] * b[2];
  r[1] = a[0] * b[1] + a[1] * b[3];
  r[2] = a[2] * b[0] + a[3] * b[2];
  r[3] = a[2] * b[1] + a[3] * b[3];
}
static void mat_herm(const cplx a[4], cplx r[4]) {
  r[0] = conj(a[0]); r[1] = conj(a[2]); r[2] = conj(a[1]); r[3] = conj(a[3]);
}
static void load_jones(const float *aterms, int32_t n_stations, int32_t N, int32_t slot,
                       int32_t station, int32_t y, int32_t x, cplx a[4]) {
  const float *p = aterms + ((((size_t)slot * n_stations + station) * N + y) * N + x) * 8;
  for (int k = 0; k < 4; ++k) a[k] = (double)p[2 * k] + I * (double)p[2 * k + 1];
}

/* ---------------------------------------------------------------------------------------
 * Gridder: Eq. 25 / Alg. 1 inner loops in the
 * polarised form of section 3.4:
 *   P[y][x] = sum_{t,c} Y[b][t][c] exp(+2 pi i (du l_x + dv m_y + dw n'_xy))
 *   Sg[y][x] = taper[y][x] A1[y][x]^H P[y][x] A2[y][x]                  (R5; c*_pk in Alg. 1)
 * with du = u_t f_c/c0 - u0 etc.  Output: subgrid images [P][4][N][N] complex128.
 * ------------------------------------------------------------------------------------- */
void oracle_gridder(const oracle_params *prm, const oracle_meta *meta, int64_t P,
                    const float *uvw, const double *freqs, const float *vis /*[B][T][C][4] c64*/,
                    const float *aterms, const float *taper, int32_t T, int32_t C,
                    int32_t n_stations, double *subgrids_out) {
  const int32_t N = prm->subgrid_size;
  const double S = prm->image_size;
#pragma omp parallel for schedule(dynamic, 1)
  for (int64_t p = 0; p < P; ++p) {
    const oracle_meta *m = &meta[p];
    double u0, v0, w0;
    subgrid_offsets(prm, m, &u0, &v0, &w0);
    cplx *sg = (cplx *)subgrids_out + (size_t)p * 4 * N * N;
    for (int32_t y = 0; y < N; ++y) {
      for (int32_t x = 0; x < N; ++x) {
        const double l = pix_l(x, N, S), mm = pix_l(y, N, S), n = pix_n(l, mm);
        if (prm->flags & ORACLE_SPAN_ATERMS) {
          /* per-sample c_pk (section 3.4, Alg. 1: c*_pk sits INSIDE the k-sum):
           * Sg = taper sum_k A1_k^H (Y_k phasor_k) A2_k with A_k the Jones matrices of the slot of timestep k */
          cplx tot[4] = {0, 0, 0, 0};
          for (int32_t t = m->time_begin; t < m->time_begin + m->n_time; ++t) {
            const float *uvw_t = uvw + ((size_t)m->baseline * T + t) * 3;
            cplx a1[4], a2[4], a1h[4];
            load_jones(aterms, n_stations, N, t / prm->aterm_interval, m->station1, y, x, a1);
            load_jones(aterms, n_stations, N, t / prm->aterm_interval, m->station2, y, x, a2);
            mat_herm(a1, a1h);
            for (int32_t c = m->chan_begin; c < m->chan_begin + m->n_chan; ++c) {
              const double k = freqs[c] / ORACLE_C0;
              const double du = (double)uvw_t[0] * k - u0;
              const double dv = (double)uvw_t[1] * k - v0;
              const double dw = (double)uvw_t[2] * k - w0;
              const double phase = ORACLE_TWO_PI * (du * l + dv * mm + dw * n);
              const cplx phasor = cos(phase) + I * sin(phase);
              const float *y4 = vis + (((size_t)m->baseline * T + t) * C + c) * 8;
              cplx yk[4], tmp[4], res[4];
              for (int k4 = 0; k4 < 4; ++k4) yk[k4] = ((double)y4[2 * k4] + I * (double)y4[2 * k4 + 1]) * phasor;
              mat_mul(a1h, yk, tmp);
              mat_mul(tmp, a2, res);
              for (int k4 = 0; k4 < 4; ++k4) tot[k4] += res[k4];
            }
          }
          const double tp = (double)taper[(size_t)y * N + x];
          for (int k4 = 0; k4 < 4; ++k4) sg[((size_t)k4 * N + y) * N + x] = tp * tot[k4];
          continue;
        }
        cplx acc[4] = {0, 0, 0, 0};
        for (int32_t t = m->time_begin; t < m->time_begin + m->n_time; ++t) {
          const float *uvw_t = uvw + ((size_t)m->baseline * T + t) * 3;
          for (int32_t c = m->chan_begin; c < m->chan_begin + m->n_chan; ++c) {
            const double k = freqs[c] / ORACLE_C0;
            const double du = (double)uvw_t[0] * k - u0;
            const double dv = (double)uvw_t[1] * k - v0;
            const double dw = (double)uvw_t[2] * k - w0;
            const double phase = ORACLE_TWO_PI * (du * l + dv * mm + dw * n);
            const cplx phasor = cos(phase) + I * sin(phase);
            const float *y4 = vis + (((size_t)m->baseline * T + t) * C + c) * 8;
            for (int k4 = 0; k4 < 4; ++k4)
              acc[k4] += ((double)y4[2 * k4] + I * (double)y4[2 * k4 + 1]) * phasor;
          }
        }
        cplx a1[4], a2[4], a1h[4], tmp[4], res[4];
        load_jones(aterms, n_stations, N, m->aterm_slot, m->station1, y, x, a1);
        load_jones(aterms, n_stations, N, m->aterm_slot, m->station2, y, x, a2);
        mat_herm(a1, a1h);
        mat_mul(a1h, acc, tmp);
        mat_mul(tmp, a2, res);
        const double tp = (double)taper[(size_t)y * N + x];
        for (int k4 = 0; k4 < 4; ++k4) sg[((size_t)k4 * N + y) * N + x] = tp * res[k4];
      }
    }
  }
}

/* ---------------------------------------------------------------------------------------
 * Subgrid FFT / IFFT ("V_p <- FFT(I_p)" PAPER.md:298-299; "I_p <- IFFT(V_p)"
 * PAPER.md:331-332).  Reading R6: forward has exp(-...), both sides centred at index
 * N/2, scale 1/N^2 in BOTH directions:
 *   out[b][a] = (1/N^2) sum_{j,i} in[j][i] exp(sign 2 pi i ((a-N/2)(i-N/2)+(b-N/2)(j-N/2))/N)
 * sign = -1 forward, +1 inverse.  The 2-D sum is evaluated one axis after the other (the
 * exponential of the sum factorises); each 1-D transform is the plain O(N^2) definition.
 * In place on [P][4][N][N] complex128.
 * ------------------------------------------------------------------------------------- */
void oracle_subgrid_fft(double *subgrids, int64_t P, int32_t N, int32_t sign) {
  cplx *w = (cplx *)malloc(sizeof(cplx) * (size_t)N * N);
  for (int32_t a = 0; a < N; ++a)
    for (int32_t i = 0; i < N; ++i) {
      /* reduce the integer product mod N before the division: exact argument */
      int64_t prod = (int64_t)(a - N / 2) * (int64_t)(i - N / 2);
      int64_t r = ((prod % N) + N) % N;
      const double ang = (double)sign * ORACLE_TWO_PI * (double)r / (double)N;
      w[(size_t)a * N + i] = cos(ang) + I * sin(ang);
    }
  const double scale = 1.0 / ((double)N * (double)N);
#pragma omp parallel for schedule(static)
  for (int64_t q = 0; q < P * 4; ++q) {
    cplx *s = (cplx *)subgrids + (size_t)q * N * N;
    cplx *tmp = (cplx *)malloc(sizeof(cplx) * (size_t)N * N);
    for (int32_t j = 0; j < N; ++j)        /* along x: tmp[j][a] = sum_i s[j][i] w[a][i] */
      for (int32_t a = 0; a < N; ++a) {
        cplx acc = 0;
        for (int32_t i = 0; i < N; ++i) acc += s[(size_t)j * N + i] * w[(size_t)a * N + i];
        tmp[(size_t)j * N + a] = acc;
      }
    for (int32_t b = 0; b < N; ++b)        /* along y: s[b][a] = sum_j tmp[j][a] w[b][j] */
      for (int32_t a = 0; a < N; ++a) {
        cplx acc = 0;
        for (int32_t j = 0; j < N; ++j) acc += tmp[(size_t)j * N + a] * w[(size_t)b * N + j];
        s[(size_t)b * N + a] = scale * acc;
      }
    free(tmp);
  }
  free(w);
}

/* ---------------------------------------------------------------------------------------
 * Adder (Eq. 24; Alg. 1; R7):
 *   grid[pol][y0+b][x0+a] += V_p[pol][b][a], no phase factor, no shift.  Accumulates.
 * grid: [4][L][L] complex128.
 * ------------------------------------------------------------------------------------- */
void oracle_adder(const oracle_meta *meta, int64_t P, const double *subgrids, int32_t N,
                  int32_t L, double *grid) {
#pragma omp parallel for schedule(static)
  for (int32_t pol = 0; pol < 4; ++pol) {
    cplx *g = (cplx *)grid + (size_t)pol * L * L;
    for (int64_t p = 0; p < P; ++p) {
      const cplx *s = (const cplx *)subgrids + ((size_t)p * 4 + pol) * N * N;
      for (int32_t b = 0; b < N; ++b)
        for (int32_t a = 0; a < N; ++a)
          g[(size_t)(meta[p].y0 + b) * L + (meta[p].x0 + a)] += s[(size_t)b * N + a];
    }
  }
}

/* Splitter (Alg. 2): V_p[pol][b][a] = grid[pol][y0+b][x0+a]. */
void oracle_splitter(const oracle_meta *meta, int64_t P, const double *grid, int32_t N, int32_t L,
                     double *subgrids) {
#pragma omp parallel for schedule(static)
  for (int64_t p = 0; p < P; ++p)
    for (int32_t pol = 0; pol < 4; ++pol) {
      const cplx *g = (const cplx *)grid + (size_t)pol * L * L;
      cplx *s = (cplx *)subgrids + ((size_t)p * 4 + pol) * N * N;
      for (int32_t b = 0; b < N; ++b)
        for (int32_t a = 0; a < N; ++a)
          s[(size_t)b * N + a] = g[(size_t)(meta[p].y0 + b) * L + (meta[p].x0 + a)];
    }
}

/* ---------------------------------------------------------------------------------------
 * Degridder: Alg. 2 inner loops (R9: I[i,j] there means I_p[i,j]),
 * polarised form, the exact adjoint of oracle_gridder:
 *   Dg[y][x] = A1[y][x] (taper[y][x] Ip[y][x]) A2[y][x]^H                 (R5; c_pk in Alg. 2)
 *   Y[b][t][c] = sum_{y,x} Dg[y][x] exp(-2 pi i (du l_x + dv m_y + dw n'_xy))
 * Input: subgrid images [P][4][N][N] complex128; output vis_out [B][T][C][4] complex128,
 * only the samples the plan covers are written.
 * ------------------------------------------------------------------------------------- */
void oracle_degridder(const oracle_params *prm, const oracle_meta *meta, int64_t P,
                      const float *uvw, const double *freqs, const double *subgrids,
                      const float *aterms, const float *taper, int32_t T, int32_t C,
                      int32_t n_stations, double *vis_out) {
  const int32_t N = prm->subgrid_size;
  const double S = prm->image_size;
#pragma omp parallel for schedule(dynamic, 1)
  for (int64_t p = 0; p < P; ++p) {
    const oracle_meta *m = &meta[p];
    double u0, v0, w0;
    subgrid_offsets(prm, m, &u0, &v0, &w0);
    const cplx *sg = (const cplx *)subgrids + (size_t)p * 4 * N * N;
    cplx *dg = (cplx *)malloc(sizeof(cplx) * 4 * (size_t)N * N);
    for (int32_t y = 0; y < N; ++y)
      for (int32_t x = 0; x < N; ++x) {
        cplx a1[4], a2[4], a2h[4], pix[4], tmp[4], res[4];
        load_jones(aterms, n_stations, N, m->aterm_slot, m->station1, y, x, a1);
        load_jones(aterms, n_stations, N, m->aterm_slot, m->station2, y, x, a2);
        const double tp = (double)taper[(size_t)y * N + x];
        for (int k4 = 0; k4 < 4; ++k4) pix[k4] = tp * sg[((size_t)k4 * N + y) * N + x];
        mat_herm(a2, a2h);
        mat_mul(a1, pix, tmp);
        mat_mul(tmp, a2h, res);
        for (int k4 = 0; k4 < 4; ++k4) dg[((size_t)k4 * N + y) * N + x] = res[k4];
      }
    for (int32_t t = m->time_begin; t < m->time_begin + m->n_time; ++t) {
      const float *uvw_t = uvw + ((size_t)m->baseline * T + t) * 3;
      if ((prm->flags & ORACLE_SPAN_ATERMS) && t / prm->aterm_interval != m->aterm_slot) {
        /* per-sample c_pk (Alg. 2): the corrected pixels of THIS timestep's slot */
        for (int32_t y = 0; y < N; ++y)
          for (int32_t x = 0; x < N; ++x) {
            cplx a1[4], a2[4], a2h[4], pix[4], tmp[4], res[4];
            load_jones(aterms, n_stations, N, t / prm->aterm_interval, m->station1, y, x, a1);
            load_jones(aterms, n_stations, N, t / prm->aterm_interval, m->station2, y, x, a2);
            const double tp = (double)taper[(size_t)y * N + x];
            for (int k4 = 0; k4 < 4; ++k4) pix[k4] = tp * sg[((size_t)k4 * N + y) * N + x];
            mat_herm(a2, a2h);
            mat_mul(a1, pix, tmp);
            mat_mul(tmp, a2h, res);
            for (int k4 = 0; k4 < 4; ++k4) dg[((size_t)k4 * N + y) * N + x] = res[k4];
          }
      }
      for (int32_t c = m->chan_begin; c < m->chan_begin + m->n_chan; ++c) {
        const double k = freqs[c] / ORACLE_C0;
        const double du = (double)uvw_t[0] * k - u0;
        const double dv = (double)uvw_t[1] * k - v0;
        const double dw = (double)uvw_t[2] * k - w0;
        cplx acc[4] = {0, 0, 0, 0};
        for (int32_t y = 0; y < N; ++y)
          for (int32_t x = 0; x < N; ++x) {
            const double l = pix_l(x, N, S), mm = pix_l(y, N, S), n = pix_n(l, mm);
            const double phase = -ORACLE_TWO_PI * (du * l + dv * mm + dw * n);
            const cplx phasor = cos(phase) + I * sin(phase);
            for (int k4 = 0; k4 < 4; ++k4) acc[k4] += dg[((size_t)k4 * N + y) * N + x] * phasor;
          }
        cplx *out = (cplx *)vis_out + (((size_t)m->baseline * T + t) * C + c) * 4;
        for (int k4 = 0; k4 < 4; ++k4) out[k4] = acc[k4];
      }
    }
    free(dg);
  }
}
