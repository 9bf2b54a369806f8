/*
 * idg_b200.h -- C ABI of the B200-native Image Domain Gridding hot path.
 *
 * Method: van der Tol, Veenboer & Offringa, "Image Domain Gridding: a fast method for
 * convolutional resampling of visibilities", arXiv 1909.07226.  Citations are lines of
 * /root/reference/PAPER.md plus the section / equation / algorithm they fall in; "R<n>"
 * names a reading of a garbled or silent passage listed in DESIGN.md.
 *
 * Conventions shared by every entry point
 *   - Every function returns int: IDG_OK (0) or a negative idg_status.  No exceptions, no
 *     aborts, nothing printed.  idg_strerror() names a code; idg_last_cuda_error() returns the
 *     cudaError_t behind the last IDG_ERR_CUDA of the calling thread.
 *   - "_dev" pointers are CUDA device pointers owned by the caller; "_host" pointers are host
 *     memory owned by the caller.  The library never frees or keeps caller memory beyond the
 *     call (asynchronous work on `cuda_stream` excepted: buffers must stay valid until the
 *     stream has run it).  `cuda_stream` is a cudaStream_t passed as void* (NULL = default).
 *   - idg_grid / idg_degrid and the stage entry points are asynchronous on `cuda_stream` and
 *     never synchronise it; idg_plan_create and the *_host entry points synchronise.
 *   - Layouts (C order, complex64 = two float32, re then im):
 *       uvw      [B][T][3]                 float32 metres (u, v, w)
 *       vis      [B][T][C][4]              complex64, polarisations XX, XY, YX, YY (row-major 2x2)
 *       aterms   [slots][stations][N][N][4] complex64 Jones matrices, pixel [y][x], row-major 2x2
 *       taper    [N][N]                    float32, pixel [y][x]
 *       subgrids [P][4][N][N]              complex64, [pol][y][x]
 *       grid     [4][L][L]                 complex64, [pol][y][x]; x <-> u <-> l fastest
 *   - A "visibility" is one (baseline, timestep, channel) sample with all four polarisations
 *     (section 5.3).
 */
#ifndef IDG_B200_H
#define IDG_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  IDG_OK = 0,
  IDG_ERR_INVALID_ARG = -1,
  IDG_ERR_OUT_OF_MEMORY = -2,
  IDG_ERR_CUDA = -3,
  IDG_ERR_PLAN_MISMATCH = -4,
  IDG_ERR_UNSUPPORTED_SUBGRID_SIZE = -5,
  IDG_ERR_SCRATCH_TOO_SMALL = -6 /* a *_static entry point was asked for more than its fixed scratch holds */
} idg_status;

#define IDG_PLAN_FORCE_BLOCKS 1 /* flags: blocks end only on max_timesteps / A-term slot (sweep mode) */
#define IDG_PLAN_SPAN_ATERMS 2  /* flags (NEXT-4): a block may span A-term slots; the slot of timestep t is
                                   t / aterm_interval and c_pk varies inside the visibility loop (section 3.4,
                                   PAPER.md:247; Alg. 1); meta.aterm_slot = slot of the first timestep */

#define IDG_PLAN_FP32_GRIDDER 4 /* flags: rows a1 and a6 always run the FP32 kernels.  Without it, plans with N = 32 and
                                   per-block A-terms run Eq. 25 (8..128 channels per block, >= 128 visibilities per block
                                   on average) and Alg. 2's inner loops (>= 384 visibilities per block on average) on the
                                   tensor cores with 22-bit (fp16 hi + lo) operands and FP32 accumulation: ~8e-6 relative
                                   L2 against float64 instead of ~1e-6 (idg_plan_uses_tensor_cores: bit 0 gridder, bit 1
                                   degridder) */

/* Partitioning parameters (section 3.2; readings R10-R12).  All explicit. */
typedef struct {
  int32_t grid_size;      /* L, even, >= subgrid_size */
  int32_t subgrid_size;   /* N in {16, 24, 32, 48} */
  int32_t kernel_size;    /* pixels reserved for taper / w / A-term support, 0 < kernel_size < N */
  int32_t max_timesteps;  /* per subgrid, >= 1 */
  int32_t max_channels;   /* per subgrid, power of two */
  int32_t aterm_interval; /* timesteps per A-term slot, >= 1 (R5: a block never spans two slots) */
  int32_t flags;          /* IDG_PLAN_FORCE_BLOCKS | IDG_PLAN_SPAN_ATERMS | IDG_PLAN_FP32_GRIDDER or 0 */
  int32_t reserved;       /* must be 0 */
  double image_size;      /* S: direction-cosine extent of the image; grid cell = 1/S wavelengths */
  double w_step;          /* w-layer thickness in wavelengths; 0 -> w0 = 0 for every subgrid (R4) */
} idg_plan_params;

/* One subgrid of the partition: 48 bytes, the bit-exact contract (Alg. 1
 * PAPER.md:276; D6 of SURVEY.md).  Centre pixel of the subgrid on the grid = (x0 + N/2, y0 + N/2);
 * u0 = (x0 + N/2 - L/2)/S (R3); w0 = (w_index + 0.5) w_step (R4). */
typedef struct {
  int32_t baseline, station1, station2, time_begin, n_time, chan_begin, n_chan, aterm_slot, x0, y0,
      w_index, reserved;
} idg_subgrid_meta;

typedef struct idg_plan idg_plan; /* opaque; owns metadata (host + device), adder work lists,
                                     the [P][4][N][N] subgrid scratch buffer and staging buffers */

/* Re-entrancy: idg_grid, idg_degrid, the *_scalar and the *_host calls WRITE the plan-owned subgrid scratch
 * (and the *_host calls the plan's staging buffers, copy stream and events) although the compute calls take a
 * `const idg_plan *`: two such calls on ONE plan must be ordered on one stream (or by events); concurrent calls on
 * one plan from two streams or two threads race.  Calls on different plans are independent.  The stage entry
 * points touch only the buffers they are given.
 * Alignment: vis, aterms, subgrids and vis_out are read / written as 16-byte vectors and must be 16-byte aligned
 * (IDG_ERR_INVALID_ARG otherwise); grid, uvw and taper need only the alignment of their element type.
 * A-term slots: every compute call takes n_slots, the first extent of the aterms (gains) array it is given; a plan
 * that indexes a slot >= n_slots is refused with IDG_ERR_PLAN_MISMATCH before anything is launched. */

const char *idg_strerror(int code);
int idg_last_cuda_error(void);
/* Number of CUDA kernels this library has launched in the process so far (all entry points, all threads);
 * the difference of two readings counts the launches in between.  Host-side bookkeeping only, never fails. */
long long idg_kernel_launches(void);

/* Measurement aid for the op-count roofline: runs the bare instruction mix of one
 * (visibility, pixel) pair of Eq. 25 -- 1 FMA + sin/cos.approx + 16 FMA as packed pairs -- on
 * registers and shared memory only, in the gridder's CTA shape, `iters` pairs per pixel, and returns the rate in
 * TFLOP-equivalents/s (36 per pair, the unit of bench.py's roofline).  variant 0: operands as in the gridder
 * (visibility pairs in vector registers, loaded from shared memory); 1: visibility pairs in uniform registers (an
 * upper bound the real kernel cannot reach from CUDA C); 2: 16 scalar FMA instead of 8 packed ones.
 * Synchronises cuda_stream; allocates and frees a small buffer. */
int idg_bench_instruction_mix(int32_t iters, int32_t variant, double *tflop_equiv_per_s, void *cuda_stream);
/* Measurement aid for the tensor-core kernels (Eq. 25 PAPER.md:230-235 and Alg. 2 PAPER.md:333-345 as contractions):
 * the issue rate of tcgen05.mma.cta_group::1.kind::f16 with M = 128, K = 16, N = n in {16, 64, 128, 256}, A operand in
 * tensor memory, B operand in shared memory -- the form csrc/gridder_tc.cu and csrc/degridder_tc.cu use with N = 16.
 * ctas_per_sm CTAs (1..4 for n <= 64, 1..2 for n = 128, 1 for n = 256) each issue n_mma MMAs (a multiple of 8) back
 * to back; the result is SM cycles per MMA, per SM.  Synchronises cuda_stream; allocates and frees a small buffer.
 * Errors: IDG_ERR_INVALID_ARG, IDG_ERR_CUDA. */
int idg_bench_mma_rate(int32_t n, int32_t ctas_per_sm, int32_t n_mma, double *cycles_per_mma_per_sm,
                       void *cuda_stream);

/* ---- planner (a0): section 3.2, Fig. 2; readings R10-R12 -----
 * Partitions every baseline's (time x channel) samples into blocks whose uv extent in grid
 * pixels plus kernel_size fits N, with one A-term slot and one w layer per block.  Runs on the
 * GPU (one walk per baseline, count -> scan -> emit), double arithmetic without FMA contraction;
 * the metadata is bit-identical to the step-by-step rule in DESIGN.md.  Synchronises the stream.
 *   uvw_dev        [B][T][3] float32 metres, device
 *   freqs_host     [C] float64 Hz, host (copied)
 *   baselines_host [B][2] int32 station pairs, host (copied)
 * Samples whose subgrid would leave the grid are skipped and counted, not an error.
 * Errors: IDG_ERR_INVALID_ARG (null pointers, bad params), IDG_ERR_UNSUPPORTED_SUBGRID_SIZE,
 * IDG_ERR_OUT_OF_MEMORY, IDG_ERR_CUDA.  *out is NULL on error. */
int idg_plan_create(idg_plan **out, const idg_plan_params *prm, const float *uvw_dev,
                    const double *freqs_host, const int32_t *baselines_host, int32_t B, int32_t T,
                    int32_t C, int32_t n_stations, void *cuda_stream);
/* Builds a plan from caller-supplied metadata (host, P entries; validated against the grid and
 * the array shapes) instead of running the planner: for tests and for externally made plans. */
int idg_plan_from_metadata(idg_plan **out, const idg_plan_params *prm,
                           const idg_subgrid_meta *meta_host, int64_t P, const double *freqs_host,
                           int32_t B, int32_t T, int32_t C, int32_t n_stations, void *cuda_stream);
int idg_plan_size(const idg_plan *plan, int64_t *n_subgrids, int64_t *n_planned_vis,
                  int64_t *n_skipped_vis);
/* Copies min(P, capacity) entries to out_host; IDG_ERR_INVALID_ARG if capacity < P. */
int idg_plan_metadata(const idg_plan *plan, idg_subgrid_meta *out_host, int64_t capacity);
/* Device pointer of the plan-owned [P][4][N][N] complex64 scratch (valid until destroy). */
int idg_plan_subgrids(const idg_plan *plan, void **subgrids_dev);
/* Number of A-term slots the plan indexes: max over subgrids of the last slot + 1 (with IDG_PLAN_SPAN_ATERMS the
 * slot of a block's last timestep decides); 0 for an empty plan. */
int idg_plan_aterm_slots(const idg_plan *plan, int32_t *n_slots);
/* Which of the plan's two contractions run on the tensor cores, as a bit mask: bit 0 (value 1) idg_gridder / idg_grid
 * (csrc/gridder_tc.cu: N = 32, one c_p per block, 8 to 128 channels in every block, mean block of 128 visibilities or
 * more), bit 1 (value 2) idg_degridder / idg_degrid (csrc/degridder_tc.cu: N = 32, one c_p per block, mean block of 384
 * visibilities or more); 0: both on the FP32 path (always with IDG_PLAN_FP32_GRIDDER). */
int idg_plan_uses_tensor_cores(const idg_plan *plan, int32_t *flag);
/* w offset of a w layer, w0 = (w_index + 0.5) w_step, or 0 when w_step = 0 (Alg. 1, R4). */
int idg_plan_w_offset(const idg_plan *plan, int32_t w_index, double *w0);
void idg_plan_destroy(idg_plan *plan);

/* ---- Algorithm 1 without its last line: gridder -> subgrid FFT -> adder.
 * ACCUMULATES into grid_dev (Alg. 1 zeroes V once; zeroing is the caller's). */
int idg_grid(const idg_plan *plan, const float *uvw_dev, const void *vis_dev,
             const void *aterms_dev, int32_t n_slots, const float *taper_dev, void *grid_dev, void *cuda_stream);
/* ---- Algorithm 2 after its first two lines: splitter -> subgrid IFFT ->
 * degridder.  Overwrites every planned visibility; skipped ones are set to 0. */
int idg_degrid(const idg_plan *plan, const float *uvw_dev, const void *grid_dev,
               const void *aterms_dev, int32_t n_slots, const float *taper_dev, void *vis_out_dev,
               void *cuda_stream);

/* ---- the same two calls on HOST buffers (pinned or pageable): copy in, run, copy out,
 * synchronise.  Device staging buffers are owned by the plan (allocated on first use).
 * idg_grid_host adds into grid_host (which is read, accumulated into on the device, and
 * written back). */
int idg_grid_host(idg_plan *plan, const float *uvw_host, const void *vis_host,
                  const void *aterms_host, int32_t n_slots, const float *taper_host,
                  void *grid_host, void *cuda_stream);
int idg_degrid_host(idg_plan *plan, const float *uvw_host, const void *grid_host,
                    const void *aterms_host, int32_t n_slots, const float *taper_host,
                    void *vis_out_host, void *cuda_stream);

/* ---- one imaging cycle on HOST buffers with the grid resident on the device: Alg. 1 of
 * vis_host into a ZEROED device grid, then Alg. 2 from that grid into vis_out_host.
 *   grid_host     [4][L][L] complex64, host, OPTIONAL (NULL: the grid is not copied back): receives the grid
 *                 (overwritten, not accumulated into)
 *   vis_out_host  [B][T][C][4] complex64, host: the predicted visibilities (skipped ones 0); may alias vis_host
 * Inputs are uploaded once, the copies overlap the kernels in both directions; synchronises like the other
 * *_host calls; same error behaviour. */
int idg_grid_degrid_host(idg_plan *plan, const float *uvw_host, const void *vis_host,
                         const void *aterms_host, int32_t n_slots, const float *taper_host,
                         void *grid_host, void *vis_out_host, void *cuda_stream);

/* ---- stage-level entry points (parity tests, per-stage timing); same conventions ------------
 * a1 gridder: Eq. 25, Alg. 1, section 3.4 PAPER.md:247-249:
 *   Sg[y][x] = taper A1^H (sum_k Y_k exp(+2 pi i (du l_x + dv m_y + dw n'_xy))) A2  -> subgrids */
int idg_gridder(const idg_plan *plan, const float *uvw_dev, const void *vis_dev,
                const void *aterms_dev, int32_t n_slots, const float *taper_dev, void *subgrids_dev,
                void *cuda_stream);
/* a2 / a5 subgrid FFT: centred 2-D DFT of every plane in place, scale 1/N^2 both ways (R6);
 * direction -1 = forward exp(-..), +1 = inverse. */
int idg_subgrid_fft(const idg_plan *plan, void *subgrids_dev, int32_t direction,
                    void *cuda_stream);
/* a3 adder: grid[pol][y0+b][x0+a] += V_p[pol][b][a] (Eq. 24). */
int idg_adder(const idg_plan *plan, const void *subgrids_dev, void *grid_dev, void *cuda_stream);
/* a4 splitter: V_p[pol][b][a] = grid[pol][y0+b][x0+a]. */
int idg_splitter(const idg_plan *plan, const void *grid_dev, void *subgrids_dev,
                 void *cuda_stream);
/* a4 + a5 in one kernel (what idg_degrid runs): the inverse subgrid FFT gathers its input from the grid window
 * instead of reading the splitter's copy, I_p = IFFT(V[pol][y0..y0+N)[x0..x0+N)).  Bit-identical
 * to idg_splitter followed by idg_subgrid_fft(+1); subgrids_dev [P][4][N][N] is written, grid_dev only read. */
int idg_splitter_ifft(const idg_plan *plan, const void *grid_dev, void *subgrids_dev,
                      void *cuda_stream);
/* a6 degridder: Alg. 2: Dg = A1 (taper Ip) A2^H per pixel, then
 *   Y_k = sum_xy Dg[y][x] exp(-2 pi i (du l_x + dv m_y + dw n'_xy)) -> vis_out (planned only). */
int idg_degridder(const idg_plan *plan, const float *uvw_dev, const void *subgrids_dev,
                  const void *aterms_dev, int32_t n_slots, const float *taper_dev, void *vis_out_dev,
                  void *cuda_stream);

/* ---- image-plane side of W-stacking (OUTSIDE the timed hot path) --------------
 * Alg. 1 last line "I <- FFT(V) / c-bar" (R8) and Alg. 2 first lines with the
 * per-subgrid w offset w0 = (w_index + 0.5) w_step (R4) resolved by W-stacking:
 * one grid per w layer; its image lacks exp(+2 pi i w0 n'(l, m)), l_x = (x - L/2) S / L (Eq. 5),
 * n' = sqrt(1 - l^2 - m^2) - 1 (R2).  The large FFT is the caller's (library).  Images are [4][L][L] complex64,
 * device; asynchronous on cuda_stream.  sign = +1 imaging, -1 prediction.
 *   idg_image_w_accumulate: acc += layer * exp(sign 2 pi i w0 n')
 *   idg_image_w_apply:      out  = in    * exp(sign 2 pi i w0 n')   (out may alias in)
 *   idg_image_divide:       image[pol][y][x] /= cbar[y][x], cbar [L][L] float32 (the image-domain taper c-bar)
 *   idg_image_taper:        c-bar itself from the subgrid taper (below)
 * Errors: IDG_ERR_INVALID_ARG, IDG_ERR_CUDA. */
int idg_image_w_accumulate(void *acc_dev, const void *layer_dev, int32_t L, double image_size, double w0,
                           int32_t sign, void *cuda_stream);
int idg_image_w_apply(void *out_dev, const void *in_dev, int32_t L, double image_size, double w0, int32_t sign,
                      void *cuda_stream);
int idg_image_divide(void *image_dev, const float *cbar_dev, int32_t L, void *cuda_stream);
/* c-bar, the image-domain taper that Alg. 1's last line divides by ("rms image domain kernel",
 * PAPER.md:278): the [N][N] subgrid taper carried to the L x L image raster by the interpolation the method itself
 * performs, section 4.2 ("the effective window is a sinc interpolation of the discrete window"): the
 * periodic (Dirichlet-kernel) interpolation of the N samples at l_i = (i - N/2) S/N onto l_x = (x - L/2) S/L, both
 * axes, real part.  FP64 arithmetic, float32 result.  taper_dev [N][N] float32, cbar_dev [L][L] float32, N in
 * {16, 24, 32, 48}, L >= N even.  Asynchronous on cuda_stream; allocates (and frees, stream-ordered) 32 L N bytes. */
int idg_image_taper(const float *taper_dev, int32_t N, float *cbar_dev, int32_t L, void *cuda_stream);
/* The same result without any allocation, for callers that cannot call cudaMalloc (CUDA graph capture, serving
 * loops): the 32 L N bytes of scratch live in a file-scope device array of the library, 8 MiB that every GPU which
 * loads the library holds until exit.  Arguments, arithmetic and result as idg_image_taper (same kernels).
 *   limit:   L * N <= IDG_IMAGE_TAPER_STATIC_MAX_LN (L <= 8192 at N = 32, L <= 5460 at N = 48); larger requests
 *            return IDG_ERR_SCRATCH_TOO_SMALL before anything is launched -- use idg_image_taper for those
 *   device:  the current device must be the one cuda_stream belongs to; the first call on each device resolves the
 *            array's device address (cudaGetSymbolAddress: no allocation) -- make that call outside stream capture
 *   sharing: every call on a device uses the SAME array, which keeps the previous call's contents (each call
 *            overwrites what it reads, nothing needs clearing); two calls that overlap on the GPU -- different
 *            streams, or captured into graphs that run concurrently -- race on it.  Calls on one stream are ordered.
 * Calls no cudaMalloc / cudaFree / allocating library routine.  Errors: IDG_ERR_INVALID_ARG,
 * IDG_ERR_SCRATCH_TOO_SMALL, IDG_ERR_CUDA. */
#define IDG_IMAGE_TAPER_STATIC_MAX_LN 262144
int idg_image_taper_static(const float *taper_dev, int32_t N, float *cbar_dev, int32_t L, void *cuda_stream);

/* ---- optimal taper (offline input of the hot path) ----------------------------------
 * Section 4.3, Appendix A: the taper c[i][j] = a_i a_j (Eq. 30) whose effective
 * window has the least side-lobe energy, averaged over the sample shifts |s| <= (N - beta + 1)/2 a kernel budget of
 * beta pixels allows: a = eigenvector of the smallest eigenvalue of R-bar = Q-bar (.) S-bar (Eq. 36-37, A.3-A.8),
 * minimised over a_1 .. a_{N-1} with a_0 = 0 so that the window is symmetric about the centre pixel N/2 (reading R16;
 * this reproduces Table 1).  beta plays the role of idg_plan_params.kernel_size.
 *   taper_dev     [N][N] float32, device, written: a_i a_j scaled to 1 at the centre pixel
 *   a_host        [N] float64, host, optional: the coefficients (a_host[N/2] = 1, a_host[0] = 0)
 *   epsilon_host  optional: the aliasing level sqrt(lambda_min) of Table 1; FP64 resolves it down to ~1e-7, below
 *                 that the window is still near-optimal but the value returned is not reliable
 * N even, 4 <= N <= 64 (every subgrid size of the library and every column of Table 1); 1 <= beta < N.
 * Runs one FP64 CTA on cuda_stream and synchronises it.  Errors: IDG_ERR_INVALID_ARG, IDG_ERR_CUDA. */
int idg_taper_optimal(int32_t N, double beta, float *taper_dev, double *a_host, double *epsilon_host,
                      void *cuda_stream);

/* ---- scalar variant: one polarisation ------------------------------------------
 * The method as the paper derives it before the 2x2 substitution (Eq. 1-25);
 * "Stokes I only" is how the classical gridder is timed in PAPER.md:481.  Complex gains g (Eq. 2):
 *   gridding   Sg = taper conj(g1) (sum_k Y_k exp(+i phase)) g2 ;  degridding  Y_k = sum_xy g1 (taper Ip) conj(g2) exp(-i phase)
 * = the XX plane of the 4-polarisation calls with Jones matrices g I_2.  Same plan object, same conventions.
 *   vis / vis_out [B][T][C] complex64, gains [slots][stations][N][N] complex64, grid [L][L] complex64,
 *   subgrids [P][N][N] complex64 (idg_grid_scalar / idg_degrid_scalar use the plan's scratch). */
int idg_grid_scalar(const idg_plan *plan, const float *uvw_dev, const void *vis_dev, const void *gains_dev, int32_t n_slots,
                    const float *taper_dev, void *grid_dev, void *cuda_stream);
int idg_degrid_scalar(const idg_plan *plan, const float *uvw_dev, const void *grid_dev, const void *gains_dev, int32_t n_slots,
                      const float *taper_dev, void *vis_out_dev, void *cuda_stream);
int idg_gridder_scalar(const idg_plan *plan, const float *uvw_dev, const void *vis_dev, const void *gains_dev, int32_t n_slots,
                       const float *taper_dev, void *subgrids_dev, void *cuda_stream);
int idg_degridder_scalar(const idg_plan *plan, const float *uvw_dev, const void *subgrids_dev, const void *gains_dev, int32_t n_slots,
                         const float *taper_dev, void *vis_out_dev, void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* IDG_B200_H */
