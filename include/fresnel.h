/*
 * fresnel.h -- C ABI of libfresnel.so: B200-native plane-to-plane Fresnel propagation.
 *
 * The hot path of arXiv 1806.06467 (Douglas & Perrin, "Accelerated Modeling of Near and Far-Field
 * Diffraction for Coronagraphic Optical Systems"): a complex N x N wavefront multiplied by quadratic
 * phase factors (thin lenses, Fresnel chirps), 2-D forward/inverse FFTs and the angular-spectrum
 * transfer function, surface after surface (BASELINE.json:north_star).
 * Citations "PAPER.md:L" are line numbers of /root/reference/PAPER.md; "gK" are the readings listed
 * in DESIGN.md where the paper is silent or garbled.
 *
 * CONVENTIONS (all entry points)
 *   Wavefront  `wf`: DEVICE pointer, row-major [batch][N][N], interleaved (re, im) of the plan's
 *              dtype (float2 for FRESNEL_C64, double2 for FRESNEL_C128), 16-byte aligned, modified
 *              IN PLACE.  The caller owns it.  Pixel [j][k] sits at y = (j - N/2)*dx, x = (k - N/2)*dx
 *              (origin on pixel N/2: the fftshift convention of PAPER.md:123, reading g8).
 *   pixel, lambda: HOST arrays of length `batch` (metres): pixel pitch dx_b and wavelength of every
 *              batch element ("repeated for all of the wavelengths").  They are consumed
 *              before the call returns.
 *   amp, opd:  DEVICE pointers to real [N][N] maps of matching precision (float / double), shared
 *              by the whole batch; either may be NULL.  The caller owns them.
 *   Execution: every call only ENQUEUES work on the plan's CUDA stream and returns without
 *              synchronising (except fresnel_plan_synchronize and plan create/destroy).  No device
 *              memory is allocated in the hot calls: the plan owns FFT twiddles, chirp tables and
 *              per-batch scalars.  All hot calls are CUDA-graph capturable.
 *   Errors:    return codes only, never exceptions or aborts.  Argument errors (INVALID_ARG, UNSUPPORTED) are
 *              detected before anything is enqueued and leave the wavefront untouched -- for a whole train in
 *              fresnel_system_run too.  FRESNEL_ERR_CUDA / FRESNEL_ERR_ALLOC raised by a launch in the middle of
 *              a call (between the row and the column pass, or between two surfaces of a train) leave the
 *              kernels enqueued so far in the stream: the wavefront contents are then unspecified.
 *                FRESNEL_ERR_INVALID_ARG  NULL plan/wf/host array, lambda <= 0, pixel <= 0, non-finite
 *                                         z, z == 0 where a division by z is needed, f == 0 or NaN,
 *                                         bad direction
 *                FRESNEL_ERR_UNSUPPORTED  grid size outside the supported set (see fresnel_plan_create), bad dtype
 *                FRESNEL_ERR_ALLOC        device/host allocation failed (plan create, fresnel_plan_reserve_tables),
 *                                         or a call needs more chirp-table slots than are free (all taken by
 *                                         captured graphs: see fresnel_plan_reserve_tables)
 *                FRESNEL_ERR_CUDA         a CUDA runtime call or launch failed
 *                FRESNEL_ERR_TOO_LARGE    fresnel_mft_noalloc only: the problem exceeds its fixed scratch array
 *   Threads:   a plan is not thread-safe; distinct plans are independent.  fresnel_mft_noalloc has no plan and shares
 *              one scratch array per device among all its calls (see there).
 *   There is no CPU fallback: without a CUDA device plan creation fails with FRESNEL_ERR_CUDA.
 */
#ifndef FRESNEL_H
#define FRESNEL_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct fresnel_plan fresnel_plan; /* opaque */

typedef enum { FRESNEL_C64 = 0, FRESNEL_C128 = 1 } fresnel_dtype;

typedef enum {
    FRESNEL_OK = 0,
    FRESNEL_ERR_INVALID_ARG = 1,
    FRESNEL_ERR_UNSUPPORTED = 2,
    FRESNEL_ERR_ALLOC = 3,
    FRESNEL_ERR_CUDA = 4,
    FRESNEL_ERR_TOO_LARGE = 5      /* fresnel_mft_noalloc only: the problem exceeds its fixed scratch array */
} fresnel_status;

enum { FRESNEL_FORWARD = +1, FRESNEL_INVERSE = -1 };

/* ---- plan ------------------------------------------------------------------------------------ */

/* Create a plan for `batch` wavefronts of N x N complex elements of `dtype` on the current CUDA
 * device.  Builds the FFT twiddle tables (host long double, rounded once) and allocates the chirp
 * table cache.  batch >= 1.  *out is set only on FRESNEL_OK.  Grid sizes:
 *   - powers of two in [64, 8192]: the register-resident radix-16 kernels (the fast path; all BASELINE configs);
 *   - N = 2800 ("N = 2800 ran faster than 4096") and 700, 1000, 1200, 1400, 1500, 2000, 2400, 3000, 3600,
 *     4000, 5000, 5600, 6000: a register-resident mixed-radix pass (mr_kernel.cuh; 2800 = 5 * 5 * 7 * 16); N = 2800 is
 *     faster per step than N = 4096 here too;
 *   - any other N in [16, 8192] (App. B calls WFIRSTSPC(npix=1025) at beam ratio 0.25, a 4100^2 grid):
 *     the shared-memory path of gen_kernel.cuh -- mixed radix when N = 2^a 3^b 5^c 7^d 11^e 13^f [x one prime 17..61]
 *     (1025 = 41 * 5^2, 4100 = 41 * 2^2 * 5^2), otherwise Bluestein (chirp x circular convolution of the next 7-smooth
 *     length >= 2N-1 x chirp), as long as two line buffers of the transform length fit one SM's shared memory (mixed
 *     radix N <= 6700, Bluestein N <= 3350 for both precisions; complex64 then takes 16-byte column tiles); beyond that
 *     FRESNEL_ERR_UNSUPPORTED.  Odd N: the grid
 *     centre is pixel N/2 (integer division), frequencies in FFT order are q/(N dx) for q <= (N-1)/2 and
 *     (q-N)/(N dx) above, and centred transforms carry phase ramps instead of (-1)^n signs.  Train-level fusion
 *     (fresnel_system_run) applies to power-of-two grids only. */
fresnel_status fresnel_plan_create(fresnel_plan **out, int N, int batch, fresnel_dtype dtype);

/* Stream all later calls enqueue on (a cudaStream_t passed as void*; NULL = legacy default stream).  The new
 * stream is made to wait for everything the plan has enqueued on the old one (its cached tables were built and
 * are read there); if either stream is being captured the cached tables are forgotten instead. */
fresnel_status fresnel_plan_set_stream(fresnel_plan *p, void *cuda_stream);

/* Chirp-table cache.  A plan owns a pool of 1-D table slots ([batch][N] complex each; 64 at creation) that cache
 * the lens / Fresnel chirps, transfer functions and 1/lambda arrays by value, least recently used first out.
 * fresnel_plan_reserve_tables makes sure at least n_tables slots are usable by eager calls (allocates device
 * memory: not while the stream is being captured -> FRESNEL_ERR_UNSUPPORTED).  A fused train
 * (fresnel_system_run) holds 2 tables per surface at once; longer trains than the pool allows are split.
 * CUDA graphs: tables built while the stream is being captured belong to that graph from then on -- replays
 * rewrite them, so they are never shared with eager calls nor evicted, only reused by later calls of the same
 * capture.  After destroying such graphs, fresnel_plan_release_graph_tables returns their slots to the pool
 * (replaying a graph captured before the release is then undefined). */
fresnel_status fresnel_plan_reserve_tables(fresnel_plan *p, int n_tables);
fresnel_status fresnel_plan_release_graph_tables(fresnel_plan *p);

/* Block the host until everything enqueued on the plan's stream has finished. */
fresnel_status fresnel_plan_synchronize(fresnel_plan *p);

/* Synchronises the plan's stream, frees everything the plan owns.  NULL is a no-op. */
fresnel_status fresnel_plan_destroy(fresnel_plan *p);

/* Number of kernels this plan has launched so far (bench.py reports it as gpu_launches). */
fresnel_status fresnel_plan_launch_count(const fresnel_plan *p, unsigned long long *count);

/* Profiling hook (used by bench.py to time the row and the column kernel inside the real timed
 * region): the NEXT two-pass call on this plan (fresnel_fft2d, fresnel_propagate_as,
 * fresnel_propagate_direct, fresnel_surface_as with z != 0) records events[0] before its row
 * pass, events[1] between the passes and events[2] after its column pass, on the plan's stream.
 * events: HOST array of 3 cudaEvent_t handles owned by the caller (passed as void*); NULL disarms. */
fresnel_status fresnel_plan_record_pass_events(fresnel_plan *p, void *const events[3]);

/* Profiling hooks of fresnel_system_run (used by bench.py for the per-kernel durations behind `roofline`).
 * fresnel_plan_record_train_events: the NEXT fresnel_system_run records events[k] right before its k-th pass
 * kernel and one more event after the last one (as far as n_events reaches), on the plan's stream; events are
 * cudaEvent_t handles owned by the caller; n_events = 0 disarms.  An event between two kernels switches off
 * their programmatic launch overlap, so instrumented trains run a few per cent slower.
 * fresnel_plan_last_schedule: the pass kernels the last fresnel_system_run enqueued, in order: direction
 * (0 along rows, 1 along columns), convolutions per resident line (0: a plain transform pass of direct Fresnel
 * or an optic-only pass, 1, or 2 for a fused pass), the surface whose optic the pass applied (or whose
 * propagation it finished), and the number of real N x N maps it read.  *count receives the total. */
typedef struct {
    int direction;
    int convolutions;
    int first_surface;
    int maps_read;
} fresnel_pass_info;
fresnel_status fresnel_plan_record_train_events(fresnel_plan *p, void *const *events, int n_events);
fresnel_status fresnel_plan_last_schedule(const fresnel_plan *p, fresnel_pass_info *out, int capacity, int *count);

/* ---- the operations of the hot path ----------------------------------------------------------- */

/* Quadratic phase factor, Eq. 2 read as (g1)
 *     wf[b][j][k] *= exp(+i*pi*(x_k^2 + y_j^2) / (lambda_b * z)),   x, y from pixel[b].
 * A thin lens of focal length f (PAPER.md:29 "treated as thin lenses", :239-244 QuadraticLens) is
 * z = -f (converging for f > 0, reading g2).  z == 0 or non-finite: FRESNEL_ERR_INVALID_ARG.
 * One pass over the wavefront; the chirp is applied as the outer product of one 1-D table. */
fresnel_status fresnel_apply_qpf(fresnel_plan *p, void *wf, const double *pixel, const double *lambda, double z);

/* Optic phasor, Eq. 3:  wf[b][j][k] *= amp[j][k] * exp(2*pi*i*opd[j][k]/lambda_b),
 * opd in metres, sign + (reading g3).  amp == NULL means 1, opd == NULL means 0; both NULL is a no-op. */
fresnel_status fresnel_apply_mask(fresnel_plan *p, void *wf, const void *amp, const void *opd, const double *lambda);

/* 2-D FFT (bottleneck #1).  direction = FRESNEL_FORWARD: unnormalised, kernel
 * exp(-2*pi*i*(j*p + k*q)/N);  FRESNEL_INVERSE: kernel exp(+...), scaled by 1/N^2 (reading g6).
 * centered != 0 computes fftshift(fft2(ifftshift(wf))) with zero extra memory
 * passes: for even N it equals s*fft2(s*wf), s = (-1)^(j+k), applied on load and on store. */
fresnel_status fresnel_fft2d(fresnel_plan *p, void *wf, int direction, int centered);

/* Angular-spectrum plane-to-plane propagation by z (BASELINE.json:north_star):
 *     wf <- fftshift(ifft2( fft2(ifftshift(wf)) * H )),   H = exp(-i*pi*lambda*z*(fx^2 + fy^2)),
 * fx, fy = FFT-order frequencies q/(N*dx).  No piston exp(ikz) (g5); unit gain; pixel pitch unchanged;
 * z < 0 allowed (g10); z == 0 is the identity (g11).  Because H = Hx (x) Hy is separable the
 * operator is a row convolution followed by a column convolution: TWO passes over the wavefront,
 * each doing FFT -> x H1 -> inverse FFT on chip; the shifts cancel exactly and cost nothing. */
fresnel_status fresnel_propagate_as(fresnel_plan *p, void *wf, const double *pixel, const double *lambda, double z);

/* Direct (single-FFT) Fresnel propagation by z != 0 (PAPER.md:29 "direct Fresnel", :53 pixelscale):
 *     wf <- (dx^2/(i*lambda*z)) * Q_dx'(z) * CFT( Q_dx(z) * wf ),    dx' = lambda*|z|/(N*dx),
 * Q_d(z) the chirp of fresnel_apply_qpf at pitch d, CFT the centred transform with the forward
 * kernel for z > 0 and the unnormalised inverse kernel for z < 0 (readings g7, g10).
 * pixel_inout (HOST, length batch) is read as dx and overwritten with dx' before the call returns. */
fresnel_status fresnel_propagate_direct(fresnel_plan *p, void *wf, double *pixel_inout, const double *lambda, double z);

/* One whole surface, fused ("add_optic(optic, distance=...)"):
 *     apply_qpf(z = -f)  [skipped if f is +-INFINITY]  ->  apply_mask(amp, opd)  ->  propagate_as(z)
 * in the same two passes as fresnel_propagate_as: the optic phasor and the x-chirp of the lens ride on
 * the load of the row pass, the y-chirp (one factor per row) on its store.  z == 0: optic only. */
fresnel_status fresnel_surface_as(fresnel_plan *p, void *wf, const double *pixel, const double *lambda,
                                  double f, const void *amp, const void *opd, double z);

/* A train of surfaces in one call (add_optic(optic, distance=...) repeated; SURVEY.md
 * sec. 8(f) NEXT-1, reduced).  Surface s = thin lens f (+-INFINITY: none), optic phasor (amp, opd; NULL: none),
 * then propagation by z with `method`:
 *     FRESNEL_METHOD_AS      angular spectrum (fresnel_surface_as): pixel pitch kept;
 *     FRESNEL_METHOD_DIRECT  direct Fresnel: pixel pitch becomes lambda*|z|/(N*dx); the lens chirp is merged
 *                            into the propagator's input chirp and the phasor rides on the row pass, so the
 *                            surface still costs two passes;
 *     FRESNEL_METHOD_AUTO    POPPY chooses from a Gaussian pilot beam (Lawrence Eq. 82-89), which the
 *                            paper does not print; reading g13b takes the sampling criterion of the two discrete
 *                            operators instead: |z| < z_c = N*dx^2/lambda -> angular spectrum, else direct.
 *                            Every batch element must fall on the same side of its own z_c, otherwise
 *                            FRESNEL_ERR_UNSUPPORTED (split the batch or force a method).
 * z == 0 applies the optic only.  pixel_inout (HOST, length batch) carries the running pixel pitch and holds the
 * final one on return; method_used (HOST, length nsurf, may be NULL) receives 0 / 1, or -1 where z == 0.
 * All surfaces are validated before anything is enqueued; the calls enqueue only, so a train can be captured
 * into one CUDA graph.
 * TRAIN-LEVEL FUSION.  The row and the column convolution of an angular-spectrum step commute, so a run of L
 * consecutive angular-spectrum surfaces is scheduled as
 *     rows_0 (optic_0 on load) | cols_0, optic_1, cols_1 | rows_1, optic_2, rows_2 | ... | last convolution:
 * L+1 passes over the wavefront instead of 2L, every inner pass holding each line on chip through
 * convolution -> optic of the next surface -> convolution ("10 optics ... 19 FFT" become 11 passes).
 * Column passes fetch the optic's map tiles by TMA.  Results equal the surface-by-surface order up to rounding
 * (the two orders differ by the commuted convolutions only).  Direct-Fresnel and z == 0 surfaces end a run. */
typedef struct {
    double f;
    const void *amp;
    const void *opd;
    double z;
    int method;
} fresnel_surface;
enum { FRESNEL_METHOD_AS = 0, FRESNEL_METHOD_DIRECT = 1, FRESNEL_METHOD_AUTO = 2 };
fresnel_status fresnel_system_run(fresnel_plan *p, void *wf, double *pixel_inout, const double *lambda,
                                  const fresnel_surface *surf, int nsurf, int *method_used);

/* A train of surfaces under the GAUSSIAN PILOT-BEAM rule ("following the methods in Ref. [6, Equation
 * 82-89]" -- Lawrence 1992, not printed in the paper; reading g21 states every convention; SURVEY.md sec.
 * 8(f) NEXT-1).  A Gaussian pilot beam per batch element -- waist radius w0 at position zw (zR = pi w0^2 / lambda),
 * current position z -- decides on which reference surface the array is kept: a plane within rayleigh_factor * zR
 * of the pilot waist, outside it a sphere centred on the waist (radius rref = z - zw) whose curvature is REMOVED
 * from the array,   U_true = U_stored * exp(i pi r^2 / (lambda rref)),   so the quadratic phases that cannot be
 * sampled far from focus never reach the grid.  A propagation from z1 to z2 takes
 *     inside -> inside    PTP(z2 - z1)                          angular spectrum, pitch kept
 *     inside -> outside   PTP(zw - z1), WTS(z2 - zw)            waist -> sphere: direct Fresnel without its output chirp
 *     outside -> inside   STW(zw - z1), PTP(z2 - zw)            sphere -> waist: direct Fresnel without its input chirp
 *     outside -> outside  STW(zw - z1), WTS(z2 - zw)            (a leg of zero length is skipped)
 * each WTS / STW leg changing the pitch to lambda |dz| / (N dx).  A thin lens f maps the pilot beam by the ABCD rule
 * 1/q' = 1/q - 1/f (q = z - zw + i zR), chooses the new reference (plane if |z - zw'| < rayleigh_factor zR', else the
 * sphere rref' = z - zw') and leaves on the array only the residual chirp exp(i pi r^2/lambda (1/rref - 1/f - 1/rref')),
 * which rides on the next pass.  Masks act on the stored array.  Surfaces: as in fresnel_system_run (`method` is
 * ignored).  state: HOST array of `batch` pilot states, read as the starting state (a collimated beam of radius R at
 * its waist: {R, 0, 0, INFINITY}) and overwritten with the final one; legs_used (HOST, 2 ints per surface, may be
 * NULL): 0 none, 1 PTP, 2 WTS, 3 STW.  Every batch element must take the same legs (and every WTS / STW leg the same
 * direction), otherwise FRESNEL_ERR_UNSUPPORTED; everything is validated before anything is enqueued.  The kernels
 * are the two-pass kernels of the other calls: only the tables differ. */
typedef struct {
    double w0;    /* waist radius of the pilot beam (m) */
    double zw;    /* position of its waist along the axis (m) */
    double z;     /* current position (m) */
    double rref;  /* radius of the reference sphere the array is stored on; +-INFINITY: planar */
} fresnel_pilot_state;
enum { FRESNEL_LEG_NONE = 0, FRESNEL_LEG_PTP = 1, FRESNEL_LEG_WTS = 2, FRESNEL_LEG_STW = 3 };
fresnel_status fresnel_system_run_pilot(fresnel_plan *p, void *wf, double *pixel_inout, const double *lambda,
                                        const fresnel_surface *surf, int nsurf, double rayleigh_factor,
                                        fresnel_pilot_state *state, int *legs_used);

/* Fraunhofer propagation by a MATRIX FOURIER TRANSFORM ("discrete matrix Fourier transforms of modest
 * sized arrays", :119; reading g22): the field in the focal plane of a lens of
 * focal length f on ANY output grid -- nb x nb pixels of pitch pixel_out[b], centred on pixel nb/2 -- from the plan's
 * N x N input of pitch pixel_in[b] (centred on pixel N/2):
 *     out[b][p][q] = s * sum_j sum_k in[b][j][k] * exp(-+ 2 pi i (x_k x'_q + y_j y'_p) / (lambda_b f)),   s = dx^2/(+- i lambda_b f)
 * (upper signs: FRESNEL_FORWARD; lower: FRESNEL_INVERSE, the inverse pair at critical sampling).  With
 * pixel_out = lambda f/(N pixel_in) and nb = N it is the Fourier core of fresnel_propagate_direct; with a finer pitch
 * and a small nb it is the high-resolution, small-field transform coronagraph models use.  The one dense contraction
 * of the library: two complex GEMMs (cost 8 (N^2 nb + N nb^2) flops) on the FP64 tensor cores (DMMA) -- complex64 plans
 * convert on load and round on store.  in: device, [batch][N][N] of the plan's dtype, read only; out: device,
 * [batch][nb][nb] of the plan's dtype, written; must not alias.  Workspace (kernel matrix and intermediate, 32 batch N nb
 * bytes) is allocated on first use of a larger nb -- call fresnel_plan_reserve_mft first to keep fresnel_mft itself
 * allocation-free (required before capturing it into a CUDA graph: FRESNEL_ERR_ALLOC otherwise). */
fresnel_status fresnel_plan_reserve_mft(fresnel_plan *p, int nb_max);
fresnel_status fresnel_mft(fresnel_plan *p, const void *in, void *out, int nb, const double *pixel_in, const double *pixel_out,
                           const double *lambda, double f, int direction);

/* The same transform for callers that may NOT allocate device memory (code under CUDA-graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc): no plan, no cudaMalloc / cudaFree / allocating library call on any path.
 * The scratch of the two GEMMs (kernel matrix and intermediate) lives in one file-scope `static __device__` array of
 * FIXED size inside the library -- 2 * FRESNEL_MFT_NOALLOC_MAX_ELEMS complex doubles = 8 MiB (+ 1.5 KiB of per-batch
 * scalars) that every GPU that loads the library holds until the process exits.  Limits: batch * nb * na <=
 * FRESNEL_MFT_NOALLOC_MAX_ELEMS (e.g. one 1024 -> 256 transform, four 512 -> 128 ones) and batch <=
 * FRESNEL_MFT_NOALLOC_MAX_BATCH; anything larger is refused with FRESNEL_ERR_TOO_LARGE and nothing is enqueued.
 * in: device, [batch][na][na] of `dtype`, read only; out: device, [batch][nb][nb] of `dtype`, written; must not alias.
 * pixel_in / pixel_out / lambda: HOST arrays of `batch` doubles; f, direction: as fresnel_mft; stream: a cudaStream_t
 * passed as void* (NULL = legacy default stream), on the CURRENT device.  Enqueues five kernels and returns (it does not
 * synchronise); results equal fresnel_mft's bit for bit (same kernels).
 * SHARED STATE: every call on a device uses the same array, which keeps the last call's contents.  Each call writes
 * every word it later reads, so nothing needs clearing -- but two calls whose kernels can overlap on the GPU (different
 * streams without an ordering between them, or two host threads) RACE on it: order them on one stream or by events. */
#define FRESNEL_MFT_NOALLOC_MAX_ELEMS 262144
#define FRESNEL_MFT_NOALLOC_MAX_BATCH 32
fresnel_status fresnel_mft_noalloc(const void *in, void *out, int na, int nb, int batch, fresnel_dtype dtype, const double *pixel_in,
                                   const double *pixel_out, const double *lambda, double f, int direction, void *stream);

/* Broadband (polychromatic) image: the incoherent, weighted sum of the batch's monochromatic intensities
 * ("calculations must be repeated for all of the wavelengths"; one process per wavelength in
 * the paper):
 *     image[j][k] += sum_b weight[b] * |wf[b][j][k]|^2
 * wf: device, [batch][N][N] complex of the plan's dtype, read only.  image: device, real [N][N] of the
 * matching precision (double for C128, float for C64), accumulated in place (zero it first for a fresh
 * image); the sum over the batch is formed in double.  weight: HOST array of length batch (consumed
 * before return; non-finite values: FRESNEL_ERR_INVALID_ARG).  One pass: reads the batch once, the image
 * once, writes the image once.  With the batch sharded over GPUs each rank accumulates its own image and
 * one sum-reduction of N*N reals finishes the job (paper_1806_06467_b200/sharding.py). */
fresnel_status fresnel_accumulate_intensity(fresnel_plan *p, const void *wf, const double *weight, void *image);

/* ---- host <-> device staging on the plan's stream (used by the end-to-end benchmark) ---------- */

/* Asynchronous copies ordered with the plan's work.  `host` should be pinned for real overlap. */
fresnel_status fresnel_memcpy_h2d(fresnel_plan *p, void *dst_device, const void *src_host, size_t bytes);
fresnel_status fresnel_memcpy_d2h(fresnel_plan *p, void *dst_host, const void *src_device, size_t bytes);

/* ---- misc -------------------------------------------------------------------------------------- */

const char *fresnel_status_string(fresnel_status s);

/* Library build string, e.g. "fresnel-b200 0.2 sm_100a". */
const char *fresnel_version(void);

#ifdef __cplusplus
}
#endif
#endif /* FRESNEL_H */
