/* epr.h — C-ABI of the B200-native fast Eikonal Phase Retrieval (EPR) hot path.
 *
 * One library, libepr.so, hand-written CUDA for sm_100a.  It implements the batched per-projection
 * iterative correction loop of arxiv 2601.22793 (§4.4) and the three operators of one
 * iteration.  No CPU fallback, no other backend.  Notation follows the paper; the readings R1..R16 of the
 * points the paper leaves open are listed in DESIGN.md.
 *
 * Conventions
 *  - Arrays are row-major [y][x], x fastest; every index is periodic (R7).
 *  - ALL array arguments are DEVICE pointers owned by the caller, contiguous, 16-byte aligned.  The library
 *    never allocates or frees them and keeps no reference once the work enqueued on `stream` has completed.
 *    (epr_retrieve_host is the one exception: it takes HOST pointers and does the copies itself.)
 *  - `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).  Calls only ENQUEUE work and
 *    return; epr_plan / epr_destroy / epr_retrieve_host may synchronise.
 *  - Every call returns an epr_status; nothing throws or exits.  On EPR_EINVAL / EPR_ESIZE nothing has been
 *    enqueued.  epr_last_error(plan) gives a NUL-terminated message owned by the plan.
 *  - A plan is not thread-safe; distinct plans are independent, also across threads and devices: a plan belongs to
 *    the CUDA device that was current in epr_plan, every call runs there (whatever device is current in the caller)
 *    and restores the caller's device.
 *  - d is the flat-field-normalised detector intensity (≈ 1 in the empty beam; Σ_s f_s = 1).
 *  - The state of the iteration is the nominal thickness field τ of Eq. (7):
 *    I_s = f_s exp(−γ_s τ).  The phase of line s is φ_s = −(δ_s/2β_s) γ_s τ (Eq. (6)).
 */
#ifndef EPR_H
#define EPR_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct epr_plan_s* epr_plan_t;

typedef enum {
  EPR_OK = 0,
  EPR_EINVAL = 1, /* bad argument (NULL pointer, non-positive size / energy / weight / step, batch > max_batch …) */
  EPR_ESIZE = 2,  /* unsupported grid: nx or ny below 8, with a prime factor other than 2, 3, 5, or above 8192 (see epr_plan) */
  EPR_ECUDA = 3,  /* a CUDA runtime call failed; message in epr_last_error */
  EPR_ENOMEM = 4  /* device allocation failed */
} epr_status;

typedef enum { EPR_LOCAL = 0, EPR_NONLOCAL = 1 } epr_solver;

/* All optional: pass NULL for the defaults, or fill with epr_default_options() first. */
typedef struct {
  int order;          /* local solver: truncation order m of P_{m,s}, 1 or 2 (default 2) */
  int wkb1;           /* local solver: include the −(ε²/4)∂(I∂Q) term of Eq. (1) (default 1) */
  int symbol;         /* Fourier symbol λ of the filter: 0 discrete 5-point (default), 1 θ²       R5 */
  float max_shift_px; /* S: clamp of each ray-map component and splat halo (default 16, ≤ 30)    R6 */
  float i_min;        /* positivity floor of the total object-plane intensity (default 1e-6) */
  int newton_iters;   /* Newton steps of the single-thickness projection (default 4)             R10 */
  int init;           /* 0: Paganin initial guess (default); 1: `out` holds τ⁰ on entry          R9 */
  int output;         /* 0: τ (default); 1: phase φ of line out_bin; 2: total intensity Σ_s I_s */
  int out_bin;
  const double* mu_rel; /* γ_s override (relative attenuation per line, length n_bins) or NULL   R11 */
  int nonlocal_wkb1;  /* non-local solver: add the local WKB1 term of Eq. (1) to the ray-map prediction (default 0)  R4 */
} epr_options;

void epr_default_options(epr_options* opt);

/* epr_plan — derive the per-line scalars and build tables / workspaces.          PAPER.md:225-233, Eq. (2),(6),(7)
 *   nx, ny        grid (x fastest).  pixel_m: detector pixel p [m].  L_m: propagation distance [m].
 *   n_bins        number of spectral lines N_s (1 = monochromatic), ≤ 16.
 *   energy_keV, weight, delta_over_beta   HOST arrays of length n_bins: E_s, spectral weight (normalised
 *                 internally to Σ f_s = 1), δ_s/β_s.
 *   solver        EPR_LOCAL: Taylor/WKB closure Eq. (1); EPR_NONLOCAL: ray map Eq. (2) + splat Eq. (3).
 *   max_batch     largest `batch` later calls may pass.  The loop's workspaces are sized for a WORK BATCH = max_batch, capped
 *                 so that they stay below 12 GB (environment EPR_WORK_BATCH = projections, read here, overrides); larger
 *                 batches pass through the loop in passes of that many projections — same results, bit for bit.
 * Grids: nx, ny >= 8 with prime factors in {2, 3, 5} (anything else: EPR_ESIZE; padding is the caller's job, R7).
 *   The tuned kernels run on 16-pixel-aligned grids whose lengths have a compiled transform (16, 32, 48, 64, 80, 96, 128,
 *   160, 256, 320, 384, 512, 640, 768, 1024, 1280, 1536, 1920, 2048, 2160, 2560, 3072, 3200, 4096); every other smooth
 *   grid up to 8192 per axis (250, 1080, 3000, odd lengths such as 375, …) runs the general path: the same steps, one
 *   pixel per thread, run-time-radix FFT — correct to the same tolerances, 2x (non-local) to 5x (local) slower per pixel.
 * Derived: k_s = 2πE_s/(hc); α_s = L/(k_s p²); a_s = α_s δ_s/(2β_s); γ_s ∝ 1/(E_s δ_s/β_s), Σ f_s γ_s = 1. */
epr_status epr_plan(epr_plan_t* plan, int nx, int ny, double pixel_m, double L_m, int n_bins,
                    const double* energy_keV, const double* weight, const double* delta_over_beta,
                    epr_solver solver, int max_batch, const epr_options* opt);

/* epr_forward — the non-linear forward model τ → Σ_s F_s[f_s e^{−γ_s τ}]         Eq. (5)
 *   tau    [batch][ny][nx]            in
 *   P_sum  [batch][ny][nx]            out: predicted detector intensity Σ_s P_s
 *   P_bins [batch][n_bins][ny][nx]    out or NULL: per-line predictions P_s
 * Local: P_s = closure Eq. (1).  Non-local: u_s = clamp(a_s D⁰ ln I_s, ±S) (Eq. (2)) and the
 * mass-conserving bilinear splat; the ray map is kept in the plan for epr_adjoint /
 * epr_transport (storage for max_batch · n_bins maps is allocated on the first non-local call). */
epr_status epr_forward(epr_plan_t plan, int batch, const float* tau, float* P_sum, float* P_bins, void* stream);

/* epr_adjoint — back-transport of per-line detector residuals                     Eq. (4)
 *   e_bins, r_bins [batch][n_bins][ny][nx].  Non-local: bilinear gather with the ray map of the last
 *   epr_forward on this plan (same batch).  Local: identity copy. */
epr_status epr_adjoint(epr_plan_t plan, int batch, const float* e_bins, float* r_bins, void* stream);

/* epr_transport — the LINEAR operator ℳ_s: splat arbitrary per-line planes with the stored ray map
 *   (Eq. (3)).  I_bins, P_bins [batch][n_bins][ny][nx].  Non-local plans only (EPR_EINVAL
 *   otherwise).  Lets ⟨ℳx,y⟩ = ⟨x,ℳ*y⟩ and mass conservation be checked on the device. */
epr_status epr_transport(epr_plan_t plan, int batch, const float* I_bins, float* P_bins, void* stream);

/* epr_precondition — q_s = IFFT2( FFT2(r_s) / (1 + a_s λ) ) per line
 *   r_bins, q_bins [batch][n_bins][ny][nx]; may alias. */
epr_status epr_precondition(epr_plan_t plan, int batch, const float* r_bins, float* q_bins, void* stream);

/* epr_retrieve — the correction loop
 *   d   [batch][ny][nx] in;  out [batch][ny][nx] out (τ, or what opt.output selects; τ⁰ in if opt.init = 1).
 *   iterations ≥ 0 correction iterations after the initial Paganin solve (0 returns the L¹/Paganin result,
 *   PAPER.md:124); step > 0 relaxation factor.
 *   Launch-bound calls (batch · n_bins · nx · ny ≤ 2^20) on a non-default stream are captured into a CUDA graph on
 *   their second occurrence and replayed while (d, out, batch, iterations, step) stay the same; the buffers' CONTENTS
 *   may change between calls.  Environment EPR_GRAPH = 0 disables this, 2 applies it to every size. */
epr_status epr_retrieve(epr_plan_t plan, int batch, const float* d, float* out, int iterations, float step,
                        void* stream);

/* epr_retrieve_oversampled — the loop on an oversampled computational grid          PAPER.md:79 (reading R16)
 *   "All reconstructions ... were computed on oversampled grids ... the local solver uses an oversampling factor of
 *   2 (i.e. a pixel size reduced by a factor 2), while the non-local solver uses an oversampling factor of 4."
 *   `plan` is the plan of the FINE grid: nx = factor · nx_d, ny = factor · ny_d, pixel_m = p / factor (so that shifts
 *   and max_shift_px count fine pixels).
 *   d   [batch][ny/factor][nx/factor] in  (detector grid);  out  same shape, out.
 *   The detector image reaches the fine grid by pixel replication (a detector pixel measures the mean intensity over
 *   its area), epr_retrieve runs there, and the result (τ, or what opt.output selects) returns as the mean over each
 *   factor x factor block — the exact left inverse of the replication.  factor ∈ 1..8 must divide nx and ny with
 *   nx / factor a multiple of 4; opt.init must be 0.  The fine-grid buffers (two planes per projection of the plan's
 *   work batch) are allocated on the first call and owned by the plan. */
epr_status epr_retrieve_oversampled(epr_plan_t plan, int factor, int batch, const float* d, float* out, int iterations,
                                    float step, void* stream);

/* epr_set_diagnostics — per-iteration diagnostics of the retrievals that follow
 *   diag: DEVICE array [batch][capacity_iters][2] of floats owned by the caller, or NULL to switch diagnostics off
 *   (the default).  For projection b of a later epr_retrieve / epr_retrieve_oversampled / epr_retrieve_host call and
 *   correction iteration n < capacity_iters:
 *     diag[b][n][0] = RMS over the pixels of the detector residual e = d − Σ_s P_s at iteration n;
 *     diag[b][n][1] = the regime indicator η of PAPER.md:53 in the sup norm: the largest unclamped shift component
 *                     max_s max_r |a_s D⁰ ln I_s| in pixels of the plan's grid (η < 1: local regime).
 *   Costs two small kernels and one pass over the residual planes per iteration; keep it off in timed runs.  While it
 *   is on, retrievals are not captured into CUDA graphs.  On a plan with an x-dependent spectrum the shift uses the
 *   scalars of the pixel's own column, a_s(x) γ_s(x) (R17(b)). */
epr_status epr_set_diagnostics(epr_plan_t plan, float* diag, int capacity_iters);

/* epr_shift_histogram — the regime diagnostic of Fig. 6
 *   "the distribution of estimated WKB0 transverse shifts (in detector-pixel units) for each sampling energy (spectral
 *   line) on a representative radiograph": for every projection b and line s the histogram over the pixels of
 *   η = ‖Δ_s‖/p = ‖a_s D⁰ ln I_s‖ (Euclidean norm, not clamped; pixels of the plan's grid) of the thickness field tau
 *   (e.g. the result of epr_retrieve).  Bin k counts η ∈ [k·bin_px, (k+1)·bin_px), the last bin is open-ended.
 *   tau  [batch][ny][nx] DEVICE in;  hist [batch][n_bins][n_hist] DEVICE unsigned out (overwritten);  2 <= n_hist <= 1024.
 *   η < 1 over most of the field: local regime; a significant fraction above 1: use the non-local solver. */
epr_status epr_shift_histogram(epr_plan_t plan, int batch, const float* tau, int n_hist, float bin_px, unsigned* hist,
                               void* stream);

/* epr_retrieve_host — same, with HOST buffers (pinned for full speed): copies d host→device, runs the loop,
 *   copies the result device→host.  The batch is cut into chunks of about 256 MB of input (never more than the plan's
 *   work batch; environment EPR_HOST_CHUNK = projections per chunk overrides) that travel on three private streams, so
 *   that the copy in of chunk i + 1 and the copy out of chunk i − 1 overlap the loop of chunk i; the first and last
 *   chunks are smaller (their copies overlap nothing).  `batch` may exceed max_batch.  The call first waits for all
 *   work enqueued earlier on the device (cudaDeviceSynchronize) and returns after its last copy has completed.
 *   Tunables (environment, read at every call): small batches are cut into 1, 2 or 4 chunks according to the share of
 *   the copies in the call, estimated from EPR_HOST_LINK_GBS (host link, default 50 GB/s — a B200 on PCIe 5 x16) and
 *   EPR_LOOP_GBS (rate at which the loop moves its algorithmic bytes, default 2500 GB/s, measured on B200); set them for
 *   another host link or GPU.  They only change the chunking, never the result. */
epr_status epr_retrieve_host(epr_plan_t plan, int batch, const float* d_host, float* out_host, int iterations,
                             float step);

/* epr_retrieve_host_async / epr_host_wait — epr_retrieve_host as a STREAMING SESSION
 *   "large acquisitions processed in chunks": a scan is thousands of radiographs handed over batch after batch.
 *   epr_retrieve_host_async enqueues one batch exactly like epr_retrieve_host (same chunks, same results bit for bit) but
 *   returns without waiting; consecutive async calls on a plan form a session in which the copy in of the next batch's first
 *   chunk overlaps the last loop of the previous batch and its last copy out overlaps the next batch's first loop.  Only the
 *   first call of a session waits for work enqueued earlier on the device.  epr_host_wait returns when everything enqueued
 *   in the session has completed — every out_host is valid from then on — and closes it; a plain epr_retrieve_host does the
 *   same before it starts.  d_host and out_host must stay valid (and should be pinned) until epr_host_wait.  Between the
 *   first async call and epr_host_wait make NO other call on this plan except epr_retrieve_host_async (the session uses
 *   the plan's workspaces on private streams).  opt.init = 1 and epr_set_diagnostics work as in epr_retrieve_host (the
 *   diagnostics rows are indexed per call: give every call its own array or read it before the next call). */
epr_status epr_retrieve_host_async(epr_plan_t plan, int batch, const float* d_host, float* out_host, int iterations,
                                   float step);
epr_status epr_host_wait(epr_plan_t plan);

/* epr_retrieve_host_multi — ONE host batch over several plans, one per GPU
 *   "when two GPUs are available ...": projections are independent, so plan k (normally created on device k; all plans on
 *   the same grid with the same physics) receives the contiguous, balanced range of the batch that rank k of n_plans gets —
 *   the first batch % n_plans plans take one projection more — as one streaming call on its own device, and the call
 *   returns when all of them have finished.  No data crosses between GPUs.  HOST buffers [batch][ny][nx], pinned for
 *   overlap.  Plans may also share a device (two pipelines on one GPU).  Returns the first error of any plan (its message
 *   is in that plan's epr_last_error). */
epr_status epr_retrieve_host_multi(epr_plan_t* plans, int n_plans, int batch, const float* d_host, float* out_host,
                                   int iterations, float step);

/* epr_shard_range — the split epr_retrieve_host_multi (and a one-process-per-GPU launcher) uses: part k of `parts` gets the
 *   projections [*start, *stop) of `total`; contiguous, balanced, the first total % parts parts take one more.  Host
 *   arithmetic only: needs no device.  EPR_EINVAL for total < 0, parts < 1, k outside 0..parts−1 or NULL pointers. */
epr_status epr_shard_range(int total, int k, int parts, int* start, int* stop);

/* epr_plan_profiles — x-dependent effective spectrum           PAPER.md:216-221 (Eq. (6) + remark), 227-229 (Eq. (7)), 431-441 (§9.2)
 *   "I_s(r) = f_s(x) exp(−γ_s(x) τ(r))", "db_s(x) = δ_s(x)/β_s(x) may be x-dependent if an x-dependent effective spectrum
 *   is used": the spectrum varies slowly across the horizontal detector coordinate x.  The paper's "blockwise
 *   interpolation strategy" is not printed; reading R17:
 *   (a) the profiles are given on n_blocks equal blocks of columns (n_blocks divides nx, <= 64); the value of column x is the
 *       linear interpolation between the two nearest block centres, constant outside the outermost centres;
 *   (b) per-line scalars are frozen at the pixel's own column: the closure stencil sees neighbouring τ through the centre
 *       column's scalars, a ray-map source carries the mass and shift of its own column (no derivative of a profile);
 *   (c) the FFT-diagonal filter is applied once per block with that block's a_s and blended with the weights of (a).
 *   weight, delta_over_beta, mu_rel: HOST arrays [n_blocks][n_bins] (mu_rel may be NULL: γ_s ∝ 1/(E_s δ_s/β_s), R11); weights
 *   are normalised per block; γ keeps ONE normalisation for the whole detector (block mean of Σ_s f_s γ_s = 1).  The energies,
 *   L, pixel and options are the plan's.  n_blocks = 1 is the uniform spectrum ("single block", §9.2).  After this call the
 *   plan runs the general path (see epr_plan); every option and entry point stays available (opt.nonlocal_wkb1 takes the
 *   WKB1 term at the detector pixel's column, epr_set_diagnostics the shift of the pixel's own column).
 *   Synchronises the device.  A ray map stored by an earlier epr_forward is dropped (call epr_forward again before
 *   epr_adjoint / epr_transport); epr_plan_lines keeps returning the uniform scalars of epr_plan — read the ones in use with
 *   epr_plan_columns.  The filter workspace (n_blocks planes per projection of the work batch) is allocated here; when it does
 *   not fit, the plan's work batch is halved until it does (larger batches simply take more passes).  If the call fails
 *   (EPR_ENOMEM, EPR_ECUDA) the plan is unchanged and stays usable with its previous spectrum. */
epr_status epr_plan_profiles(epr_plan_t plan, int n_blocks, const double* weight, const double* delta_over_beta,
                             const double* mu_rel);

/* Per-column scalars the plan uses (HOST arrays [n_bins][nx], any may be NULL): f_s(x), γ_s(x), a_s(x). */
epr_status epr_plan_columns(epr_plan_t plan, double* f, double* gamma, double* a);

/* epr_read_flags — conditions kernels detected since the flags were last cleared (synchronises the device).
 *   EPR_FLAG_SPLAT_OVERFLOW: the non-local forward accumulates each line's detector plane in 32-bit fixed point (unit
 *   2^-26 of the flat field; order-independent, exactly mass conserving).  A detector pixel of one line that collects
 *   32x the flat field or more leaves that range; the flag is raised when an accumulator reads negative, i.e. for
 *   totals in [32, 64)x (it wraps silently beyond 64x, and epr_transport, whose planes may be negative, never raises
 *   it).  Physical caustics of the paper's regime stay below ~10x.
 *   *flags receives the bits; clear != 0 resets them. */
#define EPR_FLAG_SPLAT_OVERFLOW 1u
epr_status epr_read_flags(epr_plan_t plan, unsigned* flags, int clear);

/* epr_retrieve_oversampled_host — epr_retrieve_oversampled with HOST buffers on the detector grid
 *   d_host, out_host [batch][ny/factor][nx/factor]; the same chunked schedule as epr_retrieve_host (copies of neighbouring
 *   chunks overlap the loop), every chunk replicated, retrieved and block-averaged on the device. */
epr_status epr_retrieve_oversampled_host(epr_plan_t plan, int factor, int batch, const float* d_host, float* out_host,
                                         int iterations, float step);

/* Per-line scalars epr_plan derived (HOST arrays of length n_bins, any may be NULL): f_s, γ_s, a_s, α_s.  Not changed by
 * epr_plan_profiles (see there). */
epr_status epr_plan_lines(epr_plan_t plan, double* f, double* gamma, double* a, double* alpha);

/* Number of kernel launches the plan has enqueued so far (for bench.py's gpu_launches). */
long long epr_launch_count(epr_plan_t plan);

/* Optional per-kernel timing for bench.py's roofline: while enabled, CUDA events are recorded on the launch
 * stream around every kernel launch.  epr_profile_read synchronises the device and returns, per kernel family
 * that ran, its name, total milliseconds and launch count (up to max_kernels entries; the return value is the
 * number written); reset != 0 clears the accumulators. */
epr_status epr_profile_enable(epr_plan_t plan, int on);
int epr_profile_read(epr_plan_t plan, int max_kernels, const char** names, double* total_ms, long long* count, int reset);

/* epr_residual_rms_static — the residual RMS of epr_set_diagnostics without a plan and WITHOUT ANY ALLOCATION
 *                                                                                              PAPER.md:231, 95
 *   rms[b] = sqrt( mean over the ny·nx pixels of ( Σ_s e_bins[b][s] )² ) — for e_s the per-line residuals of one loop
 *   iteration (their sum is the detector residual e = d − Σ_s P_s, "form the detector residual" PAPER.md:231) this is
 *   diag[b][n][0] of epr_set_diagnostics, the quantity whose decay over n is the convergence history of PAPER.md:95.
 *   Pass n_bins = 1 to take the RMS of a plane that is already summed.
 *     e_bins [batch][n_bins][ny][nx]  DEVICE in;   rms [batch]  DEVICE out;   1 <= n_bins <= 16;  nx·ny < 2^32, any shape.
 * For whom: callers that cannot call cudaMalloc where they want this number — a monitoring hook inside a process whose
 *   device memory has all been given to one pool (the reconstruction framework's allocator, or plans sized at start-up),
 *   where a late cudaMalloc fails or fragments that pool; and acquisition-rate loops, which cannot take the device-wide
 *   stall a cudaMalloc / cudaFree may cause.  The plan-based diagnostic allocates its reduction scratch on first use;
 *   this call does not: it calls no cudaMalloc, cudaFree or any library routine that allocates, needs no plan, and only
 *   enqueues two kernels on `stream`.
 * How: the scratch (64 doubles per projection) lives in a fixed array inside libepr.so, sized for EPR_STATIC_MAX_BATCH
 *   projections = 512 KiB.  Each GPU that loads this library's code holds its own copy of those 512 KiB until the process
 *   ends.  batch > EPR_STATIC_MAX_BATCH returns EPR_ESIZE (nothing enqueued); split larger batches into several calls.
 * Device and first call: the call works on the CURRENT device, which must own e_bins and rms (EPR_EINVAL otherwise).  The
 *   first call on each device looks up where the array sits on that device and remembers it; that first call is also
 *   when the runtime may load the library's code onto the device, so make it once during set-up, before any stream
 *   capture and before the latency-critical part of the run.  Later calls on that device do no set-up.
 * Shared scratch: all calls on a device use the same array, and it keeps whatever the previous call left there.  Nothing in
 *   it needs to be zero (every slot a call reads it has written first), so back-to-back calls on ONE stream are safe; two
 *   calls whose kernels may overlap on the GPU — different streams without an event between them, or different host
 *   threads — race on the array and return garbage.  Order them yourself.
 * Errors: epr_static_last_error() gives the message of the last failed epr_residual_rms_static of the calling thread. */
#define EPR_STATIC_MAX_BATCH 1024
epr_status epr_residual_rms_static(int batch, int n_bins, int nx, int ny, const float* e_bins, float* rms, void* stream);
const char* epr_static_last_error(void);

epr_status epr_destroy(epr_plan_t plan);
const char* epr_last_error(epr_plan_t plan);
const char* epr_version(void);

#ifdef __cplusplus
}
#endif
#endif /* EPR_H */
