// epr_internal.h — plan layout and launcher prototypes shared by the C-ABI and the kernels.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/epr.h"

#define EPR_MAX_BINS 16
#define EPR_FIX_BITS 26                       /* splat accumulators: u32 fixed point, 1.0 = 2^26 */
#define EPR_FIX_ONE 67108864.0                /* 2^26 */

// Per-line scalars, passed to kernels by value (fits the 4 KB parameter space).
struct EprLines {
  int n_bins;
  float f[EPR_MAX_BINS];        // spectral fraction f_s                       Eq. (7)
  float gamma[EPR_MAX_BINS];    // attenuation scaling γ_s                      Eq. (7)
  float a[EPR_MAX_BINS];        // a_s = α_s db_s / 2                           Eq. (1)+(6)
  float a2h[EPR_MAX_BINS];      // a_s² / 2                                     Eq. (1) WKB0
  float q4[EPR_MAX_BINS];       // α_s² / 4                                     Eq. (1) WKB1
  double fixF[EPR_MAX_BINS];    // f_s · 2^26 (double, for the splat)
  unsigned fixFi[EPR_MAX_BINS]; // rint(f_s · 2^26)
  float fixCorr[EPR_MAX_BINS];  // rint(f_s 2^26)·2^-26 − f_s
  float pj_a[EPR_MAX_BINS];     // −γ_s log2(e)          projection moments: f_s e^{−γ_s τ} = 2^(pj_a τ + pj_b)
  float pj_b[EPR_MAX_BINS];     // log2(f_s)
  float pj_g2[EPR_MAX_BINS];    // γ_s²
  float pj_g3[EPR_MAX_BINS];    // γ_s³
  float pj_G[8];                // Σ_s f_s γ_s^k, k = 0..7: the moments of the projection at τ = 0 (initial guess)
  float abar;                   // Σ f_s a_s (initial guess, R9)
  float gamma_max;              // max_s γ_s (range test of the projection's polynomial form)
  float fsum_dev;               // Σ_s (float)f_s − 1: rounding of the fp32 fractions, removed from the residual
};

// Per-column scalars of the GENERAL path (x-dependent effective spectrum, PAPER.md:216-229 / §9.2, reading R17; also
// used with constant columns for grids the tuned kernels do not take).  Device pointers, [n_bins][nx] unless stated.
struct EprColumns {
  const float* f;          // f_s(x), Σ_s f_s(x) = 1                                  Eq. (7)
  const float* gamma;      // γ_s(x)                                                   Eq. (7)
  const float* a;          // a_s(x) = α_s db_s(x)/2                                   Eq. (1)+(6)
  const unsigned* fixFi;   // rint(f_s(x) 2^26): fixed-point baseline of the splat
  const float* fixCorr;    // rint(f_s(x) 2^26) 2^-26 − f_s(x)
  const float* fsum_dev;   // [nx]  Σ_s (float)f_s(x) − 1
  const float* wblk;       // [n_blocks][nx] interpolation weights of the block filters (R17(c))
};
#define EPR_MAX_BLOCKS 64

struct epr_plan_s {
  int device;                  // CUDA device the plan was built on: every entry point runs there (DevGuard in epr_api.cu)
  int sms;                     // its SM count
  int nx, ny, n_bins, max_batch;
  int work_batch;              // projections processed per pass of the loop (workspaces are sized for it)
  int solver;                  // EPR_LOCAL / EPR_NONLOCAL
  epr_options opt;
  double h_f[EPR_MAX_BINS], h_gamma[EPR_MAX_BINS], h_a[EPR_MAX_BINS], h_alpha[EPR_MAX_BINS], h_db[EPR_MAX_BINS];
  EprLines lines;
  // tables
  float2* tw_row;              // per-pass twiddles of the nx/2-point row transform (forward radix order)
  float2* tw_r2c;              // exp(-2πi k/nx), k < nx/2 (real<->complex split)
  float2* tw_col;              // per-pass twiddles of the ny-point column transform, forward radix order
  float2* tw_col_inv;          //   … reversed radix order (inverse)
  float* lam_x;                // λ_x[kx], kx = 0..nx/2
  float* lam_y;                // λ_y[ky], ky < ny
  // workspaces (sized for max_batch)
  float* tau;                  // [work_batch][ny][nx]        state τ (when `out` is not τ) / scratch
  float* pred;                 // [work_batch][n_bins][ny][nx] P_s − f_s
  float* res;                  // [work_batch][n_bins][ny][nx] e_s then r_s
  float* res2;                 // [work_batch][n_bins][ny][nx] r_s (non-local gather output)
  float2* spec;                // [work_batch][n_bins][ny][nx/2] half spectra (packed Nyquist)
  float2* spec_sum;            // [work_batch][ny][nx/2]
  CUtensorMap map_spec;        // TMA descriptors of spec / spec_sum as [rows][nx floats], box 8 floats x 256 rows
  CUtensorMap map_spec_sum;
  int tma_ok;                  // descriptors valid (ny ≥ 256, nx % 8 == 0)
  int tma_box_rows;            // rows per TMA box: the largest divisor of ny that is ≤ 256 (256 for powers of two, 240 for 2160)
  unsigned* d_flags;           // device word of EPR_FLAG_* bits raised by kernels (epr_read_flags)
  float* gmax;                 // [work_batch][ny/16][nx/16] block maxima of |D⁰τ| (non-local: k_grad_blockmax)
  float* diag;                 // caller's diagnostics array [batch][diag_cap][2] (device) or NULL (epr_set_diagnostics)
  int diag_cap;
  double* diag_partial;        // [work_batch][64] partial sums of squares
  float* os_d;                 // [work_batch][ny][nx] up-sampled detector images (lazy, epr_retrieve_oversampled)
  float* os_out;               // [work_batch][ny][nx] fine-grid result before down-sampling (lazy)
  float2* raymap;              // [max_batch][n_bins][ny][nx] stored u_s (lazy, epr_forward non-local)
  int raymap_batch;            // batch of the stored map (0 = none)
  // host staging for epr_retrieve_host
  float* stage_in[2];
  float* stage_out[2];
  int stage_chunk;             // projections the staging buffers hold
  size_t stage_floats;         // floats each staging buffer holds
  cudaStream_t hstream[3];     // copy-in, compute, copy-out
  cudaEvent_t hev[6];          // per buffer: in-done, compute-done, out-done
  int hsession;                // 1 while epr_retrieve_host_async calls are outstanding (closed by epr_host_wait)
  long long hchunk;            // chunks enqueued in the open session (buffer = hchunk & 1)
  // CUDA graph of the last epr_retrieve (same buffers, batch, iterations, step): replayed instead of re-enqueued
  cudaGraphExec_t graph_exec;
  const float* graph_d;
  float* graph_out;
  int graph_batch, graph_iters;
  float graph_step;
  long long graph_launches;    // kernel launches inside the graph
  int graph_warm;              // an eager pass has run (function attributes are set)
  int graph_mode;              // 0 off, 1 on for launch-bound sizes (default), 2 always (EPR_GRAPH)
  // ---- general path (epr_general.cu): any {2,3,5}-smooth grid >= 8, x-dependent spectrum ----
  int general;                 // 1: the loop and the operators run the general kernels
  int fft_generic;             // 1: run-time-radix FFT (size not in the tuned table); spectra are [ny][nx/2 + 1] then
  int n_blocks;                // blocks of the x-dependent spectrum (1 = uniform)
  EprColumns cols;             // device tables (owned by the plan: cols_store)
  EprLines lines_bound;        // `lines` with a[s] = max_x a_s(x) γ_s(x), gamma[s] = 1: bounds for the tuned kernels' ring / halo / clamp tests
  void* cols_store;            // one allocation behind `cols`
  double* h_col;               // host copy [3][n_bins][nx]: f, γ, a per column (epr_plan_columns)
  float a_blk[EPR_MAX_BLOCKS][EPR_MAX_BINS];   // a_s of block b
  float abar_blk[EPR_MAX_BLOCKS];              // Σ_s f_s a_s of block b (initial guess)
  float* qblk;                 // [n_blocks][work_batch][ny][nx] filtered residual sums per block
  float2* tw_gen_x;            // exp(−2πi m/nx), m < nx   (run-time-radix FFT)
  float2* tw_gen_y;            // exp(−2πi m/ny), m < ny
  long long launches;
  int prof_on;                 // per-kernel event timing enabled
  void* prof;                  // EprProf*
  char err[256];
};

// A launcher that enqueues more than one kernel reports the extra ones here, next to the launch itself
// (epr_launch_count / bench.py's gpu_launches; the C-ABI layer counts one per launcher call).
static inline void epr_note_extra_launch(const epr_plan_s* p, int n = 1) { const_cast<epr_plan_s*>(p)->launches += n; }

// Per-device one-time setup (cudaFuncSetAttribute, occupancy queries) of a launcher: function attributes belong to the
// device, so every call site keeps one flag / value per device ordinal instead of one per process.  The calls guarded
// this way are idempotent, so two threads racing on the first use of a device both do the same harmless work.
#define EPR_MAX_DEVICES 64
struct EprPerDevice {
  long long v[EPR_MAX_DEVICES];
  long long& at(const epr_plan_s* p) { return v[(unsigned)p->device % EPR_MAX_DEVICES]; }
};

// ---- launchers (epr_kernels.cu / epr_fftk.cu); all return cudaGetLastError() ----
// planes = batch * n_bins unless stated.
// d_fuse != NULL (one line only): out = e = (d-1) - (P-1) directly; else out = pred[b][s] = P_s - f_s
cudaError_t epr_launch_forward_local(const epr_plan_s* p, int batch, const float* tau, const float* d_fuse, float* out,
                                     cudaStream_t st);
// out_mode 0: out[b][s] = P_s − f_s;  1: out[b][s] = P_s (linear transport);  2 (one line): out[b] = e = (d−1) − (P−f);
// 3 (several lines): out[b][s] = e_s = w_s e, the residual split fused into the splat (needs d)
cudaError_t epr_launch_splat(const epr_plan_s* p, int batch, const float* tau, const float* I_bins, const float2* map_in,
                             float2* map_out, float* out, int out_mode, const float* d, cudaStream_t st);
// block maxima of |D⁰τ| into p->gmax (launched by epr_launch_splat when the sources come from τ)
cudaError_t epr_launch_grad_blockmax(const epr_plan_s* p, int batch, const float* tau, cudaStream_t st);
cudaError_t epr_launch_residual(const epr_plan_s* p, int batch, const float* d, const float* pred, float* es,
                                cudaStream_t st);
cudaError_t epr_launch_pred_out(const epr_plan_s* p, int batch, const float* pred, float* P_sum, float* P_bins,
                                cudaStream_t st);
// gmax_fresh: p->gmax holds the block maxima of this tau (epr_launch_splat ran on it) -> shared-memory tile kernel
cudaError_t epr_launch_gather(const epr_plan_s* p, int batch, const float* tau, const float2* map_in, const float* es,
                              float* r, int gmax_fresh, cudaStream_t st);
cudaError_t epr_launch_rows_r2c(const epr_plan_s* p, int planes, const float* in, float in_offset, float2* spec,
                                cudaStream_t st);
// mode 0: per-plane filter with bin = plane % n_bins (out has `planes` planes);
// mode 1: sum over bins (out has planes / n_bins planes);  mode 2: single filter with abar (init).
// lines_override != NULL: the per-line filter coefficients a[] / abar are taken from it instead of p->lines (block filters)
// stage 0: whole operator; 1: forward column transform only (out[plane] = FFT_y(spec[plane]), frequency order, mode 0);
// 2: the input planes are already column-transformed (filter, Σ_s, inverse) — TMA column kernel only (power-of-two ny in
// 256 … 2048 with TMA descriptors), cudaErrorNotSupported otherwise
cudaError_t epr_launch_cols(const epr_plan_s* p, int planes, int mode, const float2* spec, float2* out, cudaStream_t st,
                            const EprLines* lines_override = nullptr, int stage = 0);
// epilogue 0: write q; 1: τ update (Newton projection) with step; init0: treat τ as 0 (initial guess)
cudaError_t epr_launch_rows_c2r(const epr_plan_s* p, int planes, const float2* spec, int epilogue, float step,
                                int tau_is_zero, float* q_or_tau, cudaStream_t st);
// oversampled grid (R16): the plan's (nx, ny) is the FINE grid; coarse planes are (ny/m) x (nx/m)
cudaError_t epr_launch_upsample(const epr_plan_s* p, int batch, int m, const float* coarse, float* fine, cudaStream_t st);
cudaError_t epr_launch_downsample(const epr_plan_s* p, int batch, int m, const float* fine, float* coarse, cudaStream_t st);
// diag[b·stride + 0] = RMS_px(Σ_s es[b][s]), diag[b·stride + 1] = max_s |c_s| · max|D⁰τ| (unclamped shift, px)
cudaError_t epr_launch_diagnostics(const epr_plan_s* p, int batch, const float* tau, const float* es, float* diag,
                                   int stride, cudaStream_t st);
// pred[b][s] −= f_s (α_s²/4) ∂i(Î ∂iQ): the WKB1 term of Eq. (1) for the non-local forward (opt.nonlocal_wkb1)
cudaError_t epr_launch_wkb1_sub(const epr_plan_s* p, int batch, const float* tau, float* pred, cudaStream_t st);
cudaError_t epr_launch_output(const epr_plan_s* p, int batch, const float* tau, float* out, cudaStream_t st);

// ---- general path (epr_general.cu / epr_fftgen.cu) ----
// a1-L: pred[b][s] = P_s − f_s(x), every line, per-column scalars frozen at the centre column (R17(b))
cudaError_t epr_gen_forward_local(const epr_plan_s* p, int batch, const float* tau, float* pred, cudaStream_t st);
// variant of R4 (opt.nonlocal_wkb1): pred[b][s] −= f_s(x)(α_s²/4) ∂i(Î ∂iQ) with the centre column's scalars
cudaError_t epr_gen_wkb1_sub(const epr_plan_s* p, int batch, const float* tau, float* pred, cudaStream_t st);
// diagnostics (epr_set_diagnostics): diag[b·stride + {0, 1}] = residual RMS of Σ_s es[b][s], largest unclamped shift component
cudaError_t epr_gen_diagnostics(const epr_plan_s* p, int batch, const float* tau, const float* es, float* diag, int stride,
                                cudaStream_t st);
// a1-N: acc[b][s] (u32 fixed point, zeroed here) += splat of line s; sources from τ (I_bins NULL; the ray map goes to map_out if
// given) or from I_bins with the stored map_in (epr_transport)
cudaError_t epr_gen_splat(const epr_plan_s* p, int batch, const float* tau, const float* I_bins, const float2* map_in,
                          float2* map_out, unsigned* acc, cudaStream_t st);
// fixed-point planes -> float, in place: mode 0: P_s − f_s(x); mode 1: P_s (transport)
cudaError_t epr_gen_fix2float(const epr_plan_s* p, int batch, unsigned* acc_inout, int mode, cudaStream_t st);
// a2: es[b][s] = w_s e from pred[b][s] = P_s − f_s (float; may alias es), fallback f_s(x)
cudaError_t epr_gen_residual(const epr_plan_s* p, int batch, const float* d, const float* pred, float* es, cudaStream_t st);
// a3: gather with the map recomputed from τ (map_in NULL) or stored
cudaError_t epr_gen_gather(const epr_plan_s* p, int batch, const float* tau, const float2* map_in, const float* es, float* r,
                           cudaStream_t st);
// a5 + a6: τ += δ(τ, step Σ_b wblk[b][x] q_b) with the column's scalars; qblk = [n_blocks][batch] planes
cudaError_t epr_gen_update(const epr_plan_s* p, int batch, const float* qblk, size_t blk_stride, float step, int tau_is_zero,
                           float* tau, cudaStream_t st);
// out (+)= wblk[b][x] · q   (epr_precondition on an x-dependent plan)
cudaError_t epr_gen_blend(const epr_plan_s* p, int planes, int b, const float* q, float* out, int accumulate, cudaStream_t st);
cudaError_t epr_gen_pred_out(const epr_plan_s* p, int batch, const float* pred, float* P_sum, float* P_bins, cudaStream_t st);
cudaError_t epr_gen_output(const epr_plan_s* p, int batch, const float* tau, float* out, cudaStream_t st);
// run-time-radix FFT (any {2,3,5}-smooth nx, ny): spectra [planes][ny][nx/2 + 1]
int epr_fftgen_supported(int n);
size_t epr_fftgen_spec_floats(const epr_plan_s* p);     // floats per spectrum plane
cudaError_t epr_fftgen_rows_r2c(const epr_plan_s* p, int planes, const float* in, float in_offset, float2* spec, cudaStream_t st);
cudaError_t epr_fftgen_cols(const epr_plan_s* p, int planes, int mode, const float2* spec, float2* out, cudaStream_t st,
                            const EprLines* lines_override);
cudaError_t epr_fftgen_rows_c2r(const epr_plan_s* p, int planes, const float2* spec, float* q, cudaStream_t st);
// per-line histogram of the unclamped shift norm (Fig. 6); hist [batch][n_bins][n_hist], zeroed by the launcher
cudaError_t epr_launch_shift_hist(const epr_plan_s* p, int batch, const float* tau, int n_hist, float bin_px, unsigned* hist,
                                  cudaStream_t st);
// tuned splat / gather of the loop with per-column tables (general path on 16-pixel-aligned grids)
cudaError_t epr_launch_splat_cols(const epr_plan_s* p, int batch, const float* tau, float* out, int out_mode, const float* d,
                                  cudaStream_t st);
cudaError_t epr_launch_gather_cols(const epr_plan_s* p, int batch, const float* tau, const float* es, float* r, cudaStream_t st);
