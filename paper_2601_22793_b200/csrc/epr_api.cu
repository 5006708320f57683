// epr_api.cu — the C-ABI of include/epr.h: plan, operators, the retrieval loop, host-streaming wrapper.
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <vector>

#include "epr_fft.cuh"
#include "epr_internal.h"

extern "C" int epr_fft_size_supported(int n);

static const double HC_KEV_M = 1.2398419843e-9;

#define FAIL(p, code, ...)                         \
  do {                                             \
    snprintf((p)->err, sizeof((p)->err), __VA_ARGS__); \
    return (code);                                 \
  } while (0)
#define CU(p, call)                                                                     \
  do {                                                                                  \
    cudaError_t e_ = (call);                                                            \
    if (e_ != cudaSuccess) FAIL(p, EPR_ECUDA, "%s: %s", #call, cudaGetErrorString(e_)); \
  } while (0)
// Kernel families, for launch counting and the optional per-kernel CUDA-event timing (epr_profile_*).
enum { K_FWD_LOCAL = 0, K_SPLAT, K_RESIDUAL, K_GATHER, K_ROWS_R2C, K_COLS, K_ROWS_C2R, K_PRED_OUT, K_OUTPUT, K_RESAMPLE, K_DIAG, K_WKB1, K_UPDATE, K_COUNT };
static const char* const K_NAMES[K_COUNT] = {"k_forward_local", "k_splat", "k_residual", "k_gather", "k_rows_r2c",
                                              "k_cols", "k_rows_c2r", "k_pred_out", "k_output", "k_resample", "k_diagnostics", "k_wkb1_sub", "k_update"};
struct EprProf {
  struct Rec { int tag; cudaEvent_t a, b; };
  std::vector<Rec> recs;
  double ms[K_COUNT];
  long long n[K_COUNT];
};

#define KL(p, ktag, st, call)                                                   \
  do {                                                                         \
    EprProf::Rec rec_;                                                         \
    if ((p)->prof_on) {                                                        \
      rec_.tag = (ktag);                                                        \
      CU(p, cudaEventCreate(&rec_.a));                                         \
      CU(p, cudaEventCreate(&rec_.b));                                         \
      CU(p, cudaEventRecord(rec_.a, (st)));                                    \
    }                                                                          \
    CU(p, call);                                                               \
    (p)->launches += 1;                                                        \
    if ((p)->prof_on) {                                                        \
      CU(p, cudaEventRecord(rec_.b, (st)));                                    \
      ((EprProf*)(p)->prof)->recs.push_back(rec_);                             \
    }                                                                          \
  } while (0)

static cudaError_t gen_r2c(epr_plan_t p, int planes, const float* in, float off, cudaStream_t cs);
static cudaError_t gen_cols(epr_plan_t p, int planes, int mode, int blk, float2* out, cudaStream_t cs, int stage);
static cudaError_t gen_c2r(epr_plan_t p, int planes, const float2* spec, float* q, cudaStream_t cs);

// Every entry point runs on the plan's device (function attributes, workspaces and streams belong to it) and restores
// the caller's current device on return.
struct DevGuard {
  int prev = -1;
  explicit DevGuard(const epr_plan_s* p) {
    if (!p) return;
    int cur = 0;
    if (cudaGetDevice(&cur) == cudaSuccess && cur != p->device) { prev = cur; cudaSetDevice(p->device); }
  }
  ~DevGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

extern "C" void epr_default_options(epr_options* o) {
  if (!o) return;
  o->order = 2; o->wkb1 = 1; o->symbol = 0; o->max_shift_px = 16.f; o->i_min = 1e-6f; o->newton_iters = 4;
  o->init = 0; o->output = 0; o->out_bin = 0; o->mu_rel = NULL; o->nonlocal_wkb1 = 0;
}

extern "C" const char* epr_version(void) { return "epr-b200 0.2.1 (sm_100a)"; }

extern "C" const char* epr_last_error(epr_plan_t p) { return p ? p->err : "null plan"; }

extern "C" long long epr_launch_count(epr_plan_t p) { return p ? p->launches : 0; }

template <typename T> static cudaError_t upload(T** dst, const std::vector<T>& v) {
  cudaError_t e = cudaMalloc((void**)dst, v.size() * sizeof(T));
  if (e != cudaSuccess) return e;
  return cudaMemcpy(*dst, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice);
}

static std::vector<float2> twiddles(int n, int count) {
  std::vector<float2> v(count);
  for (int m = 0; m < count; ++m) {
    const double th = -2.0 * M_PI * (double)m / (double)n;
    v[m] = make_float2((float)cos(th), (float)sin(th));
  }
  return v;
}

// per-pass tables of epr_fft.cuh: tab[off_i + (r−1)·P_i + k] = exp(−2πi r k/(P_i R_i))
static std::vector<float2> pass_twiddles(int n, bool rev) {
  using namespace eprfft;
  std::vector<float2> v(tw_total(n, rev) > 0 ? tw_total(n, rev) : 1, make_float2(1.f, 0.f));
  const int np = num_passes(n);
  for (int i = 1; i < np; ++i) {
    const int R = sched_radix(n, i, rev), P = sched_P(n, i, rev), off = tw_offset(n, i, rev);
    for (int r = 1; r < R; ++r)
      for (int k = 0; k < P; ++k) {
        const double th = -2.0 * M_PI * (double)r * (double)k / ((double)P * (double)R);
        v[off + (r - 1) * P + k] = make_float2((float)cos(th), (float)sin(th));
      }
  }
  return v;
}

static std::vector<float> lambda_table(int n, int count, int symbol) {
  std::vector<float> v(count);
  for (int k = 0; k < count; ++k) {
    const int kk = (k <= n / 2) ? k : k - n;
    const double th = 2.0 * M_PI * (double)kk / (double)n;
    v[k] = (float)(symbol == 0 ? 2.0 - 2.0 * cos(th) : th * th);
  }
  return v;
}

// cuTensorMapEncodeTiled through the runtime's driver entry point (no link-time dependency on libcuda)
static bool make_spec_map(CUtensorMap* map, void* base, int nx, size_t rows, int box_rows) {
  typedef CUresult (*encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
  static encode_fn fn = NULL;
  if (!fn) {
    void* ptr = NULL;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &ptr, cudaEnableDefault, &qres) != cudaSuccess || !ptr ||
        qres != cudaDriverEntryPointSuccess)
      return false;
    fn = (encode_fn)ptr;
  }
  if (rows > 0xffffffffull) return false;
  const cuuint64_t dims[2] = {(cuuint64_t)nx, (cuuint64_t)rows};
  const cuuint64_t strides[1] = {(cuuint64_t)nx * sizeof(float)};
  const cuuint32_t box[2] = {8, (cuuint32_t)box_rows};
  const cuuint32_t estr[2] = {1, 1};
  return fn(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, base, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
            CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// Per-column tables of the general path from per-block scalars (reading R17(a)): block b
// covers columns [b nx/n_blocks, (b+1) nx/n_blocks), centre c_b = (b + ½) nx/n_blocks − ½; the value of column x is the
// linear interpolation between the two nearest centres, constant outside the outermost ones.  f_blk, gamma_blk, db_blk:
// [n_blocks][n_bins] (f normalised per block, γ with its one global normalisation).  Also the per-block filter
// coefficients a_s^{(b)} = α_s db_s^{(b)}/2, ā^{(b)} = Σ_s f_s^{(b)} a_s^{(b)} (R17(c)) and the block-filter workspace.
static epr_status set_columns(epr_plan_s* p, int n_blocks, const double* f_blk, const double* gamma_blk, const double* db_blk) {
  const int nx = p->nx, nb = p->n_bins;
  const int wb = nx / n_blocks;
  std::vector<double> w((size_t)n_blocks * nx, 0.0);
  for (int x = 0; x < nx; ++x) {
    if (n_blocks == 1) { w[x] = 1.0; continue; }
    double t = ((double)x - (0.5 * wb - 0.5)) / (double)wb;            // position in units of blocks from the first centre
    t = t < 0.0 ? 0.0 : (t > n_blocks - 1.0 ? n_blocks - 1.0 : t);
    int b0 = (int)floor(t);
    if (b0 > n_blocks - 2) b0 = n_blocks - 2;
    const double fr = t - b0;
    w[(size_t)b0 * nx + x] = 1.0 - fr;
    w[(size_t)(b0 + 1) * nx + x] += fr;
  }
  // Everything new is built beside the old state and swapped in only when all of it exists: a failed allocation leaves
  // the plan exactly as it was (old tables, old n_blocks, old workspace), still usable.
  double* h_col_new = (double*)malloc(sizeof(double) * 3 * nb * nx);
  if (!h_col_new) FAIL(p, EPR_ENOMEM, "column tables");
  double *hf = h_col_new, *hg = hf + (size_t)nb * nx, *ha = hg + (size_t)nb * nx;
  for (int s = 0; s < nb; ++s)
    for (int x = 0; x < nx; ++x) {
      double f = 0, g = 0, db = 0;
      for (int b = 0; b < n_blocks; ++b) {
        const double wv = w[(size_t)b * nx + x];
        f += wv * f_blk[b * nb + s]; g += wv * gamma_blk[b * nb + s]; db += wv * db_blk[b * nb + s];
      }
      hf[(size_t)s * nx + x] = f; hg[(size_t)s * nx + x] = g; ha[(size_t)s * nx + x] = p->h_alpha[s] * db / 2.0;
    }
  // one device allocation: f, γ, a, fixCorr (float [nb][nx]), fixFi (u32 [nb][nx]), fsum_dev (float [nx]), wblk (float [n_blocks][nx])
  const size_t n1 = (size_t)nb * nx;
  std::vector<float> host(5 * n1 + nx + (size_t)n_blocks * nx);
  float *df = host.data(), *dg = df + n1, *da = dg + n1, *dc = da + n1;
  unsigned* dF = reinterpret_cast<unsigned*>(dc + n1);
  float *ds = reinterpret_cast<float*>(dF + n1), *dw = ds + nx;
  for (int x = 0; x < nx; ++x) ds[x] = 0.f;
  for (size_t i = 0; i < n1; ++i) {
    df[i] = (float)hf[i]; dg[i] = (float)hg[i]; da[i] = (float)ha[i];
    const double fix = (double)df[i] * EPR_FIX_ONE;                    // the device uses the fp32-rounded f_s(x) consistently
    dF[i] = (unsigned)llrint(fix);
    dc[i] = (float)((double)dF[i] / EPR_FIX_ONE - (double)df[i]);
  }
  for (int x = 0; x < nx; ++x) {
    double fs = 0;
    for (int s = 0; s < nb; ++s) fs += (double)df[(size_t)s * nx + x];
    ds[x] = (float)(fs - 1.0);
  }
  for (size_t i = 0; i < (size_t)n_blocks * nx; ++i) dw[i] = (float)w[i];
  void* store_new = NULL;
  float* qblk_new = NULL;
  // the general path puts work_batch · n_bins planes into gridDim.y / .z (limit 65535): small grids with a huge batch
  int work_new = p->work_batch;
  if (work_new > 65535 / nb) work_new = 65535 / nb;
  const bool need_q = !p->qblk || n_blocks > p->n_blocks;
  cudaError_t ce = cudaMalloc(&store_new, host.size() * sizeof(float));
  if (ce == cudaSuccess) ce = cudaMemcpy(store_new, host.data(), host.size() * sizeof(float), cudaMemcpyHostToDevice);
  // block-filter workspace: n_blocks planes per projection of the work batch.  The plan's work batch was sized without
  // it; when it does not fit, the work batch is halved until it does (batches are processed in passes of work_batch).
  while (ce == cudaSuccess && need_q) {
    ce = cudaMalloc((void**)&qblk_new, (size_t)n_blocks * work_new * nx * p->ny * sizeof(float));
    if (ce != cudaErrorMemoryAllocation || work_new == 1) break;
    cudaGetLastError();
    ce = cudaSuccess;
    work_new = (work_new + 1) / 2;
  }
  if (ce != cudaSuccess) {
    cudaGetLastError();
    cudaFree(store_new); cudaFree(qblk_new); free(h_col_new);
    FAIL(p, ce == cudaErrorMemoryAllocation ? EPR_ENOMEM : EPR_ECUDA, "column tables / block-filter workspace (%d blocks): %s",
         n_blocks, cudaGetErrorString(ce));
  }
  if (p->graph_exec) { cudaGraphExecDestroy(p->graph_exec); p->graph_exec = NULL; }   // it references the old tables
  free(p->h_col);
  p->h_col = h_col_new;
  cudaFree(p->cols_store);
  p->cols_store = store_new;
  if (need_q) { cudaFree(p->qblk); p->qblk = qblk_new; }
  p->work_batch = work_new;
  p->raymap_batch = 0;                                 // a stored ray map belongs to the previous scalars
  float* base = (float*)p->cols_store;
  p->cols.f = base; p->cols.gamma = base + n1; p->cols.a = base + 2 * n1; p->cols.fixCorr = base + 3 * n1;
  p->cols.fixFi = reinterpret_cast<const unsigned*>(base + 4 * n1);
  p->cols.fsum_dev = base + 5 * n1; p->cols.wblk = base + 5 * n1 + nx;
  // bounds for the tuned non-local kernels (ring width, staged halo, clamp test): the largest a_s(x) γ_s(x) of every line
  p->lines_bound = p->lines;
  for (int s = 0; s < nb; ++s) {
    float m = 0.f;
    for (int x = 0; x < nx; ++x) m = fmaxf(m, da[(size_t)s * nx + x] * dg[(size_t)s * nx + x]);
    p->lines_bound.a[s] = m * 1.000001f;               // (the kernels form a·γ in fp32 from the two table entries)
    p->lines_bound.gamma[s] = 1.f;
  }
  for (int b = 0; b < n_blocks; ++b) {
    double abar = 0;
    for (int s = 0; s < nb; ++s) {
      const double a = p->h_alpha[s] * db_blk[b * nb + s] / 2.0;
      p->a_blk[b][s] = (float)a;
      abar += f_blk[b * nb + s] * a;
    }
    p->abar_blk[b] = (float)abar;
  }
  p->n_blocks = n_blocks;
  p->general = 1;
  return EPR_OK;
}

extern "C" epr_status epr_plan(epr_plan_t* out, int nx, int ny, double pixel_m, double L_m, int n_bins,
                               const double* energy_keV, const double* weight, const double* delta_over_beta,
                               epr_solver solver, int max_batch, const epr_options* opt) {
  if (!out) return EPR_EINVAL;
  *out = NULL;
  if (!energy_keV || !weight || !delta_over_beta) return EPR_EINVAL;
  if (n_bins < 1 || n_bins > EPR_MAX_BINS || max_batch < 1 || !(pixel_m > 0) || !(L_m > 0)) return EPR_EINVAL;
  if (solver != EPR_LOCAL && solver != EPR_NONLOCAL) return EPR_EINVAL;
  if (nx < 1 || ny < 1) return EPR_EINVAL;
  if (nx < 8 || ny < 8) return EPR_ESIZE;              // include/epr.h: grids below 8 are unsupported sizes
  double wsum = 0;
  for (int s = 0; s < n_bins; ++s) {
    if (!(energy_keV[s] > 0) || !(weight[s] > 0) || !(delta_over_beta[s] > 0)) return EPR_EINVAL;
    wsum += weight[s];
  }
  epr_options o;
  epr_default_options(&o);
  if (opt) o = *opt;
  if ((o.order != 1 && o.order != 2) || (o.symbol != 0 && o.symbol != 1) || !(o.max_shift_px >= 0) ||
      o.max_shift_px > 30.f || !(o.i_min > 0) || o.newton_iters < 0 || o.newton_iters > 32 || o.output < 0 ||
      o.output > 2 || o.out_bin < 0 || o.out_bin >= n_bins)
    return EPR_EINVAL;
  // Grids: the tuned kernels take the sizes with a compiled FFT on 16-pixel-aligned grids; every other {2,3,5}-smooth
  // grid (8 … 8192 per axis) runs the general path (epr_general.cu), with the run-time-radix FFT where needed.
  const bool tuned_fft = nx % 2 == 0 && epr_fft_size_supported(nx) && epr_fft_size_supported(ny);
  const bool aligned = nx % 16 == 0 && ny % 16 == 0;
  if (!tuned_fft && !(epr_fftgen_supported(nx) && epr_fftgen_supported(ny))) return EPR_ESIZE;

  epr_plan_s* p = (epr_plan_s*)aligned_alloc(64, (sizeof(epr_plan_s) + 63) / 64 * 64);   // CUtensorMap members: 64-byte aligned
  if (!p) return EPR_ENOMEM;
  memset(p, 0, sizeof(epr_plan_s));
  *out = p;                                   // returned even on failure so that the caller can read the message
  p->nx = nx; p->ny = ny; p->n_bins = n_bins; p->max_batch = max_batch; p->solver = (int)solver; p->opt = o;
  p->opt.mu_rel = NULL;
  CU(p, cudaGetDevice(&p->device));
  CU(p, cudaDeviceGetAttribute(&p->sms, cudaDevAttrMultiProcessorCount, p->device));
  p->graph_mode = 1;
  { const char* g = getenv("EPR_GRAPH"); if (g) p->graph_mode = atoi(g); }

  // per-line scalars: k_s = 2πE/(hc); α_s = L/(k_s p²) (Eq. (2)); a_s = α_s db_s/2 (Eq. (6));
  // γ_s ∝ 1/(E_s db_s) normalised to Σ f γ = 1 (R11)
  double gsum = 0;
  for (int s = 0; s < n_bins; ++s) {
    const double k = 2.0 * M_PI * energy_keV[s] / HC_KEV_M;
    p->h_alpha[s] = L_m / (k * pixel_m * pixel_m);
    p->h_db[s] = delta_over_beta[s];
    p->h_a[s] = p->h_alpha[s] * delta_over_beta[s] / 2.0;
    p->h_f[s] = weight[s] / wsum;
    p->h_gamma[s] = o.mu_rel ? o.mu_rel[s] : 1.0 / (energy_keV[s] * delta_over_beta[s]);
    if (!(p->h_gamma[s] > 0)) FAIL(p, EPR_EINVAL, "mu_rel must be positive");
    gsum += p->h_f[s] * p->h_gamma[s];
  }
  EprLines& L = p->lines;
  L.n_bins = n_bins;
  double abar = 0;
  for (int s = 0; s < n_bins; ++s) {
    p->h_gamma[s] /= gsum;
    L.f[s] = (float)p->h_f[s];
    L.gamma[s] = (float)p->h_gamma[s];
    L.a[s] = (float)p->h_a[s];
    L.a2h[s] = (float)(0.5 * p->h_a[s] * p->h_a[s]);
    L.q4[s] = (float)(0.25 * p->h_alpha[s] * p->h_alpha[s]);
    // the device uses the fp32-rounded f_s consistently (deviation form): P_s − f_s with f_s = (float)
    L.fixF[s] = (double)L.f[s] * EPR_FIX_ONE;
    L.fixFi[s] = (unsigned)llrint(L.fixF[s]);
    L.fixCorr[s] = (float)((double)L.fixFi[s] / EPR_FIX_ONE - (double)L.f[s]);
    abar += p->h_f[s] * p->h_a[s];
  }
  L.abar = (float)abar;
  for (int s = 0; s < n_bins; ++s) {
    L.pj_a[s] = (float)(-p->h_gamma[s] * 1.4426950408889634);
    L.pj_b[s] = (float)log2(p->h_f[s]);
    L.pj_g2[s] = (float)(p->h_gamma[s] * p->h_gamma[s]);
    L.pj_g3[s] = (float)(p->h_gamma[s] * p->h_gamma[s] * p->h_gamma[s]);
  }
  for (int k = 0; k < 8; ++k) {
    double g = 0;
    for (int s = 0; s < n_bins; ++s) g += (double)L.f[s] * pow(p->h_gamma[s], k);
    L.pj_G[k] = (float)g;
  }
  L.gamma_max = 0.f;
  for (int s = 0; s < n_bins; ++s) L.gamma_max = fmaxf(L.gamma_max, L.gamma[s]);
  double fs = 0;
  for (int s = 0; s < n_bins; ++s) fs += (double)L.f[s];
  L.fsum_dev = (float)(fs - 1.0);

  const int M = nx / 2;
  p->fft_generic = tuned_fft ? 0 : 1;
  p->general = (!tuned_fft || !aligned) ? 1 : 0;
  p->n_blocks = 1;
  if (tuned_fft) {
    CU(p, upload(&p->tw_row, pass_twiddles(M, false)));
    CU(p, upload(&p->tw_r2c, twiddles(nx, M)));
    CU(p, upload(&p->tw_col, pass_twiddles(ny, false)));
    CU(p, upload(&p->tw_col_inv, pass_twiddles(ny, true)));
  } else {
    CU(p, upload(&p->tw_gen_x, twiddles(nx, nx)));
    CU(p, upload(&p->tw_gen_y, twiddles(ny, ny)));
  }
  CU(p, upload(&p->lam_x, lambda_table(nx, M + 1, o.symbol)));
  CU(p, upload(&p->lam_y, lambda_table(ny, ny, o.symbol)));

  // workspaces, sized for `work` projections at a time (≤ max_batch; bounded so that they stay within ~12 GB)
  const size_t plane = (size_t)nx * ny;
  size_t per_proj = plane * sizeof(float) * ((size_t)n_bins * (solver == EPR_NONLOCAL ? 4 : 3) + 2);
  int work = max_batch;
  const char* env = getenv("EPR_WORK_BATCH");
  size_t cap = (size_t)12 << 30;
  if (per_proj * (size_t)work > cap) work = (int)(cap / per_proj);
  if (env && atoi(env) > 0) work = atoi(env) < max_batch ? atoi(env) : max_batch;
  if (work < 1) work = 1;
  p->work_batch = work;
  const size_t wb = (size_t)work;
  cudaError_t e = cudaSuccess;
  if (e == cudaSuccess) e = cudaMalloc((void**)&p->d_flags, 4 * sizeof(unsigned));
  if (e == cudaSuccess) e = cudaMemset(p->d_flags, 0, 4 * sizeof(unsigned));
  if (e == cudaSuccess) e = cudaMalloc((void**)&p->tau, wb * plane * sizeof(float));
  if (e == cudaSuccess) e = cudaMalloc((void**)&p->pred, wb * n_bins * plane * sizeof(float));
  if (e == cudaSuccess) e = cudaMalloc((void**)&p->res, wb * n_bins * plane * sizeof(float));
  if (e == cudaSuccess && solver == EPR_NONLOCAL) e = cudaMalloc((void**)&p->res2, wb * n_bins * plane * sizeof(float));
  if (e == cudaSuccess && solver == EPR_NONLOCAL) e = cudaMalloc((void**)&p->gmax, wb * (size_t)((nx + 15) / 16) * ((ny + 15) / 16) * sizeof(float));
  const size_t spf = p->fft_generic ? epr_fftgen_spec_floats(p) : plane;     // floats per spectrum plane
  if (e == cudaSuccess) e = cudaMalloc((void**)&p->spec, wb * n_bins * spf * sizeof(float));
  if (e == cudaSuccess) e = cudaMalloc((void**)&p->spec_sum, wb * spf * sizeof(float));
  if (e != cudaSuccess) FAIL(p, e == cudaErrorMemoryAllocation ? EPR_ENOMEM : EPR_ECUDA, "workspace: %s", cudaGetErrorString(e));
  // TMA descriptors for the column kernel (power-of-two ny ≥ 256, whole 4-column tiles): the spectra seen as
  // [rows = planes·ny][nx floats], box = 8 floats (4 complex columns) x 256 rows, no swizzle.
  p->tma_ok = 0;
  if (tuned_fft && ny >= 256 && nx % 8 == 0) {
    int br = 256;
    while (ny % br != 0) --br;                       // 256 for powers of two, 240 for 2160, 160 for 320
    p->tma_box_rows = br;
    if (br >= 64 && make_spec_map(&p->map_spec, p->spec, nx, (size_t)wb * n_bins * ny, br) &&
        make_spec_map(&p->map_spec_sum, p->spec_sum, nx, (size_t)wb * ny, br))
      p->tma_ok = 1;
  }
  if (p->general) {                                    // constant columns: the uniform spectrum on the general path
    double fb[EPR_MAX_BINS], gb[EPR_MAX_BINS], dbb[EPR_MAX_BINS];
    for (int s = 0; s < n_bins; ++s) { fb[s] = p->h_f[s]; gb[s] = p->h_gamma[s]; dbb[s] = p->h_db[s]; }
    epr_status st = set_columns(p, 1, fb, gb, dbb);
    if (st != EPR_OK) return st;
  }
  return EPR_OK;
}

// Optional per-kernel timing: CUDA events are recorded around every kernel launch on the launch stream while
// enabled; epr_profile_read synchronises, accumulates and returns total ms and launch count per kernel family.
extern "C" epr_status epr_profile_enable(epr_plan_t p, int on) {
  if (!p) return EPR_EINVAL;
  if (!p->prof) {
    EprProf* pr = new EprProf();
    for (int i = 0; i < K_COUNT; ++i) { pr->ms[i] = 0; pr->n[i] = 0; }
    p->prof = pr;
  }
  p->prof_on = on ? 1 : 0;
  return EPR_OK;
}

extern "C" int epr_profile_read(epr_plan_t p, int max_kernels, const char** names, double* total_ms, long long* count,
                                int reset) {
  if (!p || !p->prof) return 0;
  DevGuard dg(p);
  EprProf* pr = (EprProf*)p->prof;
  cudaDeviceSynchronize();
  for (auto& r : pr->recs) {
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, r.a, r.b) == cudaSuccess) { pr->ms[r.tag] += ms; pr->n[r.tag] += 1; }
    cudaEventDestroy(r.a);
    cudaEventDestroy(r.b);
  }
  pr->recs.clear();
  int k = 0;
  for (int i = 0; i < K_COUNT && k < max_kernels; ++i) {
    if (!pr->n[i]) continue;
    if (names) names[k] = K_NAMES[i];
    if (total_ms) total_ms[k] = pr->ms[i];
    if (count) count[k] = pr->n[i];
    ++k;
  }
  if (reset) for (int i = 0; i < K_COUNT; ++i) { pr->ms[i] = 0; pr->n[i] = 0; }
  return k;
}

extern "C" epr_status epr_plan_lines(epr_plan_t p, double* f, double* gamma, double* a, double* alpha) {
  if (!p) return EPR_EINVAL;
  for (int s = 0; s < p->n_bins; ++s) {
    if (f) f[s] = p->h_f[s];
    if (gamma) gamma[s] = p->h_gamma[s];
    if (a) a[s] = p->h_a[s];
    if (alpha) alpha[s] = p->h_alpha[s];
  }
  return EPR_OK;
}

// x-dependent effective spectrum (reading R17): replaces the plan's uniform
// spectrum by n_blocks block profiles; the plan then runs the general path.
extern "C" epr_status epr_plan_profiles(epr_plan_t p, int n_blocks, const double* weight, const double* delta_over_beta,
                                        const double* mu_rel) {
  if (!p) return EPR_EINVAL;
  DevGuard dg(p);
  if (!weight || !delta_over_beta) FAIL(p, EPR_EINVAL, "epr_plan_profiles: NULL pointer");
  if (n_blocks < 1 || n_blocks > EPR_MAX_BLOCKS || p->nx % n_blocks != 0)
    FAIL(p, EPR_EINVAL, "epr_plan_profiles: n_blocks = %d must be in 1..%d and divide nx = %d", n_blocks, EPR_MAX_BLOCKS, p->nx);
  const int nb = p->n_bins;
  std::vector<double> f((size_t)n_blocks * nb), g((size_t)n_blocks * nb), db((size_t)n_blocks * nb);
  double G = 0;
  for (int b = 0; b < n_blocks; ++b) {
    double wsum = 0;
    for (int s = 0; s < nb; ++s) {
      const double w = weight[b * nb + s], d = delta_over_beta[b * nb + s];
      if (!(w > 0) || !(d > 0) || (mu_rel && !(mu_rel[b * nb + s] > 0)))
        FAIL(p, EPR_EINVAL, "epr_plan_profiles: weights, delta/beta and mu_rel must be positive (block %d, line %d)", b, s);
      wsum += w;
    }
    for (int s = 0; s < nb; ++s) {
      f[b * nb + s] = weight[b * nb + s] / wsum;
      db[b * nb + s] = delta_over_beta[b * nb + s];
      // γ_s ∝ 1/(E_s db_s) (R11) or the caller's relative attenuation; E_s from α_s = L/(k_s p²): 1/E_s ∝ α_s
      g[b * nb + s] = mu_rel ? mu_rel[b * nb + s] : p->h_alpha[s] / db[b * nb + s];
      G += f[b * nb + s] * g[b * nb + s];
    }
  }
  G /= n_blocks;                                       // ONE normalisation for the whole detector: τ is one thickness field
  for (auto& v : g) v /= G;
  CU(p, cudaDeviceSynchronize());                      // the tables may be in use by enqueued work
  epr_status st = set_columns(p, n_blocks, f.data(), g.data(), db.data());
  if (st != EPR_OK) return st;
  if (p->graph_exec) { cudaGraphExecDestroy(p->graph_exec); p->graph_exec = NULL; }
  return EPR_OK;
}

extern "C" epr_status epr_plan_columns(epr_plan_t p, double* f, double* gamma, double* a) {
  if (!p) return EPR_EINVAL;
  const size_t n = (size_t)p->n_bins * p->nx;
  for (int s = 0; s < p->n_bins; ++s)
    for (int x = 0; x < p->nx; ++x) {
      const size_t i = (size_t)s * p->nx + x;
      if (f) f[i] = p->h_col ? p->h_col[i] : p->h_f[s];
      if (gamma) gamma[i] = p->h_col ? p->h_col[n + i] : p->h_gamma[s];
      if (a) a[i] = p->h_col ? p->h_col[2 * n + i] : p->h_a[s];
    }
  return EPR_OK;
}

extern "C" epr_status epr_read_flags(epr_plan_t p, unsigned* flags, int clear) {
  if (!p) return EPR_EINVAL;
  if (!flags) FAIL(p, EPR_EINVAL, "epr_read_flags: NULL pointer");
  DevGuard dg(p);
  CU(p, cudaDeviceSynchronize());
  CU(p, cudaMemcpy(flags, p->d_flags, sizeof(unsigned), cudaMemcpyDeviceToHost));
  if (clear) CU(p, cudaMemset(p->d_flags, 0, sizeof(unsigned)));
  return EPR_OK;
}

extern "C" epr_status epr_destroy(epr_plan_t p) {
  if (!p) return EPR_EINVAL;
  DevGuard dg(p);
  cudaDeviceSynchronize();
  cudaFree(p->tw_row); cudaFree(p->tw_r2c); cudaFree(p->tw_col); cudaFree(p->tw_col_inv); cudaFree(p->lam_x); cudaFree(p->lam_y);
  cudaFree(p->tau); cudaFree(p->pred); cudaFree(p->res); cudaFree(p->res2); cudaFree(p->spec); cudaFree(p->spec_sum);
  cudaFree(p->d_flags); cudaFree(p->cols_store); cudaFree(p->qblk); cudaFree(p->tw_gen_x); cudaFree(p->tw_gen_y);
  free(p->h_col);
  cudaFree(p->raymap); cudaFree(p->gmax); cudaFree(p->os_d); cudaFree(p->os_out); cudaFree(p->diag_partial);
  if (p->graph_exec) cudaGraphExecDestroy(p->graph_exec);
  if (p->prof) { epr_profile_read(p, 0, NULL, NULL, NULL, 1); delete (EprProf*)p->prof; }
  for (int i = 0; i < 2; ++i) { cudaFree(p->stage_in[i]); cudaFree(p->stage_out[i]); }
  for (int i = 0; i < 3; ++i) if (p->hstream[i]) cudaStreamDestroy(p->hstream[i]);
  for (int i = 0; i < 6; ++i) if (p->hev[i]) cudaEventDestroy(p->hev[i]);
  free(p);
  return EPR_OK;
}

static epr_status check_call(epr_plan_t p, int batch) {
  if (!p) return EPR_EINVAL;
  if (batch < 1 || batch > p->max_batch) FAIL(p, EPR_EINVAL, "batch %d outside [1, max_batch = %d]", batch, p->max_batch);
  return EPR_OK;
}

// ----------------------------------------------------------------------------------------------- operators
static epr_status ensure_raymap(epr_plan_t p) {
  if (p->raymap) return EPR_OK;
  const size_t n = (size_t)p->max_batch * p->n_bins * p->nx * p->ny;       // the whole batch: epr_adjoint / epr_transport follow
  cudaError_t e = cudaMalloc((void**)&p->raymap, n * sizeof(float2));
  if (e != cudaSuccess) FAIL(p, EPR_ENOMEM, "ray map storage: %s", cudaGetErrorString(e));
  return EPR_OK;
}

extern "C" epr_status epr_forward(epr_plan_t p, int batch, const float* tau, float* P_sum, float* P_bins, void* stream) {
  epr_status st = check_call(p, batch);
  if (st != EPR_OK) return st;
  DevGuard dg(p);
  if (!tau || !P_sum) FAIL(p, EPR_EINVAL, "epr_forward: NULL tau or P_sum");
  cudaStream_t cs = (cudaStream_t)stream;
  const size_t plane = (size_t)p->nx * p->ny;
  if (p->solver == EPR_NONLOCAL && (st = ensure_raymap(p)) != EPR_OK) return st;
  for (int b0 = 0; b0 < batch; b0 += p->work_batch) {         // the prediction workspace holds work_batch projections
    const int nb = (batch - b0 < p->work_batch) ? batch - b0 : p->work_batch;
    const float* t = tau + (size_t)b0 * plane;
    float* Ps = P_sum + (size_t)b0 * plane;
    float* Pb = P_bins ? P_bins + (size_t)b0 * p->n_bins * plane : NULL;
    if (p->general) {
      if (p->solver == EPR_LOCAL) {
        KL(p, K_FWD_LOCAL, cs, epr_gen_forward_local(p, nb, t, p->pred, cs));
      } else {
        KL(p, K_SPLAT, cs, epr_gen_splat(p, nb, t, NULL, NULL, p->raymap + (size_t)b0 * p->n_bins * plane, (unsigned*)p->pred, cs));
        KL(p, K_SPLAT, cs, epr_gen_fix2float(p, nb, (unsigned*)p->pred, 0, cs));
        if (p->opt.nonlocal_wkb1) KL(p, K_WKB1, cs, epr_gen_wkb1_sub(p, nb, t, p->pred, cs));
      }
      KL(p, K_PRED_OUT, cs, epr_gen_pred_out(p, nb, p->pred, Ps, Pb, cs));
      continue;
    }
    if (p->solver == EPR_LOCAL) {
      KL(p, K_FWD_LOCAL, cs, epr_launch_forward_local(p, nb, t, NULL, p->pred, cs));
    } else {
      KL(p, K_SPLAT, cs, epr_launch_splat(p, nb, t, NULL, NULL, p->raymap + (size_t)b0 * p->n_bins * plane, p->pred, 0, NULL, cs));
      if (p->opt.nonlocal_wkb1) KL(p, K_WKB1, cs, epr_launch_wkb1_sub(p, nb, t, p->pred, cs));
    }
    KL(p, K_PRED_OUT, cs, epr_launch_pred_out(p, nb, p->pred, Ps, Pb, cs));
  }
  if (p->solver == EPR_NONLOCAL) p->raymap_batch = batch;
  return EPR_OK;
}

extern "C" epr_status epr_adjoint(epr_plan_t p, int batch, const float* e_bins, float* r_bins, void* stream) {
  epr_status st = check_call(p, batch);
  if (st != EPR_OK) return st;
  DevGuard dg(p);
  if (!e_bins || !r_bins) FAIL(p, EPR_EINVAL, "epr_adjoint: NULL pointer");
  cudaStream_t cs = (cudaStream_t)stream;
  const size_t n = (size_t)batch * p->n_bins * p->nx * p->ny;
  if (p->solver == EPR_LOCAL) {
    if (e_bins != r_bins) CU(p, cudaMemcpyAsync(r_bins, e_bins, n * sizeof(float), cudaMemcpyDeviceToDevice, cs));
    return EPR_OK;
  }
  if (e_bins == r_bins) FAIL(p, EPR_EINVAL, "epr_adjoint: the gather cannot run in place");
  if (!p->raymap || p->raymap_batch < batch) FAIL(p, EPR_EINVAL, "epr_adjoint: no ray map stored for batch %d (call epr_forward first)", batch);
  if (p->general) KL(p, K_GATHER, cs, epr_gen_gather(p, batch, NULL, p->raymap, e_bins, r_bins, cs));
  else KL(p, K_GATHER, cs, epr_launch_gather(p, batch, NULL, p->raymap, e_bins, r_bins, 0, cs));
  return EPR_OK;
}

extern "C" epr_status epr_transport(epr_plan_t p, int batch, const float* I_bins, float* P_bins, void* stream) {
  epr_status st = check_call(p, batch);
  if (st != EPR_OK) return st;
  DevGuard dg(p);
  if (!I_bins || !P_bins) FAIL(p, EPR_EINVAL, "epr_transport: NULL pointer");
  if (p->solver != EPR_NONLOCAL) FAIL(p, EPR_EINVAL, "epr_transport: non-local plans only");
  if (!p->raymap || p->raymap_batch < batch) FAIL(p, EPR_EINVAL, "epr_transport: no ray map stored for batch %d (call epr_forward first)", batch);
  cudaStream_t cs = (cudaStream_t)stream;
  const size_t plane = (size_t)p->nx * p->ny;
  if (I_bins == P_bins) FAIL(p, EPR_EINVAL, "epr_transport: the splat cannot run in place");
  if (p->general) {                                    // the caller's output planes serve as the fixed-point accumulators
    KL(p, K_SPLAT, cs, epr_gen_splat(p, batch, NULL, I_bins, p->raymap, NULL, (unsigned*)P_bins, cs));
    KL(p, K_SPLAT, cs, epr_gen_fix2float(p, batch, (unsigned*)P_bins, 1, cs));
    return EPR_OK;
  }
  KL(p, K_SPLAT, cs, epr_launch_splat(p, batch, NULL, I_bins, p->raymap, NULL, P_bins, 1, NULL, cs));
  return EPR_OK;
}

extern "C" epr_status epr_precondition(epr_plan_t p, int batch, const float* r_bins, float* q_bins, void* stream) {
  epr_status st = check_call(p, batch);
  if (st != EPR_OK) return st;
  DevGuard dg(p);
  if (!r_bins || !q_bins) FAIL(p, EPR_EINVAL, "epr_precondition: NULL pointer");
  cudaStream_t cs = (cudaStream_t)stream;
  const size_t plane = (size_t)p->nx * p->ny;
  for (int b0 = 0; b0 < batch; b0 += p->work_batch) {
    const int nb = (batch - b0 < p->work_batch) ? batch - b0 : p->work_batch;
    const int planes = nb * p->n_bins;
    const size_t off = (size_t)b0 * p->n_bins * plane;
    if (p->general) {
      // per-line filter of every block, blended with the interpolation weights (R17(c)); the input may alias the output,
      // so several blocks accumulate in a workspace first
      for (int b = 0; b < p->n_blocks; ++b) {
        KL(p, K_ROWS_R2C, cs, gen_r2c(p, planes, r_bins + off, 0.f, cs));
        KL(p, K_COLS, cs, gen_cols(p, planes, 0, b, p->spec, cs, 0));
        if (p->n_blocks == 1) { KL(p, K_ROWS_C2R, cs, gen_c2r(p, planes, p->spec, q_bins + off, cs)); break; }
        KL(p, K_ROWS_C2R, cs, gen_c2r(p, planes, p->spec, p->pred, cs));
        KL(p, K_UPDATE, cs, epr_gen_blend(p, planes, b, p->pred, p->res, b > 0, cs));
      }
      if (p->n_blocks > 1) CU(p, cudaMemcpyAsync(q_bins + off, p->res, (size_t)planes * plane * sizeof(float), cudaMemcpyDeviceToDevice, cs));
      continue;
    }
    KL(p, K_ROWS_R2C, cs, epr_launch_rows_r2c(p, planes, r_bins + off, 0.f, p->spec, cs));
    KL(p, K_COLS, cs, epr_launch_cols(p, planes, 0, p->spec, p->spec, cs));
    KL(p, K_ROWS_C2R, cs, epr_launch_rows_c2r(p, planes, p->spec, 0, 1.f, 0, q_bins + off, cs));
  }
  return EPR_OK;
}

// ----------------------------------------------------------------------------------------------- general path
// FFT back end of the general path: the tuned row / column kernels when both sizes have a compiled transform, the
// run-time-radix ones otherwise.  The filter of block b uses that block's coefficients (R17(c)).
static cudaError_t gen_r2c(epr_plan_t p, int planes, const float* in, float off, cudaStream_t cs) {
  return p->fft_generic ? epr_fftgen_rows_r2c(p, planes, in, off, p->spec, cs) : epr_launch_rows_r2c(p, planes, in, off, p->spec, cs);
}
static cudaError_t gen_cols(epr_plan_t p, int planes, int mode, int blk, float2* out, cudaStream_t cs, int stage) {
  EprLines lb = p->lines;
  for (int s = 0; s < p->n_bins; ++s) lb.a[s] = p->a_blk[blk][s];
  lb.abar = p->abar_blk[blk];
  return p->fft_generic ? epr_fftgen_cols(p, planes, mode, p->spec, out, cs, &lb) : epr_launch_cols(p, planes, mode, p->spec, out, cs, &lb, stage);
}
// Several block filters on the same residuals: transform the columns once, then filter + sum + inverse per block
// (the TMA column kernel's stages; power-of-two ny in 256 … 2048 on grids with TMA descriptors).
static bool cols_staged(epr_plan_t p) {
  const int ny = p->ny;
  return p->n_blocks > 1 && !p->fft_generic && p->tma_ok && ny >= 256 && ny <= 2048 && (ny & (ny - 1)) == 0 && (p->nx / 2) % 4 == 0;
}
static cudaError_t gen_c2r(epr_plan_t p, int planes, const float2* spec, float* q, cudaStream_t cs) {
  return p->fft_generic ? epr_fftgen_rows_c2r(p, planes, spec, q, cs) : epr_launch_rows_c2r(p, planes, spec, 0, 1.f, 0, q, cs);
}

// One pass of the loop over nb <= work_batch projections on the general path (same steps as retrieve_chunk).
static epr_status retrieve_chunk_general(epr_plan_t p, int nb, const float* d, float* tau, int iterations, float step,
                                         int b_first, cudaStream_t cs) {
  const size_t plane = (size_t)p->nx * p->ny;
  const int planes = nb * p->n_bins;
  const size_t bstride = (size_t)p->work_batch * plane;            // qblk[b] holds work_batch planes
  if (p->opt.init == 0) {
    // initial guess (R9, R17(c)): T⁰ − 1 = Σ_b wblk[b][x] IFFT(FFT(d − 1)/(1 + ā^{(b)} λ)), floored, projected
    KL(p, K_ROWS_R2C, cs, gen_r2c(p, nb, d, -1.f, cs));
    const int st2 = cols_staged(p) ? 2 : 0;
    if (st2) KL(p, K_COLS, cs, gen_cols(p, nb, 0, 0, p->spec, cs, 1));                          // columns transformed once
    for (int b = 0; b < p->n_blocks; ++b) {
      KL(p, K_COLS, cs, gen_cols(p, nb, 2, b, p->spec_sum, cs, st2));
      KL(p, K_ROWS_C2R, cs, gen_c2r(p, nb, p->spec_sum, p->qblk + b * bstride, cs));
    }
    KL(p, K_UPDATE, cs, epr_gen_update(p, nb, p->qblk, bstride, 1.f, 1, tau, cs));
  }
  for (int it = 0; it < iterations; ++it) {
    const float* r;
    if (p->solver == EPR_LOCAL) {
      KL(p, K_FWD_LOCAL, cs, epr_gen_forward_local(p, nb, tau, p->pred, cs));                   // a0 + a1-L
      KL(p, K_RESIDUAL, cs, epr_gen_residual(p, nb, d, p->pred, p->res, cs));                   // a2 (a3 = identity)
      r = p->res;
    } else if (p->nx % 16 == 0 && p->ny % 16 == 0) {
      // 16-pixel-aligned grid: the tuned tile kernels, reading the per-column tables (a0 + a1-N + a2 fused, then a3)
      if (p->opt.nonlocal_wkb1) {                      // variant: splat, WKB1 term, then the separate residual kernel
        KL(p, K_SPLAT, cs, epr_launch_splat_cols(p, nb, tau, p->pred, 0, NULL, cs));
        KL(p, K_WKB1, cs, epr_gen_wkb1_sub(p, nb, tau, p->pred, cs));
        KL(p, K_RESIDUAL, cs, epr_gen_residual(p, nb, d, p->pred, p->res, cs));
      } else {
        KL(p, K_SPLAT, cs, epr_launch_splat_cols(p, nb, tau, p->res, p->n_bins == 1 ? 2 : 3, d, cs));
      }
      r = p->res2;
    } else {
      KL(p, K_SPLAT, cs, epr_gen_splat(p, nb, tau, NULL, NULL, NULL, (unsigned*)p->res, cs));   // a0 + a1-N
      KL(p, K_SPLAT, cs, epr_gen_fix2float(p, nb, (unsigned*)p->res, 0, cs));
      if (p->opt.nonlocal_wkb1) KL(p, K_WKB1, cs, epr_gen_wkb1_sub(p, nb, tau, p->res, cs));
      KL(p, K_RESIDUAL, cs, epr_gen_residual(p, nb, d, p->res, p->res, cs));                    // a2, in place
      r = p->res2;
    }
    if (p->diag && it < p->diag_cap)                   // e_s are in p->res on every branch
      KL(p, K_DIAG, cs, epr_gen_diagnostics(p, nb, tau, p->res, p->diag + ((size_t)b_first * p->diag_cap + it) * 2, p->diag_cap * 2, cs));
    if (p->solver != EPR_LOCAL) {                      // a3
      if (p->nx % 16 == 0 && p->ny % 16 == 0) KL(p, K_GATHER, cs, epr_launch_gather_cols(p, nb, tau, p->res, p->res2, cs));
      else KL(p, K_GATHER, cs, epr_gen_gather(p, nb, tau, NULL, p->res, p->res2, cs));
    }
    KL(p, K_ROWS_R2C, cs, gen_r2c(p, planes, r, 0.f, cs));                                      // a4
    const int st2 = cols_staged(p) ? 2 : 0;
    if (st2) KL(p, K_COLS, cs, gen_cols(p, planes, 0, 0, p->spec, cs, 1));                      // columns transformed once
    for (int b = 0; b < p->n_blocks; ++b) {
      KL(p, K_COLS, cs, gen_cols(p, planes, 1, b, p->spec_sum, cs, st2));                       // Σ_s in Fourier space (R10), block b
      KL(p, K_ROWS_C2R, cs, gen_c2r(p, nb, p->spec_sum, p->qblk + b * bstride, cs));
    }
    KL(p, K_UPDATE, cs, epr_gen_update(p, nb, p->qblk, bstride, step, 0, tau, cs));             // a5 + a6
  }
  return EPR_OK;
}

// ----------------------------------------------------------------------------------------------- the loop
// One pass over `nb` ≤ work_batch projections.  tau is the state (device, [nb][ny][nx]).
// b_first: index of the chunk's first projection within the caller's batch (row of the diagnostics array).
static epr_status retrieve_chunk(epr_plan_t p, int nb, const float* d, float* tau, int iterations, float step,
                                 int b_first, cudaStream_t cs) {
  if (p->general) return retrieve_chunk_general(p, nb, d, tau, iterations, step, b_first, cs);
  const size_t plane = (size_t)p->nx * p->ny;
  const int planes = nb * p->n_bins;
  if (p->opt.init == 0) {
    // initial guess (R9): τ⁰ = project( max(IFFT(FFT(d)/(1+āλ)), i_min) ), in deviation form from d − 1
    KL(p, K_ROWS_R2C, cs, epr_launch_rows_r2c(p, nb, d, -1.f, p->spec, cs));
    KL(p, K_COLS, cs, epr_launch_cols(p, nb, 2, p->spec, p->spec_sum, cs));
    KL(p, K_ROWS_C2R, cs, epr_launch_rows_c2r(p, nb, p->spec_sum, 1, 1.f, 1, tau, cs));
  }
  for (int it = 0; it < iterations; ++it) {
    const float* r;
    if (p->solver == EPR_LOCAL) {
      if (p->n_bins == 1) {
        KL(p, K_FWD_LOCAL, cs, epr_launch_forward_local(p, nb, tau, d, p->res, cs));             // a0 + a1-L + a2 fused
      } else {
        KL(p, K_FWD_LOCAL, cs, epr_launch_forward_local(p, nb, tau, NULL, p->pred, cs));         // a0 + a1-L
        KL(p, K_RESIDUAL, cs, epr_launch_residual(p, nb, d, p->pred, p->res, cs));           // a2 (a3 = identity)
      }
      r = p->res;
      if (p->diag && it < p->diag_cap)
        KL(p, K_DIAG, cs, epr_launch_diagnostics(p, nb, tau, p->res, p->diag + ((size_t)b_first * p->diag_cap + it) * 2, p->diag_cap * 2, cs));
    } else {
      if (p->opt.nonlocal_wkb1) {                      // variant: splat, WKB1 term, then the separate residual kernel
        KL(p, K_SPLAT, cs, epr_launch_splat(p, nb, tau, NULL, NULL, NULL, p->pred, 0, NULL, cs));
        KL(p, K_WKB1, cs, epr_launch_wkb1_sub(p, nb, tau, p->pred, cs));
        KL(p, K_RESIDUAL, cs, epr_launch_residual(p, nb, d, p->pred, p->res, cs));
      } else if (p->n_bins == 1) {
        KL(p, K_SPLAT, cs, epr_launch_splat(p, nb, tau, NULL, NULL, NULL, p->res, 2, d, cs));       // a0 + a1-N + a2 fused
      } else {
        KL(p, K_SPLAT, cs, epr_launch_splat(p, nb, tau, NULL, NULL, NULL, p->res, 3, d, cs));       // a0 + a1-N + a2 fused
      }
      if (p->diag && it < p->diag_cap)
        KL(p, K_DIAG, cs, epr_launch_diagnostics(p, nb, tau, p->res, p->diag + ((size_t)b_first * p->diag_cap + it) * 2, p->diag_cap * 2, cs));
      KL(p, K_GATHER, cs, epr_launch_gather(p, nb, tau, NULL, p->res, p->res2, 1, cs));          // a3
      r = p->res2;
    }
    KL(p, K_ROWS_R2C, cs, epr_launch_rows_r2c(p, planes, r, 0.f, p->spec, cs));                 // a4
    KL(p, K_COLS, cs, epr_launch_cols(p, planes, 1, p->spec, p->spec_sum, cs));             // a4 (Σ_s in Fourier space, R10)
    KL(p, K_ROWS_C2R, cs, epr_launch_rows_c2r(p, nb, p->spec_sum, 1, step, 0, tau, cs));        // a4 + a5 + a6
  }
  return EPR_OK;
}

static epr_status retrieve_device(epr_plan_t p, int batch, const float* d, float* out, int iterations, float step,
                                  int b_first, cudaStream_t cs) {
  const size_t plane = (size_t)p->nx * p->ny;
  for (int b0 = 0; b0 < batch; b0 += p->work_batch) {
    const int nb = (batch - b0 < p->work_batch) ? batch - b0 : p->work_batch;
    float* o = out + (size_t)b0 * plane;
    float* tau = (p->opt.output == 0) ? o : p->tau;
    if (p->opt.init == 1 && tau != o) CU(p, cudaMemcpyAsync(tau, o, (size_t)nb * plane * sizeof(float), cudaMemcpyDeviceToDevice, cs));
    epr_status st = retrieve_chunk(p, nb, d + (size_t)b0 * plane, tau, iterations, step, b_first + b0, cs);
    if (st != EPR_OK) return st;
    if (p->opt.output != 0) KL(p, K_OUTPUT, cs, p->general ? epr_gen_output(p, nb, tau, o, cs) : epr_launch_output(p, nb, tau, o, cs));
  }
  return EPR_OK;
}

// Per-line distribution of the eikonal shift of a given thickness field (Fig. 6).
extern "C" epr_status epr_shift_histogram(epr_plan_t p, int batch, const float* tau, int n_hist, float bin_px, unsigned* hist,
                                          void* stream) {
  epr_status st = check_call(p, batch);
  if (st != EPR_OK) return st;
  DevGuard dg(p);
  if (!tau || !hist) FAIL(p, EPR_EINVAL, "epr_shift_histogram: NULL pointer");
  if (n_hist < 2 || n_hist > 1024 || !(bin_px > 0.f)) FAIL(p, EPR_EINVAL, "epr_shift_histogram: n_hist must be in 2..1024 and bin_px > 0");
  cudaStream_t cs = (cudaStream_t)stream;
  KL(p, K_DIAG, cs, epr_launch_shift_hist(p, batch, tau, n_hist, bin_px, hist, cs));
  return EPR_OK;
}

// Per-iteration diagnostics of the following retrievals: residual RMS and largest shift component (device array).
extern "C" epr_status epr_set_diagnostics(epr_plan_t p, float* diag, int capacity_iters) {
  if (!p) return EPR_EINVAL;
  DevGuard dg(p);
  if (diag && capacity_iters < 1) FAIL(p, EPR_EINVAL, "epr_set_diagnostics: capacity_iters must be >= 1");
  if (diag) {
    cudaError_t e = cudaSuccess;
    if (!p->diag_partial) e = cudaMalloc((void**)&p->diag_partial, (size_t)p->work_batch * 128 * sizeof(double));   // 64 x {Σe², max}
    if (e == cudaSuccess && !p->gmax && !p->general)
      e = cudaMalloc((void**)&p->gmax, (size_t)p->work_batch * (p->nx / 16) * (p->ny / 16) * sizeof(float));
    if (e != cudaSuccess) FAIL(p, e == cudaErrorMemoryAllocation ? EPR_ENOMEM : EPR_ECUDA, "diagnostics buffers: %s", cudaGetErrorString(e));
  }
  p->diag = diag;
  p->diag_cap = diag ? capacity_iters : 0;
  return EPR_OK;
}

static epr_status ensure_oversampling_buffers(epr_plan_t p) {
  if (p->os_d) return EPR_OK;
  const size_t plane = (size_t)p->nx * p->ny;
  cudaError_t e = cudaMalloc((void**)&p->os_d, (size_t)p->work_batch * plane * sizeof(float));
  if (e == cudaSuccess) e = cudaMalloc((void**)&p->os_out, (size_t)p->work_batch * plane * sizeof(float));
  if (e != cudaSuccess) FAIL(p, e == cudaErrorMemoryAllocation ? EPR_ENOMEM : EPR_ECUDA, "oversampling buffers: %s", cudaGetErrorString(e));
  return EPR_OK;
}

static epr_status check_oversampling(epr_plan_t p, int factor, const char* who) {
  if (factor < 1 || factor > 8 || p->nx % (4 * factor) != 0 || p->ny % factor != 0)
    FAIL(p, EPR_EINVAL, "%s: factor %d must be in 1..8 and divide the plan's grid %d x %d (nx / factor a multiple of 4)", who, factor, p->nx, p->ny);
  if (p->opt.init != 0) FAIL(p, EPR_EINVAL, "%s: opt.init = 1 (caller-supplied start) is not supported", who);
  return EPR_OK;
}

// replicate -> loop -> block mean for nb <= work_batch projections (coarse in / out may be any device buffers)
static epr_status retrieve_oversampled_chunk(epr_plan_t p, int factor, int nb, const float* d_coarse, float* out_coarse,
                                             int iterations, float step, int b_first, cudaStream_t cs) {
  KL(p, K_RESAMPLE, cs, epr_launch_upsample(p, nb, factor, d_coarse, p->os_d, cs));
  epr_status st = retrieve_device(p, nb, p->os_d, p->os_out, iterations, step, b_first, cs);
  if (st != EPR_OK) return st;
  KL(p, K_RESAMPLE, cs, epr_launch_downsample(p, nb, factor, p->os_out, out_coarse, cs));
  return EPR_OK;
}

// The loop on an oversampled grid (reading R16): the plan is the FINE grid's.
extern "C" epr_status epr_retrieve_oversampled(epr_plan_t p, int factor, int batch, const float* d, float* out,
                                               int iterations, float step, void* stream) {
  epr_status st = check_call(p, batch);
  if (st != EPR_OK) return st;
  DevGuard dg(p);
  if (!d || !out) FAIL(p, EPR_EINVAL, "epr_retrieve_oversampled: NULL pointer");
  if (iterations < 0 || !(step > 0.f)) FAIL(p, EPR_EINVAL, "epr_retrieve_oversampled: iterations must be >= 0 and step > 0");
  if ((st = check_oversampling(p, factor, "epr_retrieve_oversampled")) != EPR_OK) return st;
  if ((st = ensure_oversampling_buffers(p)) != EPR_OK) return st;
  cudaStream_t cs = (cudaStream_t)stream;
  const size_t plane = (size_t)p->nx * p->ny, cplane = plane / ((size_t)factor * factor);
  for (int b0 = 0; b0 < batch; b0 += p->work_batch) {
    const int nb = (batch - b0 < p->work_batch) ? batch - b0 : p->work_batch;
    st = retrieve_oversampled_chunk(p, factor, nb, d + (size_t)b0 * cplane, out + (size_t)b0 * cplane, iterations, step, b0, cs);
    if (st != EPR_OK) return st;
  }
  return EPR_OK;
}

extern "C" epr_status epr_retrieve(epr_plan_t p, int batch, const float* d, float* out, int iterations, float step,
                                   void* stream) {
  epr_status st = check_call(p, batch);
  if (st != EPR_OK) return st;
  DevGuard dg(p);
  if (!d || !out) FAIL(p, EPR_EINVAL, "epr_retrieve: NULL pointer");
  if (iterations < 0 || !(step > 0.f)) FAIL(p, EPR_EINVAL, "epr_retrieve: iterations must be >= 0 and step > 0");
  cudaStream_t cs = (cudaStream_t)stream;
  // Launch-bound sizes (a few hundred thousand pixels per launch: the kernels last microseconds): the whole loop is
  // captured once into a CUDA graph and replayed while the call's arguments stay the same.  Never under profiling
  // (events are recorded around every launch) and never on the legacy default stream (capture is illegal there).
  const size_t work = (size_t)batch * p->n_bins * p->nx * p->ny;
  bool use_graph = !p->prof_on && !p->diag && cs != 0 && cs != cudaStreamLegacy && cs != cudaStreamPerThread &&
                   (p->graph_mode == 2 || (p->graph_mode == 1 && work <= ((size_t)1 << 20)));
  if (use_graph) {                                     // a stream the caller is capturing already: just enqueue into it
    cudaStreamCaptureStatus cst = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(cs, &cst) != cudaSuccess || cst != cudaStreamCaptureStatusNone) { cudaGetLastError(); use_graph = false; }
  }
  if (!use_graph) return retrieve_device(p, batch, d, out, iterations, step, 0, cs);
  if (p->graph_exec && p->graph_d == d && p->graph_out == out && p->graph_batch == batch && p->graph_iters == iterations &&
      p->graph_step == step) {
    CU(p, cudaGraphLaunch(p->graph_exec, cs));
    p->launches += p->graph_launches;
    return EPR_OK;
  }
  if (p->graph_exec) { cudaGraphExecDestroy(p->graph_exec); p->graph_exec = NULL; }
  // one eager pass first: launchers set function attributes / query occupancy on their first call
  if (!p->graph_warm) {
    p->graph_warm = 1;
    return retrieve_device(p, batch, d, out, iterations, step, 0, cs);
  }
  // Capture is an optimisation: whatever goes wrong with it (a stream that cannot be captured, a launcher doing
  // first-use setup inside the capture, instantiation failure) ends in the eager path, never in an error.
  const long long l0 = p->launches;
  if (cudaStreamBeginCapture(cs, cudaStreamCaptureModeThreadLocal) != cudaSuccess) {
    cudaGetLastError();
    return retrieve_device(p, batch, d, out, iterations, step, 0, cs);
  }
  st = retrieve_device(p, batch, d, out, iterations, step, 0, cs);
  cudaGraph_t graph = NULL;
  cudaError_t ce = cudaStreamEndCapture(cs, &graph);
  if (st == EPR_OK && ce == cudaSuccess && graph) ce = cudaGraphInstantiate(&p->graph_exec, graph, 0);
  if (graph) cudaGraphDestroy(graph);
  if (st != EPR_OK || ce != cudaSuccess || !p->graph_exec) {
    cudaGetLastError();
    p->graph_exec = NULL;
    p->launches = l0;
    p->graph_mode = 0;                                 // do not try again on this plan
    return retrieve_device(p, batch, d, out, iterations, step, 0, cs);
  }
  p->graph_d = d; p->graph_out = out; p->graph_batch = batch; p->graph_iters = iterations; p->graph_step = step;
  p->graph_launches = p->launches - l0;
  CU(p, cudaGraphLaunch(p->graph_exec, cs));
  return EPR_OK;
}

// factor = 1: the plan's grid; factor > 1: host buffers on the detector grid, the loop on the plan's (fine) grid (R16)
// Closes a streaming session: waits for everything epr_retrieve_host_async enqueued on the plan's private streams.
static epr_status host_wait(epr_plan_t p) {
  if (!p->hsession) return EPR_OK;
  p->hsession = 0;
  p->hchunk = 0;
  CU(p, cudaStreamSynchronize(p->hstream[2]));
  CU(p, cudaStreamSynchronize(p->hstream[1]));
  CU(p, cudaStreamSynchronize(p->hstream[0]));
  return EPR_OK;
}

// async = 0: one self-contained call (waits for earlier device work on entry, returns when its last copy is done).
// async = 1: a call of a streaming session (chunk k + 1 is prepared while chunk k is processed): only the FIRST
// call of a session waits for earlier device work, no call waits at its end, and the chunk counter — which decides the
// staging buffer and the events a chunk must wait for — runs on across calls, so that the first copy in of call k + 1
// overlaps the last loop of call k and the last copy out of call k overlaps the first loop of call k + 1.
static epr_status retrieve_host_impl(epr_plan_t p, int factor, int batch, const float* d_host, float* out_host, int iterations,
                                     float step, int async) {
  if (batch < 1 || !d_host || !out_host) FAIL(p, EPR_EINVAL, "epr_retrieve_host: bad batch or NULL pointer");
  if (iterations < 0 || !(step > 0.f)) FAIL(p, EPR_EINVAL, "epr_retrieve_host: iterations must be >= 0 and step > 0");
  const size_t plane = (size_t)p->nx * p->ny / ((size_t)factor * factor);       // a plane of the HOST buffers
  // Host chunks are smaller than the device work batch so that the copies of chunk i±1 overlap the loop of chunk i:
  // about 256 MB of input per chunk (EPR_HOST_CHUNK overrides), at least min_chunks chunks per call when the batch allows
  // (C2, batch 64: chunks of 8 / 12 / 16 / 24 projections give 1012 / 1044 / 1060 / 987 projections/s end to end).
  // How many chunks a small batch is cut into follows the share of the copies: r = copy time / loop time per projection,
  // from 8 B/px over the host link (about 50 GB/s) against (iterations + 1) x the loop's algorithmic bytes at about
  // 2.5 TB/s.  Copies that are a small share (several lines: r < 0.1) are not worth loops over one or two projections,
  // whose launches underfill the GPU (measured, batch 4: C4 120.7 / 133.8 / 138.7 and C5 80.8 / 88.8 / 90.9 projections/s
  // with chunks of 1 / 2 / 4; C3, batch 8, r = 0.37: 464 / 542 / 542 / 500 with chunks of 1 / 2 / 4 / 8).
  const int nbn = p->n_bins;
  const double bpp = (p->solver == EPR_LOCAL) ? (nbn == 1 ? 40.0 : 24.0 + 24.0 * nbn) : (nbn == 1 ? 52.0 : 28.0 + 24.0 * nbn);
  // the two rates are tunables stated in include/epr.h (epr_retrieve_host): environment EPR_HOST_LINK_GBS, EPR_LOOP_GBS
  double link_gbs = 50.0, loop_gbs = 2500.0;
  { const char* e1 = getenv("EPR_HOST_LINK_GBS"); if (e1 && atof(e1) > 0) link_gbs = atof(e1); }
  { const char* e2 = getenv("EPR_LOOP_GBS"); if (e2 && atof(e2) > 0) loop_gbs = atof(e2); }
  const double r = (8.0 / link_gbs) / ((iterations + 1) * bpp * factor * factor / loop_gbs);
  const int min_chunks = r >= 0.3 ? 4 : r >= 0.15 ? 2 : 1;
  int wbch = (int)(((size_t)256 << 20) / (plane * sizeof(float)));
  if (wbch > (batch + min_chunks - 1) / min_chunks) wbch = (batch + min_chunks - 1) / min_chunks;
  if (nbn == 1 && wbch < 2) wbch = 2;              // one plane per launch leaves most SMs idle
  { const char* env = getenv("EPR_HOST_CHUNK"); if (env && atoi(env) > 0) wbch = atoi(env); }
  if (wbch < 1) wbch = 1;
  if (wbch > p->work_batch) wbch = p->work_batch;
  if (!getenv("EPR_HOST_CHUNK")) {                    // equal chunks: 16 projections in chunks of at most 15 go as 8 + 8, not 15 + 1
    const int nch = (batch + wbch - 1) / wbch;
    wbch = (batch + nch - 1) / nch;
  }
  if (!async || (p->stage_in[0] && p->stage_floats < (size_t)wbch * plane)) {
    const epr_status ws = host_wait(p);     // a self-contained call, or new staging buffers: the open session (if any) ends here
    if (ws != EPR_OK) return ws;
  }
  if (p->stage_in[0] && p->stage_floats < (size_t)wbch * plane) {           // staging buffers too small for this call: re-allocate
    CU(p, cudaDeviceSynchronize());
    for (int i = 0; i < 2; ++i) { cudaFree(p->stage_in[i]); cudaFree(p->stage_out[i]); p->stage_in[i] = p->stage_out[i] = NULL; }
  }
  if (!p->stage_in[0]) {
    for (int i = 0; i < 2; ++i) {
      CU(p, cudaMalloc((void**)&p->stage_in[i], (size_t)wbch * plane * sizeof(float)));
      CU(p, cudaMalloc((void**)&p->stage_out[i], (size_t)wbch * plane * sizeof(float)));
    }
    p->stage_chunk = wbch;
    p->stage_floats = (size_t)wbch * plane;
  }
  if (!p->hstream[0]) {
    for (int i = 0; i < 3; ++i) CU(p, cudaStreamCreateWithFlags(&p->hstream[i], cudaStreamNonBlocking));
    for (int i = 0; i < 6; ++i) CU(p, cudaEventCreateWithFlags(&p->hev[i], cudaEventDisableTiming));
  }
  cudaStream_t s_in = p->hstream[0], s_cmp = p->hstream[1], s_out = p->hstream[2];
  // The call works on private streams and on the plan's shared workspaces: whatever earlier calls on this plan enqueued
  // on the caller's streams (they only enqueue and return) must have finished first.
  if (!p->hsession) CU(p, cudaDeviceSynchronize());
  const bool head_taper = !p->hsession;     // inside a session the previous call's last loop covers this call's first copy
  if (async) p->hsession = 1;
  // Tapered schedule: the first copy in and the last copy out cannot overlap any compute, so the first and the last
  // chunks are small (wbch/4, wbch/2, wbch, …, wbch, wbch/2, wbch/4) when the batch holds at least three full chunks.
  const bool taper = wbch >= 4 && batch >= 3 * wbch;
  const int head[2] = {wbch / 4, wbch / 2};
  int chunk = 0, nb = 0;
  for (int b0 = 0; b0 < batch; b0 += nb, ++chunk) {
    const int left = batch - b0;
    nb = wbch;
    if (taper) {
      if (chunk < 2) { if (head_taper) nb = head[chunk]; }
      else if (async) { }                  // a session never knows its last call: no small chunks at the end of a call
      else if (left <= wbch / 4) nb = left;
      else if (left <= wbch / 4 + wbch / 2) nb = left - wbch / 4;
      else if (left < wbch + wbch / 4 + wbch / 2) nb = left - (wbch / 4 + wbch / 2);
    }
    if (nb > left) nb = left;
    const long long seq = async ? p->hchunk++ : (long long)chunk;         // position in the session / in this call
    const int buf = (int)(seq & 1);
    cudaEvent_t ev_in = p->hev[buf * 3 + 0], ev_cmp = p->hev[buf * 3 + 1], ev_out = p->hev[buf * 3 + 2];
    const size_t bytes = (size_t)nb * plane * sizeof(float);
    if (seq >= 2) {                       // buffers of chunk-2 must be free: its compute read stage_in, its D2H read stage_out
      CU(p, cudaStreamWaitEvent(s_in, ev_cmp, 0));
      if (p->opt.init == 1) CU(p, cudaStreamWaitEvent(s_in, ev_out, 0));
      CU(p, cudaStreamWaitEvent(s_cmp, ev_out, 0));
    }
    CU(p, cudaMemcpyAsync(p->stage_in[buf], d_host + (size_t)b0 * plane, bytes, cudaMemcpyHostToDevice, s_in));
    if (p->opt.init == 1)
      CU(p, cudaMemcpyAsync(p->stage_out[buf], out_host + (size_t)b0 * plane, bytes, cudaMemcpyHostToDevice, s_in));
    CU(p, cudaEventRecord(ev_in, s_in));
    CU(p, cudaStreamWaitEvent(s_cmp, ev_in, 0));
    epr_status st = factor == 1 ? retrieve_device(p, nb, p->stage_in[buf], p->stage_out[buf], iterations, step, b0, s_cmp)
                                : retrieve_oversampled_chunk(p, factor, nb, p->stage_in[buf], p->stage_out[buf], iterations, step, b0, s_cmp);
    if (st != EPR_OK) return st;
    CU(p, cudaEventRecord(ev_cmp, s_cmp));
    CU(p, cudaStreamWaitEvent(s_out, ev_cmp, 0));
    CU(p, cudaMemcpyAsync(out_host + (size_t)b0 * plane, p->stage_out[buf], bytes, cudaMemcpyDeviceToHost, s_out));
    CU(p, cudaEventRecord(ev_out, s_out));
  }
  if (async) return EPR_OK;
  CU(p, cudaStreamSynchronize(s_out));
  CU(p, cudaStreamSynchronize(s_cmp));
  return EPR_OK;
}

extern "C" epr_status epr_retrieve_host(epr_plan_t p, int batch, const float* d_host, float* out_host, int iterations,
                                        float step) {
  if (!p) return EPR_EINVAL;
  DevGuard dg(p);
  return retrieve_host_impl(p, 1, batch, d_host, out_host, iterations, step, 0);
}

extern "C" epr_status epr_retrieve_host_async(epr_plan_t p, int batch, const float* d_host, float* out_host, int iterations,
                                              float step) {
  if (!p) return EPR_EINVAL;
  DevGuard dg(p);
  return retrieve_host_impl(p, 1, batch, d_host, out_host, iterations, step, 1);
}

extern "C" epr_status epr_host_wait(epr_plan_t p) {
  if (!p) return EPR_EINVAL;
  DevGuard dg(p);
  return host_wait(p);
}

// Contiguous, balanced split of `total` independent projections over `parts`: part k gets [*start, *stop); the first
// total % parts parts take one more.  Pure host arithmetic (no device needed).
extern "C" epr_status epr_shard_range(int total, int k, int parts, int* start, int* stop) {
  if (total < 0 || parts < 1 || k < 0 || k >= parts || !start || !stop) return EPR_EINVAL;
  const int base = total / parts, rem = total % parts;
  *start = k * base + (k < rem ? k : rem);
  *stop = *start + base + (k < rem ? 1 : 0);
  return EPR_OK;
}

// One host batch over several plans (one per GPU): plan k takes a contiguous, balanced range of the batch
// (the split of epr_inputs.shard_range) as one streaming call, then all are awaited.
extern "C" epr_status epr_retrieve_host_multi(epr_plan_t* plans, int n_plans, int batch, const float* d_host, float* out_host,
                                              int iterations, float step) {
  if (!plans || n_plans < 1) return EPR_EINVAL;
  for (int k = 0; k < n_plans; ++k) {
    if (!plans[k]) return EPR_EINVAL;
    if (plans[k]->nx != plans[0]->nx || plans[k]->ny != plans[0]->ny) FAIL(plans[k], EPR_EINVAL, "epr_retrieve_host_multi: plans of different grids");
  }
  if (batch < 1 || !d_host || !out_host) FAIL(plans[0], EPR_EINVAL, "epr_retrieve_host_multi: bad batch or NULL pointer");
  const size_t plane = (size_t)plans[0]->nx * plans[0]->ny;
  epr_status first = EPR_OK;
  for (int k = 0; k < n_plans; ++k) {
    int b0 = 0, b1 = 0;
    epr_shard_range(batch, k, n_plans, &b0, &b1);
    if (b1 == b0) continue;
    DevGuard dg(plans[k]);
    const epr_status st = retrieve_host_impl(plans[k], 1, (int)(b1 - b0), d_host + (size_t)b0 * plane, out_host + (size_t)b0 * plane,
                                             iterations, step, 1);
    if (st != EPR_OK && first == EPR_OK) first = st;
  }
  for (int k = 0; k < n_plans; ++k) {
    DevGuard dg(plans[k]);
    const epr_status st = host_wait(plans[k]);
    if (st != EPR_OK && first == EPR_OK) first = st;
  }
  return first;
}

// Host buffers on the DETECTOR grid, the loop on the oversampled grid of the plan (R16): the same chunked,
// overlapped schedule; every chunk is replicated, retrieved and block-averaged on the device.
extern "C" epr_status epr_retrieve_oversampled_host(epr_plan_t p, int factor, int batch, const float* d_host, float* out_host,
                                                    int iterations, float step) {
  if (!p) return EPR_EINVAL;
  DevGuard dg(p);
  epr_status st = check_oversampling(p, factor, "epr_retrieve_oversampled_host");
  if (st != EPR_OK) return st;
  if ((st = ensure_oversampling_buffers(p)) != EPR_OK) return st;
  return retrieve_host_impl(p, factor, batch, d_host, out_host, iterations, step, 0);
}
