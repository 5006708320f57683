// epr_fftk.cu — the FFT-diagonal Paganin-type preconditioner P^{-1}_{1,s} as three
// hand-written kernels:   rows R2C  →  columns FFT · H_s (· Σ_s) · IFFT  →  rows C2R (+ update epilogue).
//
// Spectrum layout: [plane][ny][nx/2] float2; column kx = 0 packs the two purely real row-spectra X[0] (re)
// and X[nx/2] (im), so a plane of nx/2 complex columns holds the whole half spectrum.
// H_s(θ) = 1 / (1 + a_s λ(θ)) with λ = λx[kx] + λy[ky] from two 1-D tables (discrete or continuous symbol, R5);
// the 1/(nx·ny) normalisation is folded into H.
#include <type_traits>
#include "epr_fft.cuh"
#include "epr_internal.h"
#include "epr_math.cuh"
#include "epr_tma.cuh"

using namespace eprfft;

template <int M> struct RowCfg {                // M = nx/2 complex points per row
  static constexpr int TPC = threads_per_transform(M);   // threads per row
  static constexpr int ROWS = (TPC >= 128) ? 1 : (128 + TPC - 1) / TPC;   // rows per CTA (≥128 threads)
  static constexpr int NT = TPC * ROWS;
  static constexpr int PL = padded_len(M);
  static constexpr int PLA = (PL + 1) & ~1;      // row pitch of a stage: padded length, 16-byte aligned
  static constexpr int STAGE = ROWS * PLA;      // float2 per stage (ROWS rows; a stage is also the FFT work buffer)
  // dynamic shared memory: [2 mbarriers | pad to 128 B][stage 0][stage 1]
  static constexpr size_t OFF_STAGE = 128;
  static constexpr size_t SMEM = OFF_STAGE + 2 * (size_t)STAGE * sizeof(float2);
};

// The C2R row kernel is PERSISTENT and TMA-staged: a CTA walks over groups of ROWS consecutive rows (rows of all
// planes are contiguous, so one group is one contiguous chunk of HBM); while it transforms group i out of one
// shared-memory stage, one bulk asynchronous copy (cp.async.bulk, completion on an mbarrier) is already filling
// the other stage with group i + gridDim.x.  No warp waits on a global load inside the transform.  A stage row
// (M points, linear) is read into registers by the first pass and then REUSED in place as the padded work buffer
// of the remaining passes, so two stages are all the shared memory a CTA needs.
struct RowPipe {
  uint64_t* bar;
  float2* stage;
  const float2* src;
  int nrows, rows_per_group, M, row_pitch, stage_elems;
  __device__ __forceinline__ void issue(int grp, int buf) const {
    const int r0 = grp * rows_per_group;
    const int nr = min(rows_per_group, nrows - r0);
    const unsigned row_bytes = (unsigned)M * (unsigned)sizeof(float2);
    eprtma::fence_proxy_async();
    eprtma::mbar_expect_tx(&bar[buf], (unsigned)nr * row_bytes);
    for (int r = 0; r < nr; ++r)
      eprtma::bulk_g2s(stage + (size_t)buf * stage_elems + (size_t)r * row_pitch, src + (size_t)(r0 + r) * M, row_bytes, &bar[buf]);
  }
};

// ------------------------------------------------------------------------------------------------ rows R2C, direct
// global → registers (first pass) → shared-memory passes → registers (last pass) → pair exchange → global.
// One row group per CTA, many CTAs per SM: the forward row transform has no epilogue to hide a load behind and
// measures faster this way (6.7 vs 7.3 us per 2048² plane) than through the TMA stage, which is kept for C2R.
template <int M>
#ifndef R2C_MINB
#define R2C_MINB 1
#endif
__global__ void __launch_bounds__(RowCfg<M>::NT, (RowCfg<M>::NT <= 128) ? R2C_MINB : 1) k_rows_r2c_direct(int ny, const float* __restrict__ in, float in_offset,
                                                            const float2* __restrict__ tw, const float2* __restrict__ tw2,
                                                            float2* __restrict__ spec) {
  using C = RowCfg<M>;
  using EF = Engine<M, C::TPC, 1, false, false>;
  extern __shared__ float2 sm[];           // C::ROWS * C::PL
  const int lr = threadIdx.x / C::TPC, t = threadIdx.x - lr * C::TPC;
  const int row = blockIdx.x * C::ROWS + lr;
  const bool live = row < ny;
  const size_t rowoff = ((size_t)blockIdx.y * ny + (live ? row : 0)) * (size_t)M;
  float2* s = sm + lr * C::PL;
  const float2* src = reinterpret_cast<const float2*>(in) + rowoff;
  float2 u0[EF::G0::CNT][EF::R0], uL[EF::GL::CNT][EF::RL];
#pragma unroll
  for (int c = 0; c < EF::G0::CNT; ++c) {
    const int j = t + c * C::TPC;
#pragma unroll
    for (int r = 0; r < EF::R0; ++r) {
      float2 v = make_float2(0.f, 0.f);
      if ((EF::G0::FULL || j < EF::G0::T) && live) v = __ldg(&src[j + r * EF::G0::T]);
      u0[c][r] = make_float2(v.x + in_offset, v.y + in_offset);
    }
  }
  EF::run(u0, uL, s, 0, t, tw);
  __syncthreads();
#pragma unroll
  for (int c = 0; c < EF::GL::CNT; ++c) {
    const int j = t + c * C::TPC;
    if (EF::GL::FULL || j < EF::GL::T) {
#pragma unroll
      for (int q = 0; q < EF::RL; ++q) s[padi(j + q * EF::PL)] = uL[c][q];
    }
  }
  __syncthreads();
  // X[k] = ½(Z[k] + Z*[M−k]) − (i/2) w^k (Z[k] − Z*[M−k]),  w = e^{−2πi/nx};  k = 0: packed (X[0], X[M])
  if (live) {
    float2* dst = spec + rowoff;
#pragma unroll
    for (int c = 0; c < EF::GL::CNT; ++c) {
      const int j = t + c * C::TPC;
      if (EF::GL::FULL || j < EF::GL::T) {
#pragma unroll
        for (int q = 0; q < EF::RL; ++q) {
          const int k = j + q * EF::PL;
          const float2 zk = uL[c][q];
          if (k == 0) {
            dst[0] = make_float2(zk.x + zk.y, zk.x - zk.y);
          } else {
            const float2 zm = s[padi(M - k)];
            const float2 wk = __ldg(&tw2[k]);
            const float2 e = make_float2(0.5f * (zk.x + zm.x), 0.5f * (zk.y - zm.y));
            const float2 o = make_float2(0.5f * (zk.y + zm.y), -0.5f * (zk.x - zm.x));
            dst[k] = cadd(e, cmul(wk, o));
          }
        }
      }
    }
  }
}

// ------------------------------------------------------------------------------------------------ rows C2R
// EPI 0: out[row][x] = q.   EPI 1 / 2: τ[row][x] += δ(τ, step·q)  (projection increment, R10) for
// one line (closed form) / several lines (Newton).
#ifndef C2R_MINB
#define C2R_MINB 5
#endif
template <int M, int EPI>
__global__ void __launch_bounds__(RowCfg<M>::NT, (RowCfg<M>::NT <= 128) ? C2R_MINB : (RowCfg<M>::NT <= 192) ? 3 : 1) k_rows_c2r(EprLines L, int nrows, const float2* __restrict__ spec,
                                                            const float2* __restrict__ tw, const float2* __restrict__ tw2,
                                                            float step, int tau_is_zero, int newton_iters,
                                                            float i_min, float* __restrict__ out) {
  using C = RowCfg<M>;
  using EI = Engine<M, C::TPC, 1, true, false>;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  uint64_t* bar = reinterpret_cast<uint64_t*>(smem_raw);
  float2* stage = reinterpret_cast<float2*>(smem_raw + C::OFF_STAGE);
  const int tid = threadIdx.x;
  const int lr = tid / C::TPC, t = tid - lr * C::TPC;
  const int ngroups = (nrows + C::ROWS - 1) / C::ROWS;
  const RowPipe pipe{bar, stage, spec, nrows, C::ROWS, M, C::PLA, C::STAGE};
  __shared__ float s_f[EPR_MAX_BINS], s_gamma[EPR_MAX_BINS];
  if (EPI == 2 && tid < L.n_bins) { s_f[tid] = L.f[tid]; s_gamma[tid] = L.gamma[tid]; }
  if (tid == 0) { eprtma::mbar_init(&bar[0], 1); eprtma::mbar_init(&bar[1], 1); eprtma::mbar_fence_init(); }
  __syncthreads();
  if (tid == 0 && (int)blockIdx.x < ngroups) pipe.issue(blockIdx.x, 0);
  int it = 0;
  for (int grp = blockIdx.x; grp < ngroups; grp += gridDim.x, ++it) {
    const int buf = it & 1;
    if (tid == 0 && grp + (int)gridDim.x < ngroups) pipe.issue(grp + gridDim.x, buf ^ 1);
    float2* s = stage + (size_t)buf * C::STAGE + lr * C::PLA;
    const int row = grp * C::ROWS + lr;
    const bool live = row < nrows;
    // the τ values the epilogue will update: requested now, consumed after the transform
    float2* dst = reinterpret_cast<float2*>(out) + (size_t)(live ? row : 0) * M;
    float2 tpre[EI::GL::CNT][EI::RL];
#pragma unroll
    for (int c = 0; c < EI::GL::CNT; ++c) {
      const int j = t + c * C::TPC;
#pragma unroll
      for (int q = 0; q < EI::RL; ++q) {
        tpre[c][q] = make_float2(0.f, 0.f);
        if (EPI == 1 && !tau_is_zero && live && (EI::GL::FULL || j < EI::GL::T)) tpre[c][q] = dst[j + q * EI::PL];
      }
    }
    eprtma::mbar_wait(&bar[buf], (it >> 1) & 1);
    const float2* src = s;
    float2 u0[EI::G0::CNT][EI::R0], uL[EI::GL::CNT][EI::RL];
    // Z2[k] = (X[k] + X*[M−k]) + i w^{−k} (X[k] − X*[M−k]);  Z2[0] = (x0 + xM) + i (x0 − xM)
#pragma unroll
    for (int c = 0; c < EI::G0::CNT; ++c) {
      const int j = t + c * C::TPC;
#pragma unroll
      for (int r = 0; r < EI::R0; ++r) {
        const int k = j + r * EI::G0::T;
        float2 z = make_float2(0.f, 0.f);
        if ((EI::G0::FULL || j < EI::G0::T) && live) {
          const float2 xk = src[k];
          if (k == 0) {
            z = make_float2(xk.x + xk.y, xk.x - xk.y);
          } else {
            const float2 xm = src[M - k];
            const float2 wk = __ldg(&tw2[k]);
            const float2 e = make_float2(xk.x + xm.x, xk.y - xm.y);
            const float2 o = make_float2(-(xk.y + xm.y), xk.x - xm.x);            // i (xk − xm*)
            z = cadd(e, cmul(make_float2(wk.x, -wk.y), o));
          }
        }
        u0[c][r] = z;
      }
    }
    __syncthreads();                       // every input is in registers: the stage row becomes the work buffer
    EI::run(u0, uL, s, 0, t, tw);
    if (EPI == 2) {
      // Several lines: the projection costs hundreds of instructions per pixel.  The row goes back to shared memory in
      // natural order and is updated in a rolled loop (2 pixels per thread per pass, τ of the next pass in flight), so
      // that neither the FFT's register arrays nor 32 unrolled copies of the solver are alive in the epilogue.
      __syncthreads();                     // last-pass gathers of the row are done
#pragma unroll
      for (int c = 0; c < EI::GL::CNT; ++c) {
        const int j = t + c * C::TPC;
        if (EI::GL::FULL || j < EI::GL::T) {
#pragma unroll
          for (int q = 0; q < EI::RL; ++q) s[j + q * EI::PL] = uL[c][q];
        }
      }
      __syncthreads();
      if (live) {
        float2 tnext = tau_is_zero ? make_float2(0.f, 0.f) : dst[t];
#pragma unroll 1
        for (int i = t; i < M; i += C::TPC) {
          float2 tau = tnext;
          if (i + C::TPC < M && !tau_is_zero) tnext = dst[i + C::TPC];
          const float2 v = s[i];
          float d0, d1;
          if (tau_is_zero) {                 // the initial guess: constant moments, no exponential of τ
            d0 = epr_project_increment_tau0(L, step * v.x, s_f, s_gamma, newton_iters, i_min);
            d1 = epr_project_increment_tau0(L, step * v.y, s_f, s_gamma, newton_iters, i_min);
          } else if (!epr_project_increment_small_nb2(L, tau, make_float2(step * v.x, step * v.y), newton_iters, i_min, d0, d1)) {
            d0 = epr_project_increment(tau.x, step * v.x, s_f, s_gamma, L.n_bins, L.gamma_max, newton_iters, i_min);
            d1 = epr_project_increment(tau.y, step * v.y, s_f, s_gamma, L.n_bins, L.gamma_max, newton_iters, i_min);
          }
          tau.x += d0; tau.y += d1;
          dst[i] = tau;
        }
      }
    } else if (live) {
#pragma unroll
      for (int c = 0; c < EI::GL::CNT; ++c) {
        const int j = t + c * C::TPC;
        if (EI::GL::FULL || j < EI::GL::T) {
#pragma unroll
          for (int q = 0; q < EI::RL; ++q) {
            const int idx = j + q * EI::PL;
            float2 v = uL[c][q];
            if (EPI == 1) {
              float2 tau = tpre[c][q];
              tau.x += epr_project_increment_mono(tau.x, step * v.x, i_min);
              tau.y += epr_project_increment_mono(tau.y, step * v.y, i_min);
              v = tau;
            }
            dst[idx] = v;
          }
        }
      }
    }
    eprtma::fence_proxy_async();           // this thread's generic writes of the stage are ordered before the TMA refill
    __syncthreads();                       // stage[buf] is free for the group after next
  }
}

// ------------------------------------------------------------------------------------------------ columns
template <int N> struct ColCfg {
  static constexpr int W = 4;                    // columns per CTA (32 B per row segment)
  static constexpr int TPC = threads_per_transform(N);    // threads per column
  static constexpr int NT = TPC * W;
  static constexpr int PL = padded_len(N);
  static constexpr size_t SMEM = (size_t)PL * W * sizeof(float2);
};

// mode 0: out[plane] = IFFT( H_{plane % nb} FFT(spec[plane]) )      (per-line, epr_precondition)
// mode 1: out[b]     = IFFT( Σ_s H_s FFT(spec[b·nb + s]) )           (Fourier-space sum, R10 identity)
// mode 2: out[plane] = IFFT( H_ā FFT(spec[plane]) )                  (initial guess, R9)
// SUM (template) = mode 1 with more than one line: accumulators in registers.
// The forward transform uses the radix order (16,…), the inverse the reversed order, so the last forward pass,
// the diagonal filter and the first inverse pass all happen in registers on the same butterflies.
template <int N, bool SUM>
__global__ void __launch_bounds__(ColCfg<N>::NT, (SUM || ColCfg<N>::NT > 512) ? 1 : 2)
k_cols(EprLines L, int M, int mode, float scale, const float* __restrict__ lam_x, const float* __restrict__ lam_y,
       const float2* __restrict__ tw, const float2* __restrict__ tw_inv, const float2* __restrict__ spec,
       float2* __restrict__ out) {
  using C = ColCfg<N>;
  using EF = Engine<N, C::TPC, C::W, false, false>;
  using EI = Engine<N, C::TPC, C::W, true, true>;
  static_assert(EF::RL == EI::R0 && EF::GL::CNT == EI::G0::CNT && EF::PL == EI::G0::T, "schedules must mirror");
  extern __shared__ float2 sm[];
  const int c = threadIdx.x % C::W, t = threadIdx.x / C::W;
  const int kx = blockIdx.x * C::W + c;
  const int oplane = blockIdx.y;
  const int nb = L.n_bins;
  const int nloop = SUM ? nb : 1;
  const bool live = kx < M;
  const float lx = live ? __ldg(&lam_x[kx]) : 0.f;
  float2 acc[EF::GL::CNT][EF::RL];
  if (SUM) {
#pragma unroll
    for (int cc = 0; cc < EF::GL::CNT; ++cc)
#pragma unroll
      for (int q = 0; q < EF::RL; ++q) acc[cc][q] = make_float2(0.f, 0.f);
  }
  for (int sl = 0; sl < nloop; ++sl) {
    const size_t iplane = (mode == 1) ? (size_t)oplane * nb + sl : (size_t)oplane;
    const float a = (mode == 2) ? L.abar : L.a[(mode == 1) ? sl : (oplane % nb)];
    const float2* src = spec + iplane * (size_t)N * M + (live ? kx : 0);
    float2 u0[EF::G0::CNT][EF::R0], uL[EF::GL::CNT][EF::RL];
#pragma unroll
    for (int cc = 0; cc < EF::G0::CNT; ++cc) {
      const int j = t + cc * C::TPC;
#pragma unroll
      for (int r = 0; r < EF::R0; ++r) {
        float2 v = make_float2(0.f, 0.f);
        if ((EF::G0::FULL || j < EF::G0::T) && live) v = __ldg(&src[(size_t)(j + r * EF::G0::T) * M]);
        u0[cc][r] = v;
      }
    }
    EF::run(u0, uL, sm, c, t, tw);
    if (blockIdx.x == 0) {
      // tile 0 holds the packed column kx = 0: C = F0 + i FM (both Hermitian in ky).  With A = ½(C[ky] + C*[−ky]),
      // B = −(i/2)(C[ky] − C*[−ky]):  C'[ky] = H(0,ky) A + i H(M,ky) B,  C'[−ky] = H(0,ky) A* + i H(M,ky) B*.
      __syncthreads();
#pragma unroll
      for (int cc = 0; cc < EF::GL::CNT; ++cc) {
        const int j = t + cc * C::TPC;
        if (EF::GL::FULL || j < EF::GL::T) {
#pragma unroll
          for (int q = 0; q < EF::RL; ++q) sm[padi(j + q * EF::PL) * C::W + c] = uL[cc][q];
        }
      }
      __syncthreads();
      if (c == 0) {
        const float lxN = __ldg(&lam_x[M]);
        for (int ky = t; ky <= N / 2; ky += C::TPC) {
          const int km = (ky == 0) ? 0 : N - ky;
          const float2 ck = sm[padi(ky) * C::W], cm = sm[padi(km) * C::W];
          const float ly = __ldg(&lam_y[ky]);
          const float h0 = scale / (1.f + a * (lx + ly)), hN = scale / (1.f + a * (lxN + ly));
          const float2 A = make_float2(0.5f * (ck.x + cm.x), 0.5f * (ck.y - cm.y));
          const float2 B = make_float2(0.5f * (ck.y + cm.y), -0.5f * (ck.x - cm.x));
          sm[padi(ky) * C::W] = make_float2(h0 * A.x - hN * B.y, h0 * A.y + hN * B.x);
          if (km != ky) sm[padi(km) * C::W] = make_float2(h0 * A.x + hN * B.y, -h0 * A.y + hN * B.x);
        }
      }
      __syncthreads();
#pragma unroll
      for (int cc = 0; cc < EF::GL::CNT; ++cc) {
        const int j = t + cc * C::TPC;
        if (EF::GL::FULL || j < EF::GL::T) {
#pragma unroll
          for (int q = 0; q < EF::RL; ++q) uL[cc][q] = sm[padi(j + q * EF::PL) * C::W + c];
        }
      }
    }
    const float alx = fmaf(a, lx, 1.f);
#pragma unroll
    for (int cc = 0; cc < EF::GL::CNT; ++cc) {
      const int j = t + cc * C::TPC;
      if (EF::GL::FULL || j < EF::GL::T) {
#pragma unroll
        for (int q = 0; q < EF::RL; ++q) {
          const float h = (kx == 0) ? 1.f : __fdividef(scale, fmaf(a, __ldg(&lam_y[j + q * EF::PL]), alx));
          if (SUM) { acc[cc][q].x = fmaf(h, uL[cc][q].x, acc[cc][q].x); acc[cc][q].y = fmaf(h, uL[cc][q].y, acc[cc][q].y); }
          else { uL[cc][q].x *= h; uL[cc][q].y *= h; }
        }
      }
    }
    __syncthreads();                       // all reads of shared memory done before the next transform writes it
    if (!SUM) {
#pragma unroll
      for (int cc = 0; cc < EF::GL::CNT; ++cc)
#pragma unroll
        for (int q = 0; q < EF::RL; ++q) acc[cc][q] = uL[cc][q];
    }
  }
  float2 uo[EI::GL::CNT][EI::RL];
  EI::run(acc, uo, sm, c, t, tw_inv);
  if (live) {
    float2* dst = out + (size_t)oplane * N * M + kx;
#pragma unroll
    for (int cc = 0; cc < EI::GL::CNT; ++cc) {
      const int j = t + cc * C::TPC;
      if (EI::GL::FULL || j < EI::GL::T) {
#pragma unroll
        for (int q = 0; q < EI::RL; ++q) dst[(size_t)(j + q * EI::PL) * M] = uo[cc][q];
      }
    }
  }
}

// ------------------------------------------------------------------------------------------------ columns, TMA
// Power-of-two ny ≥ 256, nx % 8 == 0: the 4-column tile (ny rows of 32 bytes) is moved by the TMA unit
// (cp.async.bulk.tensor.2d, boxes of 256 rows) straight into shared memory and back, so the 32-byte row segments
// never pass through the LSU, registers or a scoreboard; the transform runs IN PLACE in those ny·32 bytes on the
// swizzled layout of epr_fft.cuh (no padding, conflict-free), which leaves room for two CTAs per SM.
template <int N> struct ColTmaCfg {
  static constexpr int W = 4;
  static constexpr int TPC = N / 16;
  static constexpr int NT = TPC * W;
  static constexpr int BOX = 256;                          // rows per TMA box (hardware limit)
  static constexpr size_t TILE = (size_t)N * W * sizeof(float2);
  // SUM (several lines per output tile): two tiles, so that the load of line s+1 overlaps the transform of line s
  static constexpr size_t smem(bool sum) { return (sum ? 2 : 1) * TILE + 16; }   // + two mbarriers
  static constexpr size_t smem3() { return 3 * TILE + 32; }
};

// NBUF tile buffers: 1 (one line per output tile), 2 (several lines: the load of line s + 1 under the transform of line s), 3 (stage 2
// of the block filters: no transform per line, so the loads are the whole cost and two of them are kept in flight)
template <int N, bool SUM, int NBUF = (SUM ? 2 : 1)>
__global__ void __launch_bounds__(ColTmaCfg<N>::NT, (SUM || ColTmaCfg<N>::NT > 512) ? 1 : 2)
k_cols_tma(const __grid_constant__ CUtensorMap map_in, const __grid_constant__ CUtensorMap map_out, EprLines L, int M,
           int mode, float scale, const float* __restrict__ lam_x, const float* __restrict__ lam_y,
           const float2* __restrict__ tw, const float2* __restrict__ tw_inv, int stage) {
  // stage 0: the whole operator.  Block filters of an x-dependent spectrum (R17(c)) apply several filters to the same
  // residuals, so the forward transform is done once — stage 1: out[plane] = FFT_y(spec[plane]), stored in frequency order —
  // and every block then runs stage 2: the input tiles are already transformed (filter, Σ_s, inverse only).
  using C = ColTmaCfg<N>;
  using EF = EngineSw<N, C::TPC, false, false>;
  using EI = EngineSw<N, C::TPC, true, true>;
  static_assert(EF::RL == EI::R0 && EF::GL::CNT == EI::G0::CNT && EF::PL == EI::G0::T, "schedules must mirror");
  extern __shared__ __align__(128) unsigned char smem_raw[];
  uint64_t* bar = reinterpret_cast<uint64_t*>(smem_raw + NBUF * C::TILE);
  const int c = threadIdx.x % C::W, t = threadIdx.x / C::W;
  const int kx0 = blockIdx.x * C::W, kx = kx0 + c;
  const int oplane = blockIdx.y;
  const int nb = L.n_bins;
  const int nloop = SUM ? nb : 1;
  const float lx = __ldg(&lam_x[kx]);
  if (threadIdx.x == 0) {
    for (int i = 0; i < (NBUF < 2 ? 2 : NBUF); ++i) eprtma::mbar_init(&bar[i], 1);
    eprtma::mbar_fence_init();
  }
  __syncthreads();
  auto load_tile = [&](int sl) {            // one thread: request line sl of this output tile into buffer sl % NBUF
    const int iplane = (mode == 1) ? oplane * nb + sl : oplane;
    float2* dst = reinterpret_cast<float2*>(smem_raw + (sl % NBUF) * C::TILE);
    eprtma::fence_proxy_async();
    eprtma::mbar_expect_tx(&bar[sl % NBUF], (unsigned)C::TILE);
#pragma unroll
    for (int bx = 0; bx < N / C::BOX; ++bx)
      eprtma::tensor_g2s_2d(dst + bx * C::BOX * C::W, &map_in, 2 * kx0, iplane * N + bx * C::BOX, &bar[sl % NBUF]);
  };
  if (threadIdx.x == 0)
    for (int i = 0; i < (NBUF > 1 ? NBUF - 1 : 1) && i < nloop; ++i) load_tile(i);
  float2 acc[EF::GL::CNT][EF::RL];
  if (SUM) {
#pragma unroll
    for (int cc = 0; cc < EF::GL::CNT; ++cc)
#pragma unroll
      for (int q = 0; q < EF::RL; ++q) acc[cc][q] = make_float2(0.f, 0.f);
  }
  for (int sl = 0; sl < nloop; ++sl) {
    const float a = (mode == 2) ? L.abar : L.a[(mode == 1) ? sl : (oplane % nb)];
    float2* sm = reinterpret_cast<float2*>(smem_raw + (sl % NBUF) * C::TILE);
    // buffer (sl − 1) % NBUF was last read during line sl − 1, which every thread left through the barrier closing it
    if (SUM && threadIdx.x == 0 && sl + NBUF - 1 < nloop) load_tile(sl + NBUF - 1);
    eprtma::mbar_wait(&bar[sl % NBUF], (sl / NBUF) & 1);
    float2 u0[EF::G0::CNT][EF::R0], uL[EF::GL::CNT][EF::RL];
    if (stage != 2) {
#pragma unroll
      for (int cc = 0; cc < EF::G0::CNT; ++cc)
#pragma unroll
        for (int r = 0; r < EF::R0; ++r) u0[cc][r] = sm[(t + cc * C::TPC + r * EF::G0::T) * C::W + c];   // LINEAR tile
      __syncthreads();                     // every thread has its inputs: the tile may be overwritten in place
      EF::run(u0, uL, sm, c, t, tw);
    } else {                               // the tile holds the transformed column in frequency order
#pragma unroll
      for (int cc = 0; cc < EF::GL::CNT; ++cc)
#pragma unroll
        for (int q = 0; q < EF::RL; ++q) uL[cc][q] = sm[(t + cc * C::TPC + q * EF::PL) * C::W + c];
    }
    if (stage == 1) {                      // forward only: frequency order back into the tile, TMA store, done (SUM is false)
      __syncthreads();
#pragma unroll
      for (int cc = 0; cc < EF::GL::CNT; ++cc)
#pragma unroll
        for (int q = 0; q < EF::RL; ++q) sm[(t + cc * C::TPC + q * EF::PL) * C::W + c] = uL[cc][q];
      eprtma::fence_proxy_async();
      __syncthreads();
      if (threadIdx.x == 0) {
#pragma unroll
        for (int bx = 0; bx < N / C::BOX; ++bx)
          eprtma::tensor_s2g_2d(&map_out, 2 * kx0, oplane * N + bx * C::BOX, sm + bx * C::BOX * C::W);
        eprtma::bulk_commit();
        eprtma::bulk_wait<0>();
      }
      return;
    }
    if (blockIdx.x == 0) {
      // tile 0 holds the packed column kx = 0: C = F0 + i FM (both Hermitian in ky).  With A = ½(C[ky] + C*[−ky]),
      // B = −(i/2)(C[ky] − C*[−ky]):  C'[ky] = H(0,ky) A + i H(M,ky) B,  C'[−ky] = H(0,ky) A* + i H(M,ky) B*.
      __syncthreads();
      if (stage != 2) {
#pragma unroll
        for (int cc = 0; cc < EF::GL::CNT; ++cc)
#pragma unroll
          for (int q = 0; q < EF::RL; ++q) sm[(t + cc * C::TPC + q * EF::PL) * C::W + c] = uL[cc][q];
        __syncthreads();
      }
      if (c == 0) {
        const float lxN = __ldg(&lam_x[M]);
        for (int ky = t; ky <= N / 2; ky += C::TPC) {
          const int km = (ky == 0) ? 0 : N - ky;
          const float2 ck = sm[ky * C::W], cm = sm[km * C::W];
          const float ly = __ldg(&lam_y[ky]);
          const float h0 = scale / (1.f + a * (lx + ly)), hN = scale / (1.f + a * (lxN + ly));
          const float2 A = make_float2(0.5f * (ck.x + cm.x), 0.5f * (ck.y - cm.y));
          const float2 B = make_float2(0.5f * (ck.y + cm.y), -0.5f * (ck.x - cm.x));
          sm[ky * C::W] = make_float2(h0 * A.x - hN * B.y, h0 * A.y + hN * B.x);
          if (km != ky) sm[km * C::W] = make_float2(h0 * A.x + hN * B.y, -h0 * A.y + hN * B.x);
        }
      }
      __syncthreads();
#pragma unroll
      for (int cc = 0; cc < EF::GL::CNT; ++cc)
#pragma unroll
        for (int q = 0; q < EF::RL; ++q) uL[cc][q] = sm[(t + cc * C::TPC + q * EF::PL) * C::W + c];
    }
    const float alx = fmaf(a, lx, 1.f);
#pragma unroll
    for (int cc = 0; cc < EF::GL::CNT; ++cc) {
#pragma unroll
      for (int q = 0; q < EF::RL; ++q) {
        const float h = (kx == 0) ? 1.f : __fdividef(scale, fmaf(a, __ldg(&lam_y[t + cc * C::TPC + q * EF::PL]), alx));
        if (SUM) { acc[cc][q].x = fmaf(h, uL[cc][q].x, acc[cc][q].x); acc[cc][q].y = fmaf(h, uL[cc][q].y, acc[cc][q].y); }
        else { acc[cc][q].x = h * uL[cc][q].x; acc[cc][q].y = h * uL[cc][q].y; }
      }
    }
    if (SUM) eprtma::fence_proxy_async();  // generic writes of this tile are ordered before its TMA refill (line sl + 2)
    __syncthreads();                       // all reads of the tile done before the next load / the inverse writes it
  }
  float2* sm = reinterpret_cast<float2*>(smem_raw);
  float2 uo[EI::GL::CNT][EI::RL];
  EI::run(acc, uo, sm, c, t, tw_inv);
  __syncthreads();                         // last-pass gathers done: the tile is rewritten in LINEAR order for the TMA store
#pragma unroll
  for (int cc = 0; cc < EI::GL::CNT; ++cc)
#pragma unroll
    for (int q = 0; q < EI::RL; ++q) sm[(t + cc * C::TPC + q * EI::PL) * C::W + c] = uo[cc][q];
  eprtma::fence_proxy_async();             // generic-proxy writes → visible to the async proxy
  __syncthreads();
  if (threadIdx.x == 0) {
#pragma unroll
    for (int bx = 0; bx < N / C::BOX; ++bx)
      eprtma::tensor_s2g_2d(&map_out, 2 * kx0, oplane * N + bx * C::BOX, sm + bx * C::BOX * C::W);
    eprtma::bulk_commit();
    eprtma::bulk_wait<0>();                // the CTA's shared memory must outlive the store
  }
}

// ------------------------------------------------------------------------------------------------ columns, TMA, two groups
// One line per output tile (the one-line loop, the initial guess, epr_precondition) at ny = 2048: in k_cols_tma a CTA
// loads, transforms and stores ONE tile, and a fifth of its warp time is spent at the mbarrier waiting for that tile
// (both CTAs of an SM often wait together).  Here one persistent CTA per SM runs TWO groups of 512 threads on
// different tiles with THREE 64 KB tile buffers: tile k (k = 0, 1, 2, … in this CTA's static sequence) lives in buffer
// k mod 3 and is processed by group k mod 2; the group that finishes tile k stores it and, as soon as the TMA unit has
// read the buffer, requests tile k + 3 into it — which the OTHER group will need only after finishing tile k + 1.
// The groups drift half a tile apart after the first wait, so every later tile has landed before it is wanted.
// Groups synchronise on named barriers (1 + group); the engine is the same swizzled in-place one.
template <int N>
__global__ void __launch_bounds__(2 * ColTmaCfg<N>::NT, 1)
k_cols_tma2(const __grid_constant__ CUtensorMap map_in, const __grid_constant__ CUtensorMap map_out, EprLines L, int M,
            int mode, float scale, int tiles_x, int ntiles, const float* __restrict__ lam_x,
            const float* __restrict__ lam_y, const float2* __restrict__ tw, const float2* __restrict__ tw_inv) {
  using C = ColTmaCfg<N>;
  constexpr int GT = C::NT;                                // threads per group
  using EF = EngineSw<N, C::TPC, false, false, GT>;
  using EI = EngineSw<N, C::TPC, true, true, GT>;
  static_assert(EF::RL == EI::R0 && EF::GL::CNT == EI::G0::CNT && EF::PL == EI::G0::T, "schedules must mirror");
  extern __shared__ __align__(128) unsigned char smem_raw[];
  uint64_t* bar = reinterpret_cast<uint64_t*>(smem_raw + 3 * C::TILE);
  const int g = threadIdx.x / GT, lt = threadIdx.x - g * GT;
  const int c = lt % C::W, t = lt / C::W;
  const int nb = L.n_bins;
  auto tile_of = [&](int k) { return (int)blockIdx.x + k * (int)gridDim.x; };
  auto load_tile = [&](int k) {             // one thread: request tile k of this CTA's sequence into buffer k % 3
    const int T = tile_of(k), bx = T % tiles_x, pl = T / tiles_x;
    float2* dst = reinterpret_cast<float2*>(smem_raw + (k % 3) * C::TILE);
    eprtma::fence_proxy_async();
    eprtma::mbar_expect_tx(&bar[k % 3], (unsigned)C::TILE);
#pragma unroll
    for (int b = 0; b < N / C::BOX; ++b)
      eprtma::tensor_g2s_2d(dst + b * C::BOX * C::W, &map_in, 2 * bx * C::W, pl * N + b * C::BOX, &bar[k % 3]);
  };
  if (threadIdx.x == 0) {
    for (int i = 0; i < 3; ++i) eprtma::mbar_init(&bar[i], 1);
    eprtma::mbar_fence_init();
    for (int k = 0; k < 3; ++k)
      if (tile_of(k) < ntiles) load_tile(k);
  }
  __syncthreads();
  int pending = -1;                        // thread 0 of a group: tile to request into the buffer stored last
  auto work = [&](auto bid_tag) {
    constexpr int BID = decltype(bid_tag)::value;          // named barrier of this group (compile time: no R2UR per barrier)
    for (int k = g; tile_of(k) < ntiles; k += 2) {
      const int T = tile_of(k), bx = T % tiles_x, oplane = T / tiles_x;
      const int kx = bx * C::W + c;
      const float lx = __ldg(&lam_x[kx]);
      const float a = (mode == 2) ? L.abar : L.a[oplane % nb];
      float2* sm = reinterpret_cast<float2*>(smem_raw + (k % 3) * C::TILE);
      // Refill of the buffer this group stored last: by then the TMA unit has read it (the wait returns at once), and
      // the request still leaves the other group, which wants that tile, about half a tile of lead.
      auto refill = [&]() {
        if (lt == 0 && pending >= 0) { eprtma::bulk_wait_read<0>(); load_tile(pending); pending = -1; }
      };
      eprtma::mbar_wait(&bar[k % 3], (unsigned)(k / 3) & 1u);
      float2 u0[EF::G0::CNT][EF::R0], uL[EF::GL::CNT][EF::RL], acc[EF::GL::CNT][EF::RL];
#pragma unroll
      for (int cc = 0; cc < EF::G0::CNT; ++cc)
#pragma unroll
        for (int r = 0; r < EF::R0; ++r) u0[cc][r] = sm[(t + cc * C::TPC + r * EF::G0::T) * C::W + c];   // LINEAR tile
      tile_sync<GT>(BID);                     // every thread has its inputs: the tile may be overwritten in place
      EF::run(u0, uL, sm, c, t, tw, BID, refill);
      if (bx == 0) {
        // tile 0 holds the packed column kx = 0 (see k_cols_tma)
        tile_sync<GT>(BID);
#pragma unroll
        for (int cc = 0; cc < EF::GL::CNT; ++cc)
#pragma unroll
          for (int q = 0; q < EF::RL; ++q) sm[(t + cc * C::TPC + q * EF::PL) * C::W + c] = uL[cc][q];
        tile_sync<GT>(BID);
        if (c == 0) {
          const float lxN = __ldg(&lam_x[M]);
          for (int ky = t; ky <= N / 2; ky += C::TPC) {
            const int km = (ky == 0) ? 0 : N - ky;
            const float2 ck = sm[ky * C::W], cm = sm[km * C::W];
            const float ly = __ldg(&lam_y[ky]);
            const float h0 = scale / (1.f + a * (lx + ly)), hN = scale / (1.f + a * (lxN + ly));
            const float2 A = make_float2(0.5f * (ck.x + cm.x), 0.5f * (ck.y - cm.y));
            const float2 B = make_float2(0.5f * (ck.y + cm.y), -0.5f * (ck.x - cm.x));
            sm[ky * C::W] = make_float2(h0 * A.x - hN * B.y, h0 * A.y + hN * B.x);
            if (km != ky) sm[km * C::W] = make_float2(h0 * A.x + hN * B.y, -h0 * A.y + hN * B.x);
          }
        }
        tile_sync<GT>(BID);
#pragma unroll
        for (int cc = 0; cc < EF::GL::CNT; ++cc)
#pragma unroll
          for (int q = 0; q < EF::RL; ++q) uL[cc][q] = sm[(t + cc * C::TPC + q * EF::PL) * C::W + c];
      }
      const float alx = fmaf(a, lx, 1.f);
#pragma unroll
      for (int cc = 0; cc < EF::GL::CNT; ++cc) {
#pragma unroll
        for (int q = 0; q < EF::RL; ++q) {
          const float h = (kx == 0) ? 1.f : __fdividef(scale, fmaf(a, __ldg(&lam_y[t + cc * C::TPC + q * EF::PL]), alx));
          acc[cc][q].x = h * uL[cc][q].x; acc[cc][q].y = h * uL[cc][q].y;
        }
      }
      tile_sync<GT>(BID);                     // all reads of the tile done before the inverse writes it
      float2 uo[EI::GL::CNT][EI::RL];
      EI::run(acc, uo, sm, c, t, tw_inv, BID);
      tile_sync<GT>(BID);                     // last-pass gathers done: the tile is rewritten in LINEAR order for the TMA store
#pragma unroll
      for (int cc = 0; cc < EI::GL::CNT; ++cc)
#pragma unroll
        for (int q = 0; q < EI::RL; ++q) sm[(t + cc * C::TPC + q * EI::PL) * C::W + c] = uo[cc][q];
      eprtma::fence_proxy_async();            // generic-proxy writes → visible to the async proxy
      tile_sync<GT>(BID);
      if (lt == 0) {
#pragma unroll
        for (int b = 0; b < N / C::BOX; ++b)
          eprtma::tensor_s2g_2d(&map_out, 2 * bx * C::W, oplane * N + b * C::BOX, sm + b * C::BOX * C::W);
        eprtma::bulk_commit();
        pending = tile_of(k + 3) < ntiles ? k + 3 : -1;      // refilled from the next tile's first pass (see `refill`)
      }
    }
  };
  if (g == 0) work(std::integral_constant<int, 1>{}); else work(std::integral_constant<int, 2>{});
  if (lt == 0 && pending >= 0) { eprtma::bulk_wait_read<0>(); load_tile(pending); }   // (cannot happen: kept for safety)
  if (lt == 0) eprtma::bulk_wait<0>();      // the CTA's stores are complete before it exits
}

// ------------------------------------------------------------------------------------------------ columns, TMA, any ny
// ny ≥ 256 that is not a power of two (2160 = 9 boxes of 240 rows): the 4-column tile arrives by TMA in LINEAR order in
// its own buffer(s) and the padded engine of k_cols works beside it, so that — several lines — the load of line s + 1
// runs under the transform of line s and no 32-byte row segment goes through the LSU.  The result leaves through
// tile 0 by a TMA store.  (k_cols itself has one CTA per SM at these sizes and overlaps nothing.)
template <int N> struct ColTmaPadCfg {
  using C = ColCfg<N>;
  static constexpr size_t LIN = (size_t)N * C::W * sizeof(float2);
  static constexpr size_t WORK = (C::SMEM + 15) / 16 * 16;
  // several lines: the forward twiddle table (used once per line) goes to shared memory when it still fits — with
  // ~210 KB of shared memory carved out, the L1 that is left (hit rate 29 %) cannot hold the tables
  static constexpr size_t TWB = (size_t)tw_total(N, false) * sizeof(float2);
  static constexpr bool TWS = 2 * LIN + WORK + 16 + TWB <= 227 * 1024;
  static constexpr size_t smem(bool sum) { return (sum ? 2 : 1) * LIN + WORK + 16 + ((sum && TWS) ? TWB : 0); }
};

template <int N, bool SUM>
__global__ void __launch_bounds__(ColCfg<N>::NT, 1)
k_cols_tmap(const __grid_constant__ CUtensorMap map_in, const __grid_constant__ CUtensorMap map_out, EprLines L, int M,
            int mode, float scale, int box_rows, const float* __restrict__ lam_x, const float* __restrict__ lam_y,
            const float2* __restrict__ tw, const float2* __restrict__ tw_inv) {
  using C = ColCfg<N>;
  using P = ColTmaPadCfg<N>;
  constexpr bool TWS = SUM && P::TWS;
  using EF = Engine<N, C::TPC, C::W, false, false, TWS>;
  using EI = Engine<N, C::TPC, C::W, true, true>;
  static_assert(EF::RL == EI::R0 && EF::GL::CNT == EI::G0::CNT && EF::PL == EI::G0::T, "schedules must mirror");
  extern __shared__ __align__(128) unsigned char smem_raw[];
  constexpr int NBUF = SUM ? 2 : 1;
  float2* work = reinterpret_cast<float2*>(smem_raw + NBUF * P::LIN);
  uint64_t* bar = reinterpret_cast<uint64_t*>(smem_raw + NBUF * P::LIN + P::WORK);
  float2* tw_s = reinterpret_cast<float2*>(smem_raw + NBUF * P::LIN + P::WORK + 16);
  if (TWS) {                                 // visible to everybody after the __syncthreads that follows the barrier init
    for (int i = threadIdx.x; i < tw_total(N, false); i += C::NT) tw_s[i] = __ldg(&tw[i]);
  }
  const float2* twf = TWS ? tw_s : tw;
  const int c = threadIdx.x % C::W, t = threadIdx.x / C::W;
  const int kx0 = blockIdx.x * C::W, kx = kx0 + c;
  const int oplane = blockIdx.y;
  const int nb = L.n_bins;
  const int nloop = SUM ? nb : 1;
  const int nbox = N / box_rows;
  const float lx = __ldg(&lam_x[kx]);
  if (threadIdx.x == 0) { eprtma::mbar_init(&bar[0], 1); eprtma::mbar_init(&bar[1], 1); eprtma::mbar_fence_init(); }
  __syncthreads();
  auto load_tile = [&](int sl) {            // one thread: request line sl of this output tile into buffer sl % NBUF
    const int iplane = (mode == 1) ? oplane * nb + sl : oplane;
    float2* dst = reinterpret_cast<float2*>(smem_raw + (sl % NBUF) * P::LIN);
    eprtma::fence_proxy_async();
    eprtma::mbar_expect_tx(&bar[sl % NBUF], (unsigned)P::LIN);
    for (int bx = 0; bx < nbox; ++bx)
      eprtma::tensor_g2s_2d(dst + bx * box_rows * C::W, &map_in, 2 * kx0, iplane * N + bx * box_rows, &bar[sl % NBUF]);
  };
  if (threadIdx.x == 0) load_tile(0);
  float2 acc[EF::GL::CNT][EF::RL];
#pragma unroll
  for (int cc = 0; cc < EF::GL::CNT; ++cc)
#pragma unroll
    for (int q = 0; q < EF::RL; ++q) acc[cc][q] = make_float2(0.f, 0.f);
  for (int sl = 0; sl < nloop; ++sl) {
    const float a = (mode == 2) ? L.abar : L.a[(mode == 1) ? sl : (oplane % nb)];
    const float2* lin = reinterpret_cast<const float2*>(smem_raw + (sl % NBUF) * P::LIN);
    // the other buffer was last read during line sl − 1, which every thread left through the barrier closing it
    if (SUM && threadIdx.x == 0 && sl + 1 < nloop) load_tile(sl + 1);
    eprtma::mbar_wait(&bar[sl % NBUF], (sl / NBUF) & 1);
    float2 u0[EF::G0::CNT][EF::R0], uL[EF::GL::CNT][EF::RL];
#pragma unroll
    for (int cc = 0; cc < EF::G0::CNT; ++cc) {
      const int j = t + cc * C::TPC;
#pragma unroll
      for (int r = 0; r < EF::R0; ++r) {
        float2 v = make_float2(0.f, 0.f);
        if (EF::G0::FULL || j < EF::G0::T) v = lin[(j + r * EF::G0::T) * C::W + c];
        u0[cc][r] = v;
      }
    }
    EF::run(u0, uL, work, c, t, twf);
    if (blockIdx.x == 0) {
      // tile 0 holds the packed column kx = 0: C = F0 + i FM (both Hermitian in ky).  With A = ½(C[ky] + C*[−ky]),
      // B = −(i/2)(C[ky] − C*[−ky]):  C'[ky] = H(0,ky) A + i H(M,ky) B,  C'[−ky] = H(0,ky) A* + i H(M,ky) B*.
      __syncthreads();
#pragma unroll
      for (int cc = 0; cc < EF::GL::CNT; ++cc) {
        const int j = t + cc * C::TPC;
        if (EF::GL::FULL || j < EF::GL::T) {
#pragma unroll
          for (int q = 0; q < EF::RL; ++q) work[padi(j + q * EF::PL) * C::W + c] = uL[cc][q];
        }
      }
      __syncthreads();
      if (c == 0) {
        const float lxN = __ldg(&lam_x[M]);
        for (int ky = t; ky <= N / 2; ky += C::TPC) {
          const int km = (ky == 0) ? 0 : N - ky;
          const float2 ck = work[padi(ky) * C::W], cm = work[padi(km) * C::W];
          const float ly = __ldg(&lam_y[ky]);
          const float h0 = scale / (1.f + a * (lx + ly)), hN = scale / (1.f + a * (lxN + ly));
          const float2 A = make_float2(0.5f * (ck.x + cm.x), 0.5f * (ck.y - cm.y));
          const float2 B = make_float2(0.5f * (ck.y + cm.y), -0.5f * (ck.x - cm.x));
          work[padi(ky) * C::W] = make_float2(h0 * A.x - hN * B.y, h0 * A.y + hN * B.x);
          if (km != ky) work[padi(km) * C::W] = make_float2(h0 * A.x + hN * B.y, -h0 * A.y + hN * B.x);
        }
      }
      __syncthreads();
#pragma unroll
      for (int cc = 0; cc < EF::GL::CNT; ++cc) {
        const int j = t + cc * C::TPC;
        if (EF::GL::FULL || j < EF::GL::T) {
#pragma unroll
          for (int q = 0; q < EF::RL; ++q) uL[cc][q] = work[padi(j + q * EF::PL) * C::W + c];
        }
      }
    }
    const float alx = fmaf(a, lx, 1.f);
#pragma unroll
    for (int cc = 0; cc < EF::GL::CNT; ++cc) {
      const int j = t + cc * C::TPC;
      if (EF::GL::FULL || j < EF::GL::T) {
#pragma unroll
        for (int q = 0; q < EF::RL; ++q) {
          const float h = (kx == 0) ? 1.f : __fdividef(scale, fmaf(a, __ldg(&lam_y[j + q * EF::PL]), alx));
          acc[cc][q].x = fmaf(h, uL[cc][q].x, acc[cc][q].x);
          acc[cc][q].y = fmaf(h, uL[cc][q].y, acc[cc][q].y);
        }
      }
    }
    if (SUM) eprtma::fence_proxy_async();  // generic reads of this tile are ordered before its TMA refill (line sl + 2)
    __syncthreads();                       // all reads of the tile and of the work buffer done
  }
  float2 uo[EI::GL::CNT][EI::RL];
  EI::run(acc, uo, work, c, t, tw_inv);
  float2* lin0 = reinterpret_cast<float2*>(smem_raw);     // free: every line has been consumed
#pragma unroll
  for (int cc = 0; cc < EI::GL::CNT; ++cc) {
    const int j = t + cc * C::TPC;
    if (EI::GL::FULL || j < EI::GL::T) {
#pragma unroll
      for (int q = 0; q < EI::RL; ++q) lin0[(j + q * EI::PL) * C::W + c] = uo[cc][q];
    }
  }
  eprtma::fence_proxy_async();             // generic-proxy writes → visible to the async proxy
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int bx = 0; bx < nbox; ++bx)
      eprtma::tensor_s2g_2d(&map_out, 2 * kx0, oplane * N + bx * box_rows, lin0 + bx * box_rows * C::W);
    eprtma::bulk_commit();
    eprtma::bulk_wait<0>();                // the CTA's shared memory must outlive the store
  }
}

// ------------------------------------------------------------------------------------------------ dispatch
// The instantiations are split into EPR_FFT_NGROUPS translation units (this file compiled once per group with
// -DEPR_FFT_GROUP=g, in parallel: see build.py); epr_fftd.cu routes a size to the group that holds it.
#ifndef EPR_FFT_GROUP
#error "compile with -DEPR_FFT_GROUP=<0..10> (paper_2601_22793_b200/build.py does)"
#endif
#if EPR_FFT_GROUP == 0
#define EPR_FFT_SIZES(X) X(2048) X(16) X(32)
#elif EPR_FFT_GROUP == 1
#define EPR_FFT_SIZES(X) X(2560) X(48)
#elif EPR_FFT_GROUP == 2
#define EPR_FFT_SIZES(X) X(2160) X(64)
#elif EPR_FFT_GROUP == 3
#define EPR_FFT_SIZES(X) X(1024) X(80) X(96)
#elif EPR_FFT_GROUP == 4
#define EPR_FFT_SIZES(X) X(512) X(320) X(128)
#elif EPR_FFT_GROUP == 5
#define EPR_FFT_SIZES(X) X(256) X(160)
#elif EPR_FFT_GROUP == 6
#define EPR_FFT_SIZES(X) X(4096)
#elif EPR_FFT_GROUP == 7
#define EPR_FFT_SIZES(X) X(1536) X(384)
#elif EPR_FFT_GROUP == 8
#define EPR_FFT_SIZES(X) X(1920) X(640)
#elif EPR_FFT_GROUP == 9
#define EPR_FFT_SIZES(X) X(3072) X(768)
#else
#define EPR_FFT_SIZES(X) X(3200) X(1280)
#endif
#define EPR_CAT2(a, b) a##b
#define EPR_CAT(a, b) EPR_CAT2(a, b)
#define GFN(name) EPR_CAT(name, EPR_FFT_GROUP)

int GFN(epr_fftg_has_)(int n) {
#define X(n_) if (n == n_) return 1;
  EPR_FFT_SIZES(X)
#undef X
  return 0;
}

// persistent grid: as many CTAs as are resident at once (occupancy x SMs), at most one per row group
template <typename K> static int row_grid(K kernel, int sms, int nt, size_t smem, int ngroups) {
  int occ = 0;
  cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kernel, nt, smem);
  const int g = sms * (occ > 0 ? occ : 1);
  return ngroups < g ? ngroups : g;
}

cudaError_t GFN(epr_fftg_rows_r2c_)(const epr_plan_s* p, int planes, const float* in, float in_offset, float2* spec,
                                    cudaStream_t st) {
  const int nrows = planes * p->ny;
  switch (p->nx) {
#define X(n_)                                                                                                   \
  case n_: {                                                                                                    \
    using C = RowCfg<n_ / 2>;                                                                                   \
    constexpr size_t smem = (size_t)C::ROWS * C::PL * sizeof(float2);                                           \
    static EprPerDevice attr = {};                                                                              \
    if (!attr.at(p)) {                                                                                          \
      cudaFuncSetAttribute(k_rows_r2c_direct<n_ / 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);   \
      attr.at(p) = 1;                                                                                           \
    }                                                                                                           \
    dim3 grid((p->ny + C::ROWS - 1) / C::ROWS, planes);                                                         \
    k_rows_r2c_direct<n_ / 2><<<grid, C::NT, smem, st>>>(p->ny, in, in_offset, p->tw_row, p->tw_r2c, spec);      \
  } break;
    EPR_FFT_SIZES(X)
#undef X
    default: return cudaErrorInvalidValue;
  }
  return cudaGetLastError();
}

template <int M, int EPI>
static void launch_c2r(const epr_plan_s* p, int nrows, const float2* spec, float step, int tau_is_zero, float* q_or_tau,
                       cudaStream_t st) {
  using C = RowCfg<M>;
  static EprPerDevice fullv = {};                        // resident CTAs of this kernel on the plan's device
  if (!fullv.at(p)) fullv.at(p) = row_grid(k_rows_c2r<M, EPI>, p->sms, C::NT, C::SMEM, 1 << 30);
  const int full = (int)fullv.at(p);
  const int ngroups = (nrows + C::ROWS - 1) / C::ROWS;
  k_rows_c2r<M, EPI><<<ngroups < full ? ngroups : full, C::NT, C::SMEM, st>>>(
      p->lines, nrows, spec, p->tw_row, p->tw_r2c, step, tau_is_zero, p->opt.newton_iters, p->opt.i_min, q_or_tau);
}

cudaError_t GFN(epr_fftg_rows_c2r_)(const epr_plan_s* p, int planes, const float2* spec, int epilogue, float step,
                                    int tau_is_zero, float* q_or_tau, cudaStream_t st) {
  const int nrows = planes * p->ny;
  switch (p->nx) {
#define X(n_)                                                                                                   \
  case n_: {                                                                                                    \
    if (epilogue == 0) launch_c2r<n_ / 2, 0>(p, nrows, spec, step, tau_is_zero, q_or_tau, st);                  \
    else if (p->n_bins == 1) launch_c2r<n_ / 2, 1>(p, nrows, spec, step, tau_is_zero, q_or_tau, st);            \
    else launch_c2r<n_ / 2, 2>(p, nrows, spec, step, tau_is_zero, q_or_tau, st);                                \
  } break;
    EPR_FFT_SIZES(X)
#undef X
    default: return cudaErrorInvalidValue;
  }
  return cudaGetLastError();
}

template <int N>
static bool launch_cols_tma(const epr_plan_s* p, const EprLines& LL, int oplanes, int mode, const float2* spec, float2* out,
                            float scale, cudaStream_t st, int stage) {
  if constexpr (N >= 256 && (N & (N - 1)) == 0) {
    using C = ColTmaCfg<N>;
    const int M = p->nx / 2;
    if (!p->tma_ok || M % C::W != 0 || spec != p->spec || (out != p->spec && out != p->spec_sum)) return false;
    if (mode == 1 && p->n_bins > 1 && C::smem(true) > 227 * 1024) return false;     // two tiles of 4096 rows do not fit an SM
    static EprPerDevice attr = {};
    if (!attr.at(p)) {
      cudaFuncSetAttribute(k_cols_tma<N, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::smem(false));
      if (C::smem(true) <= 227 * 1024)
        cudaFuncSetAttribute(k_cols_tma<N, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::smem(true));
      attr.at(p) = 1;
    }
    const CUtensorMap& mo = (out == p->spec) ? p->map_spec : p->map_spec_sum;
    dim3 grid(M / C::W, oplanes);
    if constexpr (2 * C::NT == 1024) {
      // one line per tile and enough tiles to keep every SM's two groups busy: persistent two-group kernel
      const int sms = p->sms;
      const int ntiles = (M / C::W) * oplanes;
      if (stage == 0 && !(mode == 1 && p->n_bins > 1) && ntiles >= 8 * sms) {
        constexpr size_t smem2 = 3 * C::TILE + 32;
        static EprPerDevice attr2 = {};
        if (!attr2.at(p)) { cudaFuncSetAttribute(k_cols_tma2<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem2); attr2.at(p) = 1; }
        k_cols_tma2<N><<<sms, 2 * C::NT, smem2, st>>>(p->map_spec, mo, LL, M, mode, scale, M / C::W, ntiles, p->lam_x, p->lam_y, p->tw_col, p->tw_col_inv);
        return true;
      }
    }
    if (mode == 1 && p->n_bins > 1 && stage == 2 && C::smem3() <= 227 * 1024) {
      static EprPerDevice attr3 = {};
      if (!attr3.at(p)) { cudaFuncSetAttribute(k_cols_tma<N, true, 3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::smem3()); attr3.at(p) = 1; }
      k_cols_tma<N, true, 3><<<grid, C::NT, C::smem3(), st>>>(p->map_spec, mo, LL, M, mode, scale, p->lam_x, p->lam_y, p->tw_col, p->tw_col_inv, stage);
    } else if (mode == 1 && p->n_bins > 1)
      k_cols_tma<N, true><<<grid, C::NT, C::smem(true), st>>>(p->map_spec, mo, LL, M, mode, scale, p->lam_x, p->lam_y, p->tw_col, p->tw_col_inv, stage);
    else
      k_cols_tma<N, false><<<grid, C::NT, C::smem(false), st>>>(p->map_spec, mo, LL, M, mode, scale, p->lam_x, p->lam_y, p->tw_col, p->tw_col_inv, stage);
    return true;
  } else if constexpr (N >= 256) {
    if (stage != 0) return false;
    using C = ColCfg<N>;
    using P = ColTmaPadCfg<N>;
    const int M = p->nx / 2;
    const bool sum = mode == 1 && p->n_bins > 1;
    if (!p->tma_ok || M % C::W != 0 || spec != p->spec || (out != p->spec && out != p->spec_sum)) return false;
    if (P::smem(sum) > 227 * 1024) return false;
    static EprPerDevice attr = {};
    if (!attr.at(p)) {
      if (P::smem(false) <= 227 * 1024)
        cudaFuncSetAttribute(k_cols_tmap<N, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)P::smem(false));
      if (P::smem(true) <= 227 * 1024)
        cudaFuncSetAttribute(k_cols_tmap<N, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)P::smem(true));
      attr.at(p) = 1;
    }
    const CUtensorMap& mo = (out == p->spec) ? p->map_spec : p->map_spec_sum;
    dim3 grid(M / C::W, oplanes);
    if (sum)
      k_cols_tmap<N, true><<<grid, C::NT, P::smem(true), st>>>(p->map_spec, mo, LL, M, mode, scale, p->tma_box_rows, p->lam_x, p->lam_y, p->tw_col, p->tw_col_inv);
    else
      k_cols_tmap<N, false><<<grid, C::NT, P::smem(false), st>>>(p->map_spec, mo, LL, M, mode, scale, p->tma_box_rows, p->lam_x, p->lam_y, p->tw_col, p->tw_col_inv);
    return true;
  } else {
    return false;
  }
}

cudaError_t GFN(epr_fftg_cols_)(const epr_plan_s* p, int planes, int mode, const float2* spec, float2* out, cudaStream_t st,
                                const EprLines* lines_override, int stage) {
  const EprLines& LL = lines_override ? *lines_override : p->lines;     // block filters pass their own a[] / abar
  const int M = p->nx / 2;
  const int oplanes = (mode == 1) ? planes / p->n_bins : planes;
  const float scale = (float)(1.0 / ((double)p->nx * (double)p->ny));
  switch (p->ny) {
#define X(n_)                                                                                                   \
  case n_: {                                                                                                    \
    using C = ColCfg<n_>;                                                                                       \
    if (launch_cols_tma<n_>(p, LL, oplanes, mode, spec, out, scale, st, stage)) break;                              \
    if (stage != 0) return cudaErrorNotSupported;           /* staged block filters: TMA column kernel only */     \
    static EprPerDevice attr = {};                                                                              \
    if (!attr.at(p)) {                                                                                          \
      cudaFuncSetAttribute(k_cols<n_, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM);       \
      cudaFuncSetAttribute(k_cols<n_, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM);        \
      attr.at(p) = 1;                                                                                           \
    }                                                                                                           \
    dim3 grid((M + C::W - 1) / C::W, oplanes);                                                                  \
    if (mode == 1 && p->n_bins > 1)                                                                             \
      k_cols<n_, true><<<grid, C::NT, C::SMEM, st>>>(LL, M, mode, scale, p->lam_x, p->lam_y, p->tw_col, p->tw_col_inv, spec, out); \
    else                                                                                                        \
      k_cols<n_, false><<<grid, C::NT, C::SMEM, st>>>(LL, M, mode, scale, p->lam_x, p->lam_y, p->tw_col, p->tw_col_inv, spec, out); \
  } break;
    EPR_FFT_SIZES(X)
#undef X
    default: return cudaErrorInvalidValue;
  }
  return cudaGetLastError();
}
