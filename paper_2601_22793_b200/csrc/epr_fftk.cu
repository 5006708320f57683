// epr_fftk.cu — the FFT-diagonal Paganin-type preconditioner P^{-1}_{1,s} as three
// hand-written kernels:   rows R2C  →  columns FFT · H_s (· Σ_s) · IFFT  →  rows C2R (+ update epilogue).
//
// Spectrum layout: [plane][ny][nx/2] float2; column kx = 0 packs the two purely real row-spectra X[0] (re)
// and X[nx/2] (im), so a plane of nx/2 complex columns holds the whole half spectrum.
// H_s(θ) = 1 / (1 + a_s λ(θ)) with λ = λx[kx] + λy[ky] from two 1-D tables (discrete or continuous symbol, R5);
// the 1/(nx·ny) normalisation is folded into H.
#include "epr_fft.cuh"
#include "epr_internal.h"
#include "epr_math.cuh"

using namespace eprfft;

template <int M> struct RowCfg {                // M = nx/2 complex points per row
  static constexpr int TPC = (M + 15) / 16;     // threads per row
  static constexpr int ROWS = (TPC >= 128) ? 1 : (128 + TPC - 1) / TPC;   // rows per CTA (≥128 threads)
  static constexpr int NT = TPC * ROWS;
  static constexpr int PL = padded_len(M);
};

// ------------------------------------------------------------------------------------------------ rows R2C
template <int M>
__global__ void __launch_bounds__(RowCfg<M>::NT) k_rows_r2c(int ny, const float* __restrict__ in, float in_offset,
                                                            const float2* __restrict__ tw, const float2* __restrict__ tw2,
                                                            float2* __restrict__ spec) {
  using C = RowCfg<M>;
  __shared__ float2 sm[C::ROWS * C::PL];
  const int lr = threadIdx.x / C::TPC, t = threadIdx.x - lr * C::TPC;
  const int row = blockIdx.x * C::ROWS + lr;
  const bool live = row < ny;
  const size_t plane = blockIdx.y;
  float2* s = sm + lr * C::PL;
  if (live) {
    const float2* src = reinterpret_cast<const float2*>(in + (plane * ny + row) * (size_t)(2 * M));
    for (int j = t; j < M; j += C::TPC) {
      float2 v = __ldg(&src[j]);
      s[padi(j)] = make_float2(v.x + in_offset, v.y + in_offset);
    }
  }
  __syncthreads();
  fft_smem<M, C::TPC, 1, false>(s, 0, t, tw);
  // post-process pairs (k, M-k):  X[k] = ½(Z[k] + Z*[M−k]) − (i/2) w^k (Z[k] − Z*[M−k]),  w = e^{−2πi/nx}
  float2* dst = spec + (plane * ny + row) * (size_t)M;
  if (live) {
    for (int k = t; k <= M / 2; k += C::TPC) {
      if (k == 0) {
        const float2 z = s[0];
        dst[0] = make_float2(z.x + z.y, z.x - z.y);          // packed: re = X[0], im = X[M]
      } else {
        const float2 zk = s[padi(k)], zm = s[padi(M - k)];
        const float2 wk = __ldg(&tw2[k]), wm = __ldg(&tw2[M - k]);
        {
          const float2 e = make_float2(0.5f * (zk.x + zm.x), 0.5f * (zk.y - zm.y));
          const float2 o = make_float2(0.5f * (zk.y + zm.y), -0.5f * (zk.x - zm.x));   // −(i/2)(zk − zm*)
          dst[k] = cadd(e, cmul(wk, o));
        }
        if (k != M - k) {
          const float2 e = make_float2(0.5f * (zm.x + zk.x), 0.5f * (zm.y - zk.y));
          const float2 o = make_float2(0.5f * (zm.y + zk.y), -0.5f * (zm.x - zk.x));
          dst[M - k] = cadd(e, cmul(wm, o));
        }
      }
    }
  }
}

// ------------------------------------------------------------------------------------------------ rows C2R
// epilogue 0: out[plane][y][x] = q.   epilogue 1: τ[plane][y][x] += δ(τ, step·q)  (projection increment, R10)
template <int M>
__global__ void __launch_bounds__(RowCfg<M>::NT) k_rows_c2r(EprLines L, int ny, const float2* __restrict__ spec,
                                                            const float2* __restrict__ tw, const float2* __restrict__ tw2,
                                                            int epilogue, float step, int tau_is_zero, int newton_iters,
                                                            float i_min, float* __restrict__ out) {
  using C = RowCfg<M>;
  __shared__ float2 sm[C::ROWS * C::PL];
  const int lr = threadIdx.x / C::TPC, t = threadIdx.x - lr * C::TPC;
  const int row = blockIdx.x * C::ROWS + lr;
  const bool live = row < ny;
  const size_t plane = blockIdx.y;
  float2* s = sm + lr * C::PL;
  const float2* src = spec + (plane * ny + row) * (size_t)M;
  // Z2[k] = (X[k] + X*[M−k]) + i w^{−k} (X[k] − X*[M−k]);  Z2[0] = (x0 + xM) + i (x0 − xM)
  if (live) {
    for (int k = t; k <= M / 2; k += C::TPC) {
      if (k == 0) {
        const float2 x = __ldg(&src[0]);
        s[0] = make_float2(x.x + x.y, x.x - x.y);
      } else {
        const float2 xk = __ldg(&src[k]), xm = __ldg(&src[M - k]);
        const float2 wk = __ldg(&tw2[k]), wm = __ldg(&tw2[M - k]);
        {
          const float2 e = make_float2(xk.x + xm.x, xk.y - xm.y);
          const float2 dlt = make_float2(xk.x - xm.x, xk.y + xm.y);            // xk − xm*
          const float2 o = make_float2(-dlt.y, dlt.x);                          // i (xk − xm*)
          s[padi(k)] = cadd(e, cmul(make_float2(wk.x, -wk.y), o));
        }
        if (k != M - k) {
          const float2 e = make_float2(xm.x + xk.x, xm.y - xk.y);
          const float2 dlt = make_float2(xm.x - xk.x, xm.y + xk.y);
          const float2 o = make_float2(-dlt.y, dlt.x);
          s[padi(M - k)] = cadd(e, cmul(make_float2(wm.x, -wm.y), o));
        }
      }
    }
  }
  __syncthreads();
  fft_smem<M, C::TPC, 1, true>(s, 0, t, tw);
  if (live) {
    float2* dst = reinterpret_cast<float2*>(out + (plane * ny + row) * (size_t)(2 * M));
    for (int j = t; j < M; j += C::TPC) {
      float2 q = s[padi(j)];
      if (epilogue == 1) {
        float2 tau = tau_is_zero ? make_float2(0.f, 0.f) : dst[j];
        tau.x += epr_project_increment(tau.x, step * q.x, L, newton_iters, i_min);
        tau.y += epr_project_increment(tau.y, step * q.y, L, newton_iters, i_min);
        q = tau;
      }
      dst[j] = q;
    }
  }
}

// ------------------------------------------------------------------------------------------------ columns
template <int N> struct ColCfg {
  static constexpr int W = 4;                    // columns per CTA (32 B per row segment)
  static constexpr int TPC = (N + 15) / 16;      // threads per column
  static constexpr int NT = TPC * W;
  static constexpr int PL = padded_len(N);
  static constexpr int OWN = (N + TPC - 1) / TPC;
  static constexpr size_t SMEM = (size_t)PL * W * sizeof(float2);
};

// mode 0: out[plane] = IFFT( H_{plane % nb} FFT(spec[plane]) )      (per-line, epr_precondition)
// mode 1: out[b]     = IFFT( Σ_s H_s FFT(spec[b·nb + s]) )           (Fourier-space sum, R10 identity)
// mode 2: out[plane] = IFFT( H_ā FFT(spec[plane]) )                  (initial guess, R9)
template <int N>
__global__ void __launch_bounds__(ColCfg<N>::NT) k_cols(EprLines L, int M, int mode, float scale,
                                                        const float* __restrict__ lam_x, const float* __restrict__ lam_y,
                                                        const float2* __restrict__ tw, const float2* __restrict__ spec,
                                                        float2* __restrict__ out) {
  using C = ColCfg<N>;
  extern __shared__ float2 sm[];
  const int c = threadIdx.x % C::W, t = threadIdx.x / C::W;
  const int kx = blockIdx.x * C::W + c;
  const int oplane = blockIdx.y;
  const int nb = L.n_bins;
  const int nloop = (mode == 1) ? nb : 1;
  const bool live = kx < M;
  const float lx = live ? __ldg(&lam_x[kx]) : 0.f;
  const float lxN = __ldg(&lam_x[M]);            // λx at the Nyquist column (packed into kx = 0)
  float2 acc[C::OWN];
#pragma unroll
  for (int m = 0; m < C::OWN; ++m) acc[m] = make_float2(0.f, 0.f);

  for (int sl = 0; sl < nloop; ++sl) {
    const size_t iplane = (mode == 1) ? (size_t)oplane * nb + sl : (size_t)oplane;
    const float a = (mode == 2) ? L.abar : L.a[(mode == 1) ? sl : (oplane % nb)];
    const float2* src = spec + iplane * (size_t)N * M;
    for (int i = threadIdx.x; i < N * C::W; i += C::NT) {
      const int ky = i / C::W, cc = i - ky * C::W;
      const int k2 = blockIdx.x * C::W + cc;
      sm[padi(ky) * C::W + cc] = (k2 < M) ? __ldg(&src[(size_t)ky * M + k2]) : make_float2(0.f, 0.f);
    }
    __syncthreads();
    fft_smem<N, C::TPC, C::W, false>(sm, c, t, tw);
    if (kx == 0) {
      // packed column: C = F0 + i FM with F0, FM Hermitian in ky.  A = ½(C[ky] + C*[−ky]), B = −(i/2)(C[ky] − C*[−ky]);
      // C'[ky] = H(0,ky) A + i H(M,ky) B,  C'[−ky] = H(0,ky) A* + i H(M,ky) B*
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
    for (int m = 0; m < C::OWN; ++m) {
      const int ky = t + m * C::TPC;
      if (C::OWN * C::TPC == N || ky < N) {
        const float2 v = sm[padi(ky) * C::W + c];
        const float h = (kx == 0) ? 1.f : scale / (1.f + a * (lx + __ldg(&lam_y[ky])));
        acc[m].x = fmaf(h, v.x, acc[m].x);
        acc[m].y = fmaf(h, v.y, acc[m].y);
      }
    }
    __syncthreads();
  }
#pragma unroll
  for (int m = 0; m < C::OWN; ++m) {
    const int ky = t + m * C::TPC;
    if (C::OWN * C::TPC == N || ky < N) sm[padi(ky) * C::W + c] = acc[m];
  }
  __syncthreads();
  fft_smem<N, C::TPC, C::W, true>(sm, c, t, tw);
  float2* dst = out + (size_t)oplane * N * M;
  for (int i = threadIdx.x; i < N * C::W; i += C::NT) {
    const int ky = i / C::W, cc = i - ky * C::W;
    const int k2 = blockIdx.x * C::W + cc;
    if (k2 < M) dst[(size_t)ky * M + k2] = sm[padi(ky) * C::W + cc];
  }
}

// ------------------------------------------------------------------------------------------------ dispatch
#define EPR_FFT_SIZES(X) X(16) X(32) X(48) X(64) X(80) X(96) X(128) X(160) X(256) X(320) X(512) X(1024) X(2048) X(2160) X(2560)

extern "C" int epr_fft_size_supported(int n) {
#define X(n_) if (n == n_) return 1;
  EPR_FFT_SIZES(X)
#undef X
  return 0;
}

cudaError_t epr_launch_rows_r2c(const epr_plan_s* p, int planes, const float* in, float in_offset, float2* spec,
                                cudaStream_t st) {
  switch (p->nx) {
#define X(n_)                                                                                                   \
  case n_: {                                                                                                    \
    using C = RowCfg<n_ / 2>;                                                                                   \
    dim3 grid((p->ny + C::ROWS - 1) / C::ROWS, planes);                                                         \
    k_rows_r2c<n_ / 2><<<grid, C::NT, 0, st>>>(p->ny, in, in_offset, p->tw_row, p->tw_r2c, spec);                \
  } break;
    EPR_FFT_SIZES(X)
#undef X
    default: return cudaErrorInvalidValue;
  }
  return cudaGetLastError();
}

cudaError_t epr_launch_rows_c2r(const epr_plan_s* p, int planes, const float2* spec, int epilogue, float step,
                                int tau_is_zero, float* q_or_tau, cudaStream_t st) {
  switch (p->nx) {
#define X(n_)                                                                                                   \
  case n_: {                                                                                                    \
    using C = RowCfg<n_ / 2>;                                                                                   \
    dim3 grid((p->ny + C::ROWS - 1) / C::ROWS, planes);                                                         \
    k_rows_c2r<n_ / 2><<<grid, C::NT, 0, st>>>(p->lines, p->ny, spec, p->tw_row, p->tw_r2c, epilogue, step,       \
                                               tau_is_zero, p->opt.newton_iters, p->opt.i_min, q_or_tau);       \
  } break;
    EPR_FFT_SIZES(X)
#undef X
    default: return cudaErrorInvalidValue;
  }
  return cudaGetLastError();
}

cudaError_t epr_launch_cols(const epr_plan_s* p, int planes, int mode, const float2* spec, float2* out, cudaStream_t st) {
  const int M = p->nx / 2;
  const int oplanes = (mode == 1) ? planes / p->n_bins : planes;
  const float scale = (float)(1.0 / ((double)p->nx * (double)p->ny));
  switch (p->ny) {
#define X(n_)                                                                                                   \
  case n_: {                                                                                                    \
    using C = ColCfg<n_>;                                                                                       \
    static bool attr = false;                                                                                   \
    if (!attr) { cudaFuncSetAttribute(k_cols<n_>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM); attr = true; } \
    dim3 grid((M + C::W - 1) / C::W, oplanes);                                                                  \
    k_cols<n_><<<grid, C::NT, C::SMEM, st>>>(p->lines, M, mode, scale, p->lam_x, p->lam_y, p->tw_col, spec, out); \
  } break;
    EPR_FFT_SIZES(X)
#undef X
    default: return cudaErrorInvalidValue;
  }
  return cudaGetLastError();
}
