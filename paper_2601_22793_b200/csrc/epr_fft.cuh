// epr_fft.cuh — shared-memory mixed-radix Stockham FFT engine (radices 16/8/4/2/5/3), sm_100a.
//
// Used by the FFT-diagonal Paganin-type preconditioner P^{-1}_{1,s}: row R2C,
// column FFT · H_s · column IFFT, row C2R.  The data of one transform live in shared memory as float2
// at  s[pad(i) * STRIDE + off];  each pass is done by TPC cooperating threads which hold their
// butterflies in registers (read all → barrier → write all → barrier), so no ping-pong buffer is needed.
// Natural order in, natural order out (autosort).  Forward sign e^{-i…}; INV gives the unnormalised inverse.
#pragma once
#include <cuda_runtime.h>

namespace eprfft {

// Greedy radix choice.  The composite odd / semi-odd radices 15, 10, 9, 6 (nested 3x5, 2x5, 3x3, 2x3 butterflies in
// registers) keep the mixed sizes at three passes: 2160 = 16·15·9, 2560 = 16·16·10, 1080 = 8·15·9.
__host__ __device__ constexpr int pick_radix(int rem) {
  return (rem % 16 == 0) ? 16 : (rem % 8 == 0) ? 8 : (rem % 4 == 0) ? 4 : (rem % 15 == 0) ? 15 : (rem % 10 == 0) ? 10
       : (rem % 9 == 0) ? 9 : (rem % 6 == 0) ? 6 : (rem % 2 == 0) ? 2 : (rem % 5 == 0) ? 5 : (rem % 3 == 0) ? 3 : 0;
}
__host__ __device__ constexpr bool supported(int n) {
  while (n > 1) { int r = pick_radix(n); if (!r) return false; n /= r; }
  return true;
}
// shared-memory padding: one extra element every 16 keeps stride-R first-pass writes off a single bank
__host__ __device__ constexpr int padi(int i) { return i + (i >> 4); }
__host__ __device__ constexpr int padded_len(int n) { return padi(n - 1) + 1; }

__device__ __forceinline__ float2 cmul(float2 a, float2 b) {
  return make_float2(fmaf(a.x, b.x, -a.y * b.y), fmaf(a.x, b.y, a.y * b.x));
}
// (packed add.f32x2 / fma.rn.f32x2 were tried here: fewer FP instructions but more register-pair moves and
// address arithmetic; the column kernel got 10 % slower, so the scalar forms stay)
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
template <bool INV> __device__ __forceinline__ float2 rot90(float2 a) {   // multiply by -i (fwd) / +i (inv)
  return INV ? make_float2(-a.y, a.x) : make_float2(a.y, -a.x);
}
template <bool INV> __device__ __forceinline__ float2 conj_if(float2 a) { return INV ? make_float2(a.x, -a.y) : a; }

template <bool INV> __device__ __forceinline__ void dft2(float2* v) {
  float2 a = v[0], b = v[1];
  v[0] = cadd(a, b); v[1] = csub(a, b);
}
template <bool INV> __device__ __forceinline__ void dft4(float2& a0, float2& a1, float2& a2, float2& a3) {
  float2 t0 = cadd(a0, a2), t1 = csub(a0, a2), t2 = cadd(a1, a3), t3 = rot90<INV>(csub(a1, a3));
  a0 = cadd(t0, t2); a2 = csub(t0, t2); a1 = cadd(t1, t3); a3 = csub(t1, t3);
}
template <bool INV> __device__ __forceinline__ void dft3(float2* v) {
  const float s = INV ? 0.86602540378443864676f : -0.86602540378443864676f;   // Im of w3
  float2 t = cadd(v[1], v[2]), d = csub(v[1], v[2]);
  float2 m = make_float2(fmaf(-0.5f, t.x, v[0].x), fmaf(-0.5f, t.y, v[0].y));
  float2 r = make_float2(-s * d.y, s * d.x);                                  // i*s*d
  v[0] = cadd(v[0], t); v[1] = cadd(m, r); v[2] = csub(m, r);
}
template <bool INV> __device__ __forceinline__ void dft5(float2* v) {
  const float c1 = 0.30901699437494742410f, c2 = -0.80901699437494742410f;
  const float s1 = INV ? 0.95105651629515357212f : -0.95105651629515357212f;
  const float s2 = INV ? 0.58778525229247312917f : -0.58778525229247312917f;
  float2 a = cadd(v[1], v[4]), b = csub(v[1], v[4]), c = cadd(v[2], v[3]), d = csub(v[2], v[3]);
  float2 m1 = make_float2(v[0].x + c1 * a.x + c2 * c.x, v[0].y + c1 * a.y + c2 * c.y);
  float2 m2 = make_float2(v[0].x + c2 * a.x + c1 * c.x, v[0].y + c2 * a.y + c1 * c.y);
  float2 r1 = make_float2(-(s1 * b.y + s2 * d.y), s1 * b.x + s2 * d.x);       // i*(s1 b + s2 d)
  float2 r2 = make_float2(-(s2 * b.y - s1 * d.y), s2 * b.x - s1 * d.x);       // i*(s2 b - s1 d)
  v[0] = cadd(v[0], cadd(a, c));
  v[1] = cadd(m1, r1); v[4] = csub(m1, r1); v[2] = cadd(m2, r2); v[3] = csub(m2, r2);
}
template <bool INV> __device__ __forceinline__ void dft8(float2* v) {
  const float h = 0.70710678118654752440f;
  float2 e0 = v[0], e1 = v[2], e2 = v[4], e3 = v[6], o0 = v[1], o1 = v[3], o2 = v[5], o3 = v[7];
  dft4<INV>(e0, e1, e2, e3);
  dft4<INV>(o0, o1, o2, o3);
  // o_k *= w8^k, w8 = e^{∓iπ/4}
  float2 p1 = INV ? make_float2(h * (o1.x - o1.y), h * (o1.x + o1.y)) : make_float2(h * (o1.x + o1.y), h * (o1.y - o1.x));
  float2 p2 = rot90<INV>(o2);
  float2 p3 = INV ? make_float2(-h * (o3.x + o3.y), h * (o3.x - o3.y)) : make_float2(h * (o3.y - o3.x), -h * (o3.x + o3.y));
  v[0] = cadd(e0, o0); v[4] = csub(e0, o0);
  v[1] = cadd(e1, p1); v[5] = csub(e1, p1);
  v[2] = cadd(e2, p2); v[6] = csub(e2, p2);
  v[3] = cadd(e3, p3); v[7] = csub(e3, p3);
}
template <bool INV> __device__ __forceinline__ void dft16(float2* v) {
  // X[k1 + 4 k2] = Σ_{n2} w16^{n2 k1} ( Σ_{n1} x[4 n1 + n2] w4^{n1 k1} ) w4^{n2 k2}
  const float c1 = 0.92387953251128675613f, s1 = 0.38268343236508977173f, h = 0.70710678118654752440f;
#pragma unroll
  for (int n2 = 0; n2 < 4; ++n2) dft4<INV>(v[n2], v[4 + n2], v[8 + n2], v[12 + n2]);   // v[4 k1 + n2] = Y[n2][k1]
  // twiddles w16^{n2 k1}, w16 = e^{∓iπ/8}
  const float2 w1 = conj_if<INV>(make_float2(c1, -s1)), w2 = conj_if<INV>(make_float2(h, -h)),
               w3 = conj_if<INV>(make_float2(s1, -c1)), w6 = conj_if<INV>(make_float2(-h, -h)),
               w9 = conj_if<INV>(make_float2(-c1, s1));
  v[4 + 1] = cmul(v[4 + 1], w1); v[4 + 2] = cmul(v[4 + 2], w2); v[4 + 3] = cmul(v[4 + 3], w3);
  v[8 + 1] = cmul(v[8 + 1], w2); v[8 + 2] = rot90<INV>(v[8 + 2]); v[8 + 3] = cmul(v[8 + 3], w6);
  v[12 + 1] = cmul(v[12 + 1], w3); v[12 + 2] = cmul(v[12 + 2], w6); v[12 + 3] = cmul(v[12 + 3], w9);
#pragma unroll
  for (int k1 = 0; k1 < 4; ++k1) dft4<INV>(v[4 * k1], v[4 * k1 + 1], v[4 * k1 + 2], v[4 * k1 + 3]);   // → v[4 k1 + k2]
  // natural order X[k1 + 4 k2] ← v[4 k1 + k2]: transpose the 4x4
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = i + 1; j < 4; ++j) { float2 t = v[4 * i + j]; v[4 * i + j] = v[4 * j + i]; v[4 * j + i] = t; }
}
// e^{∓iθ} from (cos θ, sin θ): forward sign −, inverse +
template <bool INV> __device__ __forceinline__ float2 wconst(float c, float sn) { return make_float2(c, INV ? sn : -sn); }

// Composite radix N1·N2 by Cooley-Tukey in registers: n = N2 n1 + n2, k = k1 + N1 k2,
//   X[k1 + N1 k2] = Σ_{n2} w_{N2}^{n2 k2} · w_N^{n2 k1} · ( Σ_{n1} x[N2 n1 + n2] w_{N1}^{n1 k1} ).
template <bool INV> __device__ __forceinline__ void dft6(float2* v) {          // 2 x 3
  float2 y[6];
#pragma unroll
  for (int n2 = 0; n2 < 3; ++n2) { float2 a[2] = {v[n2], v[3 + n2]}; dft2<INV>(a); y[n2] = a[0]; y[3 + n2] = a[1]; }
  y[3 + 1] = cmul(y[3 + 1], wconst<INV>(0.5f, 0.86602540378443864676f));
  y[3 + 2] = cmul(y[3 + 2], wconst<INV>(-0.5f, 0.86602540378443864676f));
#pragma unroll
  for (int k1 = 0; k1 < 2; ++k1) {
    float2 a[3] = {y[3 * k1], y[3 * k1 + 1], y[3 * k1 + 2]};
    dft3<INV>(a);
#pragma unroll
    for (int k2 = 0; k2 < 3; ++k2) v[k1 + 2 * k2] = a[k2];
  }
}
template <bool INV> __device__ __forceinline__ void dft9(float2* v) {          // 3 x 3
  float2 y[9];
#pragma unroll
  for (int n2 = 0; n2 < 3; ++n2) {
    float2 a[3] = {v[n2], v[3 + n2], v[6 + n2]};
    dft3<INV>(a);
    y[n2] = a[0]; y[3 + n2] = a[1]; y[6 + n2] = a[2];
  }
  y[3 + 1] = cmul(y[3 + 1], wconst<INV>(0.76604444311897803520f, 0.64278760968653932632f));    // w9^1
  y[3 + 2] = cmul(y[3 + 2], wconst<INV>(0.17364817766693034885f, 0.98480775301220805937f));    // w9^2
  y[6 + 1] = cmul(y[6 + 1], wconst<INV>(0.17364817766693034885f, 0.98480775301220805937f));    // w9^2
  y[6 + 2] = cmul(y[6 + 2], wconst<INV>(-0.93969262078590838405f, 0.34202014332566873304f));   // w9^4
#pragma unroll
  for (int k1 = 0; k1 < 3; ++k1) {
    float2 a[3] = {y[3 * k1], y[3 * k1 + 1], y[3 * k1 + 2]};
    dft3<INV>(a);
#pragma unroll
    for (int k2 = 0; k2 < 3; ++k2) v[k1 + 3 * k2] = a[k2];
  }
}
template <bool INV> __device__ __forceinline__ void dft10(float2* v) {         // 2 x 5
  float2 y[10];
#pragma unroll
  for (int n2 = 0; n2 < 5; ++n2) { float2 a[2] = {v[n2], v[5 + n2]}; dft2<INV>(a); y[n2] = a[0]; y[5 + n2] = a[1]; }
  y[5 + 1] = cmul(y[5 + 1], wconst<INV>(0.80901699437494742410f, 0.58778525229247312917f));    // w10^1
  y[5 + 2] = cmul(y[5 + 2], wconst<INV>(0.30901699437494742410f, 0.95105651629515357212f));    // w10^2
  y[5 + 3] = cmul(y[5 + 3], wconst<INV>(-0.30901699437494742410f, 0.95105651629515357212f));   // w10^3
  y[5 + 4] = cmul(y[5 + 4], wconst<INV>(-0.80901699437494742410f, 0.58778525229247312917f));   // w10^4
#pragma unroll
  for (int k1 = 0; k1 < 2; ++k1) {
    float2 a[5] = {y[5 * k1], y[5 * k1 + 1], y[5 * k1 + 2], y[5 * k1 + 3], y[5 * k1 + 4]};
    dft5<INV>(a);
#pragma unroll
    for (int k2 = 0; k2 < 5; ++k2) v[k1 + 2 * k2] = a[k2];
  }
}
template <bool INV> __device__ __forceinline__ void dft15(float2* v) {         // 3 x 5
  float2 y[15];
#pragma unroll
  for (int n2 = 0; n2 < 5; ++n2) {
    float2 a[3] = {v[n2], v[5 + n2], v[10 + n2]};
    dft3<INV>(a);
    y[n2] = a[0]; y[5 + n2] = a[1]; y[10 + n2] = a[2];
  }
  // w15^{n2 k1}: k1 = 1 → exponents 1..4; k1 = 2 → 2, 4, 6, 8
  y[5 + 1] = cmul(y[5 + 1], wconst<INV>(0.91354545764260089550f, 0.40673664307580020775f));
  y[5 + 2] = cmul(y[5 + 2], wconst<INV>(0.66913060635885821383f, 0.74314482547739423501f));
  y[5 + 3] = cmul(y[5 + 3], wconst<INV>(0.30901699437494742410f, 0.95105651629515357212f));
  y[5 + 4] = cmul(y[5 + 4], wconst<INV>(-0.10452846326765347140f, 0.99452189536827333692f));
  y[10 + 1] = cmul(y[10 + 1], wconst<INV>(0.66913060635885821383f, 0.74314482547739423501f));
  y[10 + 2] = cmul(y[10 + 2], wconst<INV>(-0.10452846326765347140f, 0.99452189536827333692f));
  y[10 + 3] = cmul(y[10 + 3], wconst<INV>(-0.80901699437494742410f, 0.58778525229247312917f));
  y[10 + 4] = cmul(y[10 + 4], wconst<INV>(-0.97814760073380563793f, -0.20791169081775933710f));
#pragma unroll
  for (int k1 = 0; k1 < 3; ++k1) {
    float2 a[5] = {y[5 * k1], y[5 * k1 + 1], y[5 * k1 + 2], y[5 * k1 + 3], y[5 * k1 + 4]};
    dft5<INV>(a);
#pragma unroll
    for (int k2 = 0; k2 < 5; ++k2) v[k1 + 3 * k2] = a[k2];
  }
}
template <int R, bool INV> __device__ __forceinline__ void dft(float2* v) {
  if constexpr (R == 2) dft2<INV>(v);
  else if constexpr (R == 3) dft3<INV>(v);
  else if constexpr (R == 4) dft4<INV>(v[0], v[1], v[2], v[3]);
  else if constexpr (R == 5) dft5<INV>(v);
  else if constexpr (R == 6) dft6<INV>(v);
  else if constexpr (R == 8) dft8<INV>(v);
  else if constexpr (R == 9) dft9<INV>(v);
  else if constexpr (R == 10) dft10<INV>(v);
  else if constexpr (R == 15) dft15<INV>(v);
  else dft16<INV>(v);
}

// ---- radix schedule: forward order greedy (16,…,8,4,2,5,3); the inverse uses the REVERSED order, so that the
// last forward pass and the first inverse pass act on the same butterflies (indices j + r·N/R) and a diagonal
// filter can be applied between them in registers. ----
__host__ __device__ constexpr int num_passes(int n) { int c = 0; while (n > 1) { n /= pick_radix(n); ++c; } return c; }
__host__ __device__ constexpr int fwd_radix(int n, int i) {
  int r = pick_radix(n);
  while (i-- > 0) { n /= r; r = pick_radix(n); }
  return r;
}
// radix of pass i (0-based) in schedule DIR (false: forward order, true: reversed order)
__host__ __device__ constexpr int sched_radix(int n, int i, bool rev) { return fwd_radix(n, rev ? num_passes(n) - 1 - i : i); }
__host__ __device__ constexpr int sched_P(int n, int i, bool rev) {   // product of the radices before pass i
  int p = 1;
  for (int k = 0; k < i; ++k) p *= sched_radix(n, k, rev);
  return p;
}

// Per-pass twiddle tables: pass i ≥ 1 of a schedule uses tab[off_i + (r−1)·P_i + k] = exp(−2πi r k /(P_i R_i)),
// k < P_i, 1 ≤ r < R_i — laid out so that threads with consecutive k read consecutive addresses (one or two
// 128-byte lines per warp load instead of up to 4r lines with a single stride-indexed table).
__host__ __device__ constexpr int tw_offset(int n, int i, bool rev) {
  int off = 0;
  for (int k = 1; k < i; ++k) off += (sched_radix(n, k, rev) - 1) * sched_P(n, k, rev);
  return off;
}
__host__ __device__ constexpr int tw_total(int n, bool rev) { return tw_offset(n, num_passes(n), rev); }

// Threads cooperating on one transform: 16 points each, but never fewer than the butterflies of a radix-15 pass
// (N/15 > N/16 would otherwise cost a whole second, almost empty, round of 15-point butterflies).
__host__ __device__ constexpr int threads_per_transform(int n) {
  int t = (n + 15) / 16;
  for (int i = 0; i < num_passes(n); ++i)
    if (fwd_radix(n, i) == 15 && n / 15 > t) t = n / 15;
  return t;
}

template <int N, int R, int TPC> struct PassGeom {
  static constexpr int T = N / R;                       // butterflies per transform
  static constexpr int CNT = (T + TPC - 1) / TPC;       // butterflies per thread
  static constexpr bool FULL = (CNT * TPC == T);
};

// Butterfly + Stockham scatter of one thread's butterflies held in u[c][r] (inputs x[j + r·T], j = t + c·TPC):
// twiddle (P > 1), radix-R DFT; afterwards u[c][q] is output element j0 + q·P, j0 = (j − j%P)·R + j%P.
// TWS: the twiddle table lives in shared memory (plain loads) instead of global memory (read-only path)
template <int N, int P, int R, int TPC, bool INV, bool TWS = false>
__device__ __forceinline__ void bfly(float2 (&u)[PassGeom<N, R, TPC>::CNT][R], int t, const float2* __restrict__ tw) {
  using G = PassGeom<N, R, TPC>;
#pragma unroll
  for (int c = 0; c < G::CNT; ++c) {
    const int j = t + c * TPC;
    if (G::FULL || j < G::T) {
      if constexpr (P > 1) {
        const int k = j % P;
#pragma unroll
        for (int r = 1; r < R; ++r) u[c][r] = cmul(u[c][r], conj_if<INV>(TWS ? tw[(r - 1) * P + k] : __ldg(&tw[(r - 1) * P + k])));
      }
      dft<R, INV>(u[c]);
    }
  }
}
template <int N, int R, int TPC, int STRIDE>
__device__ __forceinline__ void smem_gather(float2 (&u)[PassGeom<N, R, TPC>::CNT][R], const float2* s, int off, int t) {
  using G = PassGeom<N, R, TPC>;
#pragma unroll
  for (int c = 0; c < G::CNT; ++c) {
    const int j = t + c * TPC;
    if (G::FULL || j < G::T) {
#pragma unroll
      for (int r = 0; r < R; ++r) u[c][r] = s[padi(j + r * G::T) * STRIDE + off];
    }
  }
}
template <int N, int P, int R, int TPC, int STRIDE>
__device__ __forceinline__ void smem_scatter(const float2 (&u)[PassGeom<N, R, TPC>::CNT][R], float2* s, int off, int t) {
  using G = PassGeom<N, R, TPC>;
#pragma unroll
  for (int c = 0; c < G::CNT; ++c) {
    const int j = t + c * TPC;
    if (G::FULL || j < G::T) {
      const int k = (P == 1) ? 0 : j % P;
      const int j0 = (j - k) * R + k;
#pragma unroll
      for (int q = 0; q < R; ++q) s[padi(j0 + q * P) * STRIDE + off] = u[c][q];
    }
  }
}

// Engine for one transform size/schedule.  REV selects the reversed radix order (used for inverses).
// Usage (n = NP passes):  first pass inputs come from registers (filled by the caller from global memory:
// element index of u[c][r] is (t + c·TPC) + r·T0), last pass outputs stay in registers (element index of
// u[c][q] is (t + c·TPC) + q·PL).  Passes in between go through shared memory.
template <int N, int TPC, int STRIDE, bool INV, bool REV, bool TWS = false> struct Engine {
  static constexpr int NP = num_passes(N);
  static constexpr int R0 = sched_radix(N, 0, REV);                 // first radix
  static constexpr int RL = sched_radix(N, NP - 1, REV);            // last radix
  static constexpr int PL = sched_P(N, NP - 1, REV);                // = N / RL
  using G0 = PassGeom<N, R0, TPC>;
  using GL = PassGeom<N, RL, TPC>;

  template <int I> __device__ static __forceinline__ void middle(float2* s, int off, int t, const float2* __restrict__ tw) {
    if constexpr (I < NP - 1) {
      constexpr int R = sched_radix(N, I, REV), P = sched_P(N, I, REV);
      float2 u[PassGeom<N, R, TPC>::CNT][R];
      smem_gather<N, R, TPC, STRIDE>(u, s, off, t);
      __syncthreads();
      bfly<N, P, R, TPC, INV, TWS>(u, t, tw + tw_offset(N, I, REV));
      smem_scatter<N, P, R, TPC, STRIDE>(u, s, off, t);
      __syncthreads();
      middle<I + 1>(s, off, t, tw);
    }
  }
  // u0: first-pass inputs (registers) → … → uL: last-pass outputs (registers).  For NP == 1, u0 and uL are the
  // same butterflies: pass the same array type (R0 == RL) and the result is left in uL.
  __device__ static __forceinline__ void run(float2 (&u0)[G0::CNT][R0], float2 (&uL)[GL::CNT][RL], float2* s, int off, int t,
                                             const float2* __restrict__ tw) {
    if constexpr (NP == 1) {
      bfly<N, 1, R0, TPC, INV, TWS>(u0, t, tw);
#pragma unroll
      for (int c = 0; c < G0::CNT; ++c)
#pragma unroll
        for (int r = 0; r < R0; ++r) uL[c][r] = u0[c][r];
    } else {
      bfly<N, 1, R0, TPC, INV, TWS>(u0, t, tw);
      smem_scatter<N, 1, R0, TPC, STRIDE>(u0, s, off, t);
      __syncthreads();
      middle<1>(s, off, t, tw);
      smem_gather<N, RL, TPC, STRIDE>(uL, s, off, t);
      bfly<N, PL, RL, TPC, INV, TWS>(uL, t, tw + tw_offset(N, NP - 1, REV));
    }
  }
};

}  // namespace eprfft

// =====================================================================================================
// Swizzled in-place variant for power-of-two column transforms whose tile is staged by TMA.
// A tile is N rows of W = 4 complex columns (32 bytes per row), exactly as the TMA box lands it: LINEAR layout,
// element (row, c) at float2 index row·4 + c, no padding (N·32 bytes in all).  After the first pass the data live
// in the SAME N·32 bytes in a SWIZZLED layout  (row ^ h(row))·4 + c  with
//     h(row) = ((row>>3 ^ row>>5) & 1) | ((row>>4 & 1) << 1),
// a bijection that only permutes the 4 rows of a 128-byte group.  A warp is 8 butterflies x 4 columns, and a
// 64-bit shared access is served per half-warp (4 butterflies x 4 columns = 128 bytes if the 4 rows differ mod 4):
// with h, the 4 rows are distinct mod 4 for consecutive rows and for rows 8 or 16 apart — every gather / scatter
// pattern of the (16,16,8 | 8,16,16) schedules — so all passes are bank-conflict free without padding.
// Addresses: a thread's rows in one pass are rb + off with rb (run time) and off (compile time) on disjoint bits, so
// (rb + off) ^ h(rb + off) = [rb ^ h(rb)] ^ h(off) + off: ONE base register per pass (xor-ed with a 2-bit
// constant) plus immediate offsets — no per-access index arithmetic.
// =====================================================================================================
namespace eprfft {

__host__ __device__ constexpr int hsw(int row) { return (((row >> 3) ^ (row >> 5)) & 1) | (((row >> 4) & 1) << 1); }

// float2 index of row (rb + OFF), given e0 = ((rb ^ h(rb)) << 2) + c
template <int OFF> __device__ __forceinline__ int sw_index(int e0) {
  constexpr int x = (OFF & 3) ^ hsw(OFF);
  return (e0 ^ (x << 2)) + ((OFF & ~3) << 2);
}
__device__ __forceinline__ int sw_base(int rb, int c) { return ((rb ^ hsw(rb)) << 2) + c; }

template <int N, int R, int TPC, int CC, int RR>
__device__ __forceinline__ void sw_gather_one(float2 (&u)[PassGeom<N, R, TPC>::CNT][R], const float2* s, int e0) {
  using G = PassGeom<N, R, TPC>;
  u[CC][RR] = s[sw_index<CC * TPC + RR * G::T>(e0)];
  if constexpr (RR + 1 < R) sw_gather_one<N, R, TPC, CC, RR + 1>(u, s, e0);
  else if constexpr (CC + 1 < G::CNT) sw_gather_one<N, R, TPC, CC + 1, 0>(u, s, e0);
}
// rows t + cc·TPC + r·T: rb = t
template <int N, int R, int TPC>
__device__ __forceinline__ void sw_gather(float2 (&u)[PassGeom<N, R, TPC>::CNT][R], const float2* s, int c, int t) {
  static_assert(PassGeom<N, R, TPC>::FULL, "power-of-two sizes only");
  sw_gather_one<N, R, TPC, 0, 0>(u, s, sw_base(t, c));
}
template <int N, int P, int R, int TPC, int CC, int Q>
__device__ __forceinline__ void sw_scatter_q(const float2 (&u)[PassGeom<N, R, TPC>::CNT][R], float2* s, int e0) {
  s[sw_index<Q * P>(e0)] = u[CC][Q];
  if constexpr (Q + 1 < R) sw_scatter_q<N, P, R, TPC, CC, Q + 1>(u, s, e0);
}
template <int N, int P, int R, int TPC, int CC>
__device__ __forceinline__ void sw_scatter_cc(const float2 (&u)[PassGeom<N, R, TPC>::CNT][R], float2* s, int c, int t) {
  using G = PassGeom<N, R, TPC>;
  const int j = t + CC * TPC;
  const int k = (P == 1) ? 0 : j % P;
  const int j0 = (j - k) * R + k;                 // rows j0 + q·P: rb = j0
  sw_scatter_q<N, P, R, TPC, CC, 0>(u, s, sw_base(j0, c));
  if constexpr (CC + 1 < G::CNT) sw_scatter_cc<N, P, R, TPC, CC + 1>(u, s, c, t);
}
template <int N, int P, int R, int TPC>
__device__ __forceinline__ void sw_scatter(const float2 (&u)[PassGeom<N, R, TPC>::CNT][R], float2* s, int c, int t) {
  sw_scatter_cc<N, P, R, TPC, 0>(u, s, c, t);
}

// Same pass structure as Engine (STRIDE = 4 columns per tile), on the swizzled layout.
//  run_first: first-pass inputs already in registers (read by the caller from the LINEAR tile, followed by a barrier)
//  the last pass leaves its outputs in registers (element index of uL[c][q] is (t + c·TPC) + q·PL).
// barrier of the threads that share a tile: the whole CTA (GROUP = 0, __syncthreads) or a named barrier `id` of GROUP
// threads (two 512-thread groups of one CTA working on different tiles)
template <int GROUP> __device__ __forceinline__ void tile_sync(int id) {
  if constexpr (GROUP == 0) __syncthreads();
  else asm volatile("bar.sync %0, %1;" ::"r"(id), "n"(GROUP) : "memory");
}

template <int N, int TPC, bool INV, bool REV, int GROUP = 0> struct EngineSw {
  using E = Engine<N, TPC, 4, INV, REV>;
  static constexpr int NP = E::NP, R0 = E::R0, RL = E::RL, PL = E::PL;
  using G0 = typename E::G0;
  using GL = typename E::GL;
  static_assert(NP >= 2, "at least two passes");

  template <int I> __device__ static __forceinline__ void middle(float2* s, int c, int t, const float2* __restrict__ tw, int bar) {
    if constexpr (I < NP - 1) {
      constexpr int R = sched_radix(N, I, REV), P = sched_P(N, I, REV);
      float2 u[PassGeom<N, R, TPC>::CNT][R];
      sw_gather<N, R, TPC>(u, s, c, t);
      tile_sync<GROUP>(bar);
      bfly<N, P, R, TPC, INV>(u, t, tw + tw_offset(N, I, REV));
      sw_scatter<N, P, R, TPC>(u, s, c, t);
      tile_sync<GROUP>(bar);
      middle<I + 1>(s, c, t, tw, bar);
    }
  }
  struct NoHook { __device__ __forceinline__ void operator()() const {} };
  // hook: called once by every thread after its first-pass scatter, before the first barrier (a place where one
  // thread can do a little bookkeeping while the others are still computing)
  template <class HOOK = NoHook>
  __device__ static __forceinline__ void run(float2 (&u0)[G0::CNT][R0], float2 (&uL)[GL::CNT][RL], float2* s, int c, int t,
                                             const float2* __restrict__ tw, int bar = 0, HOOK hook = HOOK()) {
    bfly<N, 1, R0, TPC, INV>(u0, t, tw);
    sw_scatter<N, 1, R0, TPC>(u0, s, c, t);
    hook();
    tile_sync<GROUP>(bar);
    middle<1>(s, c, t, tw, bar);
    sw_gather<N, RL, TPC>(uL, s, c, t);
    bfly<N, PL, RL, TPC, INV>(uL, t, tw + tw_offset(N, NP - 1, REV));
  }
};

}  // namespace eprfft
