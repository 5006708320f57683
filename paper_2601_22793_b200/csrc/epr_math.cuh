// epr_math.cuh — per-pixel device arithmetic of the EPR iteration (deviation form, fp32).
//
// fp32 near 1 is too coarse for the retrieved phase (φ = (db/2) ln I with db/2 = 100…500), so the device
// path never stores or differences O(1) intensities: the state is τ (Eq. (7)), line
// intensities enter as J_s = I_s/f_s − 1 = expm1(−γ_s τ), the data as d − 1, predictions as P_s − f_s,
// and the projection is solved for the increment δτ.
#pragma once
#include "epr_internal.h"

__device__ __forceinline__ int wrap1(int i, int n) { return i < 0 ? i + n : (i >= n ? i - n : i); }   // -n <= i < 2n
__device__ __forceinline__ int wrapm(int i, int n) { i %= n; return i < 0 ? i + n : i; }               // any i

// expm1 to ~2 ulp RELATIVE accuracy without the slow path of expm1f: Taylor (degree 8) for |x| < 0.35
// (truncation x^8/9! < 1e-9 relative), exp(x) − 1 with the MUFU exponential beyond (|result| > 0.29 there, so
// the 2^-22 relative error of ex2.approx stays below 1e-6 relative).  Both branches are evaluated (no divergence).
// Taylor branch alone (valid for |x| < 0.35): callers test the range once per warp and row.
__device__ __forceinline__ float epr_expm1_small(float x) {
  float q = fmaf(x, 2.48015873e-5f, 1.98412698e-4f);
  q = fmaf(x, q, 1.38888889e-3f);
  q = fmaf(x, q, 8.33333333e-3f);
  q = fmaf(x, q, 4.16666667e-2f);
  q = fmaf(x, q, 1.66666667e-1f);
  q = fmaf(x, q, 0.5f);
  return fmaf(x * x, q, x);
}

// Taylor degree 5 for |x| < 0.09: truncation x^6/720, 1e-8 relative to x at the limit (below fp32 rounding)
__device__ __forceinline__ float epr_expm1_tiny(float x) {
  float q = fmaf(x, 8.33333333e-3f, 4.16666667e-2f);
  q = fmaf(x, q, 1.66666667e-1f);
  q = fmaf(x, q, 0.5f);
  return fmaf(x * x, q, x);
}

// e^x by the MUFU exponential alone (ex2.approx.ftz, 2^-22 relative; no denormal rescue: callers' results saturate)
__device__ __forceinline__ float epr_exp_fast(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x * 1.4426950408889634f));
  return y;
}

__device__ __forceinline__ float epr_expm1(float x) {
  float q = fmaf(x, 2.48015873e-5f, 1.98412698e-4f);
  q = fmaf(x, q, 1.38888889e-3f);
  q = fmaf(x, q, 8.33333333e-3f);
  q = fmaf(x, q, 4.16666667e-2f);
  q = fmaf(x, q, 1.66666667e-1f);
  q = fmaf(x, q, 0.5f);
  const float small = fmaf(x * x, q, x);
  const float big = __expf(x) - 1.f;
  return fabsf(x) < 0.35f ? small : big;
}

// log1p to ~2 ulp relative accuracy: 2 atanh(z/(2+z)) series for |z| < 0.25 (s^10/11 < 1e-10), log(1+z) beyond.
__device__ __forceinline__ float epr_log1p(float z) {
  const float s = __fdividef(z, 2.f + z);
  const float s2 = s * s;
  float q = fmaf(s2, 0.111111111f, 0.142857143f);
  q = fmaf(s2, q, 0.2f);
  q = fmaf(s2, q, 0.333333333f);
  q = fmaf(s2, q, 1.f);
  const float small = 2.f * s * q;
  const float big = __logf(1.f + z);
  return fabsf(z) < 0.25f ? small : big;
}

// out-of-line copy for rare paths (keeps the unrolled epilogues small)
static __device__ __noinline__ float epr_log1p_cold(float z) { return epr_log1p(z); }

// One spectral line (f = γ = 1, I = e^{−τ}):  δ = −log1p(ΔT e^{τ}), with the floor I + ΔT ≥ i_min ⇔ 1 + z ≥ i_min e^{τ}.
// log1p: alternating series (degree 8, |z| < 0.1: z^9/9 < 1.2e-10) on the common path, atanh series / log beyond.
__device__ __forceinline__ float epr_project_increment_mono(float tau, float dT, float i_min) {
  const float E = __expf(tau);
  float z = dT * E;
  z = fmaxf(z, fmaf(i_min, E, -1.f));
  if (fabsf(z) < 0.1f) {
    float q = fmaf(z, -0.125f, 0.142857143f);
    q = fmaf(z, q, -0.166666667f);
    q = fmaf(z, q, 0.2f);
    q = fmaf(z, q, -0.25f);
    q = fmaf(z, q, 0.333333333f);
    q = fmaf(z, q, -0.5f);
    return -fmaf(z * z, q, z);
  }
  return -epr_log1p_cold(z);
}

// Converging iterations of the projection (R10) for a compile-time number of lines: |γ_max δ| < 0.01, where the cubic
// Taylor polynomial of F(δ) = Σ_s I_s expm1(−γ_s δ) − ΔT is exact to (γδ)³/24 < 5e-8 relative.  The per-line constants
// are read straight from the kernel's parameter bank (L by value, s unrolled): one FFMA + one MUFU.EX2 for I_s and one
// FFMA per moment, no table loads.  Returns false when the step is too large or the floor could bind: the caller then
// takes the general routine below.
template <int NB>
__device__ __forceinline__ bool epr_project_increment_small(const EprLines& L, float tau, float dT, int newton_iters,
                                                            float i_min, float& delta_out) {
  float G0 = 0.f, G1 = 0.f, G2 = 0.f, G3 = 0.f;
#pragma unroll
  for (int s = 0; s < NB; ++s) {
    float p;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(p) : "f"(fmaf(tau, L.pj_a[s], L.pj_b[s])));
    G0 += p;
    G1 = fmaf(p, L.gamma[s], G1);
    G2 = fmaf(p, L.pj_g2[s], G2);
    G3 = fmaf(p, L.pj_g3[s], G3);
  }
  const float rc1 = -__fdividef(1.f, G1);            // 1 / c1
  float delta = dT * rc1;                            // y = ΔT / c1: first order
  // straight-line code (no early return): the caller runs two pixels through it back to back and the two chains of
  // exponentials and divisions interleave; a result with ok == false is discarded
  const bool ok = fabsf(delta) * L.gamma_max < 0.01f && G0 + dT >= i_min;
  if (newton_iters > 0) {
    // No loop, no divergence: second-order series reversion δ₁ = y − (c2/c1) y² (relative error (γ y)²/3 < 4e-5), then
    // ONE Newton step on the cubic, which squares it (< 1e-9: below fp32).  The loop this replaces took three
    // iterations with a division each from the first-order guess and left the warp waiting for its slowest lane.
    const float c1 = -G1, c2 = 0.5f * G2, c3 = -1.66666667e-1f * G3;
    delta = fmaf(-(c2 * rc1) * delta, delta, delta);
    const float F = fmaf(fmaf(fmaf(c3, delta, c2), delta, c1), delta, -dT);
    const float dF = fmaf(fmaf(3.f * c3, delta, 2.f * c2), delta, c1);
    delta -= __fdividef(F, dF);
  }
  delta_out = delta;
  return ok;
}

// the line counts with an unrolled instance: 8 (BASELINE configs C4, C5), 5 and 10 (the paper's own runs);
// two pixels at once (the C2R epilogue's float2): both small-step solutions in one basic block; false if either needs
// the general routine (the caller then takes it for both: the general routine repeats the small test itself)
__device__ __forceinline__ bool epr_project_increment_small_nb2(const EprLines& L, float2 tau, float2 dT, int newton_iters,
                                                                float i_min, float& d0, float& d1) {
  bool ok0, ok1;
  switch (L.n_bins) {
    case 8: ok0 = epr_project_increment_small<8>(L, tau.x, dT.x, newton_iters, i_min, d0);
            ok1 = epr_project_increment_small<8>(L, tau.y, dT.y, newton_iters, i_min, d1); break;
    case 5: ok0 = epr_project_increment_small<5>(L, tau.x, dT.x, newton_iters, i_min, d0);
            ok1 = epr_project_increment_small<5>(L, tau.y, dT.y, newton_iters, i_min, d1); break;
    case 10: ok0 = epr_project_increment_small<10>(L, tau.x, dT.x, newton_iters, i_min, d0);
             ok1 = epr_project_increment_small<10>(L, tau.y, dT.y, newton_iters, i_min, d1); break;
    default: return false;
  }
  return ok0 && ok1;
}

// Projection to the single-thickness manifold, Eq. (7) + PAPER.md:233 (R10), as an increment:
//   given τ and ΔT, find δ with Σ_s I_s(τ) expm1(−γ_s δ) = ΔT, clamped so that Σ_s I_s + ΔT ≥ i_min.
// Newton from the Jensen bound δ0 = −log1p(ΔT/ΣI)/γ̄_I (monotone; exact for one line).
// The exponentials are evaluated ONCE, as the moments G_k = Σ_s I_s γ_s^k; then F(δ) = Σ_k (−δ)^k G_k / k! − ΔT is
// a polynomial and Newton runs on it with no further transcendental: k ≤ 4 when |γ_max δ| < 0.03 (the converging
// iterations; truncation < 2e-10 relative), k ≤ 7 when |γ_max δ| < 0.25 (< 4e-10).  Otherwise: Newton on the exact
// sum (the initial guess, thick objects).
// f, gamma: the per-line tables (any address space; the row kernel keeps a copy in shared memory).  Out of line on
// purpose: the C2R epilogue calls it 32 times per thread and the unrolled copies would not fit the instruction cache.
static __device__ __noinline__ float epr_project_increment(float tau, float dT, const float* __restrict__ f,
                                                           const float* __restrict__ gamma, int nb, float gamma_max,
                                                           int newton_iters, float i_min) {
  if (nb == 1) return epr_project_increment_mono(tau, dT, i_min);
  // tier 1 (converging iterations, |γ_max δ| < 0.03): moments up to G_4, truncation (γδ)^5/5! < 2e-10 relative
  {
    float G0 = 0.f, G1 = 0.f, G2 = 0.f, G3 = 0.f, G4 = 0.f;
    for (int s = 0; s < nb; ++s) {
      const float g = gamma[s];
      float p = f[s] * __expf(-g * tau);
      G0 += p; p *= g;
      G1 += p; p *= g;
      G2 += p; p *= g;
      G3 += p; p *= g;
      G4 += p;
    }
    const float rG1 = __fdividef(1.f, G1);
    float delta = -dT * rG1;                          // first order; the floor cannot bind for so small a step
    if (fabsf(delta) * gamma_max < 0.03f && G0 + dT >= i_min) {
      const float c1 = -G1, c2 = 0.5f * G2, c3 = -1.66666667e-1f * G3, c4 = 4.16666667e-2f * G4;
      for (int it = 0; it < newton_iters; ++it) {
        float P = c4, dP = 0.f;
        dP = fmaf(dP, delta, P); P = fmaf(P, delta, c3);
        dP = fmaf(dP, delta, P); P = fmaf(P, delta, c2);
        dP = fmaf(dP, delta, P); P = fmaf(P, delta, c1);
        const float F = fmaf(P, delta, -dT), dF = fmaf(dP, delta, P);
        const float stp = __fdividef(F, dF);
        delta -= stp;
        if (fabsf(stp) <= 1e-7f * fabsf(delta) + 1e-12f) break;
      }
      return delta;
    }
  }
  float G0 = 0.f, G1 = 0.f, G2 = 0.f, G3 = 0.f, G4 = 0.f, G5 = 0.f, G6 = 0.f, G7 = 0.f;
  for (int s = 0; s < nb; ++s) {
    const float g = gamma[s];
    float p = f[s] * __expf(-g * tau);
    G0 += p; p *= g;
    G1 += p; p *= g;
    G2 += p; p *= g;
    G3 += p; p *= g;
    G4 += p; p *= g;
    G5 += p; p *= g;
    G6 += p; p *= g;
    G7 += p;
  }
  if (G0 + dT < i_min) dT = i_min - G0;
  float delta = -epr_log1p(__fdividef(dT, G0)) * __fdividef(G0, G1);
  if (fabsf(delta) * gamma_max < 0.25f) {
    // c_k = (−1)^k G_k / k!
    const float c1 = -G1, c2 = 0.5f * G2, c3 = -1.66666667e-1f * G3, c4 = 4.16666667e-2f * G4,
                c5 = -8.33333333e-3f * G5, c6 = 1.38888889e-3f * G6, c7 = -1.98412698e-4f * G7;
    for (int it = 0; it < newton_iters; ++it) {
      float P = c7, dP = 0.f;
      dP = fmaf(dP, delta, P); P = fmaf(P, delta, c6);
      dP = fmaf(dP, delta, P); P = fmaf(P, delta, c5);
      dP = fmaf(dP, delta, P); P = fmaf(P, delta, c4);
      dP = fmaf(dP, delta, P); P = fmaf(P, delta, c3);
      dP = fmaf(dP, delta, P); P = fmaf(P, delta, c2);
      dP = fmaf(dP, delta, P); P = fmaf(P, delta, c1);
      const float F = fmaf(P, delta, -dT), dF = fmaf(dP, delta, P);
      const float stp = __fdividef(F, dF);
      delta -= stp;
      if (fabsf(stp) <= 1e-7f * fabsf(delta) + 1e-12f) break;
    }
    return delta;
  }
  for (int it = 0; it < newton_iters; ++it) {
    float F = -dT, dF = 0.f;
    for (int s = 0; s < nb; ++s) {
      const float I = f[s] * __expf(-gamma[s] * tau);
      const float em = epr_expm1(-gamma[s] * delta);
      F = fmaf(I, em, F);
      dF = fmaf(-gamma[s] * I, 1.f + em, dF);
    }
    const float stp = __fdividef(F, dF);
    delta -= stp;
    if (fabsf(stp) <= 1e-7f * fabsf(delta) + 1e-12f) break;      // converged to fp32 (Newton is quadratic)
  }
  return delta;
}

// The projection of the INITIAL guess (τ = 0, R9): I_s = f_s, so the moments G_k = Σ_s f_s γ_s^k are constants of the plan
// (L.pj_G) and no exponential of τ is needed: Newton on the degree-7 polynomial for |γ_max δ| < 0.25, on the exact sum
// Σ_s f_s expm1(−γ_s δ) = ΔT beyond (thick objects).  Same tiers, start and stopping rule as epr_project_increment.
static __device__ __noinline__ float epr_project_increment_tau0(const EprLines& L, float dT, const float* __restrict__ f,
                                                                const float* __restrict__ gamma, int newton_iters, float i_min) {
  const float G0 = L.pj_G[0], G1 = L.pj_G[1];
  if (G0 + dT < i_min) dT = i_min - G0;
  float delta = -epr_log1p(__fdividef(dT, G0)) * __fdividef(G0, G1);
  if (fabsf(delta) * L.gamma_max < 0.25f) {
    const float c1 = -G1, c2 = 0.5f * L.pj_G[2], c3 = -1.66666667e-1f * L.pj_G[3], c4 = 4.16666667e-2f * L.pj_G[4],
                c5 = -8.33333333e-3f * L.pj_G[5], c6 = 1.38888889e-3f * L.pj_G[6], c7 = -1.98412698e-4f * L.pj_G[7];
    for (int it = 0; it < newton_iters; ++it) {
      float P = c7, dP = 0.f;
      dP = fmaf(dP, delta, P); P = fmaf(P, delta, c6);
      dP = fmaf(dP, delta, P); P = fmaf(P, delta, c5);
      dP = fmaf(dP, delta, P); P = fmaf(P, delta, c4);
      dP = fmaf(dP, delta, P); P = fmaf(P, delta, c3);
      dP = fmaf(dP, delta, P); P = fmaf(P, delta, c2);
      dP = fmaf(dP, delta, P); P = fmaf(P, delta, c1);
      const float F = fmaf(P, delta, -dT), dF = fmaf(dP, delta, P);
      const float stp = __fdividef(F, dF);
      delta -= stp;
      if (fabsf(stp) <= 1e-7f * fabsf(delta) + 1e-12f) break;
    }
    return delta;
  }
  for (int it = 0; it < newton_iters; ++it) {
    float F = -dT, dF = 0.f;
    for (int s = 0; s < L.n_bins; ++s) {
      const float em = epr_expm1(-gamma[s] * delta);
      F = fmaf(f[s], em, F);
      dF = fmaf(-gamma[s] * f[s], 1.f + em, dF);
    }
    const float stp = __fdividef(F, dF);
    delta -= stp;
    if (fabsf(stp) <= 1e-7f * fabsf(delta) + 1e-12f) break;
  }
  return delta;
}
