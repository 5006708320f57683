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

// Projection to the single-thickness manifold, Eq. (7) + PAPER.md:233 (R10), as an increment:
//   given τ and ΔT, find δ with Σ_s I_s(τ) expm1(−γ_s δ) = ΔT, clamped so that Σ_s I_s + ΔT ≥ i_min.
// Newton from the Jensen bound δ0 = −log1p(ΔT/ΣI)/γ̄_I (monotone; exact for one line).
__device__ __forceinline__ float epr_project_increment(float tau, float dT, const EprLines& L, int newton_iters,
                                                       float i_min) {
  const int nb = L.n_bins;
  float Tsum = 0.f, G = 0.f;
  for (int s = 0; s < nb; ++s) {
    const float I = L.f[s] * expf(-L.gamma[s] * tau);
    Tsum += I;
    G = fmaf(L.gamma[s], I, G);
  }
  if (Tsum + dT < i_min) dT = i_min - Tsum;
  float delta = -log1pf(dT / Tsum) * (Tsum / G);
  if (nb > 1) {
    for (int it = 0; it < newton_iters; ++it) {
      float F = -dT, dF = 0.f;
      for (int s = 0; s < nb; ++s) {
        const float I = L.f[s] * expf(-L.gamma[s] * tau);
        const float x = -L.gamma[s] * delta;
        F = fmaf(I, expm1f(x), F);
        dF = fmaf(-L.gamma[s] * I, expf(x), dF);
      }
      delta -= F / dF;
    }
  }
  return delta;
}
