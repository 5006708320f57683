// epr_kernels.cu — stencil, splat, gather and pointwise kernels of the EPR iteration (sm_100a).
#include <cstdlib>
#include <type_traits>
#include "epr_internal.h"
#include "epr_math.cuh"
#include "epr_tma.cuh"

// =====================================================================================================
// a1-L  local O(L²) closure, Eq. (1) PAPER.md:146 (readings R1-R3), in deviation form, fused (one line) with
// a2, the detector residual (a3 is the identity for the local solver).
//   P_s/f_s − 1 = J − a ∇²₅J + (a²/2)[D²x(Î gx²) + D²y(Î gy²) + 2 D⁰xD⁰y(Î gx gy)] − (α²/4) Σ_i D⁻_i(Ī_i D⁺_i Q)
//   with A = exp(−γτ/2) = 1 + Ad,  Î = I/f = A²,  J = Î − 1 = Ad(2+Ad),  g = −γ D⁰τ,  Q = ∇²₅A / A.
//   One line: out = e = (d − 1) − (P − 1);  several lines: out[b][s] = P_s − f_s for k_residual.
// The kernel is bound by fp32 issue (≈ 90 instructions per pixel and line), not by HBM: see DESIGN.md.
// =====================================================================================================
// -----------------------------------------------------------------------------------------------------
// k_local_march — the closure (fused with the residual for one spectral line, the hot configuration), register marching.
// A warp owns a band of 128 columns (lane l: 4 consecutive pixels; lanes 0 and 31 are halo providers, lanes
// 1..30 write 120 output columns) and marches down LM_MR output rows.  Every row of τ and d is fetched ONCE
// (cp.async ring, see below); all x-neighbours come from warp shuffles and all y-neighbours from rolling
// registers; no barriers.  The arithmetic is organised so that every neighbour difference is formed once:
//   * each stage-2 row m SCATTERS its contributions into three rolling accumulator rows (m−1, m, m+1) instead of
//     every output row gathering from three stored rows of Î gx², Î gy², Î gx gy and Q;
//   * y-differences (J, A, Q, fluxes) are shared between the two rows they separate, x-differences between the
//     two pixels they separate;
//   * constant factors are folded: S'_ij = c2 Î ∂_iτ ∂_jτ with c2 = (a²/2)(γ/2)², H = ½Î (the flux mean).
//   v[o] = J[o] − a ∇²₅J + [D²x S'xx + D²y S'yy + 2 D⁰xD⁰y S'xy] − (α²/4) Σ_i D⁻_i(Ī_i D⁺_i Q),  out = (d − 1) − v.
// Rolling rows (suffix a = m−1, b = m, c = m+1 = newest row n); output row o = m − 1 is final after stage 2 of m.
// ≈ 62 fp32 instructions per pixel: bound by fp32 issue, not by HBM (12 B/px) — DESIGN.md §7.
// -----------------------------------------------------------------------------------------------------
// LM_MR output rows per warp and LM_WPC warps (bands) per CTA are template parameters: (128, 1) when the launch has
// enough bands x row blocks x projections to fill the GPU (row halo 4/128, 12.4 us per 2048² plane), (32, 4) otherwise.
#define LM_BW 120                    // output columns per warp
#ifndef LM_D
#define LM_D 4                       // cp.async ring depth: rows are requested LM_D − 1 steps ahead
#endif
#ifndef LM_UNROLL
#define LM_UNROLL 4
#endif
#define EPR_PRAGMA(x) _Pragma(#x)
#define EPR_UNROLL(n) EPR_PRAGMA(unroll n)

struct F4 { float v[4]; };
__device__ __forceinline__ float shfl_l(float x) { return __shfl_up_sync(0xffffffffu, x, 1); }     // from lane-1
__device__ __forceinline__ float shfl_r(float x) { return __shfl_down_sync(0xffffffffu, x, 1); }   // from lane+1

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((unsigned)__cvta_generic_to_shared(smem)), "l"(gmem) : "memory");
}
// shared-memory access by 32-bit shared address (volatile: program order among themselves is kept, so a kernel can
// place the loads of the next step before the atomics of the current one)
__device__ __forceinline__ float lds_f32(unsigned a) {
  float v;
  asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(a));
  return v;
}
__device__ __forceinline__ void red_shared_u32(unsigned a, unsigned v) {
  asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(a), "r"(v) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

struct W6 { float w[6]; };
__device__ __forceinline__ W6 window(const F4& v) {
  W6 r;
  r.w[0] = shfl_l(v.v[3]);
  r.w[1] = v.v[0]; r.w[2] = v.v[1]; r.w[3] = v.v[2]; r.w[4] = v.v[3];
  r.w[5] = shfl_r(v.v[0]);
  return r;
}

// PRED (several lines): blockIdx.z = projection · n_bins + line; out[b][s] = P_s − f_s = f_s v for k_residual, no d.
template <int LM_MR, int LM_WPC, bool PRED>
__global__ void __launch_bounds__(32 * LM_WPC) k_local_march(EprLines L, int nx, int ny, int order, int wkb1,
                                                     const float* __restrict__ tau, const float* __restrict__ d,
                                                     float* __restrict__ out) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int band = blockIdx.x * LM_WPC + warp;
  const int xs = band * LM_BW - 4 + 4 * lane;
  if (band * LM_BW >= nx) return;
  const int y0 = blockIdx.y * LM_MR;
  const unsigned plane = (unsigned)nx * (unsigned)ny;
  const int ls = PRED ? (int)(blockIdx.z % L.n_bins) : 0;                  // spectral line
  const size_t bz = PRED ? blockIdx.z / L.n_bins : blockIdx.z;             // projection
  const float* tb = tau + bz * plane;
  const float* db = PRED ? nullptr : d + bz * plane;
  float* ob = out + (size_t)blockIdx.z * plane;
  const int xw = wrapm(xs, nx);
  const bool writer = lane >= 1 && lane <= 30 && xs < nx;
  const float cg = -0.5f * L.gamma[ls], a = L.a[ls], q4 = L.q4[ls], fs = L.f[ls];
  const float c2 = L.a2h[ls] * cg * cg;
  const bool o2 = order == 2, wk = o2 && wkb1;

  F4 t_a, t_b, t_c, A_b, dA_lo, J_a, J_b, H_a, Q_a, ACC_a, ACC_b;
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    t_a.v[k] = t_b.v[k] = t_c.v[k] = A_b.v[k] = dA_lo.v[k] = J_a.v[k] = J_b.v[k] = 0.f;
    H_a.v[k] = 0.5f; Q_a.v[k] = ACC_a.v[k] = ACC_b.v[k] = 0.f;
  }
  __shared__ float4 ring_t[LM_D][32 * LM_WPC], ring_d[LM_D][32 * LM_WPC];
  const unsigned tid = threadIdx.x;
  // row pointers advance by one row per request (τ rows wrap periodically, d / out rows never leave the plane)
  int yr = wrapm(y0 - 2, ny);
  const float* tp = tb + (unsigned)yr * nx + xw;
  const float* dp = PRED ? nullptr : db + (unsigned)y0 * nx + xs;
  float* op = ob + (unsigned)y0 * nx + xs;
#pragma unroll
  for (int i = 0; i < LM_D - 1; ++i) {
    cp_async16(&ring_t[i][tid], tp);
    tp += nx;
    if (++yr == ny) { yr = 0; tp -= plane; }
    cp_async_commit();                             // (no d row is due before step 4 > LM_D − 2)
  }
  static_assert(LM_D <= 5, "d rows of the prologue are not requested");
  EPR_UNROLL(LM_UNROLL)
  for (int step = 0; step < LM_MR + 4; ++step) {
    const int n = y0 - 2 + step;
    {
      const int sl = (step + LM_D - 1) % LM_D, ahead = step + LM_D - 1;
      if (ahead < LM_MR + 4) {
        cp_async16(&ring_t[sl][tid], tp);
        tp += nx;
        if (++yr == ny) { yr = 0; tp -= plane; }
        if (!PRED && ahead >= 4) {                   // d row of output row y0 − 4 + ahead
          if (y0 - 4 + ahead < ny && writer) cp_async16(&ring_d[sl][tid], dp);
          dp += nx;
        }
      }
      cp_async_commit();
      cp_async_wait<LM_D - 1>();
    }
    const float4 tv = ring_t[step % LM_D][tid];
    float4 dd = make_float4(0.f, 0.f, 0.f, 0.f);
    if (!PRED) dd = ring_d[step % LM_D][tid];
    // ---- rotate ----
    t_a = t_b; t_b = t_c;
    t_c.v[0] = tv.x; t_c.v[1] = tv.y; t_c.v[2] = tv.z; t_c.v[3] = tv.w;
    // ---- stage 1 on the new row n: A, J, and the y-difference of A towards row m ----
    F4 A_c, J_c, dA_hi;
    {
      const float x0 = cg * t_c.v[0], x1 = cg * t_c.v[1], x2 = cg * t_c.v[2], x3 = cg * t_c.v[3];
      const float mx = fmaxf(fmaxf(fabsf(x0), fabsf(x1)), fmaxf(fabsf(x2), fabsf(x3)));
      if (!__any_sync(0xffffffffu, mx >= 0.09f)) {       // weak absorption (most rows): a shorter series is exact in fp32
        A_c.v[0] = epr_expm1_tiny(x0); A_c.v[1] = epr_expm1_tiny(x1);
        A_c.v[2] = epr_expm1_tiny(x2); A_c.v[3] = epr_expm1_tiny(x3);
      } else if (__any_sync(0xffffffffu, mx >= 0.35f)) {  // rare (thick object): both branches of epr_expm1
        A_c.v[0] = epr_expm1(x0); A_c.v[1] = epr_expm1(x1); A_c.v[2] = epr_expm1(x2); A_c.v[3] = epr_expm1(x3);
      } else {
        A_c.v[0] = epr_expm1_small(x0); A_c.v[1] = epr_expm1_small(x1);
        A_c.v[2] = epr_expm1_small(x2); A_c.v[3] = epr_expm1_small(x3);
      }
    }
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      J_c.v[k] = A_c.v[k] * (2.f + A_c.v[k]);
      dA_hi.v[k] = A_c.v[k] - A_b.v[k];
    }
    // ---- stage 2 on row m = n − 1: scatter into ACC_a (row m−1, final after this), ACC_b (row m), ACC_c (row m+1) ----
    F4 ACC_c, H_b, Q_b;
    {
      const W6 Jw = window(J_b);
      float dJ[5];
#pragma unroll
      for (int i = 0; i < 5; ++i) dJ[i] = Jw.w[i + 1] - Jw.w[i];
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const float g = J_b.v[k] - J_a.v[k];                       // y-difference of J across m−½
        ACC_b.v[k] = fmaf(-a, dJ[k + 1] - dJ[k], fmaf(a, g, ACC_b.v[k]));
        ACC_a.v[k] = fmaf(-a, g, ACC_a.v[k]);
        ACC_c.v[k] = 0.f;
        H_b.v[k] = fmaf(0.5f, J_b.v[k], 0.5f);
        Q_b.v[k] = 0.f;
      }
      if (o2) {
        const W6 tw = window(t_b);
        F4 Sxx, Sxy;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          const float dx = tw.w[k + 2] - tw.w[k], dy = t_c.v[k] - t_a.v[k];
          const float Ic = fmaf(c2, J_b.v[k], c2), tt = Ic * dx, Syy = Ic * dy * dy;
          Sxx.v[k] = tt * dx; Sxy.v[k] = tt * dy;
          ACC_c.v[k] = Syy;
          ACC_b.v[k] = fmaf(-2.f, Syy, ACC_b.v[k]);
          ACC_a.v[k] += Syy;
        }
        const W6 xw6 = window(Sxx), yw6 = window(Sxy);
        float dS[5];
#pragma unroll
        for (int i = 0; i < 5; ++i) dS[i] = xw6.w[i + 1] - xw6.w[i];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          const float cx = yw6.w[k + 2] - yw6.w[k];
          ACC_b.v[k] += dS[k + 1] - dS[k];
          ACC_c.v[k] = fmaf(-0.5f, cx, ACC_c.v[k]);
          ACC_a.v[k] = fmaf(0.5f, cx, ACC_a.v[k]);
        }
        if (wk) {
          const W6 Aw = window(A_b);
          float dAx[5];
#pragma unroll
          for (int i = 0; i < 5; ++i) dAx[i] = Aw.w[i + 1] - Aw.w[i];
#pragma unroll
          for (int k = 0; k < 4; ++k)
            Q_b.v[k] = __fdividef((dAx[k + 1] - dAx[k]) + (dA_hi.v[k] - dA_lo.v[k]), 1.f + A_b.v[k]);
          const W6 Qw = window(Q_b);
          float Hw[6], Fx[5];
#pragma unroll
          for (int i = 0; i < 6; ++i) Hw[i] = fmaf(0.5f, Jw.w[i], 0.5f);
#pragma unroll
          for (int i = 0; i < 5; ++i) Fx[i] = (Hw[i + 1] + Hw[i]) * (Qw.w[i + 1] - Qw.w[i]);
#pragma unroll
          for (int k = 0; k < 4; ++k) {
            const float Fy = (H_b.v[k] + H_a.v[k]) * (Q_b.v[k] - Q_a.v[k]);    // flux across m−½
            ACC_b.v[k] = fmaf(-q4, Fx[k + 1] - Fx[k], fmaf(q4, Fy, ACC_b.v[k]));
            ACC_a.v[k] = fmaf(-q4, Fy, ACC_a.v[k]);
          }
        }
      }
    }
    // ---- output row o = n − 2 = m − 1 ----
    const int o = n - 2;
    if (step >= 4 && o < ny && writer) {
      if (PRED)
        *reinterpret_cast<float4*>(op + (unsigned)(step - 4) * nx) =
            make_float4(fs * (J_a.v[0] + ACC_a.v[0]), fs * (J_a.v[1] + ACC_a.v[1]), fs * (J_a.v[2] + ACC_a.v[2]),
                        fs * (J_a.v[3] + ACC_a.v[3]));
      else
        *reinterpret_cast<float4*>(op + (unsigned)(step - 4) * nx) =
            make_float4((dd.x - 1.f) - (J_a.v[0] + ACC_a.v[0]), (dd.y - 1.f) - (J_a.v[1] + ACC_a.v[1]),
                        (dd.z - 1.f) - (J_a.v[2] + ACC_a.v[2]), (dd.w - 1.f) - (J_a.v[3] + ACC_a.v[3]));
    }
    // ---- rotate the row windows ----
    A_b = A_c; dA_lo = dA_hi; J_a = J_b; J_b = J_c; H_a = H_b; Q_a = Q_b; ACC_a = ACC_b; ACC_b = ACC_c;
  }
}

cudaError_t epr_launch_forward_local(const epr_plan_s* p, int batch, const float* tau, const float* d_fuse, float* out,
                                     cudaStream_t st) {
  // one line fused with the residual (d_fuse), or line by line into pred (several lines: blockIdx.z = projection · n_bins + line)
  const int bands = (p->nx + LM_BW - 1) / LM_BW;
  const int nz = d_fuse ? batch : batch * p->n_bins;
  const int sms = p->sms;
  // the tallest row block that still gives every SM about a dozen warps (all CTAs resident at once: no tail wave)
  const long long need = 12ll * sms;
#define EPR_MARCH(MR, WPC, GX, GY, NT)                                                                               \
  do {                                                                                                              \
    dim3 grid(GX, GY, nz);                                                                                          \
    if (d_fuse) k_local_march<MR, WPC, false><<<grid, NT, 0, st>>>(p->lines, p->nx, p->ny, p->opt.order, p->opt.wkb1, tau, d_fuse, out); \
    else k_local_march<MR, WPC, true><<<grid, NT, 0, st>>>(p->lines, p->nx, p->ny, p->opt.order, p->opt.wkb1, tau, nullptr, out);       \
  } while (0)
  if ((long long)bands * ((p->ny + 127) / 128) * nz >= need) EPR_MARCH(128, 1, bands, (p->ny + 127) / 128, 32);
  else if ((long long)bands * ((p->ny + 63) / 64) * nz >= need) EPR_MARCH(64, 2, (bands + 1) / 2, (p->ny + 63) / 64, 64);
  else EPR_MARCH(32, 4, (bands + 3) / 4, (p->ny + 31) / 32, 128);
#undef EPR_MARCH
  return cudaGetLastError();
}

// =====================================================================================================
// Helper of a1-N / a3: gmax[b][y/16][x/16] = max over the 16x16-pixel block of max(|τ[x+1] − τ[x−1]|, |τ[y+1] − τ[y−1]|)
// (periodic; nx, ny are multiples of 16).  With u_s = c_s D⁰τ (Eq. (2)) it bounds the ray shifts of a
// block, which tells the splat how wide a ring of foreign sources can reach a detector tile and the gather how wide a
// halo of the residual a tile needs — before either loads anything.  One pass over τ (4 B/px).
// A warp owns 128 columns x 16 rows = 8 blocks and walks down the rows with the column's three current rows in registers
// (18 row loads of 512 B for 16 rows; x-neighbours by shuffles, the two strip edges by one scalar load each);
// CTA = 8 warps stacked in y.
// =====================================================================================================
__global__ void __launch_bounds__(256) k_grad_blockmax(int nx, int ny, const float* __restrict__ tau, float* __restrict__ gmax) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int x = blockIdx.x * 128 + 4 * lane, by = blockIdx.y * 8 + warp;       // block row
  if (by * 16 >= ny) return;
  const bool xin = x < nx;
  const int xs = xin ? x : 0;
  const float* tb = tau + (size_t)blockIdx.z * nx * ny;
  const int xm = xs == 0 ? nx - 1 : xs - 1, xp = xs + 4 >= nx ? 0 : xs + 4;
  const int y0 = by * 16;
  auto row4 = [&](int y) { return __ldg(reinterpret_cast<const float4*>(tb + (size_t)(y < 0 ? y + ny : (y >= ny ? y - ny : y)) * nx + xs)); };
  float4 n = row4(y0 - 1), c = row4(y0);
  float m = 0.f;
#pragma unroll 8
  for (int r = 0; r < 16; ++r) {
    const float4 s4 = row4(y0 + r + 1);
    float l = __shfl_up_sync(0xffffffffu, c.w, 1), rr = __shfl_down_sync(0xffffffffu, c.x, 1);
    const float* row = tb + (size_t)(y0 + r) * nx;
    if (lane == 0 || x == 0) l = __ldg(row + xm);
    if (lane == 31 || x + 4 >= nx) rr = __ldg(row + xp);
    m = fmaxf(m, fmaxf(fmaxf(fabsf(c.y - l), fabsf(c.z - c.x)), fmaxf(fabsf(c.w - c.y), fabsf(rr - c.z))));
    m = fmaxf(m, fmaxf(fmaxf(fabsf(s4.x - n.x), fabsf(s4.y - n.y)), fmaxf(fabsf(s4.z - n.z), fabsf(s4.w - n.w))));
    n = c; c = s4;
  }
  if (!xin) m = 0.f;
  m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, 1));
  m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, 2));
  const int nbx = nx >> 4;
  if ((lane & 3) == 0 && xin) gmax[((size_t)blockIdx.z * (ny >> 4) + by) * nbx + (x >> 4)] = m;
}

cudaError_t epr_launch_grad_blockmax(const epr_plan_s* p, int batch, const float* tau, cudaStream_t st) {
  dim3 grid((p->nx + 127) / 128, (p->ny / 16 + 7) / 8, batch);
  k_grad_blockmax<<<grid, 256, 0, st>>>(p->nx, p->ny, tau, p->gmax);
  return cudaGetLastError();
}

// =====================================================================================================
// a1-N  ray map (Eq. (2), clamp R6) + mass-conserving bilinear splat,
//       DETECTOR-TILE-OWNED: one CTA owns ST_W x ST_H detector pixels of one projection and walks over every
//       source pixel that can reach them (the tile grown by H = ceil(S) + 1), so the 4-way scatter is resolved
//       entirely by NATIVE u32 shared-memory atomics on the CTA's own accumulator tile: no global atomics, no
//       zero-initialised global plane, no second pass over the prediction.
//   Accumulation is u32 fixed point (unit 2^-26): independent of the order of the atomics (bit-reproducible) and
//   exactly mass conserving — the 4th corner receives the source mass minus the other three corners, in integers.
//   Source mass: tot = rint(f_s 2^26) + rint(f_s 2^26 J), J = expm1(−γ_s τ) (deviation form: the fp32 rounding
//   acts on the small J only), or rint(I 2^26) for an arbitrary plane (epr_transport).  Corner masses:
//   (tot · rint(w 2^24) + 2^23) >> 24 in 64-bit integers.
//   Sources: I_s from τ (I_bins == NULL) or a given plane; u from τ (map_in == NULL; written to map_out by the
//   tile that owns the source pixel) or from a stored map.
//   Output (out_mode): 0  out[b][s] = P_s − f_s (float);  1  out[b][s] = P_s;  3  out[b][s] = e_s = w_s e (the residual
//   split a2 of several lines, fused: see the end of the kernel);  2 (one line)  out[b] = e =
//   (d − 1) − (P − f): the detector residual a2 fused into the flush.
// =====================================================================================================
#define ST_W 128
#define ST_H 64                       // tile height (template parameter TH of the kernel: 64, or 32 for large S)
#define ST_AP (ST_W + 8)              // accumulator pitch: 4 columns of (aligned) border left, 1 used right
#define ST_AROWS (ST_H + 2)
#define ST_LCAP 2048                  // capacity of the ring-candidate list (several lines); beyond it the ring is walked           // one border row above and below: out-of-tile corners land there, unflushed

// FROM_TAU: sources and ray map from the τ tile staged in shared memory (the loop's configuration);
// otherwise (epr_transport) both are read from global planes.
// ST_NT threads per CTA: 512 when two CTAs fit an SM, 1024 when the halo (large S) leaves room for one only
// COLS: x-dependent effective spectrum (reading R17): the per-line scalars of a SOURCE come from its own column's tables C
// (mass f_s(x), γ_s(x), shift coefficient a_s(x)γ_s(x)), the baseline / split fractions of a DETECTOR pixel from its column;
// L then only carries bounds (a[s]·gamma[s] = max over columns of a_s(x)γ_s(x)) for the ring width and the clamp test.
template <bool FROM_TAU, bool MAP_OUT, int ST_NT, int TH, bool COLS = false>
__global__ void __launch_bounds__(ST_NT) k_splat_tile(EprLines L, EprColumns C, int nx, int ny, float S, int H,
                                                    const float* __restrict__ tau, const float* __restrict__ I_bins,
                                                    const float2* __restrict__ map_in, float2* __restrict__ map_out,
                                                    float* __restrict__ out, int out_mode, const float* __restrict__ d,
                                                    const float* __restrict__ gmax, int use_list,
                                                    unsigned* __restrict__ flags) {
  extern __shared__ __align__(16) unsigned char st_raw[];
  unsigned* s_acc = reinterpret_cast<unsigned*>(st_raw);                              // [(TH + 2)][ST_AP]
  float* s_tau = reinterpret_cast<float*>(st_raw + ST_AP * (TH + 2) * sizeof(unsigned));   // [TH + 2 H + 2][TP]
  const int b = blockIdx.z, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  constexpr int NW = ST_NT / 32;
  const int x0 = blockIdx.x * ST_W, y0 = blockIdx.y * TH;
  const int Ha = (H + 1 + 3) & ~3;                     // τ tile halo in x, rounded up to whole 16-byte chunks
  const int TP = ST_W + 2 * Ha;                        // τ tile pitch; tile column of tile-relative x is x + Ha
  const unsigned plane = (unsigned)nx * (unsigned)ny;

  // Largest |D⁰τ| (times 2) among the sources in the ring of width H around the tile (s_maxd) and in the tile itself
  // (s_maxd_in), from the 16x16-block maxima of k_grad_blockmax: a source at distance D from the tile reaches it only
  // if ⌊|u|⌋ + 1 ≥ D, so the ring that has to be walked (and loaded) is He ≤ H wide.
  __shared__ unsigned s_maxd, s_maxd_in, s_cnt;
  // several lines: the few ring sources that can reach the tile at all, found once (see below), 16 bits each
  unsigned short* s_list = reinterpret_cast<unsigned short*>(st_raw + ST_AP * (TH + 2) * sizeof(unsigned) +
                                                             (size_t)TP * (TH + 2 * H + 2) * sizeof(float));
  if (FROM_TAU) {
    if (tid == 0) { s_maxd = 0u; s_maxd_in = 0u; }
    __syncthreads();
    const int nbx = nx >> 4, nby = ny >> 4;
    const int nsx = (ST_W + 2 * H + 15) / 16 + 1, nsy = (TH + 2 * H + 15) / 16 + 1;
    const float* gm = gmax + (size_t)b * nbx * nby;
    for (int i = tid; i < nsx * nsy; i += ST_NT) {
      const int j = i / nsx, ii = i - j * nsx;
      const int px = min(-H + 16 * ii, ST_W - 1 + H), py = min(-H + 16 * j, TH - 1 + H);   // tile-relative sample
      const bool inside = (unsigned)px < ST_W && (unsigned)py < TH;
      const float v = __ldg(&gm[(wrapm(y0 + py, ny) >> 4) * nbx + (wrapm(x0 + px, nx) >> 4)]);
      atomicMax(inside ? &s_maxd_in : &s_maxd, __float_as_uint(v));
    }
    __syncthreads();
    float csmax = 0.f;
    for (int s = 0; s < L.n_bins; ++s) csmax = fmaxf(csmax, 0.5f * L.a[s] * L.gamma[s]);
    const int Hl = min(H, (int)fminf(csmax * __uint_as_float(s_maxd), S) + 1);      // widest ring of any line
    // τ tile rows y0 − Hl − 1 … y0 + TH + Hl (tile rows H − Hl … H + TH + 1 + Hl), columns x0 − Ha …:
    // 16-byte cp.async chunks (nx % 4 == 0: a chunk never straddles the wrap), spread evenly over the threads
    const float* tb = tau + (size_t)b * plane;
    const int cpr = TP / 4, nrows = TH + 2 + 2 * Hl;
    const float inv_cpr = 1.f / (float)cpr;
    const bool big = nx >= 2 * (ST_W + 2 * Ha) && ny >= 2 * (TH + 2 * H + 2);
    for (int i = tid; i < nrows * cpr; i += ST_NT) {
      const int r = (int)(((float)i + 0.5f) * inv_cpr), cx = i - r * cpr;
      const int ly = H - Hl + r;
      int gy = y0 - H - 1 + ly, gx = x0 - Ha + 4 * cx;
      if (big) { gy = wrap1(gy, ny); gx = wrap1(gx, nx); } else { gy = wrapm(gy, ny); gx = wrapm(gx, nx); }
      cp_async16(s_tau + ly * TP + 4 * cx, tb + (unsigned)gy * nx + gx);
    }
    cp_async_commit();
    if (use_list) {
      // Ring candidates of ALL lines in one walk.  u_s = c_s D⁰τ with c_s < 0 for every line, so the shift of any line
      // is the strongest line's shift scaled by t ∈ (0, 1]: ⌊u_s⌋ lies between min(⌊u_max⌋, 0) and max(⌊u_max⌋, −1) on
      // each axis (fp32 products and the clamp are monotone in |c_s|).  A source none of whose possible targets touches
      // the tile is dropped here once instead of being rejected by every line; the per-line walk below repeats the
      // exact test on what is left (a few per cent of the tile's own sources).
      if (tid == 0) s_cnt = 0u;
      cp_async_wait<0>();
      __syncthreads();
      const int RWl = ST_W + 2 * Hl, n_tbl = 2 * Hl * RWl, n_wl = n_tbl + 2 * TH * Hl;
      const float inv_rwl = 1.f / (float)RWl, inv_2hl = 1.f / (float)(2 * Hl);
      for (int i = tid; i < n_wl; i += ST_NT) {
        int sx, sy;
        if (i < n_tbl) {
          sy = (int)(((float)i + 0.5f) * inv_rwl); sx = i - sy * RWl;
          if (sy >= Hl) sy += TH;
        } else {
          const int j = i - n_tbl;
          sy = (int)(((float)j + 0.5f) * inv_2hl); sx = j - sy * 2 * Hl;
          sy += Hl;
          if (sx >= Hl) sx += ST_W;
        }
        const int tx0 = sx - Hl, ty0 = sy - Hl;
        const float* tp = s_tau + (ty0 + H + 1) * TP + (tx0 + Ha);
        const float ux = fminf(fmaxf(-csmax * (tp[1] - tp[-1]), -S), S);
        const float uy = fminf(fmaxf(-csmax * (tp[TP] - tp[-TP]), -S), S);
        const int fx = __float2int_rd(ux), fy = __float2int_rd(uy);
        if (tx0 + max(fx, -1) >= -1 && tx0 + min(fx, 0) <= ST_W - 1 && ty0 + max(fy, -1) >= -1 && ty0 + min(fy, 0) <= TH - 1) {
          const unsigned k = atomicAdd(&s_cnt, 1u);
          if (k < ST_LCAP) s_list[k] = (unsigned short)(((ty0 + 64) << 8) | (tx0 + 64));
        }
      }
    }
  }
  // one line with the residual fused (out_mode 2): the d values of this thread's flush groups are requested now, so that
  // the flush does not wait on them (the load used to be 21 % of the kernel's stall samples)
  // Flush geometry: a thread owns the same NFL groups of 4 pixels for every line — column group tid % 32, rows
  // fty + FRS·k — so the shared-memory offsets are immediates and the global offset advances by FRS·nx per group
  // (the generic index arithmetic i = tid + k·NT → (ty, tx) cost 21 of the 66 instructions of a group).
  constexpr int NFL = ST_W * TH / 4 / ST_NT;         // flush groups (4 pixels) per thread
  constexpr int FRS = ST_NT / (ST_W / 4);            // rows between a thread's consecutive groups
  const int ftx = 4 * (tid % (ST_W / 4)), fty = tid / (ST_W / 4);
  const bool fxin = x0 + ftx < nx;
  const int frows = ny - y0 - fty;                   // group k is inside the image iff fxin && FRS·k < frows
  const unsigned fg0 = (unsigned)(y0 + fty) * nx + (x0 + ftx), fgs = (unsigned)FRS * nx;
  unsigned* facc = s_acc + (fty + 1) * ST_AP + 4 + ftx;
  float4 dpre[NFL];
  if (out_mode == 2) {
    const float* dg = d + (size_t)b * plane + fg0;
#pragma unroll
    for (int k = 0; k < NFL; ++k) {
      dpre[k] = make_float4(0.f, 0.f, 0.f, 0.f);
      if (fxin && FRS * k < frows) dpre[k] = __ldg(reinterpret_cast<const float4*>(dg + k * fgs));
    }
  }
  for (int s = 0; s < L.n_bins; ++s) {
    const size_t pl = ((size_t)b * L.n_bins + s) * plane;
    // The accumulator tile is zeroed once; afterwards the flush of a line zeroes what it reads (and the unflushed
    // border), so a line costs two barriers — after the scatter, after the flush — and no separate clearing pass.
    if (s == 0) {
      __syncthreads();                                 // (the candidate list above reads the τ tile; s_acc is untouched so far)
      for (int i = tid; i < ST_AP * (TH + 2) / 4; i += ST_NT) reinterpret_cast<uint4*>(s_acc)[i] = make_uint4(0u, 0u, 0u, 0u);
      if (FROM_TAU) cp_async_wait<0>();
    }
    __syncthreads();                                   // accumulators clear (first line) / previous line flushed and cleared
    const float cs = -0.5f * L.a[s] * L.gamma[s], gam = L.gamma[s], fixFf = (float)L.fixF[s];
    const int Fi = (int)L.fixFi[s];
    // a source at distance D from the tile reaches it only if ⌊|u|⌋ + 1 ≥ D
    int He = H;
    if (FROM_TAU) He = min(H, (int)fminf(fabsf(cs) * __uint_as_float(s_maxd), S) + 1);
    const int RWe = ST_W + 2 * He, RHe = TH + 2 * He;
    // Every periodic image of a source pixel inside the region is a distinct candidate: its targets differ by whole
    // periods, and exactly one image puts a given corner on a given detector pixel — that IS the periodic wrap (R7).
    if (FROM_TAU) {
      // (1) The tile's own ST_W x TH sources (nearly all of them hit): a warp owns a 32-column strip and marches
      // down its rows with the column's τ values in registers (3 shared loads per source instead of 5, no index
      // arithmetic: one address per array advances by a row); the loads of row r + 1 are issued before the atomics
      // of row r.  32-bit shared addresses are formed once (the compiler otherwise rebuilds them per source).
      // The clamp of u is skipped when |c_s| · max|D⁰τ| over the tile cannot exceed S.
      constexpr int RG = NW / 4, ROWS = TH / RG;
      const int x = (warp & 3) * 32 + lane, yb = (warp >> 2) * ROWS;
      float csx = cs, gamx = gam, fixFfx = fixFf;      // scalars of THIS thread's source column
      int Fix = Fi;
      if (COLS) {
        const size_t ci = (size_t)s * nx + wrapm(x0 + x, nx);
        gamx = __ldg(&C.gamma[ci]);
        csx = -0.5f * __ldg(&C.a[ci]) * gamx;
        fixFfx = __ldg(&C.f[ci]) * 67108864.f;
        Fix = (int)__ldg(&C.fixFi[ci]);
      }
      const unsigned TP4 = 4u * TP;
      const unsigned rb0 = (unsigned)__cvta_generic_to_shared(s_tau) + 4u * (unsigned)((yb + H + 1) * TP + x + Ha);
      const unsigned ab0 = (unsigned)__cvta_generic_to_shared(s_acc) + 4u * (unsigned)((yb + 1) * ST_AP + x + 4);
      auto interior = [&](auto clamp_tag) {
        constexpr bool CLAMP = decltype(clamp_tag)::value;
        unsigned rb = rb0, ab = ab0;
        float tn = lds_f32(rb - TP4), tc = lds_f32(rb), ts = lds_f32(rb + TP4), tl = lds_f32(rb - 4), tr = lds_f32(rb + 4);
        float2* mo = MAP_OUT ? map_out + pl + (size_t)(y0 + yb) * nx + (x0 + x) : nullptr;
#pragma unroll 8
        for (int r = 0; r < ROWS; ++r) {
          rb += TP4;                                   // one row beyond the strip at the last r: still inside the τ tile
          const float ts2 = lds_f32(rb + TP4), tl2 = lds_f32(rb - 4), tr2 = lds_f32(rb + 4);
          const float gx = tr - tl, gy = ts - tn;
          float ux = csx * gx, uy = csx * gy;
          if (CLAMP) { ux = fminf(fmaxf(ux, -S), S); uy = fminf(fmaxf(uy, -S), S); }
          if (MAP_OUT) {
            if (x0 + x < nx && y0 + yb + r < ny) *mo = make_float2(ux, uy);
            mo += nx;
          }
          const int fx = __float2int_rd(ux), fy = __float2int_rd(uy);
          const float dx = ux - (float)fx, dy = uy - (float)fy;
          const float xe = -gamx * tc;
          float J = epr_expm1_small(xe);               // MUFU branch only where a lane of the warp needs it
          if (__any_sync(0xffffffffu, fabsf(xe) >= 0.35f)) J = fabsf(xe) < 0.35f ? J : epr_exp_fast(xe) - 1.f;
          const int tot = Fix + __float2int_rn(fixFfx * J);
          const float totf = (float)tot, te = totf * (1.f - dy), td = totf * dy, ex = 1.f - dx;
          const int c00 = __float2int_rn(te * ex), c10 = __float2int_rn(te * dx), c01 = __float2int_rn(td * ex);
          const int c11 = tot - c00 - c10 - c01;
          // ax = x + fx ∈ [−1, ST_W − 1], ay ∈ [−1, TH − 1]: all four corners are inside the bordered accumulator
          if ((unsigned)(x + fx + 1) <= ST_W && (unsigned)(yb + r + fy + 1) <= TH) {
            const unsigned a0 = ab + 4u * (unsigned)(fy * ST_AP + fx);
            red_shared_u32(a0, (unsigned)c00);
            red_shared_u32(a0 + 4, (unsigned)c10);
            red_shared_u32(a0 + 4 * ST_AP, (unsigned)c01);
            red_shared_u32(a0 + 4 * ST_AP + 4, (unsigned)c11);
          }
          tn = tc; tc = ts; ts = ts2; tl = tl2; tr = tr2;
          ab += 4u * ST_AP;
        }
      };
      if (fabsf(cs) * __uint_as_float(s_maxd_in) <= S) interior(std::false_type{});
      else interior(std::true_type{});
    }
    // (2) FROM_TAU: the ring of width He around the tile (two bands of He rows, two of He columns), few of whose
    // sources reach the tile; otherwise (epr_transport): the whole region, row-major.
    const bool listed = FROM_TAU && use_list && s_cnt <= ST_LCAP;      // s_cnt is final: barriers above (uniform)
    const int n_tb = 2 * He * RWe, n_walk = listed ? (int)s_cnt : FROM_TAU ? n_tb + 2 * TH * He : RWe * RHe;
    const float inv_rw = 1.f / (float)RWe, inv_2he = 1.f / (float)(2 * He);
    for (int i = tid; i < n_walk; i += ST_NT) {
      int sx, sy;                                      // quotients by float reciprocal: exact for these ranges
      if (listed) {
        const unsigned e = s_list[i];
        sx = (int)(e & 255u) - 64 + He; sy = (int)(e >> 8) - 64 + He;
      } else if (!FROM_TAU || i < n_tb) {
        sy = (int)(((float)i + 0.5f) * inv_rw); sx = i - sy * RWe;
        if (FROM_TAU && sy >= He) sy += TH;
      } else {
        const int j = i - n_tb;
        sy = (int)(((float)j + 0.5f) * inv_2he); sx = j - sy * 2 * He;
        sy += He;
        if (sx >= He) sx += ST_W;
      }
      const int tx0 = sx - He, ty0 = sy - He;          // source pixel relative to the tile
      float ux, uy, tc = 0.f;
      unsigned gidx = 0;
      float csx = cs, gamx = gam, fixFfx = fixFf;      // scalars of the source's column
      int Fix = Fi;
      if (COLS && FROM_TAU) {
        const size_t ci = (size_t)s * nx + wrapm(x0 + tx0, nx);
        gamx = __ldg(&C.gamma[ci]);
        csx = -0.5f * __ldg(&C.a[ci]) * gamx;
        fixFfx = __ldg(&C.f[ci]) * 67108864.f;
        Fix = (int)__ldg(&C.fixFi[ci]);
      }
      if (FROM_TAU) {
        // u = a D⁰ ln I_s = −a γ D⁰τ, clamped to ±S
        const float* tp = s_tau + (ty0 + H + 1) * TP + (tx0 + Ha);
        tc = tp[0];
        ux = fminf(fmaxf(csx * (tp[1] - tp[-1]), -S), S);
        uy = fminf(fmaxf(csx * (tp[TP] - tp[-TP]), -S), S);
        if (MAP_OUT && (unsigned)tx0 < ST_W && (unsigned)ty0 < TH && x0 + tx0 < nx && y0 + ty0 < ny)
          map_out[pl + (unsigned)(y0 + ty0) * nx + (x0 + tx0)] = make_float2(ux, uy);
      } else {
        gidx = (unsigned)wrapm(y0 + ty0, ny) * nx + wrapm(x0 + tx0, nx);
        const float2 m = __ldg(&map_in[pl + gidx]);
        ux = m.x; uy = m.y;
      }
      const int fx = __float2int_rd(ux), fy = __float2int_rd(uy);
      const int ax = tx0 + fx, ay = ty0 + fy;          // top-left target, tile coordinates
      if ((unsigned)(ax + 1) > ST_W || (unsigned)(ay + 1) > TH) continue;      // cannot touch this tile
      const float dx = ux - (float)fx, dy = uy - (float)fy;
      int tot;                                         // signed: epr_transport accepts planes of either sign
      if (FROM_TAU) {
        // the same arithmetic as the interior walk, operation for operation: a source is an interior source of its
        // own tile and a ring source of its neighbours, and all of them must agree on its four corner masses
        const float xe = -gamx * tc;
        const float J = fabsf(xe) < 0.35f ? epr_expm1_small(xe) : epr_exp_fast(xe) - 1.f;
        tot = Fix + __float2int_rn(fixFfx * J);
      } else {
        tot = __float2int_rn(__ldg(&I_bins[pl + gidx]) * 67108864.f);
      }
      // corner masses in fp32 (± 2 units of 2^-26), the 4th corner takes the exact remainder
      const float totf = (float)tot, te = totf * (1.f - dy), td = totf * dy, ex = 1.f - dx;
      const int c00 = __float2int_rn(te * ex), c10 = __float2int_rn(te * dx), c01 = __float2int_rn(td * ex);
      const int c11 = tot - c00 - c10 - c01;
      // ax ∈ [−1, ST_W − 1], ay ∈ [−1, TH − 1]: all four corners are inside the bordered accumulator
      unsigned* a0 = s_acc + (ay + 1) * ST_AP + (ax + 4);
      atomicAdd(a0, (unsigned)c00);
      atomicAdd(a0 + 1, (unsigned)c10);
      atomicAdd(a0 + ST_AP, (unsigned)c01);
      atomicAdd(a0 + ST_AP + 1, (unsigned)c11);
    }
    __syncthreads();
    // flush the tile: 4 pixels per thread per pass
    const float sc = 1.0f / (float)EPR_FIX_ONE, corr = L.fixCorr[s];
    float* ol = out + pl + fg0;
    // border cells (4 columns left and right of every row, the rows above and below): out-of-tile corners, never flushed
    if (tid < 2 * (TH + 2)) {
      const int r = tid >> 1;
      *reinterpret_cast<uint4*>(s_acc + r * ST_AP + ((tid & 1) ? ST_W + 4 : 0)) = make_uint4(0u, 0u, 0u, 0u);
    } else if (tid < 2 * (TH + 2) + 2 * (ST_W / 4)) {
      const int j = tid - 2 * (TH + 2), r = (j & 1) ? TH + 1 : 0;
      *reinterpret_cast<uint4*>(s_acc + r * ST_AP + 4 + 4 * (j >> 1)) = make_uint4(0u, 0u, 0u, 0u);
    }
#pragma unroll
    for (int k = 0; k < NFL; ++k) {
      const uint4 v = *reinterpret_cast<const uint4*>(facc + k * FRS * ST_AP);
      *reinterpret_cast<uint4*>(facc + k * FRS * ST_AP) = make_uint4(0u, 0u, 0u, 0u);      // cleared for the next line
      if (!(fxin && FRS * k < frows)) continue;
      float4 o;
      if (out_mode == 1) {
        o = make_float4((float)(int)v.x * sc, (float)(int)v.y * sc, (float)(int)v.z * sc, (float)(int)v.w * sc);
      } else {
        // Sources from τ are positive, so an accumulator that reads negative has passed 32x the flat field (u32 fixed
        // point, 1.0 = 2^26, wraps at 64x): reported through the plan's flag word (epr_read_flags), never silently.
        // (The exact-remainder corner may be a few units NEGATIVE when a weight vanishes, so a pixel fed by such corners
        // alone legitimately reads −1 … −8 units: those are not overflows, hence the offset.)
        if (min(min((int)v.x, (int)v.y), min((int)v.z, (int)v.w)) < -1024) atomicOr(flags, EPR_FLAG_SPLAT_OVERFLOW);
        // An EMPTY detector pixel (no source reaches it: the shadow side of a caustic) is written as exactly −f_s, so that
        // P_s = f_s + (P_s − f_s) is exactly 0 downstream and the split's decision "Σ_t P_t⁺ = 0 → w_s = f_s" (R8) is
        // taken on the integers, where an empty pixel is exactly empty — (float)(−Fi) alone would leave ±3e-8 there.
        if (COLS) {                                    // baseline, its fp32 remainder and f_s of the four DETECTOR columns
          const size_t ci = (size_t)s * nx + (x0 + ftx);
          const uint4 F4 = __ldg(reinterpret_cast<const uint4*>(C.fixFi + ci));
          const float4 c4 = __ldg(reinterpret_cast<const float4*>(C.fixCorr + ci)), f4 = __ldg(reinterpret_cast<const float4*>(C.f + ci));
          o = make_float4(v.x ? fmaf((float)((int)v.x - (int)F4.x), sc, c4.x) : -f4.x, v.y ? fmaf((float)((int)v.y - (int)F4.y), sc, c4.y) : -f4.y,
                          v.z ? fmaf((float)((int)v.z - (int)F4.z), sc, c4.z) : -f4.z, v.w ? fmaf((float)((int)v.w - (int)F4.w), sc, c4.w) : -f4.w);
        } else {
          const float nf = -L.f[s];
          o = make_float4(v.x ? fmaf((float)((int)v.x - Fi), sc, corr) : nf, v.y ? fmaf((float)((int)v.y - Fi), sc, corr) : nf,
                          v.z ? fmaf((float)((int)v.z - Fi), sc, corr) : nf, v.w ? fmaf((float)((int)v.w - Fi), sc, corr) : nf);
        }
        if (out_mode == 2) {
          const float4 dd = dpre[k];
          float4 off = make_float4(1.f + L.fsum_dev, 1.f + L.fsum_dev, 1.f + L.fsum_dev, 1.f + L.fsum_dev);
          if (COLS) {
            const float4 fd = __ldg(reinterpret_cast<const float4*>(C.fsum_dev + (x0 + ftx)));
            off = make_float4(1.f + fd.x, 1.f + fd.y, 1.f + fd.z, 1.f + fd.w);
          }
          o = make_float4((dd.x - off.x) - o.x, (dd.y - off.y) - o.y, (dd.z - off.z) - o.z, (dd.w - off.w) - o.w);
        }
      }
      *reinterpret_cast<float4*>(ol + k * fgs) = o;
    }
  }
  if (out_mode == 3) {
    // a2 fused (several lines): e = (d − 1) − Σ_s (P_s − f_s), e_s = w_s e with w_s = P_s⁺ / Σ_t P_t⁺ (fallback f_s),
    // PAPER.md:231, reading R8 — the arithmetic of k_residual, in place.  Every thread re-reads exactly the values
    // P_s − f_s it stored above (same thread, same addresses: program order makes them visible; they are still in L2)
    // and overwrites them with e_s, so the N prediction planes never come back from HBM.
    float4 off = make_float4(1.f + L.fsum_dev, 1.f + L.fsum_dev, 1.f + L.fsum_dev, 1.f + L.fsum_dev);
    if (COLS && fxin) {
      const float4 fd = __ldg(reinterpret_cast<const float4*>(C.fsum_dev + (x0 + ftx)));
      off = make_float4(1.f + fd.x, 1.f + fd.y, 1.f + fd.z, 1.f + fd.w);
    }
    // f_s of the thread's four detector columns: the line's scalar, or (COLS) the columns' table entries
    auto f4_of = [&](int s) {
      if (COLS) return __ldg(reinterpret_cast<const float4*>(C.f + (size_t)s * nx + (x0 + ftx)));
      const float f = L.f[s];
      return make_float4(f, f, f, f);
    };
    float* ob = out + (size_t)b * L.n_bins * plane + fg0;
    const float* dg = d + (size_t)b * plane + fg0;
#pragma unroll 1
    for (int k = 0; k < NFL; ++k) {
      if (!(fxin && FRS * k < frows)) continue;
      float* og = ob + k * fgs;
      float4 sum = make_float4(0.f, 0.f, 0.f, 0.f), den = sum;
      #pragma unroll 4                                  // four independent L2 loads in flight per thread (8: slower)
      for (int s = 0; s < L.n_bins; ++s) {
        const float4 pd = __ldcg(reinterpret_cast<const float4*>(og + (size_t)s * plane));
        const float4 f = f4_of(s);
        sum.x += pd.x; sum.y += pd.y; sum.z += pd.z; sum.w += pd.w;
        den.x += fmaxf(f.x + pd.x, 0.f); den.y += fmaxf(f.y + pd.y, 0.f); den.z += fmaxf(f.z + pd.z, 0.f); den.w += fmaxf(f.w + pd.w, 0.f);
      }
      const float4 dd = __ldg(reinterpret_cast<const float4*>(dg + k * fgs));
      const float4 e = make_float4((dd.x - off.x) - sum.x, (dd.y - off.y) - sum.y, (dd.z - off.z) - sum.z, (dd.w - off.w) - sum.w);
      // e_s = P_s⁺ q + f_s fb:  q = e/Σ_t P_t⁺, fb = 0 where the sum is positive;  q = 0, fb = e (weights f_s) where it is not
      const float4 q = make_float4(den.x > 0.f ? e.x / den.x : 0.f, den.y > 0.f ? e.y / den.y : 0.f,
                                   den.z > 0.f ? e.z / den.z : 0.f, den.w > 0.f ? e.w / den.w : 0.f);
      const float4 fb = make_float4(den.x > 0.f ? 0.f : e.x, den.y > 0.f ? 0.f : e.y, den.z > 0.f ? 0.f : e.z, den.w > 0.f ? 0.f : e.w);
      #pragma unroll 4
      for (int s = 0; s < L.n_bins; ++s) {
        const float4 pd = __ldcg(reinterpret_cast<const float4*>(og + (size_t)s * plane));
        const float4 f = f4_of(s);
        float4 o;
        o.x = fmaf(fmaxf(f.x + pd.x, 0.f), q.x, f.x * fb.x);
        o.y = fmaf(fmaxf(f.y + pd.y, 0.f), q.y, f.y * fb.y);
        o.z = fmaf(fmaxf(f.z + pd.z, 0.f), q.z, f.z * fb.z);
        o.w = fmaf(fmaxf(f.w + pd.w, 0.f), q.w, f.w * fb.w);
        *reinterpret_cast<float4*>(og + (size_t)s * plane) = o;
      }
    }
  }
}

template <bool FROM_TAU, bool MAP_OUT, int NT, int TH, bool COLS>
static cudaError_t launch_splat_v(const epr_plan_s* p, int batch, int H, size_t smem, const float* tau, const float* I_bins,
                                  const float2* map_in, float2* map_out, float* out, int out_mode, const float* d,
                                  cudaStream_t st) {
  static EprPerDevice attr = {};                         // largest dynamic shared memory set so far, per device
  if ((long long)smem > attr.at(p)) {
    cudaFuncSetAttribute(k_splat_tile<FROM_TAU, MAP_OUT, NT, TH, COLS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    attr.at(p) = (long long)smem;
  }
  dim3 grid((p->nx + ST_W - 1) / ST_W, (p->ny + TH - 1) / TH, batch);
  // several lines share one list of ring candidates (the coordinates are packed in 8 bits each: H ≤ 64)
  const int use_list = FROM_TAU && p->lines.n_bins > 1 && H <= 64;
  k_splat_tile<FROM_TAU, MAP_OUT, NT, TH, COLS><<<grid, NT, smem, st>>>(COLS ? p->lines_bound : p->lines, p->cols, p->nx, p->ny,
                                                                         p->opt.max_shift_px, H, tau, I_bins, map_in, map_out, out,
                                                                         out_mode, d, p->gmax, use_list, p->d_flags);
  return cudaGetLastError();
}

template <bool FROM_TAU, bool MAP_OUT, bool COLS = false>
static cudaError_t launch_splat_t(const epr_plan_s* p, int batch, const float* tau, const float* I_bins, const float2* map_in,
                                  float2* map_out, float* out, int out_mode, const float* d, cudaStream_t st) {
  const int H = (int)ceilf(p->opt.max_shift_px) + 1;
  const int Ha = (H + 1 + 3) & ~3;
  auto smem_of = [&](int th) {
    return (size_t)ST_AP * (th + 2) * sizeof(unsigned) + (FROM_TAU ? (size_t)(ST_W + 2 * Ha) * (th + 2 * H + 2) * sizeof(float) + ST_LCAP * sizeof(unsigned short) : 0);
  };
  if (FROM_TAU) {                                      // block maxima of |D⁰τ| (also used by the gather of this τ)
    const cudaError_t e = epr_launch_grad_blockmax(p, batch, tau, st);
    if (e != cudaSuccess) return e;
    epr_note_extra_launch(p);
  }
  const size_t half = 113 * 1024;                      // half of the 227 KB an SM offers: two CTAs per SM
  // 128 x 64 tiles with 512 threads when two CTAs fit an SM; large S (C5: S = 24): 128 x 32 tiles still bring two;
  // beyond that one 1024-thread CTA per SM
  if (smem_of(ST_H) <= half)
    return launch_splat_v<FROM_TAU, MAP_OUT, 512, ST_H, COLS>(p, batch, H, smem_of(ST_H), tau, I_bins, map_in, map_out, out, out_mode, d, st);
  if (smem_of(ST_H / 2) <= half)
    return launch_splat_v<FROM_TAU, MAP_OUT, 512, ST_H / 2, COLS>(p, batch, H, smem_of(ST_H / 2), tau, I_bins, map_in, map_out, out, out_mode, d, st);
  return launch_splat_v<FROM_TAU, MAP_OUT, 1024, ST_H, COLS>(p, batch, H, smem_of(ST_H), tau, I_bins, map_in, map_out, out, out_mode, d, st);
}

cudaError_t epr_launch_splat(const epr_plan_s* p, int batch, const float* tau, const float* I_bins, const float2* map_in,
                             float2* map_out, float* out, int out_mode, const float* d, cudaStream_t st) {
  if (!tau) return launch_splat_t<false, false>(p, batch, tau, I_bins, map_in, map_out, out, out_mode, d, st);
  if (map_out) return launch_splat_t<true, true>(p, batch, tau, I_bins, map_in, map_out, out, out_mode, d, st);
  return launch_splat_t<true, false>(p, batch, tau, I_bins, map_in, map_out, out, out_mode, d, st);
}

// The loop's splat with the per-column tables of an x-dependent spectrum (16-pixel-aligned grids; reading R17(b))
cudaError_t epr_launch_splat_cols(const epr_plan_s* p, int batch, const float* tau, float* out, int out_mode, const float* d,
                                  cudaStream_t st) {
  return launch_splat_t<true, false, true>(p, batch, tau, nullptr, nullptr, nullptr, out, out_mode, d, st);
}

// =====================================================================================================
// a2  detector residual and positivity-weighted split (reading R8), deviation form:
//   e = (d − 1) − Σ_s (P_s − f_s);   w_s = P_s⁺ / Σ_t P_t⁺ (fallback f_s);   es_s = w_s e
//   pred holds P_s − f_s (float), written by k_local_march (several lines) or k_splat_tile.
// =====================================================================================================
// one thread = 4 consecutive pixels (plane % 4 == 0)
__global__ void __launch_bounds__(256) k_residual(EprLines L, unsigned plane, const float* __restrict__ d,
                                                  const float* __restrict__ pred, float* __restrict__ es) {
  const unsigned i = (blockIdx.x * 256u + threadIdx.x) * 4u;
  const int b = blockIdx.y;
  if (i >= plane) return;
  const size_t base = (size_t)b * L.n_bins * plane + i;
  float4 sum = make_float4(0.f, 0.f, 0.f, 0.f), den = sum;
  for (int s = 0; s < L.n_bins; ++s) {
    const float4 pd = __ldg(reinterpret_cast<const float4*>(pred + base + (size_t)s * plane));
    const float f = L.f[s];
    sum.x += pd.x; sum.y += pd.y; sum.z += pd.z; sum.w += pd.w;
    den.x += fmaxf(f + pd.x, 0.f); den.y += fmaxf(f + pd.y, 0.f); den.z += fmaxf(f + pd.z, 0.f); den.w += fmaxf(f + pd.w, 0.f);
  }
  const float4 dd = __ldg(reinterpret_cast<const float4*>(d + (size_t)b * plane + i));
  const float off = 1.f + L.fsum_dev;
  const float4 e = make_float4((dd.x - off) - sum.x, (dd.y - off) - sum.y, (dd.z - off) - sum.z, (dd.w - off) - sum.w);
  // e/den once per pixel; w_s e = P_s⁺ (e/den), fallback f_s e where den <= 0
  const float4 q = make_float4(den.x > 0.f ? e.x / den.x : 0.f, den.y > 0.f ? e.y / den.y : 0.f,
                               den.z > 0.f ? e.z / den.z : 0.f, den.w > 0.f ? e.w / den.w : 0.f);
  for (int s = 0; s < L.n_bins; ++s) {
    const float4 pd = __ldg(reinterpret_cast<const float4*>(pred + base + (size_t)s * plane));
    const float f = L.f[s];
    float4 o;
    o.x = den.x > 0.f ? fmaxf(f + pd.x, 0.f) * q.x : f * e.x;
    o.y = den.y > 0.f ? fmaxf(f + pd.y, 0.f) * q.y : f * e.y;
    o.z = den.z > 0.f ? fmaxf(f + pd.z, 0.f) * q.z : f * e.z;
    o.w = den.w > 0.f ? fmaxf(f + pd.w, 0.f) * q.w : f * e.w;
    *reinterpret_cast<float4*>(es + base + (size_t)s * plane) = o;
  }
}

cudaError_t epr_launch_residual(const epr_plan_s* p, int batch, const float* d, const float* pred, float* es,
                                cudaStream_t st) {
  const unsigned plane = (unsigned)p->nx * p->ny;
  dim3 grid((plane / 4 + 255) / 256, batch);
  k_residual<<<grid, 256, 0, st>>>(p->lines, plane, d, pred, es);
  return cudaGetLastError();
}

// epr_forward output: P_s = f_s + (P_s − f_s), P = Σ_s P_s.
__global__ void __launch_bounds__(256) k_pred_out(EprLines L, size_t plane, const float* __restrict__ pred,
                                                  float* __restrict__ P_sum, float* __restrict__ P_bins) {
  const size_t i = (size_t)blockIdx.x * 256 + threadIdx.x;
  const int b = blockIdx.y;
  if (i >= plane) return;
  const size_t base = (size_t)b * L.n_bins * plane + i;
  float sum = 0.f;
  for (int s = 0; s < L.n_bins; ++s) {
    const float v = L.f[s] + __ldg(&pred[base + s * plane]);
    sum += v;
    if (P_bins) P_bins[base + s * plane] = v;
  }
  if (P_sum) P_sum[(size_t)b * plane + i] = sum;
}

cudaError_t epr_launch_pred_out(const epr_plan_s* p, int batch, const float* pred, float* P_sum, float* P_bins,
                                cudaStream_t st) {
  const size_t plane = (size_t)p->nx * p->ny;
  dim3 grid((unsigned)((plane + 255) / 256), batch);
  k_pred_out<<<grid, 256, 0, st>>>(p->lines, plane, pred, P_sum, P_bins);
  return cudaGetLastError();
}

// =====================================================================================================
// a3  adjoint ℳ*_s: bilinear gather at the mapped coordinates, Eq. (4), with the SAME
//     x0, y0, w as the splat of this iteration (ray map recomputed from τ, or the stored one).
// =====================================================================================================
template <bool BIG, bool COLS = false>          // BIG: nx, ny > 32 ≥ |shift| + 1, so one conditional add wraps an index; COLS: per-column a_s γ_s
__global__ void __launch_bounds__(256) k_gather(EprLines L, EprColumns C, int nx, int ny, float S, const float* __restrict__ tau,
                                                const float2* __restrict__ map_in, const float* __restrict__ es,
                                                float* __restrict__ r) {
  // one thread = 4 consecutive pixels of one row (nx % 4 == 0)
  const int x = 4 * (blockIdx.x * 64 + (threadIdx.x & 63)), y = blockIdx.y * 4 + (threadIdx.x >> 6);
  const int b = blockIdx.z;
  if (x >= nx || y >= ny) return;
  const unsigned plane = (unsigned)nx * (unsigned)ny, row = (unsigned)y * nx;
  float dtx[4] = {0.f, 0.f, 0.f, 0.f}, dty[4] = {0.f, 0.f, 0.f, 0.f};
  if (!map_in) {
    const float* tb = tau + (size_t)b * plane;
    const int xm = x == 0 ? nx - 1 : x - 1, xp = x + 4 == nx ? 0 : x + 4;
    const int ym = y == 0 ? ny - 1 : y - 1, yp = y + 1 == ny ? 0 : y + 1;
    const float4 c = __ldg(reinterpret_cast<const float4*>(tb + row + x));
    const float4 n = __ldg(reinterpret_cast<const float4*>(tb + (unsigned)ym * nx + x));
    const float4 s4 = __ldg(reinterpret_cast<const float4*>(tb + (unsigned)yp * nx + x));
    const float l = __ldg(tb + row + xm), rr = __ldg(tb + row + xp);
    dtx[0] = c.y - l; dtx[1] = c.z - c.x; dtx[2] = c.w - c.y; dtx[3] = rr - c.z;
    dty[0] = s4.x - n.x; dty[1] = s4.y - n.y; dty[2] = s4.z - n.z; dty[3] = s4.w - n.w;
  }
  const size_t p0 = (size_t)b * L.n_bins * plane;
  const float* eb = es + p0;
  float* rb = r + p0 + row + x;
  const float2* mb = map_in ? map_in + p0 + row + x : nullptr;
  for (int s = 0; s < L.n_bins; ++s, eb += plane, rb += plane) {
    float c4[4];
    c4[0] = c4[1] = c4[2] = c4[3] = -0.5f * L.a[s] * L.gamma[s];
    if (COLS) {                                        // the pixel's own column (the map of the splat of this column's sources)
      const float4 a4 = __ldg(reinterpret_cast<const float4*>(C.a + (size_t)s * nx + x));
      const float4 g4 = __ldg(reinterpret_cast<const float4*>(C.gamma + (size_t)s * nx + x));
      c4[0] = -0.5f * a4.x * g4.x; c4[1] = -0.5f * a4.y * g4.y; c4[2] = -0.5f * a4.z * g4.z; c4[3] = -0.5f * a4.w * g4.w;
    }
    float o[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      float ux, uy;
      if (map_in) {
        const float2 m = __ldg(mb + k);
        ux = m.x; uy = m.y;
      } else {
        ux = fminf(fmaxf(c4[k] * dtx[k], -S), S);
        uy = fminf(fmaxf(c4[k] * dty[k], -S), S);
      }
      const int fx = __float2int_rd(ux), fy = __float2int_rd(uy);
      const float dx = ux - (float)fx, dy = uy - (float)fy;
      const int ix0 = BIG ? wrap1(x + k + fx, nx) : wrapm(x + k + fx, nx);
      const int iy0 = BIG ? wrap1(y + fy, ny) : wrapm(y + fy, ny);
      const int ix1 = ix0 + 1 == nx ? 0 : ix0 + 1, iy1 = iy0 + 1 == ny ? 0 : iy0 + 1;
      const unsigned r0 = (unsigned)iy0 * nx, r1 = (unsigned)iy1 * nx;
      const float e00 = __ldg(eb + (r0 + ix0)), e10 = __ldg(eb + (r0 + ix1));
      const float e01 = __ldg(eb + (r1 + ix0)), e11 = __ldg(eb + (r1 + ix1));
      // Eq. (4): Σ_ab w_ab e[y0+b][x0+a], w00 = (1−dx)(1−dy), w10 = dx(1−dy), w01 = (1−dx)dy, w11 = dx dy
      const float ex = 1.f - dx, ey = 1.f - dy;
      o[k] = ey * (ex * e00 + dx * e10) + dy * (ex * e01 + dx * e11);
    }
    if (map_in) mb += plane;
    *reinterpret_cast<float4*>(rb) = make_float4(o[0], o[1], o[2], o[3]);
  }
}

// -----------------------------------------------------------------------------------------------------
// a3 through shared memory (the loop's configuration: ray map recomputed from τ, block maxima of |D⁰τ| at hand).
// One CTA = GT_W x GT_H pixels of one projection.  The tile's own max|u_s| (from p->gmax) gives the halo Hg of the
// residual it can touch; e_s[tile + Hg] is staged by 16-byte cp.async (line s + 1 under the gather of line s) and the
// four corners are plain shared loads at consecutive lanes — one wavefront each instead of the ~4.5 lines a scattered
// global load touches.  The τ differences are formed once and reused for every line.  Lines whose halo exceeds
// GT_HG fall back to global loads inside the same kernel.
#define GT_W 128
#define GT_H 64
#define GT_HG 8                        // largest halo served from shared memory (multiple of 4)
#define GT_EP (GT_W + 2 * GT_HG)       // pitch of a staged tile
#define GT_ER (GT_H + 2 * GT_HG)
#define GT_NT 512
#define GT_PPT (GT_W * GT_H / GT_NT)   // pixels per thread (rows y = (tid >> 7) + 4 k of column tid & 127)

template <bool BIG, bool COLS = false>          // BIG: nx, ny ≥ 2 (tile + halo), so one conditional add wraps an index
__global__ void __launch_bounds__(GT_NT, 2) k_gather_tile(EprLines L, EprColumns C, int nx, int ny, float S, const float* __restrict__ tau,
                                                        const float* __restrict__ gmax, const float* __restrict__ es,
                                                        float* __restrict__ r) {
  extern __shared__ __align__(128) float s_e[];       // [2][GT_ER][GT_EP]
  __shared__ unsigned s_max;
  __shared__ __align__(8) uint64_t s_bar[2];
  const int tid = threadIdx.x, b = blockIdx.z;
  const int x0 = blockIdx.x * GT_W, y0 = blockIdx.y * GT_H;
  const unsigned plane = (unsigned)nx * (unsigned)ny;
  if (tid == 0) { s_max = 0u; eprtma::mbar_init(&s_bar[0], 1); eprtma::mbar_init(&s_bar[1], 1); eprtma::mbar_fence_init(); }
  __syncthreads();
  if (tid < 32) {
    const int px = x0 + 16 * (tid & 7), py = y0 + 16 * (tid >> 3);
    if (px < nx && py < ny) atomicMax(&s_max, __float_as_uint(__ldg(&gmax[((size_t)b * (ny >> 4) + (py >> 4)) * (nx >> 4) + (px >> 4)])));
  }
  __syncthreads();
  const float maxd = __uint_as_float(s_max);
  const size_t p0 = (size_t)b * L.n_bins * plane;
  // reads reach x + fx … x + fx + 1 with fx ∈ [−Hg, Hg − 1], Hg = ⌊max|u|⌋ + 1
  auto halo = [&](int s) { return (int)fminf(0.5f * L.a[s] * L.gamma[s] * maxd, S) + 1; };
  // request e_s[tile + halo] into buffer s & 1: one bulk copy (TMA, cp.async.bulk) per row — two where the row
  // crosses the periodic boundary — issued by the first 64 + 2 Hg threads, completion counted on s_bar[s & 1]
  auto stage = [&](int s) {
    const int Hg = halo(s);
    if (Hg > GT_HG) return;
    const int Hga = (Hg + 3) & ~3, rows = GT_H + 2 * Hg, len = GT_W + 2 * Hga;
    if (tid == 0) eprtma::mbar_expect_tx(&s_bar[s & 1], (unsigned)(rows * len) * 4u);
    if (tid < rows) {
      const float* erow = es + p0 + (size_t)s * plane + (size_t)(BIG ? wrap1(y0 - Hg + tid, ny) : wrapm(y0 - Hg + tid, ny)) * nx;
      float* dst = s_e + (s & 1) * (GT_ER * GT_EP) + (GT_HG - Hg + tid) * GT_EP + (GT_HG - Hga);
      int gx = BIG ? wrap1(x0 - Hga, nx) : wrapm(x0 - Hga, nx), left = len;
      while (left > 0) {
        const int n = min(left, nx - gx);
        eprtma::bulk_g2s(dst, erow + gx, (unsigned)n * 4u, &s_bar[s & 1]);
        dst += n; left -= n; gx = 0;
      }
    }
  };
  stage(0);
  // τ differences of this thread's pixels (column x, rows yy + 4 k), formed once for all lines
  const int x = tid & (GT_W - 1), yy = tid >> 7;
  const bool xin = x0 + x < nx;
  float dtx[GT_PPT], dty[GT_PPT];
  {
    const float* tb = tau + (size_t)b * plane;
    const int gx = xin ? x0 + x : 0;
    const int xm = gx == 0 ? nx - 1 : gx - 1, xp = gx + 1 == nx ? 0 : gx + 1;
#pragma unroll
    for (int k = 0; k < GT_PPT; ++k) {
      const int gy = min(y0 + yy + 4 * k, ny - 1);
      const int ym = gy == 0 ? ny - 1 : gy - 1, yp = gy + 1 == ny ? 0 : gy + 1;
      const float* row = tb + (unsigned)gy * nx;
      dtx[k] = __ldg(row + xp) - __ldg(row + xm);
      dty[k] = __ldg(tb + (unsigned)yp * nx + gx) - __ldg(tb + (unsigned)ym * nx + gx);
      // Pixels outside the image (ragged last tile) only keep the lanes busy: their shifts must be ZERO, not those of
      // column 0 / row ny − 1, whose gradients the tile's block maxima (and so the staged halo Hg) do not bound — the
      // corner loads below are unpredicated and would leave the staged tile.
      if (!xin || y0 + yy + 4 * k >= ny) dtx[k] = dty[k] = 0.f;
    }
  }
  unsigned nfill = 0u;                                 // bit i: parity of the fills of buffer i (lines served by global loads skip theirs)
  for (int s = 0; s < L.n_bins; ++s) {
    if (s + 1 < L.n_bins) stage(s + 1);                // buffer (s + 1) & 1 was released by the barrier ending line s − 1
    // COLS: L carries the bound max_x a_s(x) γ_s(x) (halo, clamp test); the thread's pixels share its column's coefficient
    const float cb = -0.5f * L.a[s] * L.gamma[s];
    const float c = COLS ? -0.5f * __ldg(&C.a[(size_t)s * nx + (xin ? x0 + x : 0)]) * __ldg(&C.gamma[(size_t)s * nx + (xin ? x0 + x : 0)]) : cb;
    const int Hg = halo(s);
    if (Hg <= GT_HG) {                                 // phase parity = how often this buffer has been filled before
      eprtma::mbar_wait(&s_bar[s & 1], (nfill >> (s & 1)) & 1u);
      nfill ^= 1u << (s & 1);
    }
    float* rb = r + p0 + (size_t)s * plane + (size_t)(y0 + yy) * nx + (x0 + x);
    if (Hg <= GT_HG) {
      const unsigned base = (unsigned)__cvta_generic_to_shared(s_e + (s & 1) * (GT_ER * GT_EP)) +
                            4u * (unsigned)((yy + GT_HG) * GT_EP + x + GT_HG);
      const size_t nx4 = 4 * (size_t)nx;
      // CLAMP: some |u| of the tile may exceed S;  FULL: the whole tile lies inside the image (no per-pixel test)
      auto body = [&](auto clamp_tag, auto full_tag) {
        constexpr bool CLAMP = decltype(clamp_tag)::value, FULL = decltype(full_tag)::value;
#pragma unroll
        for (int k = 0; k < GT_PPT; ++k) {
          float ux = c * dtx[k], uy = c * dty[k];
          if (CLAMP) { ux = fminf(fmaxf(ux, -S), S); uy = fminf(fmaxf(uy, -S), S); }
          const int fx = __float2int_rd(ux), fy = __float2int_rd(uy);
          const float dx = ux - (float)fx, dy = uy - (float)fy;
          const unsigned a = base + 4u * (unsigned)(fy * GT_EP + fx);
          // the row offsets 16 k GT_EP are compile-time after unrolling: ptxas folds them into the load
          const float e00 = lds_f32(a + 16 * k * GT_EP), e10 = lds_f32(a + 16 * k * GT_EP + 4);
          const float e01 = lds_f32(a + (16 * k + 4) * GT_EP), e11 = lds_f32(a + (16 * k + 4) * GT_EP + 4);
          // Eq. (4): Σ_ab w_ab e[y0+b][x0+a], w00 = (1−dx)(1−dy), w10 = dx(1−dy), w01 = (1−dx)dy, w11 = dx dy
          const float t0 = fmaf(dx, e10 - e00, e00), t1 = fmaf(dx, e11 - e01, e01);
          if (FULL || (xin && y0 + yy + 4 * k < ny)) rb[k * nx4] = fmaf(dy, t1 - t0, t0);
        }
      };
      const bool clamp = fabsf(cb) * maxd > S, full = x0 + GT_W <= nx && y0 + GT_H <= ny;
      if (clamp) { if (full) body(std::true_type{}, std::true_type{}); else body(std::true_type{}, std::false_type{}); }
      else { if (full) body(std::false_type{}, std::true_type{}); else body(std::false_type{}, std::false_type{}); }
    } else if (xin) {
      const float* eb = es + p0 + (size_t)s * plane;
      for (int k = 0; k < GT_PPT; ++k) {
        const int gy = y0 + yy + 4 * k;
        if (gy >= ny) break;
        const float ux = fminf(fmaxf(c * dtx[k], -S), S), uy = fminf(fmaxf(c * dty[k], -S), S);
        const int fx = __float2int_rd(ux), fy = __float2int_rd(uy);
        const float dx = ux - (float)fx, dy = uy - (float)fy;
        const int ix0 = wrapm(x0 + x + fx, nx), iy0 = wrapm(gy + fy, ny);
        const int ix1 = ix0 + 1 == nx ? 0 : ix0 + 1, iy1 = iy0 + 1 == ny ? 0 : iy0 + 1;
        const unsigned r0 = (unsigned)iy0 * nx, r1 = (unsigned)iy1 * nx;
        const float e00 = __ldg(eb + (r0 + ix0)), e10 = __ldg(eb + (r0 + ix1));
        const float e01 = __ldg(eb + (r1 + ix0)), e11 = __ldg(eb + (r1 + ix1));
        const float ex = 1.f - dx, ey = 1.f - dy;
        rb[(size_t)(4 * k) * nx] = ey * (ex * e00 + dx * e10) + dy * (ex * e01 + dx * e11);
      }
    }
    eprtma::fence_proxy_async();                       // this thread's reads of the buffer precede its refill by the TMA unit
    __syncthreads();                                   // buffer s & 1 is free for line s + 2
  }
}

template <bool COLS>
static cudaError_t launch_gather_t(const epr_plan_s* p, int batch, const float* tau, const float2* map_in, const float* es,
                                   float* r, int gmax_fresh, cudaStream_t st) {
  const EprLines& LL = COLS ? p->lines_bound : p->lines;
  if (tau && !map_in && gmax_fresh && p->gmax && p->n_bins > 1) {
    // the loop: p->gmax holds the block maxima of this τ (written ahead of the splat of the same iteration).
    // Several lines only: with one line there is nothing to stage ahead and nothing to share, and the direct kernel
    // below measures faster (14.1 vs 15.5 us per 2048² plane).
    constexpr size_t smem = 2 * (size_t)GT_ER * GT_EP * sizeof(float);
    static EprPerDevice attr = {};
    if (!attr.at(p)) {
      cudaFuncSetAttribute(k_gather_tile<true, COLS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
      cudaFuncSetAttribute(k_gather_tile<false, COLS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
      attr.at(p) = 1;
    }
    dim3 grid((p->nx + GT_W - 1) / GT_W, (p->ny + GT_H - 1) / GT_H, batch);
    if (p->nx >= 2 * GT_EP && p->ny >= 2 * GT_ER)
      k_gather_tile<true, COLS><<<grid, GT_NT, smem, st>>>(LL, p->cols, p->nx, p->ny, p->opt.max_shift_px, tau, p->gmax, es, r);
    else
      k_gather_tile<false, COLS><<<grid, GT_NT, smem, st>>>(LL, p->cols, p->nx, p->ny, p->opt.max_shift_px, tau, p->gmax, es, r);
    return cudaGetLastError();
  }
  dim3 grid((p->nx / 4 + 63) / 64, (p->ny + 3) / 4, batch);
  if (p->nx > 32 && p->ny > 32) k_gather<true, COLS><<<grid, 256, 0, st>>>(LL, p->cols, p->nx, p->ny, p->opt.max_shift_px, tau, map_in, es, r);
  else k_gather<false, COLS><<<grid, 256, 0, st>>>(LL, p->cols, p->nx, p->ny, p->opt.max_shift_px, tau, map_in, es, r);
  return cudaGetLastError();
}

cudaError_t epr_launch_gather(const epr_plan_s* p, int batch, const float* tau, const float2* map_in, const float* es,
                              float* r, int gmax_fresh, cudaStream_t st) {
  return launch_gather_t<false>(p, batch, tau, map_in, es, r, gmax_fresh, st);
}

// the loop's gather with the per-column tables of an x-dependent spectrum (after epr_launch_splat_cols on the same τ)
cudaError_t epr_launch_gather_cols(const epr_plan_s* p, int batch, const float* tau, const float* es, float* r, cudaStream_t st) {
  return launch_gather_t<true>(p, batch, tau, nullptr, es, r, 1, st);
}

// Final output conversion: τ | φ of one line (Eq. (6): φ_s = −(db_s/2) γ_s τ) | Σ_s I_s (Eq. (7)).
__global__ void __launch_bounds__(256) k_output(EprLines L, size_t n, int mode, float phase_coef,
                                                const float* __restrict__ tau, float* __restrict__ out) {
  const size_t i = (size_t)blockIdx.x * 256 + threadIdx.x;
  if (i >= n) return;
  const float t = tau[i];
  float v = t;
  if (mode == 1) v = phase_coef * t;
  else if (mode == 2) {
    v = 0.f;
    for (int s = 0; s < L.n_bins; ++s) v += L.f[s] * expf(-L.gamma[s] * t);
  }
  out[i] = v;
}

cudaError_t epr_launch_output(const epr_plan_s* p, int batch, const float* tau, float* out, cudaStream_t st) {
  const size_t n = (size_t)p->nx * p->ny * batch;
  const int sb = p->opt.out_bin;
  const float coef = (float)(-0.5 * p->h_db[sb] * p->h_gamma[sb]);
  k_output<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(p->lines, n, p->opt.output, coef, tau, out);
  return cudaGetLastError();
}

// =====================================================================================================
// Oversampled computational grid (reading R16): the loop runs on a grid refined m times; the detector
// image reaches it by pixel replication (a detector pixel measures the mean intensity over its area) and the result
// returns by the mean over each m x m block — the exact left inverse.  Both kernels are plain HBM streams.
// =====================================================================================================
// fine[b][Y][X] = coarse[b][Y / m][X / m];  one thread = 4 consecutive fine pixels (nx_f % 4 == 0)
__global__ void __launch_bounds__(256) k_upsample(int nx_f, int ny_f, int m, const float* __restrict__ coarse,
                                                  float* __restrict__ fine) {
  const int X = 4 * (blockIdx.x * 256 + threadIdx.x), Y = blockIdx.y, b = blockIdx.z;
  if (X >= nx_f) return;
  const int nx_c = nx_f / m, ny_c = ny_f / m;
  const float* row = coarse + ((size_t)b * ny_c + Y / m) * nx_c;
  float4 o;
  if (m == 2) { const float2 v = __ldg(reinterpret_cast<const float2*>(row + X / 2)); o = make_float4(v.x, v.x, v.y, v.y); }
  else if (m % 4 == 0) { const float v = __ldg(row + X / m); o = make_float4(v, v, v, v); }
  else o = make_float4(__ldg(row + X / m), __ldg(row + (X + 1) / m), __ldg(row + (X + 2) / m), __ldg(row + (X + 3) / m));
  *reinterpret_cast<float4*>(fine + ((size_t)b * ny_f + Y) * nx_f + X) = o;
}

// coarse[b][y][x] = mean of fine[b][m y + j][m x + i], i, j < m;  one thread = one coarse pixel
__global__ void __launch_bounds__(256) k_downsample(int nx_c, int ny_c, int m, const float* __restrict__ fine,
                                                    float* __restrict__ coarse) {
  const int x = blockIdx.x * 256 + threadIdx.x, y = blockIdx.y, b = blockIdx.z;
  if (x >= nx_c) return;
  const int nx_f = nx_c * m;
  const float* src = fine + ((size_t)b * ny_c * m + (size_t)y * m) * nx_f + (size_t)x * m;
  float acc = 0.f;
  for (int j = 0; j < m; ++j) {
    float r = 0.f;
    for (int i = 0; i < m; ++i) r += __ldg(src + (size_t)j * nx_f + i);
    acc += r;
  }
  coarse[((size_t)b * ny_c + y) * nx_c + x] = acc / (float)(m * m);
}

cudaError_t epr_launch_upsample(const epr_plan_s* p, int batch, int m, const float* coarse, float* fine, cudaStream_t st) {
  dim3 grid((p->nx / 4 + 255) / 256, p->ny, batch);
  k_upsample<<<grid, 256, 0, st>>>(p->nx, p->ny, m, coarse, fine);
  return cudaGetLastError();
}

cudaError_t epr_launch_downsample(const epr_plan_s* p, int batch, int m, const float* fine, float* coarse, cudaStream_t st) {
  dim3 grid((p->nx / m + 255) / 256, p->ny / m, batch);
  k_downsample<<<grid, 256, 0, st>>>(p->nx / m, p->ny / m, m, fine, coarse);
  return cudaGetLastError();
}

// =====================================================================================================
// Diagnostics of the loop (off unless epr_set_diagnostics was called; never in timed runs): per projection and
// iteration, the RMS of the detector residual e = d − Σ_s P_s = Σ_s e_s and the regime indicator
// η as the largest unclamped shift component max_s |c_s| · max|D⁰τ| from the block maxima.
// Two launches, fixed summation order (bit-reproducible).
// =====================================================================================================
#define DG_BLK 64
__global__ void __launch_bounds__(256) k_diag_partial(int n_bins, unsigned plane, const float* __restrict__ es,
                                                      double* __restrict__ partial) {
  __shared__ double s_sum[256];
  const int b = blockIdx.y;
  const float* eb = es + (size_t)b * n_bins * plane;
  double acc = 0.0;
  for (unsigned i = (blockIdx.x * 256u + threadIdx.x) * 4u; i < plane; i += DG_BLK * 256u * 4u) {
    float4 e = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int s = 0; s < n_bins; ++s) {
      const float4 v = __ldg(reinterpret_cast<const float4*>(eb + (size_t)s * plane + i));
      e.x += v.x; e.y += v.y; e.z += v.z; e.w += v.w;
    }
    acc += (double)e.x * e.x + (double)e.y * e.y + (double)e.z * e.z + (double)e.w * e.w;
  }
  s_sum[threadIdx.x] = acc;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if (threadIdx.x < o) s_sum[threadIdx.x] += s_sum[threadIdx.x + o];
    __syncthreads();
  }
  if (threadIdx.x == 0) partial[(size_t)b * DG_BLK + blockIdx.x] = s_sum[0];
}

__global__ void __launch_bounds__(256) k_diag_final(unsigned plane, int nblocks, float cmax, const double* __restrict__ partial,
                                                    const float* __restrict__ gmax, float* __restrict__ diag, int stride) {
  __shared__ float s_max[256];
  const int b = blockIdx.x;
  float m = 0.f;
  for (int i = threadIdx.x; i < nblocks; i += 256) m = fmaxf(m, __ldg(&gmax[(size_t)b * nblocks + i]));
  s_max[threadIdx.x] = m;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if (threadIdx.x < o) s_max[threadIdx.x] = fmaxf(s_max[threadIdx.x], s_max[threadIdx.x + o]);
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    double sum = 0.0;
    for (int i = 0; i < DG_BLK; ++i) sum += partial[(size_t)b * DG_BLK + i];
    diag[(size_t)b * stride] = (float)sqrt(sum / (double)plane);
    diag[(size_t)b * stride + 1] = cmax * s_max[0];
  }
}

cudaError_t epr_launch_diagnostics(const epr_plan_s* p, int batch, const float* tau, const float* es, float* diag,
                                   int stride, cudaStream_t st) {
  const unsigned plane = (unsigned)p->nx * p->ny;
  if (p->solver == EPR_LOCAL) {                       // the non-local splat has already refreshed p->gmax for this τ
    const cudaError_t e = epr_launch_grad_blockmax(p, batch, tau, st);
    if (e != cudaSuccess) return e;
    epr_note_extra_launch(p);
  }
  float cmax = 0.f;
  for (int s = 0; s < p->n_bins; ++s) cmax = fmaxf(cmax, 0.5f * p->lines.a[s] * p->lines.gamma[s]);
  epr_note_extra_launch(p);                            // two kernels below
  k_diag_partial<<<dim3(DG_BLK, batch), 256, 0, st>>>(p->n_bins, plane, es, p->diag_partial);
  k_diag_final<<<batch, 256, 0, st>>>(plane, (p->nx / 16) * (p->ny / 16), cmax, p->diag_partial, p->gmax, diag, stride);
  return cudaGetLastError();
}

// =====================================================================================================
// Variant of reading R4 (opt.nonlocal_wkb1, off by default): the leading wave-optics correction of Eq. (1)
// PAPER.md:146, −(ε²/4) ∂i(I ∂iQ) with Q = ∇²√I/√I (Eq. (S15)), added to the ray-map prediction as the
// same LOCAL term ("when complemented by the second-order corrections"):
//   pred[b][s] −= f_s (α_s²/4) Σ_i D⁻_i( ½(Î[+1] + Î) D⁺_i Q ),  Î = A², A = 1 + Ad, Ad = expm1(−γ_s τ/2), Q = ∇²₅Ad / A.
// The paper finds the term "consistently negligible"; this is a plain tile kernel, not a tuned one.
// CTA = 32 x 8 pixels; Ad on the tile + 2, Q on the tile + 1, both in shared memory.
// =====================================================================================================
#define WK_TX 32
#define WK_TY 8
__global__ void __launch_bounds__(256) k_wkb1_sub(EprLines L, int nx, int ny, const float* __restrict__ tau,
                                                  float* __restrict__ pred) {
  __shared__ float s_ad[WK_TY + 4][WK_TX + 4], s_q[WK_TY + 2][WK_TX + 2];
  const int tid = threadIdx.x, b = blockIdx.z;
  const int x0 = blockIdx.x * WK_TX, y0 = blockIdx.y * WK_TY;
  const unsigned plane = (unsigned)nx * (unsigned)ny;
  const float* tb = tau + (size_t)b * plane;
  for (int s = 0; s < L.n_bins; ++s) {
    const float cg = -0.5f * L.gamma[s];
    __syncthreads();                                   // the previous line's tiles are no longer read
    for (int i = tid; i < (WK_TY + 4) * (WK_TX + 4); i += 256) {
      const int ly = i / (WK_TX + 4), lx = i - ly * (WK_TX + 4);
      s_ad[ly][lx] = epr_expm1(cg * __ldg(tb + (unsigned)wrapm(y0 - 2 + ly, ny) * nx + wrapm(x0 - 2 + lx, nx)));
    }
    __syncthreads();
    for (int i = tid; i < (WK_TY + 2) * (WK_TX + 2); i += 256) {
      const int ly = i / (WK_TX + 2), lx = i - ly * (WK_TX + 2);
      const float ac = s_ad[ly + 1][lx + 1];
      s_q[ly][lx] = __fdividef(((s_ad[ly + 1][lx + 2] - ac) + (s_ad[ly + 1][lx] - ac)) +
                               ((s_ad[ly][lx + 1] - ac) + (s_ad[ly + 2][lx + 1] - ac)), 1.f + ac);
    }
    __syncthreads();
    const int tx = tid & (WK_TX - 1), ty = tid / WK_TX;
    const int gx = x0 + tx, gy = y0 + ty;
    if (gx < nx && gy < ny) {
      auto I = [&](int dy, int dx) { const float a = 1.f + s_ad[ty + 2 + dy][tx + 2 + dx]; return a * a; };
      auto Q = [&](int dy, int dx) { return s_q[ty + 1 + dy][tx + 1 + dx]; };
      const float Ic = I(0, 0), Qc = Q(0, 0);
      const float fxp = 0.5f * (I(0, 1) + Ic) * (Q(0, 1) - Qc), fxm = 0.5f * (Ic + I(0, -1)) * (Qc - Q(0, -1));
      const float fyp = 0.5f * (I(1, 0) + Ic) * (Q(1, 0) - Qc), fym = 0.5f * (Ic + I(-1, 0)) * (Qc - Q(-1, 0));
      float* o = pred + ((size_t)b * L.n_bins + s) * plane + (unsigned)gy * nx + gx;
      *o -= L.f[s] * L.q4[s] * ((fxp - fxm) + (fyp - fym));
    }
  }
}

cudaError_t epr_launch_wkb1_sub(const epr_plan_s* p, int batch, const float* tau, float* pred, cudaStream_t st) {
  dim3 grid((p->nx + WK_TX - 1) / WK_TX, (p->ny + WK_TY - 1) / WK_TY, batch);
  k_wkb1_sub<<<grid, 256, 0, st>>>(p->lines, p->nx, p->ny, tau, pred);
  return cudaGetLastError();
}
