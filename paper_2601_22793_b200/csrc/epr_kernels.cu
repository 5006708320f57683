// epr_kernels.cu — stencil, splat, gather and pointwise kernels of the EPR iteration (sm_100a).
#include "epr_internal.h"
#include "epr_math.cuh"

// =====================================================================================================
// a1-L  local O(L²) closure, Eq. (1) PAPER.md:146 (readings R1-R3), in deviation form.
//   out: pred[b][s][y][x] = P_s − f_s
//   P_s/f_s − 1 = J − a ∇²₅J + (a²/2)[D²x(Î gx²) + D²y(Î gy²) + 2 D⁰xD⁰y(Î gx gy)] − (α²/4) Σ_i D⁻_i(Ī_i D⁺_i Q)
//   with A = exp(−γτ/2) = 1 + Ad,  Î = I/f = A²,  J = Î − 1 = Ad(2+Ad),  g = −γ D⁰τ,  Q = ∇²₅A / A.
// One CTA = 64x16 output pixels; τ and Ad staged in shared memory with a 2-pixel halo, g and Q with 1.
// =====================================================================================================
#define FL_TX 64
#define FL_TY 16
#define FL_SX (FL_TX + 4)
#define FL_SY (FL_TY + 4)

__global__ void __launch_bounds__(256) k_forward_local(EprLines L, int nx, int ny, int order, int wkb1,
                                                       const float* __restrict__ tau, float* __restrict__ pred) {
  __shared__ float s_tau[FL_SY][FL_SX], s_ad[FL_SY][FL_SX], s_gx[FL_SY][FL_SX], s_gy[FL_SY][FL_SX], s_q[FL_SY][FL_SX];
  const int b = blockIdx.z;
  const int x0 = blockIdx.x * FL_TX - 2, y0 = blockIdx.y * FL_TY - 2;
  const size_t plane = (size_t)nx * ny;
  const float* tb = tau + (size_t)b * plane;
  const int tid = threadIdx.x;

  for (int i = tid; i < FL_SX * FL_SY; i += 256) {
    const int ly = i / FL_SX, lx = i - ly * FL_SX;
    int gx_ = x0 + lx, gy_ = y0 + ly;
    gx_ = wrapm(gx_, nx);
    gy_ = wrapm(gy_, ny);
    s_tau[ly][lx] = __ldg(&tb[(size_t)gy_ * nx + gx_]);
  }
  for (int s = 0; s < L.n_bins; ++s) {
    const float gam = L.gamma[s];
    __syncthreads();
    for (int i = tid; i < FL_SX * FL_SY; i += 256) {
      const int ly = i / FL_SX, lx = i - ly * FL_SX;
      s_ad[ly][lx] = expm1f(-0.5f * gam * s_tau[ly][lx]);
    }
    __syncthreads();
    if (order == 2) {
      for (int i = tid; i < (FL_SX - 2) * (FL_SY - 2); i += 256) {
        const int ly = i / (FL_SX - 2) + 1, lx = i - (ly - 1) * (FL_SX - 2) + 1;
        s_gx[ly][lx] = -0.5f * gam * (s_tau[ly][lx + 1] - s_tau[ly][lx - 1]);
        s_gy[ly][lx] = -0.5f * gam * (s_tau[ly + 1][lx] - s_tau[ly - 1][lx]);
        const float c = s_ad[ly][lx];
        s_q[ly][lx] = ((s_ad[ly][lx + 1] - c) + (s_ad[ly][lx - 1] - c) + (s_ad[ly + 1][lx] - c) + (s_ad[ly - 1][lx] - c)) / (1.f + c);
      }
    }
    __syncthreads();
    float* out = pred + ((size_t)b * L.n_bins + s) * plane;
    for (int i = tid; i < FL_TX * FL_TY; i += 256) {
      const int ty = i / FL_TX, tx = i - ty * FL_TX;
      const int gxx = x0 + 2 + tx, gyy = y0 + 2 + ty;
      if (gxx >= nx || gyy >= ny) continue;
      const int ly = ty + 2, lx = tx + 2;
#define AD(dy, dx) s_ad[ly + (dy)][lx + (dx)]
#define IH(dy, dx) ((1.f + AD(dy, dx)) * (1.f + AD(dy, dx)))
#define JJ(dy, dx) (AD(dy, dx) * (2.f + AD(dy, dx)))
      const float Jc = JJ(0, 0);
      const float lapJ = (JJ(0, 1) - Jc) + (JJ(0, -1) - Jc) + (JJ(1, 0) - Jc) + (JJ(-1, 0) - Jc);
      float v = Jc - L.a[s] * lapJ;
      if (order == 2) {
#define GX(dy, dx) s_gx[ly + (dy)][lx + (dx)]
#define GY(dy, dx) s_gy[ly + (dy)][lx + (dx)]
#define QQ(dy, dx) s_q[ly + (dy)][lx + (dx)]
        const float Ic = IH(0, 0), Ixp = IH(0, 1), Ixm = IH(0, -1), Iyp = IH(1, 0), Iym = IH(-1, 0);
        const float sxx = Ixp * GX(0, 1) * GX(0, 1) - 2.f * Ic * GX(0, 0) * GX(0, 0) + Ixm * GX(0, -1) * GX(0, -1);
        const float syy = Iyp * GY(1, 0) * GY(1, 0) - 2.f * Ic * GY(0, 0) * GY(0, 0) + Iym * GY(-1, 0) * GY(-1, 0);
        const float sxy = 0.25f * (IH(1, 1) * GX(1, 1) * GY(1, 1) - IH(1, -1) * GX(1, -1) * GY(1, -1)
                                   - IH(-1, 1) * GX(-1, 1) * GY(-1, 1) + IH(-1, -1) * GX(-1, -1) * GY(-1, -1));
        v = fmaf(L.a2h[s], sxx + syy + 2.f * sxy, v);
        if (wkb1) {
          const float Qc = QQ(0, 0);
          const float div = 0.5f * ((Ixp + Ic) * (QQ(0, 1) - Qc) - (Ic + Ixm) * (Qc - QQ(0, -1))
                                    + (Iyp + Ic) * (QQ(1, 0) - Qc) - (Ic + Iym) * (Qc - QQ(-1, 0)));
          v = fmaf(-L.q4[s], div, v);
        }
      }
      out[(size_t)gyy * nx + gxx] = L.f[s] * v;
    }
  }
}

cudaError_t epr_launch_forward_local(const epr_plan_s* p, int batch, const float* tau, float* pred, cudaStream_t st) {
  dim3 grid((p->nx + FL_TX - 1) / FL_TX, (p->ny + FL_TY - 1) / FL_TY, batch);
  k_forward_local<<<grid, 256, 0, st>>>(p->lines, p->nx, p->ny, p->opt.order, p->opt.wkb1, tau, pred);
  return cudaGetLastError();
}

// =====================================================================================================
// a1-N  ray map (Eq. (2), clamp R6) + mass-conserving bilinear splat.
//   One CTA = 64x32 source pixels.  The 4-way scatter is resolved with NATIVE u32 shared-memory atomics on a
//   fixed-point (2^-26) accumulator tile that covers the source tile plus the halo actually reached by this
//   tile's rays (h = 1 + max |floor u|, found by a block reduction), then flushed once to the global
//   fixed-point plane with RED.ADD.  Integer accumulation makes the result independent of the order of the
//   atomics (deterministic) and conserves mass exactly: the 4th corner gets rint(I·2^26) minus the other three.
//   Sources: I_s = f_s(1+J) from τ (I_bins == NULL) or an arbitrary plane (epr_transport);
//            u from τ (map_in == NULL; optionally written to map_out) or from a stored map.
// =====================================================================================================
#define SP_TX 64
#define SP_TY 32
#define SP_PX ((SP_TX * SP_TY) / 256)

__global__ void __launch_bounds__(256) k_splat(EprLines L, int nx, int ny, float S, int hmax,
                                               const float* __restrict__ tau, const float* __restrict__ I_bins,
                                               const float2* __restrict__ map_in, float2* __restrict__ map_out,
                                               unsigned* __restrict__ pfix) {
  extern __shared__ unsigned s_acc[];                 // (SP_TY + 2 hmax) x (SP_TX + 2 hmax)
  __shared__ float s_tau[SP_TY + 2][SP_TX + 2];
  __shared__ int s_h;
  const int b = blockIdx.z, tid = threadIdx.x;
  const int x0 = blockIdx.x * SP_TX, y0 = blockIdx.y * SP_TY;
  const size_t plane = (size_t)nx * ny;
  const int aw = SP_TX + 2 * hmax;

  if (tau) {
    const float* tb = tau + (size_t)b * plane;
    for (int i = tid; i < (SP_TX + 2) * (SP_TY + 2); i += 256) {
      const int ly = i / (SP_TX + 2), lx = i - ly * (SP_TX + 2);
      s_tau[ly][lx] = __ldg(&tb[(size_t)wrapm(y0 - 1 + ly, ny) * nx + wrapm(x0 - 1 + lx, nx)]);
    }
  }
  for (int s = 0; s < L.n_bins; ++s) {
    const size_t pl = ((size_t)b * L.n_bins + s) * plane;
    if (tid == 0) s_h = 0;
    __syncthreads();                                   // also orders the previous bin's flush before re-zeroing
    float ux[SP_PX], uy[SP_PX];
    int hloc = 0;
#pragma unroll
    for (int k = 0; k < SP_PX; ++k) {
      const int i = tid + k * 256, ty = i / SP_TX, tx = i - ty * SP_TX;
      const int gx = x0 + tx, gy = y0 + ty;
      ux[k] = uy[k] = 0.f;
      if (gx < nx && gy < ny) {
        if (map_in) {
          const float2 m = __ldg(&map_in[pl + (size_t)gy * nx + gx]);
          ux[k] = m.x; uy[k] = m.y;
        } else {
          // u = a D⁰ ln I_s = −a γ D⁰τ, clamped to ±S
          const float c = -0.5f * L.a[s] * L.gamma[s];
          ux[k] = fminf(fmaxf(c * (s_tau[ty + 1][tx + 2] - s_tau[ty + 1][tx]), -S), S);
          uy[k] = fminf(fmaxf(c * (s_tau[ty + 2][tx + 1] - s_tau[ty][tx + 1]), -S), S);
          if (map_out) map_out[pl + (size_t)gy * nx + gx] = make_float2(ux[k], uy[k]);
        }
        const int fx = (int)floorf(ux[k]), fy = (int)floorf(uy[k]);
        hloc = max(hloc, max(max(-fx, fx + 1), max(-fy, fy + 1)));
      }
    }
    atomicMax(&s_h, hloc);
    __syncthreads();
    const int h = min(s_h, hmax);
    const int rw = SP_TX + 2 * h, rh = SP_TY + 2 * h;
    for (int i = tid; i < rw * rh; i += 256) { const int ry = i / rw; s_acc[ry * aw + (i - ry * rw)] = 0u; }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < SP_PX; ++k) {
      const int i = tid + k * 256, ty = i / SP_TX, tx = i - ty * SP_TX;
      const int gx = x0 + tx, gy = y0 + ty;
      if (gx < nx && gy < ny) {
        const float fxf = floorf(ux[k]), fyf = floorf(uy[k]);
        const double dx = (double)(ux[k] - fxf), dy = (double)(uy[k] - fyf);
        double Id;                                     // source mass in fixed-point units
        if (I_bins) Id = (double)__ldg(&I_bins[pl + (size_t)gy * nx + gx]) * EPR_FIX_ONE;
        else Id = L.fixF[s] * (1.0 + (double)expm1f(-L.gamma[s] * s_tau[ty + 1][tx + 1]));
        const long long tot = __double2ll_rn(Id);
        const long long c00 = __double2ll_rn(Id * (1.0 - dx) * (1.0 - dy));
        const long long c10 = __double2ll_rn(Id * dx * (1.0 - dy));
        const long long c01 = __double2ll_rn(Id * (1.0 - dx) * dy);
        const long long c11 = tot - c00 - c10 - c01;
        const int ax = tx + h + (int)fxf, ay = ty + h + (int)fyf;
        unsigned* a0 = &s_acc[ay * aw + ax];
        atomicAdd(a0, (unsigned)c00);
        atomicAdd(a0 + 1, (unsigned)c10);
        atomicAdd(a0 + aw, (unsigned)c01);
        atomicAdd(a0 + aw + 1, (unsigned)c11);
      }
    }
    __syncthreads();
    unsigned* pb = pfix + pl;
    for (int i = tid; i < rw * rh; i += 256) {
      const int ry = i / rw, rx = i - ry * rw;
      const unsigned v = s_acc[ry * aw + rx];
      if (v) atomicAdd(&pb[(size_t)wrapm(y0 - h + ry, ny) * nx + wrapm(x0 - h + rx, nx)], v);
    }
  }
}

cudaError_t epr_launch_splat(const epr_plan_s* p, int batch, const float* tau, const float* I_bins, const float2* map_in,
                             float2* map_out, unsigned* pfix, cudaStream_t st) {
  const int hmax = (int)ceilf(p->opt.max_shift_px) + 1;
  const size_t smem = (size_t)(SP_TX + 2 * hmax) * (SP_TY + 2 * hmax) * sizeof(unsigned);
  static bool attr_set = false;
  if (!attr_set) {
    cudaFuncSetAttribute(k_splat, cudaFuncAttributeMaxDynamicSharedMemorySize, 160 * 1024);
    attr_set = true;
  }
  dim3 grid((p->nx + SP_TX - 1) / SP_TX, (p->ny + SP_TY - 1) / SP_TY, batch);
  k_splat<<<grid, 256, smem, st>>>(p->lines, p->nx, p->ny, p->opt.max_shift_px, hmax, tau, I_bins, map_in, map_out, pfix);
  return cudaGetLastError();
}

// =====================================================================================================
// a2  detector residual and positivity-weighted split (reading R8), deviation form:
//   e = (d − 1) − Σ_s (P_s − f_s);   w_s = P_s⁺ / Σ_t P_t⁺ (fallback f_s);   es_s = w_s e
//   pred is either float P_s − f_s (local) or the u32 fixed-point splat plane (non-local).
// =====================================================================================================
__device__ __forceinline__ float pred_dev(const void* pred, size_t idx, int fixed, const EprLines& L, int s) {
  if (fixed) {
    const unsigned v = __ldg(&((const unsigned*)pred)[idx]);
    return (float)(int)(v - L.fixFi[s]) * (1.0f / (float)EPR_FIX_ONE) + L.fixCorr[s];
  }
  return __ldg(&((const float*)pred)[idx]);
}

__global__ void __launch_bounds__(256) k_residual(EprLines L, size_t plane, const float* __restrict__ d,
                                                  const void* __restrict__ pred, int fixed, float* __restrict__ es) {
  const size_t i = (size_t)blockIdx.x * 256 + threadIdx.x;
  const int b = blockIdx.y;
  if (i >= plane) return;
  const size_t base = (size_t)b * L.n_bins * plane + i;
  float sum = 0.f, den = 0.f;
  for (int s = 0; s < L.n_bins; ++s) {
    const float pd = pred_dev(pred, base + s * plane, fixed, L, s);
    sum += pd;
    den += fmaxf(L.f[s] + pd, 0.f);
  }
  const float e = (__ldg(&d[(size_t)b * plane + i]) - 1.f) - sum - L.fsum_dev;
  for (int s = 0; s < L.n_bins; ++s) {
    const float pd = pred_dev(pred, base + s * plane, fixed, L, s);
    const float w = den > 0.f ? fmaxf(L.f[s] + pd, 0.f) / den : L.f[s];
    es[base + s * plane] = w * e;
  }
}

cudaError_t epr_launch_residual(const epr_plan_s* p, int batch, const float* d, const void* pred, int fixed,
                                float* es, cudaStream_t st) {
  const size_t plane = (size_t)p->nx * p->ny;
  dim3 grid((unsigned)((plane + 255) / 256), batch);
  k_residual<<<grid, 256, 0, st>>>(p->lines, plane, d, pred, fixed, es);
  return cudaGetLastError();
}

// epr_forward / epr_transport output: P_s = f_s + (P_s − f_s) (linear = 1: plain fixed-point value), P = Σ_s P_s.
__global__ void __launch_bounds__(256) k_pred_out(EprLines L, size_t plane, const void* __restrict__ pred, int fixed,
                                                  int linear, float* __restrict__ P_sum, float* __restrict__ P_bins) {
  const size_t i = (size_t)blockIdx.x * 256 + threadIdx.x;
  const int b = blockIdx.y;
  if (i >= plane) return;
  const size_t base = (size_t)b * L.n_bins * plane + i;
  float sum = 0.f;
  for (int s = 0; s < L.n_bins; ++s) {
    float v;
    if (linear) v = (float)(int)__ldg(&((const unsigned*)pred)[base + s * plane]) * (1.0f / (float)EPR_FIX_ONE);
    else v = L.f[s] + pred_dev(pred, base + s * plane, fixed, L, s);
    sum += v;
    if (P_bins) P_bins[base + s * plane] = v;
  }
  if (P_sum) P_sum[(size_t)b * plane + i] = sum;
}

cudaError_t epr_launch_pred_out(const epr_plan_s* p, int batch, const void* pred, int fixed, int linear, float* P_sum,
                                float* P_bins, cudaStream_t st) {
  const size_t plane = (size_t)p->nx * p->ny;
  dim3 grid((unsigned)((plane + 255) / 256), batch);
  k_pred_out<<<grid, 256, 0, st>>>(p->lines, plane, pred, fixed, linear, P_sum, P_bins);
  return cudaGetLastError();
}

// =====================================================================================================
// a3  adjoint ℳ*_s: bilinear gather at the mapped coordinates, Eq. (4), with the SAME
//     x0, y0, w as the splat of this iteration (ray map recomputed from τ, or the stored one).
// =====================================================================================================
__global__ void __launch_bounds__(256) k_gather(EprLines L, int nx, int ny, float S, const float* __restrict__ tau,
                                                const float2* __restrict__ map_in, const float* __restrict__ es,
                                                float* __restrict__ r) {
  const int x = blockIdx.x * 64 + (threadIdx.x & 63), y = blockIdx.y * 4 + (threadIdx.x >> 6);
  const int b = blockIdx.z;
  if (x >= nx || y >= ny) return;
  const size_t plane = (size_t)nx * ny;
  const int xm = wrap1(x - 1, nx), xp = wrap1(x + 1, nx), ym = wrap1(y - 1, ny), yp = wrap1(y + 1, ny);
  float dtx = 0.f, dty = 0.f;
  if (!map_in) {
    const float* tb = tau + (size_t)b * plane;
    dtx = __ldg(&tb[(size_t)y * nx + xp]) - __ldg(&tb[(size_t)y * nx + xm]);
    dty = __ldg(&tb[(size_t)yp * nx + x]) - __ldg(&tb[(size_t)ym * nx + x]);
  }
  for (int s = 0; s < L.n_bins; ++s) {
    const size_t pl = ((size_t)b * L.n_bins + s) * plane;
    float ux, uy;
    if (map_in) {
      const float2 m = __ldg(&map_in[pl + (size_t)y * nx + x]);
      ux = m.x; uy = m.y;
    } else {
      const float c = -0.5f * L.a[s] * L.gamma[s];
      ux = fminf(fmaxf(c * dtx, -S), S);
      uy = fminf(fmaxf(c * dty, -S), S);
    }
    const float fx = floorf(ux), fy = floorf(uy);
    const float dx = ux - fx, dy = uy - fy;
    const int ix0 = wrapm(x + (int)fx, nx), iy0 = wrapm(y + (int)fy, ny);
    const int ix1 = wrap1(ix0 + 1, nx), iy1 = wrap1(iy0 + 1, ny);
    const float* eb = es + pl;
    const float e00 = __ldg(&eb[(size_t)iy0 * nx + ix0]), e10 = __ldg(&eb[(size_t)iy0 * nx + ix1]);
    const float e01 = __ldg(&eb[(size_t)iy1 * nx + ix0]), e11 = __ldg(&eb[(size_t)iy1 * nx + ix1]);
    r[pl + (size_t)y * nx + x] = (1.f - dx) * (1.f - dy) * e00 + dx * (1.f - dy) * e10 + (1.f - dx) * dy * e01 + dx * dy * e11;
  }
}

cudaError_t epr_launch_gather(const epr_plan_s* p, int batch, const float* tau, const float2* map_in, const float* es,
                              float* r, cudaStream_t st) {
  dim3 grid((p->nx + 63) / 64, (p->ny + 3) / 4, batch);
  k_gather<<<grid, 256, 0, st>>>(p->lines, p->nx, p->ny, p->opt.max_shift_px, tau, map_in, es, r);
  return cudaGetLastError();
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

cudaError_t epr_launch_zero(void* ptr, size_t bytes, cudaStream_t st) { return cudaMemsetAsync(ptr, 0, bytes, st); }
