// epr_general.cu — the GENERAL path of the EPR iteration (sm_100a): the same steps a0 … a6 as epr_kernels.cu, with
//   * every per-line scalar read per COLUMN from small device tables — the x-dependent effective spectrum
//     f_s(x), γ_s(x), db_s(x) of PAPER.md:216-221 (Eq. (6) + remark), 227-229 (Eq. (7)), 431-441 (§9.2), reading R17:
//     the scalars are frozen at the pixel's own column (no derivative of a profile is ever taken) and the
//     FFT-diagonal filter is applied per block and blended (epr_api.cu);
//   * no alignment requirement on the grid: any nx, ny >= 8 (one pixel per thread, scalar accesses), so that it also
//     serves {2,3,5}-smooth grids the tuned kernels do not take (nx % 4 != 0, ny % 16 != 0, …).
// The tuned kernels of epr_kernels.cu remain the path of the uniform spectrum on aligned grids; these kernels favour
// plain structure over the last factor of two (they are bound by instruction issue at about 3x the tuned cost).
// Arithmetic is the same deviation form: state τ, J = expm1(−γτ), data d − 1, predictions P_s − f_s(x),
// splat in u32 fixed point with the exact-remainder corner.
#include "epr_internal.h"
#include "epr_math.cuh"

#define GN_TX 32
#define GN_TY 16
// pointwise kernels: one thread = one pixel; x = blockIdx.x·256 + threadIdx.x, y = blockIdx.y, projection (or plane) = blockIdx.z
// — the column (for the per-column tables) comes without a division
#define GN_PIX(nx)                                                              \
  const int x = blockIdx.x * 256 + threadIdx.x;                                 \
  if (x >= (nx)) return;                                                        \
  const size_t i = (size_t)blockIdx.y * (nx) + x;
static inline dim3 gn_grid(const epr_plan_s* p, int nz) { return dim3((p->nx + 255) / 256, p->ny, nz); }

// =====================================================================================================
// a1-L  local O(L²) closure, Eq. (1) PAPER.md:146 (readings R1-R3), scalars of the CENTRE column (R17(b)):
//   P_s/f_s − 1 = J − a ∇²₅J + (a²/2)[D²x(Î gx²) + D²y(Î gy²) + 2 D⁰xD⁰y(Î gx gy)] − (α²/4) Σ_i D⁻_i(Ī_i D⁺_i Q)
//   A = exp(−γτ/2) = 1 + Ad, Î = A², J = Ad(2 + Ad), g = −γ D⁰τ, Q = ∇²₅A / A; neighbour values formed with the centre's γ.
// One thread = one pixel, every line; τ tile + 2 in shared memory.
// =====================================================================================================
// term_only (variant of reading R4, opt.nonlocal_wkb1): pred −= f_s(x)(α²/4) Σ_i D⁻_i(Ī_i D⁺_i Q) alone — the WKB1 term
// added to the ray-map prediction as the same LOCAL term ("when complemented by the second-order corrections").
__global__ void __launch_bounds__(GN_TX * GN_TY) k_gen_local(EprLines L, EprColumns C, int nx, int ny, int order, int wkb1,
                                                            int term_only, const float* __restrict__ tau, float* pred) {
  __shared__ float s_t[GN_TY + 4][GN_TX + 4];
  const int tid = threadIdx.y * GN_TX + threadIdx.x, b = blockIdx.z;
  const int x0 = blockIdx.x * GN_TX, y0 = blockIdx.y * GN_TY;
  const size_t plane = (size_t)nx * ny;
  const float* tb = tau + (size_t)b * plane;
  // (the periodic wrap by one conditional add where the grid is larger than a tile + halo: the integer modulo of the general
  // case was a quarter of the kernel's instructions and half of its stall samples)
  const bool big = nx >= GN_TX + 4 && ny >= GN_TY + 4;
  for (int i = tid; i < (GN_TY + 4) * (GN_TX + 4); i += GN_TX * GN_TY) {
    const int ly = i / (GN_TX + 4), lx = i - ly * (GN_TX + 4);
    const int gy = big ? wrap1(y0 - 2 + ly, ny) : wrapm(y0 - 2 + ly, ny), gx = big ? wrap1(x0 - 2 + lx, nx) : wrapm(x0 - 2 + lx, nx);
    s_t[ly][lx] = __ldg(tb + (size_t)gy * nx + gx);
  }
  __syncthreads();
  const int x = x0 + threadIdx.x, y = y0 + threadIdx.y;
  if (x >= nx || y >= ny) return;
  // τ on the 5 x 5 neighbourhood (corners unused)
  float t[5][5];
#pragma unroll
  for (int j = 0; j < 5; ++j)
#pragma unroll
    for (int i = 0; i < 5; ++i) t[j][i] = s_t[threadIdx.y + j][threadIdx.x + i];
  const bool o2 = order == 2, wk = o2 && wkb1;
  float tmax = 0.f;                                    // largest |τ| of the diamond: picks the series of expm1 per warp and line
#pragma unroll
  for (int j = 0; j < 5; ++j)
#pragma unroll
    for (int i = 0; i < 5; ++i)
      if (abs(i - 2) + abs(j - 2) <= 2) tmax = fmaxf(tmax, fabsf(t[j][i]));
  for (int s = 0; s < L.n_bins; ++s) {
    const float gam = __ldg(&C.gamma[(size_t)s * nx + x]), a = __ldg(&C.a[(size_t)s * nx + x]), fs = __ldg(&C.f[(size_t)s * nx + x]);
    const float cg = -0.5f * gam, c2 = 0.5f * a * a * cg * cg, q4 = L.q4[s];
    // Ad on the 13-point diamond |dx| + |dy| <= 2 (index [dy + 2][dx + 2]): every neighbour seen through THIS column's γ, so
    // nothing can be shared with the neighbouring threads; the series is as short as the warp's largest argument allows
    float A[5][5];
    const float amax = fabsf(cg) * tmax;
    const int tier = __any_sync(__activemask(), amax >= 0.35f) ? 2 : (__any_sync(__activemask(), amax >= 0.09f) ? 1 : 0);
    auto fill = [&](auto fn) {
#pragma unroll
      for (int j = 0; j < 5; ++j)
#pragma unroll
        for (int i = 0; i < 5; ++i) A[j][i] = (abs(i - 2) + abs(j - 2) <= 2) ? fn(cg * t[j][i]) : 0.f;
    };
    if (tier == 0) fill([](float v) { return epr_expm1_tiny(v); });
    else if (tier == 1) fill([](float v) { return epr_expm1_small(v); });
    else fill([](float v) { return epr_expm1(v); });
    auto J = [&](int dy, int dx) { const float v = A[dy + 2][dx + 2]; return v * (2.f + v); };
    auto Ih = [&](int dy, int dx) { const float v = 1.f + A[dy + 2][dx + 2]; return v * v; };
    const float J0 = J(0, 0);
    float v = term_only ? 0.f : J0 - a * (((J(0, 1) - J0) + (J(0, -1) - J0)) + ((J(1, 0) - J0) + (J(-1, 0) - J0)));
    if (o2 && !term_only) {
      auto tx = [&](int dy, int dx) { return t[dy + 2][dx + 3] - t[dy + 2][dx + 1]; };
      auto ty = [&](int dy, int dx) { return t[dy + 3][dx + 2] - t[dy + 1][dx + 2]; };
      auto Sxx = [&](int dx) { const float g = tx(0, dx); return Ih(0, dx) * g * g; };
      auto Syy = [&](int dy) { const float g = ty(dy, 0); return Ih(dy, 0) * g * g; };
      auto Sxy = [&](int dy, int dx) { return Ih(dy, dx) * tx(dy, dx) * ty(dy, dx); };
      const float sx0 = Sxx(0), sy0 = Syy(0);
      const float d2x = (Sxx(1) - sx0) - (sx0 - Sxx(-1)), d2y = (Syy(1) - sy0) - (sy0 - Syy(-1));
      const float cross = 0.5f * ((Sxy(1, 1) - Sxy(1, -1)) - (Sxy(-1, 1) - Sxy(-1, -1)));
      v = fmaf(c2, d2x + d2y + cross, v);
    }
    if (wk) {
      auto Q = [&](int dy, int dx) {
        const float ac = A[dy + 2][dx + 2];
        return __fdividef(((A[dy + 2][dx + 3] - ac) + (A[dy + 2][dx + 1] - ac)) + ((A[dy + 3][dx + 2] - ac) + (A[dy + 1][dx + 2] - ac)), 1.f + ac);
      };
      const float Q0 = Q(0, 0), I0 = Ih(0, 0);
      const float fxp = 0.5f * (Ih(0, 1) + I0) * (Q(0, 1) - Q0), fxm = 0.5f * (I0 + Ih(0, -1)) * (Q0 - Q(0, -1));
      const float fyp = 0.5f * (Ih(1, 0) + I0) * (Q(1, 0) - Q0), fym = 0.5f * (I0 + Ih(-1, 0)) * (Q0 - Q(-1, 0));
      v = fmaf(-q4, (fxp - fxm) + (fyp - fym), v);
    }
    float* o = pred + ((size_t)b * L.n_bins + s) * plane + (size_t)y * nx + x;
    *o = term_only ? fmaf(fs, v, *o) : fs * v;
  }
}

cudaError_t epr_gen_forward_local(const epr_plan_s* p, int batch, const float* tau, float* pred, cudaStream_t st) {
  dim3 grid((p->nx + GN_TX - 1) / GN_TX, (p->ny + GN_TY - 1) / GN_TY, batch), blk(GN_TX, GN_TY);
  k_gen_local<<<grid, blk, 0, st>>>(p->lines, p->cols, p->nx, p->ny, p->opt.order, p->opt.wkb1, 0, tau, pred);
  return cudaGetLastError();
}

cudaError_t epr_gen_wkb1_sub(const epr_plan_s* p, int batch, const float* tau, float* pred, cudaStream_t st) {
  dim3 grid((p->nx + GN_TX - 1) / GN_TX, (p->ny + GN_TY - 1) / GN_TY, batch), blk(GN_TX, GN_TY);
  k_gen_local<<<grid, blk, 0, st>>>(p->lines, p->cols, p->nx, p->ny, 2, 1, 1, tau, pred);
  return cudaGetLastError();
}

// =====================================================================================================
// a1-N  ray map (Eq. (2), clamp R6) + mass-conserving bilinear splat, scalars of
// the SOURCE's column (R17(b)).  One thread = one source pixel, every line; the 4-way scatter goes to a u32 fixed-point
// plane in global memory (unit 2^-26, zero-initialised by the launcher) with native integer atomics: order-independent
// (bit-reproducible) and exactly mass conserving — the 4th corner takes the integer remainder, as in k_splat_tile.
// =====================================================================================================
template <bool FROM_TAU>
__global__ void __launch_bounds__(256) k_gen_splat(EprLines L, EprColumns C, int nx, int ny, float S,
                                                   const float* __restrict__ tau, const float* __restrict__ I_bins,
                                                   const float2* __restrict__ map_in, float2* __restrict__ map_out,
                                                   unsigned* __restrict__ acc) {
  const int x = blockIdx.x * 64 + (threadIdx.x & 63), y = blockIdx.y * 4 + (threadIdx.x >> 6), b = blockIdx.z;
  if (x >= nx || y >= ny) return;
  const size_t plane = (size_t)nx * ny, pix = (size_t)y * nx + x;
  float tc = 0.f, dtx = 0.f, dty = 0.f;
  if (FROM_TAU) {
    const float* tb = tau + (size_t)b * plane;
    const int xm = x == 0 ? nx - 1 : x - 1, xp = x + 1 == nx ? 0 : x + 1;
    const int ym = y == 0 ? ny - 1 : y - 1, yp = y + 1 == ny ? 0 : y + 1;
    tc = __ldg(tb + pix);
    dtx = __ldg(tb + (size_t)y * nx + xp) - __ldg(tb + (size_t)y * nx + xm);
    dty = __ldg(tb + (size_t)yp * nx + x) - __ldg(tb + (size_t)ym * nx + x);
  }
  for (int s = 0; s < L.n_bins; ++s) {
    const size_t pl = ((size_t)b * L.n_bins + s) * plane;
    float ux, uy;
    int tot;
    if (FROM_TAU) {
      const float gam = __ldg(&C.gamma[(size_t)s * nx + x]), a = __ldg(&C.a[(size_t)s * nx + x]), fs = __ldg(&C.f[(size_t)s * nx + x]);
      const float cs = -0.5f * a * gam;                 // u = a D⁰ ln I_s = −a γ D⁰τ
      ux = fminf(fmaxf(cs * dtx, -S), S);
      uy = fminf(fmaxf(cs * dty, -S), S);
      if (map_out) map_out[pl + pix] = make_float2(ux, uy);
      const float xe = -gam * tc;
      const float J = fabsf(xe) < 0.35f ? epr_expm1_small(xe) : epr_exp_fast(xe) - 1.f;
      tot = (int)__ldg(&C.fixFi[(size_t)s * nx + x]) + __float2int_rn(fs * 67108864.f * J);
    } else {
      const float2 m = __ldg(&map_in[pl + pix]);
      ux = m.x; uy = m.y;
      tot = __float2int_rn(__ldg(&I_bins[pl + pix]) * 67108864.f);
    }
    const int fx = __float2int_rd(ux), fy = __float2int_rd(uy);
    const float dx = ux - (float)fx, dy = uy - (float)fy;
    const float totf = (float)tot, te = totf * (1.f - dy), td = totf * dy, ex = 1.f - dx;
    const int c00 = __float2int_rn(te * ex), c10 = __float2int_rn(te * dx), c01 = __float2int_rn(td * ex);
    const int c11 = tot - c00 - c10 - c01;
    const int ix0 = wrapm(x + fx, nx), iy0 = wrapm(y + fy, ny);
    const int ix1 = ix0 + 1 == nx ? 0 : ix0 + 1, iy1 = iy0 + 1 == ny ? 0 : iy0 + 1;
    unsigned* ap = acc + pl;
    atomicAdd(ap + (size_t)iy0 * nx + ix0, (unsigned)c00);
    atomicAdd(ap + (size_t)iy0 * nx + ix1, (unsigned)c10);
    atomicAdd(ap + (size_t)iy1 * nx + ix0, (unsigned)c01);
    atomicAdd(ap + (size_t)iy1 * nx + ix1, (unsigned)c11);
  }
}

cudaError_t epr_gen_splat(const epr_plan_s* p, int batch, const float* tau, const float* I_bins, const float2* map_in,
                          float2* map_out, unsigned* acc, cudaStream_t st) {
  const size_t n = (size_t)batch * p->n_bins * p->nx * p->ny;
  cudaError_t e = cudaMemsetAsync(acc, 0, n * sizeof(unsigned), st);
  if (e != cudaSuccess) return e;
  dim3 grid((p->nx + 63) / 64, (p->ny + 3) / 4, batch);
  if (tau) k_gen_splat<true><<<grid, 256, 0, st>>>(p->lines, p->cols, p->nx, p->ny, p->opt.max_shift_px, tau, nullptr, nullptr, map_out, acc);
  else k_gen_splat<false><<<grid, 256, 0, st>>>(p->lines, p->cols, p->nx, p->ny, p->opt.max_shift_px, nullptr, I_bins, map_in, nullptr, acc);
  return cudaGetLastError();
}

// fixed point -> float in place.  mode 0: P_s − f_s(x) of the detector pixel's column (an EMPTY pixel is written as exactly
// −f_s(x), so that P_s = 0 exactly downstream: the split's fallback decision, R8); mode 1: P_s (epr_transport, signed).
__global__ void __launch_bounds__(256) k_gen_fix2float(int n_bins, EprColumns C, int nx, size_t plane, int mode,
                                                       unsigned* __restrict__ acc, unsigned* __restrict__ flags) {
  GN_PIX(nx)
  const float sc = 1.0f / (float)EPR_FIX_ONE;
  for (int s = 0; s < n_bins; ++s) {
    unsigned* ap = acc + ((size_t)blockIdx.z * n_bins + s) * plane + i;
    const unsigned v = *ap;
    float o;
    if (mode == 1) {
      o = (float)(int)v * sc;
    } else {
      if ((v + 1024u) & 0x80000000u) atomicOr(flags, EPR_FLAG_SPLAT_OVERFLOW);
      const int Fi = (int)__ldg(&C.fixFi[(size_t)s * nx + x]);
      o = v ? fmaf((float)((int)v - Fi), sc, __ldg(&C.fixCorr[(size_t)s * nx + x])) : -__ldg(&C.f[(size_t)s * nx + x]);
    }
    *reinterpret_cast<float*>(ap) = o;
  }
}

cudaError_t epr_gen_fix2float(const epr_plan_s* p, int batch, unsigned* acc, int mode, cudaStream_t st) {
  const size_t plane = (size_t)p->nx * p->ny;
  k_gen_fix2float<<<gn_grid(p, batch), 256, 0, st>>>(p->n_bins, p->cols, p->nx, plane, mode, acc, p->d_flags);
  return cudaGetLastError();
}

// =====================================================================================================
// a2  residual and positivity-weighted split (R8) with the column's f_s(x):
//   e = (d − 1) − Σ_s (P_s − f_s) − (Σ_s (float)f_s(x) − 1);  w_s = P_s⁺/Σ_t P_t⁺ (fallback f_s(x));  es_s = w_s e.  pred may alias es.
// =====================================================================================================
__global__ void __launch_bounds__(256) k_gen_residual(int n_bins, EprColumns C, int nx, size_t plane, const float* __restrict__ d,
                                                      const float* pred, float* es) {
  GN_PIX(nx)
  const int b = blockIdx.z;
  const size_t base = (size_t)b * n_bins * plane + i;
  float sum = 0.f, den = 0.f;
  for (int s = 0; s < n_bins; ++s) {                    // two passes over the lines (the second hits L1/L2): no per-thread array
    const float pd = pred[base + (size_t)s * plane];
    sum += pd;
    den += fmaxf(__ldg(&C.f[(size_t)s * nx + x]) + pd, 0.f);           // P_s⁺
  }
  const float e = (__ldg(&d[(size_t)b * plane + i]) - (1.f + __ldg(&C.fsum_dev[x]))) - sum;
  const float q = den > 0.f ? e / den : 0.f;
  for (int s = 0; s < n_bins; ++s) {
    const float f = __ldg(&C.f[(size_t)s * nx + x]);
    const float pp = fmaxf(f + pred[base + (size_t)s * plane], 0.f);
    es[base + (size_t)s * plane] = den > 0.f ? pp * q : f * e;
  }
}

// the same for four consecutive pixels per thread (nx % 4 == 0): 16-byte accesses
__global__ void __launch_bounds__(256) k_gen_residual4(int n_bins, EprColumns C, int nx, size_t plane, const float* __restrict__ d,
                                                       const float* pred, float* es) {
  const int x = 4 * (blockIdx.x * 256 + threadIdx.x);
  if (x >= nx) return;
  const size_t i = (size_t)blockIdx.y * nx + x;
  const int b = blockIdx.z;
  const size_t base = (size_t)b * n_bins * plane + i;
  float4 sum = make_float4(0.f, 0.f, 0.f, 0.f), den = sum;
  for (int s = 0; s < n_bins; ++s) {
    const float4 pd = *reinterpret_cast<const float4*>(pred + base + (size_t)s * plane);
    const float4 f = __ldg(reinterpret_cast<const float4*>(C.f + (size_t)s * nx + x));
    sum.x += pd.x; sum.y += pd.y; sum.z += pd.z; sum.w += pd.w;
    den.x += fmaxf(f.x + pd.x, 0.f); den.y += fmaxf(f.y + pd.y, 0.f); den.z += fmaxf(f.z + pd.z, 0.f); den.w += fmaxf(f.w + pd.w, 0.f);
  }
  const float4 dd = __ldg(reinterpret_cast<const float4*>(d + (size_t)b * plane + i));
  const float4 fd = __ldg(reinterpret_cast<const float4*>(C.fsum_dev + x));
  const float4 e = make_float4((dd.x - (1.f + fd.x)) - sum.x, (dd.y - (1.f + fd.y)) - sum.y, (dd.z - (1.f + fd.z)) - sum.z, (dd.w - (1.f + fd.w)) - sum.w);
  const float4 q = make_float4(den.x > 0.f ? e.x / den.x : 0.f, den.y > 0.f ? e.y / den.y : 0.f, den.z > 0.f ? e.z / den.z : 0.f, den.w > 0.f ? e.w / den.w : 0.f);
  for (int s = 0; s < n_bins; ++s) {
    const float4 pd = *reinterpret_cast<const float4*>(pred + base + (size_t)s * plane);
    const float4 f = __ldg(reinterpret_cast<const float4*>(C.f + (size_t)s * nx + x));
    float4 o;
    o.x = den.x > 0.f ? fmaxf(f.x + pd.x, 0.f) * q.x : f.x * e.x;
    o.y = den.y > 0.f ? fmaxf(f.y + pd.y, 0.f) * q.y : f.y * e.y;
    o.z = den.z > 0.f ? fmaxf(f.z + pd.z, 0.f) * q.z : f.z * e.z;
    o.w = den.w > 0.f ? fmaxf(f.w + pd.w, 0.f) * q.w : f.w * e.w;
    *reinterpret_cast<float4*>(es + base + (size_t)s * plane) = o;
  }
}

cudaError_t epr_gen_residual(const epr_plan_s* p, int batch, const float* d, const float* pred, float* es, cudaStream_t st) {
  const size_t plane = (size_t)p->nx * p->ny;
  if (p->nx % 4 == 0)
    k_gen_residual4<<<dim3((p->nx / 4 + 255) / 256, p->ny, batch), 256, 0, st>>>(p->n_bins, p->cols, p->nx, plane, d, pred, es);
  else
    k_gen_residual<<<gn_grid(p, batch), 256, 0, st>>>(p->n_bins, p->cols, p->nx, plane, d, pred, es);
  return cudaGetLastError();
}

// =====================================================================================================
// a3  adjoint gather, Eq. (4), with the SAME x0, y0, w as the splat: the map of the pixel's own column.
// =====================================================================================================
__global__ void __launch_bounds__(256) k_gen_gather(EprLines L, EprColumns C, int nx, int ny, float S, const float* __restrict__ tau,
                                                    const float2* __restrict__ map_in, const float* __restrict__ es,
                                                    float* __restrict__ r) {
  const int x = blockIdx.x * 64 + (threadIdx.x & 63), y = blockIdx.y * 4 + (threadIdx.x >> 6), b = blockIdx.z;
  if (x >= nx || y >= ny) return;
  const size_t plane = (size_t)nx * ny, pix = (size_t)y * nx + x;
  float dtx = 0.f, dty = 0.f;
  if (!map_in) {
    const float* tb = tau + (size_t)b * plane;
    const int xm = x == 0 ? nx - 1 : x - 1, xp = x + 1 == nx ? 0 : x + 1;
    const int ym = y == 0 ? ny - 1 : y - 1, yp = y + 1 == ny ? 0 : y + 1;
    dtx = __ldg(tb + (size_t)y * nx + xp) - __ldg(tb + (size_t)y * nx + xm);
    dty = __ldg(tb + (size_t)yp * nx + x) - __ldg(tb + (size_t)ym * nx + x);
  }
  for (int s = 0; s < L.n_bins; ++s) {
    const size_t pl = ((size_t)b * L.n_bins + s) * plane;
    float ux, uy;
    if (map_in) {
      const float2 m = __ldg(&map_in[pl + pix]);
      ux = m.x; uy = m.y;
    } else {
      const float cs = -0.5f * __ldg(&C.a[(size_t)s * nx + x]) * __ldg(&C.gamma[(size_t)s * nx + x]);
      ux = fminf(fmaxf(cs * dtx, -S), S);
      uy = fminf(fmaxf(cs * dty, -S), S);
    }
    const int fx = __float2int_rd(ux), fy = __float2int_rd(uy);
    const float dx = ux - (float)fx, dy = uy - (float)fy;
    const int ix0 = wrapm(x + fx, nx), iy0 = wrapm(y + fy, ny);
    const int ix1 = ix0 + 1 == nx ? 0 : ix0 + 1, iy1 = iy0 + 1 == ny ? 0 : iy0 + 1;
    const float* eb = es + pl;
    const float e00 = __ldg(eb + (size_t)iy0 * nx + ix0), e10 = __ldg(eb + (size_t)iy0 * nx + ix1);
    const float e01 = __ldg(eb + (size_t)iy1 * nx + ix0), e11 = __ldg(eb + (size_t)iy1 * nx + ix1);
    const float t0 = fmaf(dx, e10 - e00, e00), t1 = fmaf(dx, e11 - e01, e01);
    r[pl + pix] = fmaf(dy, t1 - t0, t0);
  }
}

cudaError_t epr_gen_gather(const epr_plan_s* p, int batch, const float* tau, const float2* map_in, const float* es, float* r,
                           cudaStream_t st) {
  dim3 grid((p->nx + 63) / 64, (p->ny + 3) / 4, batch);
  k_gen_gather<<<grid, 256, 0, st>>>(p->lines, p->cols, p->nx, p->ny, p->opt.max_shift_px, tau, map_in, es, r);
  return cudaGetLastError();
}

// =====================================================================================================
// a5 + a6  relaxed update and projection to the single-thickness manifold (R10) as an increment, with
// the scalars of the pixel's column:  ΔT = step · Σ_b wblk[b][x] q_b  (R17(c): block filters blended),
//   τ += δ,  Σ_s f_s(x) e^{−γ_s(x) τ} expm1(−γ_s(x) δ) = ΔT,  floored so that Σ_s I_s + ΔT >= i_min.
// =====================================================================================================
// δ of one pixel of column x: given τ and ΔT, Σ_s f_s(x) e^{−γ_s(x) τ} expm1(−γ_s(x) δ) = ΔT (floored)
__device__ __forceinline__ float gen_delta(int n_bins, const EprColumns& C, int nx, int x, float t, float dT, int newton_iters, float i_min) {
  if (n_bins == 1) {
    const float g = __ldg(&C.gamma[x]);                 // one line: f = 1; δ = −log1p(ΔT e^{γτ})/γ in closed form
    return epr_project_increment_mono(g * t, dT, i_min) / g;
  }
  // converging iterations (|γ_max δ| < 0.01): the moments G_k = Σ_s I_s γ_s^k of the column's lines once, the cubic of
  // F(δ) = Σ_s I_s expm1(−γ_s δ) − ΔT solved without a loop (series reversion + one Newton step) — the arithmetic of
  // epr_project_increment_small (epr_math.cuh) with run-time line count and per-column scalars
  float G0 = 0.f, G1 = 0.f, G2 = 0.f, G3 = 0.f, gmax = 0.f;
#pragma unroll 4
  for (int s = 0; s < n_bins; ++s) {
    const float g = __ldg(&C.gamma[(size_t)s * nx + x]);
    const float pI = __ldg(&C.f[(size_t)s * nx + x]) * epr_exp_fast(-g * t);
    gmax = fmaxf(gmax, g);
    G0 += pI;
    float pg = pI * g; G1 += pg;
    pg *= g; G2 += pg;
    G3 = fmaf(pg, g, G3);
  }
  const float rc1 = -__fdividef(1.f, G1);
  float delta = dT * rc1;
  if (fabsf(delta) * gmax < 0.01f && G0 + dT >= i_min && newton_iters > 0) {
    const float c1 = -G1, c2 = 0.5f * G2, c3 = -1.66666667e-1f * G3;
    delta = fmaf(-(c2 * rc1) * delta, delta, delta);
    const float F = fmaf(fmaf(fmaf(c3, delta, c2), delta, c1), delta, -dT);
    const float dF = fmaf(fmaf(3.f * c3, delta, 2.f * c2), delta, c1);
    return delta - __fdividef(F, dF);
  }
  float f[EPR_MAX_BINS], g[EPR_MAX_BINS];
  for (int s = 0; s < n_bins; ++s) {
    f[s] = __ldg(&C.f[(size_t)s * nx + x]);
    g[s] = __ldg(&C.gamma[(size_t)s * nx + x]);
  }
  return epr_project_increment(t, dT, f, g, n_bins, gmax, newton_iters, i_min);
}

// V pixels per thread: 1 (any nx) or 4 (nx % 4 == 0: 16-byte accesses)
template <int V>
__global__ void __launch_bounds__(256) k_gen_update(int n_bins, EprColumns C, int nx, size_t plane, int n_blocks,
                                                    const float* __restrict__ qblk, size_t blk_stride, float step,
                                                    int tau_is_zero, int newton_iters, float i_min, float* __restrict__ tau) {
  const int x = V * (blockIdx.x * 256 + threadIdx.x);
  if (x >= nx) return;
  const size_t i = (size_t)blockIdx.y * nx + x;
  const int b = blockIdx.z;
  float q[V], t[V];
#pragma unroll
  for (int v = 0; v < V; ++v) q[v] = 0.f;
  for (int k = 0; k < n_blocks; ++k) {
    const float* wp = C.wblk + (size_t)k * nx + x;
    const float* qp = qblk + (size_t)k * blk_stride + (size_t)b * plane + i;
    if (V == 4) {
      const float4 w = __ldg(reinterpret_cast<const float4*>(wp));
      if (w.x != 0.f || w.y != 0.f || w.z != 0.f || w.w != 0.f) {
        const float4 qq = __ldg(reinterpret_cast<const float4*>(qp));
        q[0] = fmaf(w.x, qq.x, q[0]); q[1 % V] = fmaf(w.y, qq.y, q[1 % V]); q[2 % V] = fmaf(w.z, qq.z, q[2 % V]); q[3 % V] = fmaf(w.w, qq.w, q[3 % V]);
      }
    } else {
      const float w = __ldg(wp);
      if (w != 0.f) q[0] = fmaf(w, __ldg(qp), q[0]);
    }
  }
  float* tp = tau + (size_t)b * plane + i;
  if (V == 4) {
    const float4 tv = tau_is_zero ? make_float4(0.f, 0.f, 0.f, 0.f) : *reinterpret_cast<const float4*>(tp);
    t[0] = tv.x; t[1 % V] = tv.y; t[2 % V] = tv.z; t[3 % V] = tv.w;
  } else {
    t[0] = tau_is_zero ? 0.f : *tp;
  }
#pragma unroll
  for (int v = 0; v < V; ++v) t[v] += gen_delta(n_bins, C, nx, x + v, t[v], step * q[v], newton_iters, i_min);
  if (V == 4) *reinterpret_cast<float4*>(tp) = make_float4(t[0], t[1 % V], t[2 % V], t[3 % V]);
  else *tp = t[0];
}

cudaError_t epr_gen_update(const epr_plan_s* p, int batch, const float* qblk, size_t blk_stride, float step, int tau_is_zero,
                           float* tau, cudaStream_t st) {
  const size_t plane = (size_t)p->nx * p->ny;
  if (p->nx % 4 == 0)
    k_gen_update<4><<<dim3((p->nx / 4 + 255) / 256, p->ny, batch), 256, 0, st>>>(p->n_bins, p->cols, p->nx, plane, p->n_blocks, qblk, blk_stride,
                                                                                 step, tau_is_zero, p->opt.newton_iters, p->opt.i_min, tau);
  else
    k_gen_update<1><<<gn_grid(p, batch), 256, 0, st>>>(p->n_bins, p->cols, p->nx, plane, p->n_blocks, qblk, blk_stride, step, tau_is_zero,
                                                       p->opt.newton_iters, p->opt.i_min, tau);
  return cudaGetLastError();
}

// out (+)= wblk[b][x] q over `planes` planes (epr_precondition with block filters)
__global__ void __launch_bounds__(256) k_gen_blend(const float* __restrict__ w, int nx, size_t plane, const float* __restrict__ q,
                                                   float* __restrict__ out, int accumulate) {
  GN_PIX(nx)
  const size_t j = (size_t)blockIdx.z * plane + i;
  const float v = __ldg(&w[x]) * __ldg(&q[j]);
  out[j] = accumulate ? out[j] + v : v;
}

cudaError_t epr_gen_blend(const epr_plan_s* p, int planes, int b, const float* q, float* out, int accumulate, cudaStream_t st) {
  k_gen_blend<<<gn_grid(p, planes), 256, 0, st>>>(p->cols.wblk + (size_t)b * p->nx, p->nx, (size_t)p->nx * p->ny, q, out, accumulate);
  return cudaGetLastError();
}

// epr_forward output: P_s = f_s(x) + (P_s − f_s), P = Σ_s P_s
__global__ void __launch_bounds__(256) k_gen_pred_out(int n_bins, EprColumns C, int nx, size_t plane, const float* __restrict__ pred,
                                                      float* __restrict__ P_sum, float* __restrict__ P_bins) {
  GN_PIX(nx)
  const int b = blockIdx.z;
  const size_t base = (size_t)b * n_bins * plane + i;
  float sum = 0.f;
  for (int s = 0; s < n_bins; ++s) {
    const float v = __ldg(&C.f[(size_t)s * nx + x]) + __ldg(&pred[base + (size_t)s * plane]);
    sum += v;
    if (P_bins) P_bins[base + (size_t)s * plane] = v;
  }
  if (P_sum) P_sum[(size_t)b * plane + i] = sum;
}

cudaError_t epr_gen_pred_out(const epr_plan_s* p, int batch, const float* pred, float* P_sum, float* P_bins, cudaStream_t st) {
  const size_t plane = (size_t)p->nx * p->ny;
  k_gen_pred_out<<<gn_grid(p, batch), 256, 0, st>>>(p->n_bins, p->cols, p->nx, plane, pred, P_sum, P_bins);
  return cudaGetLastError();
}

// output conversion with the column's scalars: τ | φ of line out_bin = −(db_s(x)/2) γ_s(x) τ (Eq. (6)) | Σ_s I_s (Eq. (7))
__global__ void __launch_bounds__(256) k_gen_output(int n_bins, EprColumns C, int nx, size_t plane, int mode, int bin, float inv_alpha,
                                                    const float* __restrict__ tau_b, float* __restrict__ out_b) {
  GN_PIX(nx)
  const float* tau = tau_b + (size_t)blockIdx.z * plane;
  float* out = out_b + (size_t)blockIdx.z * plane;
  const float t = tau[i];
  float v = t;
  if (mode == 1) v = -(__ldg(&C.a[(size_t)bin * nx + x]) * inv_alpha) * __ldg(&C.gamma[(size_t)bin * nx + x]) * t;   // db/2 = a/α
  else if (mode == 2) {
    v = 0.f;
    for (int s = 0; s < n_bins; ++s) v += __ldg(&C.f[(size_t)s * nx + x]) * expf(-__ldg(&C.gamma[(size_t)s * nx + x]) * t);
  }
  out[i] = v;
}

cudaError_t epr_gen_output(const epr_plan_s* p, int batch, const float* tau, float* out, cudaStream_t st) {
  const size_t n = (size_t)p->nx * p->ny;
  const int sb = p->opt.out_bin;
  k_gen_output<<<gn_grid(p, batch), 256, 0, st>>>(p->n_bins, p->cols, p->nx, n, p->opt.output, sb,
                                                             (float)(1.0 / p->h_alpha[sb]), tau, out);
  return cudaGetLastError();
}

// =====================================================================================================
// Regime diagnostic (Fig. 6): per projection and line, the histogram over the pixels of
// η = ‖Δ_s‖/p = a_s γ_s ‖D⁰τ‖ (Euclidean norm of the UNCLAMPED eikonal shift, Eq. (2)), bins [k·bin_px, (k+1)·bin_px), the last
// one open-ended.  hist: [batch][n_bins][n_hist] unsigned, accumulated (the launcher zeroes it).  Works on both paths: the
// scalars come from the column tables when the plan has them, from the uniform per-line scalars otherwise.
// One thread = one pixel; counts are collected per CTA in shared memory first.
// =====================================================================================================
__global__ void __launch_bounds__(256) k_shift_hist(EprLines L, EprColumns C, int use_cols, int nx, int ny, int n_hist, int s0,
                                                    int ns, float inv_bin, const float* __restrict__ tau,
                                                    unsigned* __restrict__ hist) {
  extern __shared__ unsigned s_h[];                     // [ns][n_hist]: lines s0 … s0 + ns − 1
  const int nb = L.n_bins, b = blockIdx.z;
  for (int i = threadIdx.x; i < ns * n_hist; i += 256) s_h[i] = 0u;
  __syncthreads();
  const int x = blockIdx.x * 64 + (threadIdx.x & 63), y = blockIdx.y * 4 + (threadIdx.x >> 6);
  if (x < nx && y < ny) {
    const float* tb = tau + (size_t)b * nx * ny;
    const int xm = x == 0 ? nx - 1 : x - 1, xp = x + 1 == nx ? 0 : x + 1;
    const int ym = y == 0 ? ny - 1 : y - 1, yp = y + 1 == ny ? 0 : y + 1;
    const float dtx = __ldg(tb + (size_t)y * nx + xp) - __ldg(tb + (size_t)y * nx + xm);
    const float dty = __ldg(tb + (size_t)yp * nx + x) - __ldg(tb + (size_t)ym * nx + x);
    const float g = 0.5f * sqrtf(dtx * dtx + dty * dty);                      // ‖D⁰τ‖
    for (int j = 0; j < ns; ++j) {
      const int s = s0 + j;
      const float c = use_cols ? __ldg(&C.a[(size_t)s * nx + x]) * __ldg(&C.gamma[(size_t)s * nx + x]) : L.a[s] * L.gamma[s];
      const int k = min((int)(c * g * inv_bin), n_hist - 1);
      atomicAdd(&s_h[j * n_hist + k], 1u);
    }
  }
  __syncthreads();
  for (int i = threadIdx.x; i < ns * n_hist; i += 256)
    if (s_h[i]) atomicAdd(&hist[((size_t)b * nb + s0) * n_hist + i], s_h[i]);
}

// The per-CTA counters stay within the 48 KB of shared memory every kernel may use without opting in: the lines are
// taken in passes of at most 12288 / n_hist (16 lines x 1024 bins = 64 KB goes in two passes of 12 and 4 lines).
cudaError_t epr_launch_shift_hist(const epr_plan_s* p, int batch, const float* tau, int n_hist, float bin_px, unsigned* hist,
                                  cudaStream_t st) {
  const size_t n = (size_t)batch * p->n_bins * n_hist;
  cudaError_t e = cudaMemsetAsync(hist, 0, n * sizeof(unsigned), st);
  if (e != cudaSuccess) return e;
  const int per_pass = (48 * 1024 / (int)sizeof(unsigned)) / n_hist;        // n_hist <= 1024: at least 12
  bool first = true;
  for (int b0 = 0; b0 < batch; b0 += 65535) {                               // gridDim.z <= 65535
    const int nbat = batch - b0 < 65535 ? batch - b0 : 65535;
    dim3 grid((p->nx + 63) / 64, (p->ny + 3) / 4, nbat);
    for (int s0 = 0; s0 < p->n_bins; s0 += per_pass) {
      const int ns = p->n_bins - s0 < per_pass ? p->n_bins - s0 : per_pass;
      if (!first) epr_note_extra_launch(p);
      first = false;
      k_shift_hist<<<grid, 256, (size_t)ns * n_hist * sizeof(unsigned), st>>>(
          p->lines, p->cols, p->general, p->nx, p->ny, n_hist, s0, ns, 1.f / bin_px, tau + (size_t)b0 * p->nx * p->ny,
          hist + (size_t)b0 * p->n_bins * n_hist);
    }
  }
  return cudaGetLastError();
}

// =====================================================================================================
// Diagnostics of the loop on the general path (epr_set_diagnostics; never in timed runs): per projection, the RMS of the
// detector residual e = Σ_s e_s and the regime indicator as the largest UNCLAMPED shift
// component max_s a_s(x) γ_s(x) · max(|D⁰xτ|, |D⁰yτ|) with the scalars of the pixel's own column (R17(b)).
// Two launches, fixed summation order (bit-reproducible): 64 partial sums / maxima per projection, then one thread each.
// =====================================================================================================
#define GD_BLK 64
__global__ void __launch_bounds__(256) k_gen_diag_partial(int n_bins, EprColumns C, int nx, int ny, const float* __restrict__ tau,
                                                          const float* __restrict__ es, double* __restrict__ partial) {
  __shared__ double s_sum[256];
  __shared__ float s_max[256];
  const int b = blockIdx.y;
  const size_t plane = (size_t)nx * ny;
  const float* tb = tau + (size_t)b * plane;
  const float* eb = es + (size_t)b * n_bins * plane;
  double acc = 0.0;
  float m = 0.f;
  for (int x = threadIdx.x; x < nx; x += 256) {
    float c = 0.f;
    for (int s = 0; s < n_bins; ++s) c = fmaxf(c, __ldg(&C.a[(size_t)s * nx + x]) * __ldg(&C.gamma[(size_t)s * nx + x]));
    const int xm = x == 0 ? nx - 1 : x - 1, xp = x + 1 == nx ? 0 : x + 1;
    for (int y = blockIdx.x; y < ny; y += GD_BLK) {
      const int ym = y == 0 ? ny - 1 : y - 1, yp = y + 1 == ny ? 0 : y + 1;
      const size_t i = (size_t)y * nx + x;
      float e = 0.f;
      for (int s = 0; s < n_bins; ++s) e += __ldg(eb + (size_t)s * plane + i);
      acc += (double)e * e;
      const float dtx = __ldg(tb + (size_t)y * nx + xp) - __ldg(tb + (size_t)y * nx + xm);
      const float dty = __ldg(tb + (size_t)yp * nx + x) - __ldg(tb + (size_t)ym * nx + x);
      m = fmaxf(m, 0.5f * c * fmaxf(fabsf(dtx), fabsf(dty)));
    }
  }
  s_sum[threadIdx.x] = acc;
  s_max[threadIdx.x] = m;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if (threadIdx.x < o) {
      s_sum[threadIdx.x] += s_sum[threadIdx.x + o];
      s_max[threadIdx.x] = fmaxf(s_max[threadIdx.x], s_max[threadIdx.x + o]);
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    partial[((size_t)b * GD_BLK + blockIdx.x) * 2] = s_sum[0];
    partial[((size_t)b * GD_BLK + blockIdx.x) * 2 + 1] = (double)s_max[0];
  }
}

__global__ void __launch_bounds__(32) k_gen_diag_reduce(int batch, size_t plane, const double* __restrict__ partial,
                                                        float* __restrict__ diag, int stride) {
  const int b = blockIdx.x * 32 + threadIdx.x;
  if (b >= batch) return;
  double sum = 0.0, m = 0.0;
  for (int i = 0; i < GD_BLK; ++i) {
    sum += partial[((size_t)b * GD_BLK + i) * 2];
    m = fmax(m, partial[((size_t)b * GD_BLK + i) * 2 + 1]);
  }
  diag[(size_t)b * stride] = (float)sqrt(sum / (double)plane);
  diag[(size_t)b * stride + 1] = (float)m;
}

// partial: [batch][GD_BLK][2] doubles (epr_set_diagnostics allocates it)
cudaError_t epr_gen_diagnostics(const epr_plan_s* p, int batch, const float* tau, const float* es, float* diag, int stride,
                                cudaStream_t st) {
  epr_note_extra_launch(p);                              // two kernels
  k_gen_diag_partial<<<dim3(GD_BLK, batch), 256, 0, st>>>(p->n_bins, p->cols, p->nx, p->ny, tau, es, p->diag_partial);
  k_gen_diag_reduce<<<(batch + 31) / 32, 32, 0, st>>>(batch, (size_t)p->nx * p->ny, p->diag_partial, diag, stride);
  return cudaGetLastError();
}
