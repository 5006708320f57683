// epr_fftgen.cu — run-time-radix FFT for the FFT-diagonal preconditioner on any
// {2,3,5}-smooth grid (8 <= n <= 8192) that has no compile-time instantiation in epr_fftk.cu.
//
// Same three steps (rows R2C → columns FFT · H_s (· Σ_s) · IFFT → rows C2R) with the plain layout of a real
// transform: spectra are [plane][ny][nx/2 + 1] float2 (kx = 0 … ⌊nx/2⌋; odd nx allowed), no packed Nyquist column.
// Stockham autosort in shared memory, ping-pong between two buffers, radix 4 / 2 / 3 / 5 chosen per pass at run time;
// twiddles from one table exp(−2πi m/n) per axis.  A row transform is a full complex transform of length nx (the
// half-length trick of the tuned kernels needs an even nx); this path trades that factor of two for generality.
#include "epr_fft.cuh"
#include "epr_internal.h"

namespace {

struct Sched { int np; int radix[16]; };

Sched make_sched(int n) {
  Sched s;
  s.np = 0;
  while (n % 4 == 0) { s.radix[s.np++] = 4; n /= 4; }
  while (n % 2 == 0) { s.radix[s.np++] = 2; n /= 2; }
  while (n % 3 == 0) { s.radix[s.np++] = 3; n /= 3; }
  while (n % 5 == 0) { s.radix[s.np++] = 5; n /= 5; }
  return s;
}

// One Stockham pass of W interleaved transforms of length N (element i of transform c at [i·W + c]):
//   out[j0 + q·P] = Σ_r w^{r k rest·…} in[j + r·T],  T = N/R,  k = j mod P,  j0 = (j − k)·R + k,  twiddle exp(∓2πi r k/(P R)).
template <int R, bool INV>
__device__ __forceinline__ void gen_pass(const float2* __restrict__ src, float2* __restrict__ dst, int N, int P, int W,
                                         const float2* __restrict__ tab) {
  const int T = N / R, rest = T / P;                    // N = P·R·rest
  for (int idx = threadIdx.x; idx < T * W; idx += blockDim.x) {
    const int j = idx / W, c = idx - j * W;
    const int k = j % P;
    float2 u[R];
#pragma unroll
    for (int r = 0; r < R; ++r) u[r] = src[(j + r * T) * W + c];
    if (P > 1) {
#pragma unroll
      for (int r = 1; r < R; ++r) u[r] = eprfft::cmul(u[r], eprfft::conj_if<INV>(__ldg(&tab[r * k * rest])));
    }
    eprfft::dft<R, INV>(u);
    const int j0 = (j - k) * R + k;
#pragma unroll
    for (int q = 0; q < R; ++q) dst[(j0 + q * P) * W + c] = u[q];
  }
}

// all passes; returns the buffer that holds the result (a or b)
template <bool INV>
__device__ __forceinline__ float2* gen_fft(float2* a, float2* b, int N, int W, const Sched& sc, const float2* __restrict__ tab) {
  int P = 1;
  for (int i = 0; i < sc.np; ++i) {
    const int R = sc.radix[i];
    if (R == 4) gen_pass<4, INV>(a, b, N, P, W, tab);
    else if (R == 2) gen_pass<2, INV>(a, b, N, P, W, tab);
    else if (R == 3) gen_pass<3, INV>(a, b, N, P, W, tab);
    else gen_pass<5, INV>(a, b, N, P, W, tab);
    __syncthreads();
    P *= R;
    float2* t = a; a = b; b = t;
  }
  return a;
}

__global__ void __launch_bounds__(256) k_gen_rows_r2c(int nx, int ny, Sched sc, const float* __restrict__ in, float in_offset,
                                                      const float2* __restrict__ tab, float2* __restrict__ spec) {
  extern __shared__ float2 sm[];                        // 2 x nx
  const size_t row = (size_t)blockIdx.y * ny + blockIdx.x;
  const float* src = in + row * nx;
  for (int i = threadIdx.x; i < nx; i += blockDim.x) sm[i] = make_float2(__ldg(&src[i]) + in_offset, 0.f);
  __syncthreads();
  const float2* res = gen_fft<false>(sm, sm + nx, nx, 1, sc, tab);
  const int Mg = nx / 2 + 1;
  float2* dst = spec + row * Mg;
  for (int k = threadIdx.x; k < Mg; k += blockDim.x) dst[k] = res[k];
}

__global__ void __launch_bounds__(256) k_gen_rows_c2r(int nx, int ny, Sched sc, const float2* __restrict__ spec,
                                                      const float2* __restrict__ tab, float* __restrict__ out) {
  extern __shared__ float2 sm[];
  const size_t row = (size_t)blockIdx.y * ny + blockIdx.x;
  const int Mg = nx / 2 + 1;
  const float2* src = spec + row * Mg;
  for (int k = threadIdx.x; k < Mg; k += blockDim.x) {   // Hermitian completion: X[nx − k] = X*[k]
    const float2 v = __ldg(&src[k]);
    sm[k] = v;
    if (k > 0 && 2 * k != nx) sm[nx - k] = make_float2(v.x, -v.y);
  }
  __syncthreads();
  const float2* res = gen_fft<true>(sm, sm + nx, nx, 1, sc, tab);
  float* dst = out + row * nx;
  for (int i = threadIdx.x; i < nx; i += blockDim.x) dst[i] = res[i].x;
}

// mode 0: out[plane] = IFFT(H_{plane % nb} FFT(spec[plane])); 1: out[b] = IFFT(Σ_s H_s FFT(spec[b nb + s])); 2: H_ā.
// H = scale / (1 + a (λx[kx] + λy[ky])).  Tile = W columns x ny rows; three shared buffers (ping, pong, accumulator).
__global__ void __launch_bounds__(256) k_gen_cols(EprLines L, int Mg, int ny, int W, int mode, float scale, Sched sc,
                                                  const float* __restrict__ lam_x, const float* __restrict__ lam_y,
                                                  const float2* __restrict__ tab, const float2* __restrict__ spec,
                                                  float2* __restrict__ out) {
  extern __shared__ float2 sm[];                        // 3 x ny x W
  float2 *a = sm, *b = sm + (size_t)ny * W, *acc = sm + 2 * (size_t)ny * W;
  const int kx0 = blockIdx.x * W, oplane = blockIdx.y, nb = L.n_bins;
  const int nloop = (mode == 1) ? nb : 1;
  for (int i = threadIdx.x; i < ny * W; i += blockDim.x) acc[i] = make_float2(0.f, 0.f);
  for (int sl = 0; sl < nloop; ++sl) {
    const size_t iplane = (mode == 1) ? (size_t)oplane * nb + sl : (size_t)oplane;
    const float av = (mode == 2) ? L.abar : L.a[(mode == 1) ? sl : (oplane % nb)];
    const float2* src = spec + iplane * (size_t)ny * Mg;
    __syncthreads();
    for (int i = threadIdx.x; i < ny * W; i += blockDim.x) {
      const int r = i / W, c = i - r * W;
      a[i] = (kx0 + c < Mg) ? __ldg(&src[(size_t)r * Mg + kx0 + c]) : make_float2(0.f, 0.f);
    }
    __syncthreads();
    const float2* res = gen_fft<false>(a, b, ny, W, sc, tab);
    for (int i = threadIdx.x; i < ny * W; i += blockDim.x) {
      const int r = i / W, c = i - r * W;
      const int kx = min(kx0 + c, Mg - 1);
      const float h = __fdividef(scale, fmaf(av, __ldg(&lam_x[kx]) + __ldg(&lam_y[r]), 1.f));
      acc[i].x = fmaf(h, res[i].x, acc[i].x);
      acc[i].y = fmaf(h, res[i].y, acc[i].y);
    }
  }
  __syncthreads();
  // inverse from the accumulator: ping = acc, pong = a (free)
  const float2* res = gen_fft<true>(acc, a, ny, W, sc, tab);
  float2* dst = out + (size_t)oplane * ny * Mg;
  for (int i = threadIdx.x; i < ny * W; i += blockDim.x) {
    const int r = i / W, c = i - r * W;
    if (kx0 + c < Mg) dst[(size_t)r * Mg + kx0 + c] = res[i];
  }
}

int cols_width(int ny) {                                // widest tile whose three buffers fit 200 KB
  int W = 8;
  while (W > 1 && (size_t)3 * ny * W * sizeof(float2) > 200 * 1024) W >>= 1;
  return W;
}

}  // namespace

int epr_fftgen_supported(int n) {
  if (n < 8 || n > 8192) return 0;
  while (n % 2 == 0) n /= 2;
  while (n % 3 == 0) n /= 3;
  while (n % 5 == 0) n /= 5;
  return n == 1;
}

size_t epr_fftgen_spec_floats(const epr_plan_s* p) { return (size_t)2 * (p->nx / 2 + 1) * p->ny; }

cudaError_t epr_fftgen_rows_r2c(const epr_plan_s* p, int planes, const float* in, float in_offset, float2* spec, cudaStream_t st) {
  const size_t smem = (size_t)2 * p->nx * sizeof(float2);
  static EprPerDevice attr = {};
  if ((long long)smem > attr.at(p)) {
    cudaFuncSetAttribute(k_gen_rows_r2c, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    attr.at(p) = (long long)smem;
  }
  k_gen_rows_r2c<<<dim3(p->ny, planes), 256, smem, st>>>(p->nx, p->ny, make_sched(p->nx), in, in_offset, p->tw_gen_x, spec);
  return cudaGetLastError();
}

cudaError_t epr_fftgen_rows_c2r(const epr_plan_s* p, int planes, const float2* spec, float* q, cudaStream_t st) {
  const size_t smem = (size_t)2 * p->nx * sizeof(float2);
  static EprPerDevice attr = {};
  if ((long long)smem > attr.at(p)) {
    cudaFuncSetAttribute(k_gen_rows_c2r, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    attr.at(p) = (long long)smem;
  }
  k_gen_rows_c2r<<<dim3(p->ny, planes), 256, smem, st>>>(p->nx, p->ny, make_sched(p->nx), spec, p->tw_gen_x, q);
  return cudaGetLastError();
}

cudaError_t epr_fftgen_cols(const epr_plan_s* p, int planes, int mode, const float2* spec, float2* out, cudaStream_t st,
                            const EprLines* lines_override) {
  const int Mg = p->nx / 2 + 1, W = cols_width(p->ny);
  const int oplanes = (mode == 1) ? planes / p->n_bins : planes;
  const size_t smem = (size_t)3 * p->ny * W * sizeof(float2);
  static EprPerDevice attr = {};
  if ((long long)smem > attr.at(p)) {
    cudaFuncSetAttribute(k_gen_cols, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    attr.at(p) = (long long)smem;
  }
  const float scale = (float)(1.0 / ((double)p->nx * (double)p->ny));
  k_gen_cols<<<dim3((Mg + W - 1) / W, oplanes), 256, smem, st>>>(lines_override ? *lines_override : p->lines, Mg, p->ny, W, mode,
                                                                  scale, make_sched(p->ny), p->lam_x, p->lam_y, p->tw_gen_y, spec, out);
  return cudaGetLastError();
}
