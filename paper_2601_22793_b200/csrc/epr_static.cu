// epr_static.cu — epr_residual_rms_static: the residual-RMS convergence monitor ("form the detector
// residual"; PAPER.md:95 convergence history) for callers that must not allocate device memory.
//
// Who cannot allocate.  A beamline reconstruction process usually hands (nearly) all of the GPU's memory to ONE pool —
// the tomography framework's caching allocator, or the plans of this library sized at start-up for the largest batch —
// so a cudaMalloc issued later from a monitoring hook fails with out-of-memory, or succeeds only by fragmenting what
// the pool expects to get back.  And cudaMalloc / cudaFree are not stream-ordered: they may stall every stream of the
// device, which an acquisition-rate loop (chunk k + 1 uploading while chunk k iterates) cannot afford in
// a per-iteration diagnostic.  Such callers own their inputs and outputs already; what they lack is the reduction's
// scratch.  The plan-based route (epr_set_diagnostics) takes that scratch from cudaMalloc on its first use; this file
// keeps it in the library image instead.
//
// The scratch is g_rms_partial below: 64 partial sums (double) per projection, EPR_STATIC_MAX_BATCH projections,
// 512 KiB, in a file-scope __device__ array.  Every GPU on which this library's code gets loaded holds its own copy
// from that moment until the process exits — that is the price, and the reason the maximum is modest.
//
// The array's name is usable as an address only in DEVICE code.  In host code the same identifier is a host-side
// shadow the runtime uses as a lookup key; handing it to a kernel as a pointer would make the kernel read and write
// whatever lies at that host address (a fault, or — on systems where the GPU can reach host memory — silent
// corruption).  The host side therefore asks the runtime for the device address, once per device and with that device
// current (scratch_on_current_device), and passes that pointer to the kernels.
//
// This file is self-contained on purpose: array, address look-up, kernels and launch all live in one translation unit
// (a static __device__ symbol is not visible from another), and it changes nothing in the plan-based path.
#include <cuda_runtime.h>

#include <cstdio>
#include <mutex>

#include "../../include/epr.h"

#define RS_BLK 64                    // partial sums per projection: the same 64 x 256-thread layout as k_diag_partial
#define RS_MAX_DEVICES 64
#define RS_MAX_BINS 16               // N_s limit of every other entry point (epr_plan)

static __device__ __align__(256) double g_rms_partial[(size_t)EPR_STATIC_MAX_BATCH * RS_BLK];

static std::mutex g_mu;                                   // guards g_scratch (first call per device)
static double* g_scratch[RS_MAX_DEVICES] = {};            // DEVICE address of g_rms_partial, per device ordinal
static thread_local char t_err[256] = "";

#define RS_FAIL(code, ...) do { snprintf(t_err, sizeof t_err, __VA_ARGS__); return (code); } while (0)

// Stage 1.  Block (k, b) adds up e² = (Σ_s e_s)² over its strided share of projection b and WRITES slot [b][k] —
// every slot a call later reads is written by that call first (also when the share is empty), so nothing in the
// scratch has to start at zero and the previous call's leftovers are harmless.  VEC: four pixels per load
// (plane % 4 == 0 and a 16-byte aligned base); otherwise one pixel per load, same block-to-pixel assignment modulo 4.
template <bool VEC>
__global__ void __launch_bounds__(256) k_rms_partial_static(int n_bins, unsigned plane, const float* __restrict__ es,
                                                            double* __restrict__ partial) {
  __shared__ double s_sum[256];
  const int b = blockIdx.y;
  const float* eb = es + (size_t)b * n_bins * plane;
  double acc = 0.0;
  if (VEC) {
    for (unsigned i = (blockIdx.x * 256u + threadIdx.x) * 4u; i < plane; i += RS_BLK * 256u * 4u) {
      float4 e = make_float4(0.f, 0.f, 0.f, 0.f);
      for (int s = 0; s < n_bins; ++s) {
        const float4 v = __ldg(reinterpret_cast<const float4*>(eb + (size_t)s * plane + i));
        e.x += v.x; e.y += v.y; e.z += v.z; e.w += v.w;
      }
      acc += (double)e.x * e.x + (double)e.y * e.y + (double)e.z * e.z + (double)e.w * e.w;
    }
  } else {
    for (size_t i = (size_t)blockIdx.x * 256u + threadIdx.x; i < plane; i += (size_t)RS_BLK * 256u) {
      float e = 0.f;
      for (int s = 0; s < n_bins; ++s) e += __ldg(eb + (size_t)s * plane + i);
      acc += (double)e * e;
    }
  }
  s_sum[threadIdx.x] = acc;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if (threadIdx.x < o) s_sum[threadIdx.x] += s_sum[threadIdx.x + o];
    __syncthreads();
  }
  if (threadIdx.x == 0) partial[(size_t)b * RS_BLK + blockIdx.x] = s_sum[0];
}

// Stage 2.  One thread per projection adds its 64 slots in index order (fixed order: the result is bit-reproducible).
__global__ void __launch_bounds__(64) k_rms_final_static(int batch, unsigned plane, const double* __restrict__ partial,
                                                         float* __restrict__ rms) {
  const int b = blockIdx.x * 64 + threadIdx.x;
  if (b >= batch) return;
  double sum = 0.0;
  for (int i = 0; i < RS_BLK; ++i) sum += partial[(size_t)b * RS_BLK + i];
  rms[b] = (float)sqrt(sum / (double)plane);
}

// Device address of g_rms_partial on the CURRENT device; looked up on the first call per device, cached afterwards.
// cudaGetSymbolAddress allocates nothing itself, but the first use of anything in this library on a device makes
// the runtime load the library's code there (which is when the array comes to exist on that device) — so the first
// call on a device belongs before any stream capture and outside latency-critical sections.
static cudaError_t scratch_on_current_device(int dev, double** out) {
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_scratch[dev]) {
    void* p = NULL;
    const cudaError_t e = cudaGetSymbolAddress(&p, g_rms_partial);
    if (e != cudaSuccess) return e;
    g_scratch[dev] = (double*)p;
  }
  *out = g_scratch[dev];
  return cudaSuccess;
}

// True when `p` is device (or managed) memory that the device `dev` owns.
static bool on_device(const void* p, int dev) {
  cudaPointerAttributes at;
  if (cudaPointerGetAttributes(&at, p) != cudaSuccess) { cudaGetLastError(); return false; }
  return (at.type == cudaMemoryTypeDevice && at.device == dev) || at.type == cudaMemoryTypeManaged;
}

extern "C" epr_status epr_residual_rms_static(int batch, int n_bins, int nx, int ny, const float* e_bins, float* rms,
                                              void* stream) {
  t_err[0] = 0;
  if (!e_bins || !rms) RS_FAIL(EPR_EINVAL, "epr_residual_rms_static: e_bins and rms must not be NULL");
  if (batch < 1 || nx < 1 || ny < 1) RS_FAIL(EPR_EINVAL, "epr_residual_rms_static: batch, nx, ny must be positive");
  if (n_bins < 1 || n_bins > RS_MAX_BINS)
    RS_FAIL(EPR_EINVAL, "epr_residual_rms_static: n_bins = %d outside 1..%d", n_bins, RS_MAX_BINS);
  if (batch > EPR_STATIC_MAX_BATCH)
    RS_FAIL(EPR_ESIZE, "epr_residual_rms_static: batch = %d exceeds EPR_STATIC_MAX_BATCH = %d (the built-in scratch holds %d "
                       "partial sums for each of that many projections and is never enlarged); split the batch",
            batch, EPR_STATIC_MAX_BATCH, RS_BLK);
  const unsigned long long plane64 = (unsigned long long)nx * (unsigned long long)ny;
  if (plane64 >= (1ull << 32))
    RS_FAIL(EPR_ESIZE, "epr_residual_rms_static: nx * ny = %llu does not fit 32 bits", plane64);
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) RS_FAIL(EPR_ECUDA, "epr_residual_rms_static: cudaGetDevice: %s", cudaGetErrorString(e));
  if (dev < 0 || dev >= RS_MAX_DEVICES)
    RS_FAIL(EPR_EINVAL, "epr_residual_rms_static: device ordinal %d outside 0..%d", dev, RS_MAX_DEVICES - 1);
  if (!on_device(e_bins, dev) || !on_device(rms, dev))
    RS_FAIL(EPR_EINVAL, "epr_residual_rms_static: e_bins and rms must be device memory of the current device (%d)", dev);
  double* scratch = NULL;
  e = scratch_on_current_device(dev, &scratch);
  if (e != cudaSuccess) {
    cudaGetLastError();
    RS_FAIL(EPR_ECUDA, "epr_residual_rms_static: cudaGetSymbolAddress on device %d: %s", dev, cudaGetErrorString(e));
  }
  const unsigned plane = (unsigned)plane64;
  const cudaStream_t st = (cudaStream_t)stream;
  const dim3 grid(RS_BLK, batch);
  if (plane % 4u == 0 && ((size_t)e_bins & 15u) == 0)
    k_rms_partial_static<true><<<grid, 256, 0, st>>>(n_bins, plane, e_bins, scratch);
  else
    k_rms_partial_static<false><<<grid, 256, 0, st>>>(n_bins, plane, e_bins, scratch);
  k_rms_final_static<<<(batch + 63) / 64, 64, 0, st>>>(batch, plane, scratch, rms);
  e = cudaGetLastError();
  if (e != cudaSuccess) RS_FAIL(EPR_ECUDA, "epr_residual_rms_static: launch: %s", cudaGetErrorString(e));
  return EPR_OK;
}

extern "C" const char* epr_static_last_error(void) { return t_err; }
