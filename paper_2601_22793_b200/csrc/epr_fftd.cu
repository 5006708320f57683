// epr_fftd.cu — routes an FFT launch to the translation unit (group) that instantiates its size.
// epr_fftk.cu is compiled EPR_FFT_NGROUPS times (-DEPR_FFT_GROUP=g), each with a subset of the supported sizes.
#include "epr_internal.h"

#ifdef EPR_FFT_DEV          /* developer build: only group 0 (2048, 16, 32) is compiled */
#define EPR_FFT_GROUPS(G) G(0)
#else
#define EPR_FFT_GROUPS(G) G(0) G(1) G(2) G(3) G(4) G(5) G(6) G(7) G(8) G(9) G(10)
#endif

#define G(g)                                                                                                          \
  int epr_fftg_has_##g(int n);                                                                                        \
  cudaError_t epr_fftg_rows_r2c_##g(const epr_plan_s*, int, const float*, float, float2*, cudaStream_t);               \
  cudaError_t epr_fftg_rows_c2r_##g(const epr_plan_s*, int, const float2*, int, float, int, float*, cudaStream_t);     \
  cudaError_t epr_fftg_cols_##g(const epr_plan_s*, int, int, const float2*, float2*, cudaStream_t, const EprLines*, int);
EPR_FFT_GROUPS(G)
#undef G

extern "C" int epr_fft_size_supported(int n) {
#define G(g) if (epr_fftg_has_##g(n)) return 1;
  EPR_FFT_GROUPS(G)
#undef G
  return 0;
}

cudaError_t epr_launch_rows_r2c(const epr_plan_s* p, int planes, const float* in, float in_offset, float2* spec,
                                cudaStream_t st) {
#define G(g) if (epr_fftg_has_##g(p->nx)) return epr_fftg_rows_r2c_##g(p, planes, in, in_offset, spec, st);
  EPR_FFT_GROUPS(G)
#undef G
  return cudaErrorInvalidValue;
}

cudaError_t epr_launch_rows_c2r(const epr_plan_s* p, int planes, const float2* spec, int epilogue, float step,
                                int tau_is_zero, float* q_or_tau, cudaStream_t st) {
#define G(g) if (epr_fftg_has_##g(p->nx)) return epr_fftg_rows_c2r_##g(p, planes, spec, epilogue, step, tau_is_zero, q_or_tau, st);
  EPR_FFT_GROUPS(G)
#undef G
  return cudaErrorInvalidValue;
}

cudaError_t epr_launch_cols(const epr_plan_s* p, int planes, int mode, const float2* spec, float2* out, cudaStream_t st,
                            const EprLines* lines_override, int stage) {
#define G(g) if (epr_fftg_has_##g(p->ny)) return epr_fftg_cols_##g(p, planes, mode, spec, out, st, lines_override, stage);
  EPR_FFT_GROUPS(G)
#undef G
  return cudaErrorInvalidValue;
}
