"""B200-native fast Eikonal Phase Retrieval (EPR) hot path — thin Python binding over libepr.so.

The binding only marshals arguments (torch CUDA tensors -> raw device pointers, the current torch stream ->
cudaStream_t).  Every step of the path runs in the hand-written sm_100a kernels behind the C-ABI declared in
`include/epr.h`; there is no CPU fallback: without the compiled library, or without a CUDA device, calls raise.
"""
from .binding import (EPR_LOCAL, EPR_NONLOCAL, EprError, Options, Plan, epr_adjoint, epr_forward, epr_plan, epr_plan_profiles,  # noqa: F401
                      epr_precondition, epr_retrieve, epr_retrieve_host, epr_retrieve_oversampled, epr_set_diagnostics, epr_shift_histogram, epr_transport, lib_path,
                      EPR_STATIC_MAX_BATCH, epr_residual_rms_static, epr_host_wait, epr_retrieve_host_multi, epr_shard_range,
                      load_library)
