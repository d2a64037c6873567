"""sagecal-b200: the data-parallel hot path of SAGECal direction-dependent calibration on one NVIDIA B200.

Thin ctypes binding of libsagecal_b200.so (C ABI: include/sagecal_b200.h).  The functions here have the names of
the C entry points and only marshal arguments: torch is used for device memory and streams, every step of the path
runs in the library's CUDA kernels.  There is no CPU fallback: if the shared library is missing the import of any
entry point raises.
"""
from ._binding import (  # noqa: F401
    COH_FULL,
    COH_SCALAR,
    LM_COMPRESSED,
    LM_DIRECT,
    LM_FULLGN,
    LM_PERCLUSTER,
    SagecalError,
    apply_flags,
    canonical_to_rows,
    rows_to_canonical,
    calibrate_interval_host,
    host_sync,
    host_trim,
    corrupt_subtract,
    kernel_kinds,
    launch_count,
    lib_path,
    lm_cost_grad_jtj,
    load_library,
    predict_coherencies,
    predict_coherencies_static,
    predict_static_bytes,
    predict_residual,
    predict_set_form,
    profile_dfma_peak,
    profile_dmma_peak,
    profile_enable,
    profile_read,
    sage_calibrate,
    version,
    workspace_bytes,
)

__all__ = [
    "COH_FULL", "COH_SCALAR", "LM_COMPRESSED", "LM_DIRECT", "LM_FULLGN", "LM_PERCLUSTER", "SagecalError", "apply_flags", "canonical_to_rows", "rows_to_canonical", "calibrate_interval_host", "host_sync", "host_trim", "corrupt_subtract", "kernel_kinds",
    "launch_count", "lib_path", "lm_cost_grad_jtj", "load_library", "predict_coherencies", "predict_coherencies_static", "predict_static_bytes", "predict_residual", "predict_set_form", "profile_dfma_peak", "profile_dmma_peak", "profile_enable",
    "profile_read", "sage_calibrate", "version", "workspace_bytes",
]
