"""hclooc-b200: out-of-core FP64 matrix multiplication (the MMOOC of arXiv 1808.05056) on one B200.

Thin ctypes binding over the C ABI in include/hclooc.h -- same names, argument marshalling only;
every step of the hot path (plan, schedule, copies, events, the DMMA tile kernel) runs inside
libhclooc_b200.so.  There is no CPU fallback: if the library cannot be built or loaded, importing
the binding's functions raises.
"""
from ._binding import (  # noqa: F401
    HclError, lib, HostMatrix, Plan, ResidentPlan, Stats,
    hclooc_plan, hclooc_plan_ex, hclooc_plan_trans, hclooc_plan_resident, hclooc_resident_schedule, hclooc_shard_rows, hclooc_schedule, hclMatrixPartitioner,
    hclooc_ctx_create, hclooc_ctx_destroy, hclooc_ctx_set_trace, hclooc_ctx_get_trace, hclooc_ctx_set_direct, hclooc_ctx_set_debug, hclooc_calibrate_link, TRACE_DTYPE, hclooc_dgemm, hclooc_dgemm_ex, hclooc_dgemm_t, hclooc_dsyrk, hclooc_dsyr2k, hclooc_dtrsm, hclooc_dtrsm_plan, hclooc_dtrsm_side, hclooc_dpotrf, hclooc_dpotrf_plan, hclooc_dgetrf, hclooc_dgetrf_plan, hclDgetrf, hclooc_dtrmm, hclooc_dsymm, hclooc_dgemm_fig2, hclooc_dgemm_nsteps,
    hclMalloc, hclFree, hclGetMemSize, hclStreamCreate, hclStreamDestroy, hclEventDestroy,
    hclMemcpy, hclMemcpyAsync, hclMemcpy2DAsync, hclDgemmAsync, hclDgemmAsyncEx, hclDgemmAsyncT, hclDgemmNoAlloc, hclDgemmNoAllocScratchBytes, hclDtrsmAsync, hclDpotrfAsync, hclWaitEvent,
    hclStreamSynchronize, hclDeviceSynchronize,
    hclooc_host_alloc, hclooc_host_free, hclooc_host_register, hclooc_host_unregister,
    hclooc_strerror, hclooc_last_cuda_error, hclooc_version, hclooc_probe_fp64,
    HCL_H2D, HCL_D2H, HCL_OP_N, HCL_OP_T, HCL_UPLO_LOWER, HCL_UPLO_UPPER, HCL_DIAG_NONUNIT, HCL_DIAG_UNIT, HCL_SIDE_LEFT, HCL_SIDE_RIGHT, EXPORTS, OP_DTYPE,
)
