"""ctypes marshalling for include/hclooc.h.  No arithmetic of the method lives here."""
from __future__ import annotations

import ctypes
from ctypes import POINTER, byref, c_char_p, c_double, c_int, c_int32, c_int64, c_size_t, c_uint64, c_void_p

import numpy as np

from . import build as _build

HCL_H2D, HCL_D2H = 0, 1
HCL_OP_N, HCL_OP_T = 0, 1
HCL_UPLO_LOWER, HCL_UPLO_UPPER = 0, 1
HCL_DIAG_NONUNIT, HCL_DIAG_UNIT = 0, 1
HCL_SIDE_LEFT, HCL_SIDE_RIGHT = 0, 1

# every symbol include/hclooc.h declares (tests check the .so exports all of them)
EXPORTS = [
    "hclooc_plan", "hclooc_plan_ex", "hclooc_plan_trans", "hclooc_plan_resident", "hclooc_resident_schedule", "hclooc_shard_rows", "hclMatrixPartitioner", "hclooc_schedule", "hclooc_ctx_create", "hclooc_ctx_destroy",
    "hclooc_ctx_set_trace", "hclooc_ctx_get_trace", "hclooc_ctx_set_direct", "hclooc_ctx_set_debug", "hclooc_calibrate_link",
    "hclooc_dgemm", "hclooc_dgemm_ex", "hclooc_dgemm_t", "hclooc_dsyrk", "hclooc_dsyr2k", "hclooc_dtrsm", "hclooc_dtrsm_plan", "hclooc_dtrsm_side", "hclooc_dpotrf", "hclooc_dpotrf_plan", "hclooc_dgetrf", "hclooc_dgetrf_plan", "hclDgetrf", "hclooc_dtrmm", "hclooc_dsymm", "hclooc_dgemm_fig2", "hclooc_dgemm_nsteps", "hclMalloc", "hclFree", "hclGetMemSize", "hclStreamCreate",
    "hclStreamDestroy", "hclEventDestroy", "hclMemcpy", "hclMemcpyAsync", "hclMemcpy2DAsync",
    "hclDgemmAsync", "hclDgemmAsyncEx", "hclDgemmAsyncT", "hclDgemmNoAlloc", "hclDgemmNoAllocScratchBytes", "hclDtrsmAsync", "hclDpotrfAsync", "hclWaitEvent", "hclStreamSynchronize", "hclDeviceSynchronize",
    "hclooc_host_alloc", "hclooc_host_free", "hclooc_host_register", "hclooc_host_unregister",
    "hclooc_strerror", "hclooc_last_cuda_error", "hclooc_version", "hclooc_probe_fp64",
]


class ResidentPlan(ctypes.Structure):
    _fields_ = [("applies", c_int32), ("ring", c_int32), ("mb", c_int64), ("h", c_int64), ("kb", c_int64), ("npanels", c_int64),
                ("p_switch", c_int64), ("lda_dev", c_int64), ("ldb_dev", c_int64), ("ldc_dev", c_int64), ("workspace_bytes", c_uint64),
                ("t_flop_s", c_double), ("t_link_s", c_double), ("t_model_s", c_double),
                ("panel_k0", c_int64 * 128), ("panel_kk", c_int64 * 128)]


class Plan(ctypes.Structure):
    _fields_ = [("M", c_int64), ("N", c_int64), ("K", c_int64),
                ("mb", c_int64), ("nb", c_int64), ("kb", c_int64),
                ("h", c_int64), ("w", c_int64), ("kpanels", c_int64), ("n_steps", c_int64),
                ("n_sets", c_int32), ("n_bbuf", c_int32), ("beta_nonzero", c_int32), ("scale_only", c_int32),
                ("ksplit", c_int32), ("n_abuf", c_int32),
                ("lda_dev", c_int64), ("ldb_dev", c_int64), ("ldc_dev", c_int64),
                ("bytes_a_buf", c_uint64), ("bytes_b_buf", c_uint64), ("bytes_c_buf", c_uint64),
                ("workspace_bytes", c_uint64), ("bytes_h2d", c_uint64), ("bytes_d2h", c_uint64),
                ("n_copies_h2d", c_uint64), ("n_copies_d2h", c_uint64),
                ("flops", c_double), ("t_flop_s", c_double), ("t_link_s", c_double), ("t_model_s", c_double),
                ("n_scratch", c_int32), ("c_on_device", c_int32), ("bytes_scratch", c_uint64),
                ("direct", c_int32), ("direct_cm", c_int32), ("direct_cn", c_int32), ("tri", c_int32), ("resident", c_int32), ("trans", c_int32)]

    def asdict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


class Stats(ctypes.Structure):
    _fields_ = [("plan", Plan), ("bytes_h2d", c_uint64), ("bytes_d2h", c_uint64), ("n_kernels", c_uint64),
                ("n_copies_h2d", c_uint64), ("n_copies_d2h", c_uint64), ("t_total_s", c_double), ("t_enqueue_s", c_double)]

    def asdict(self):
        d = {k: getattr(self, k) for k, _ in self._fields_ if k != "plan"}
        d["plan"] = self.plan.asdict()
        return d


OP_DTYPE = np.dtype([("kind", "<i4"), ("stream", "<i4"), ("event", "<i4"), ("buf", "<i4"), ("buf2", "<i4"), ("buf3", "<i4"),
                     ("r0", "<i8"), ("nr", "<i8"), ("c0", "<i8"), ("nc", "<i8"), ("dev_r0", "<i8"),
                     ("k0", "<i8"), ("kk", "<i8"), ("step", "<i8"), ("beta", "<f8")], align=True)


class HclError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        msg = lib().hclooc_strerror(status).decode()
        extra = f", cuda error {lib().hclooc_last_cuda_error()}" if status == 3 else ""
        super().__init__(f"{where}: status {status} ({msg}{extra})")


_lib = None


def lib():
    """Load (building first if stale) libhclooc_b200.so.  Raises if that is impossible."""
    global _lib
    if _lib is None:
        L = ctypes.CDLL(_build.build())
        i64, dbl, vp, sz = c_int64, c_double, c_void_p, c_size_t
        L.hclooc_plan.argtypes = [i64, i64, i64, c_int, c_int, sz, POINTER(Plan)]
        L.hclooc_plan_resident.argtypes = [i64, i64, i64, c_int, sz, dbl, POINTER(ResidentPlan)]
        L.hclooc_resident_schedule.argtypes = [POINTER(ResidentPlan), i64, i64, i64, c_int, c_int, vp, sz, POINTER(sz)]
        L.hclooc_shard_rows.argtypes = [i64, c_int, c_int, i64, POINTER(i64), POINTER(i64)]
        L.hclooc_plan_ex.argtypes = [i64, i64, i64, c_int, c_int, sz, c_int, POINTER(Plan)]
        L.hclooc_plan_trans.argtypes = [i64, i64, i64, c_int, c_int, sz, c_int, c_int, c_int, POINTER(Plan)]
        L.hclMatrixPartitioner.argtypes = [i64, i64, i64, i64, POINTER(i64), POINTER(i64)]
        L.hclooc_schedule.argtypes = [POINTER(Plan), c_int, vp, sz, POINTER(sz)]
        L.hclooc_ctx_create.argtypes = [POINTER(vp), c_int, vp, sz, vp, vp, POINTER(vp), c_int]
        L.hclooc_ctx_destroy.argtypes = [vp]
        L.hclooc_ctx_set_trace.argtypes = [vp, c_int]
        L.hclooc_ctx_get_trace.argtypes = [vp, vp, sz, POINTER(sz)]
        L.hclooc_ctx_set_direct.argtypes = [vp, c_int]
        L.hclooc_ctx_set_debug.argtypes = [vp, c_uint64, c_int]
        L.hclooc_calibrate_link.argtypes = [vp, POINTER(c_double), POINTER(c_double), POINTER(c_double)]
        L.hclooc_dgemm.argtypes = [i64, i64, i64, dbl, vp, i64, vp, i64, dbl, vp, i64, sz]
        L.hclooc_dgemm_ex.argtypes = [vp, i64, i64, i64, dbl, vp, i64, vp, i64, dbl, vp, i64, sz, POINTER(Stats)]
        L.hclooc_dgemm_t.argtypes = [vp, c_int, c_int, i64, i64, i64, dbl, vp, i64, vp, i64, dbl, vp, i64, sz, POINTER(Stats)]
        L.hclooc_dsyrk.argtypes = [vp, c_int, c_int, i64, i64, dbl, vp, i64, dbl, vp, i64, sz, POINTER(Stats)]
        L.hclooc_dtrsm_plan.argtypes = [i64, i64, sz, c_int, POINTER(i64), POINTER(i64), POINTER(c_int), POINTER(ctypes.c_uint64)]
        L.hclooc_dtrsm.argtypes = [vp, c_int, c_int, c_int, i64, i64, dbl, vp, i64, vp, i64, sz, POINTER(Stats)]
        L.hclooc_dtrsm_side.argtypes = [vp, c_int, c_int, c_int, c_int, i64, i64, dbl, vp, i64, vp, i64, sz, POINTER(Stats)]
        L.hclooc_dtrmm.argtypes = [vp, c_int, c_int, c_int, c_int, i64, i64, dbl, vp, i64, vp, i64, sz, POINTER(Stats)]
        L.hclooc_dsymm.argtypes = [vp, c_int, c_int, i64, i64, dbl, vp, i64, vp, i64, dbl, vp, i64, sz, POINTER(Stats)]
        L.hclooc_dpotrf.argtypes = [vp, c_int, i64, vp, i64, sz, POINTER(i64), POINTER(Stats)]
        L.hclooc_dpotrf_plan.argtypes = [i64, sz, POINTER(i64), POINTER(ctypes.c_uint64)]
        L.hclooc_dgetrf.argtypes = [vp, i64, i64, vp, i64, vp, sz, POINTER(i64), POINTER(Stats)]
        L.hclooc_dgetrf_plan.argtypes = [i64, i64, sz, POINTER(i64), POINTER(ctypes.c_uint64)]
        L.hclDgetrf.argtypes = [i64, i64, vp, i64, vp, POINTER(i64), vp]
        L.hclooc_dsyr2k.argtypes = [vp, c_int, c_int, i64, i64, dbl, vp, i64, vp, i64, dbl, vp, i64, sz, POINTER(Stats)]
        L.hclooc_dgemm_nsteps.argtypes = [vp, i64, i64, i64, dbl, vp, i64, vp, i64, dbl, vp, i64, sz, c_int, POINTER(c_int), POINTER(Stats)]
        L.hclooc_dgemm_fig2.argtypes = [i64, i64, i64, dbl, vp, i64, vp, i64, dbl, vp, i64, sz, POINTER(Stats)]
        L.hclMalloc.argtypes = [POINTER(vp), sz]
        L.hclFree.argtypes = [vp]
        L.hclGetMemSize.argtypes = [c_int, POINTER(sz)]
        L.hclStreamCreate.argtypes = [POINTER(vp)]
        L.hclStreamDestroy.argtypes = [vp]
        L.hclEventDestroy.argtypes = [vp]
        L.hclMemcpy.argtypes = [vp, vp, sz, c_int]
        L.hclMemcpyAsync.argtypes = [vp, vp, sz, c_int, vp, POINTER(vp)]
        L.hclMemcpy2DAsync.argtypes = [vp, sz, vp, sz, sz, sz, c_int, vp, POINTER(vp)]
        L.hclDgemmAsync.argtypes = [i64, i64, i64, dbl, vp, i64, vp, i64, dbl, vp, i64, vp, POINTER(vp)]
        L.hclDgemmNoAlloc.argtypes = [i64, i64, i64, dbl, vp, i64, vp, i64, dbl, vp, i64, vp]
        L.hclDgemmNoAllocScratchBytes.argtypes = []
        L.hclDgemmNoAllocScratchBytes.restype = sz
        L.hclDgemmAsyncEx.argtypes = [i64, i64, i64, dbl, vp, i64, vp, i64, dbl, vp, i64, vp, POINTER(vp), c_int]
        L.hclDgemmAsyncT.argtypes = [c_int, c_int, i64, i64, i64, dbl, vp, i64, vp, i64, dbl, vp, i64, vp, POINTER(vp), c_int]
        L.hclDtrsmAsync.argtypes = [c_int, c_int, c_int, c_int, i64, i64, dbl, vp, i64, vp, i64, vp, POINTER(vp)]
        L.hclDpotrfAsync.argtypes = [c_int, i64, vp, i64, vp, vp, POINTER(vp)]
        L.hclWaitEvent.argtypes = [vp, vp]
        L.hclStreamSynchronize.argtypes = [vp]
        L.hclDeviceSynchronize.argtypes = [c_int]
        L.hclooc_host_alloc.argtypes = [sz]
        L.hclooc_host_alloc.restype = vp
        L.hclooc_host_free.argtypes = [vp]
        L.hclooc_host_register.argtypes = [vp, sz]
        L.hclooc_host_unregister.argtypes = [vp]
        L.hclooc_strerror.argtypes = [c_int]
        L.hclooc_strerror.restype = c_char_p
        L.hclooc_last_cuda_error.argtypes = []
        L.hclooc_version.restype = c_char_p
        L.hclooc_probe_fp64.argtypes = [c_int, c_int, dbl, POINTER(dbl)]
        for name in EXPORTS:
            if name not in ("hclooc_host_alloc", "hclooc_strerror", "hclooc_version"):
                getattr(L, name).restype = c_int
        _lib = L
    return _lib


def _ptr(x) -> int | None:
    """Address of a host/device buffer: int, None, numpy array, torch tensor or HostMatrix."""
    if x is None:
        return None
    if isinstance(x, int):
        return x
    if isinstance(x, HostMatrix):
        return x.ptr
    if isinstance(x, np.ndarray):
        return x.ctypes.data
    if hasattr(x, "data_ptr"):
        return x.data_ptr()
    if hasattr(x, "cuda_stream"):      # torch.cuda.Stream
        return x.cuda_stream
    raise TypeError(type(x))


def _check(status: int, where: str) -> None:
    if status != 0:
        raise HclError(status, where)


# ------------------------------------------------------------------ pinned host memory
def hclooc_host_alloc(nbytes: int) -> int:
    p = lib().hclooc_host_alloc(nbytes)
    if not p:
        raise HclError(4, "hclooc_host_alloc")
    return p


def hclooc_host_free(p) -> None:
    _check(lib().hclooc_host_free(_ptr(p)), "hclooc_host_free")


def hclooc_host_register(p, nbytes: int) -> None:
    _check(lib().hclooc_host_register(_ptr(p), nbytes), "hclooc_host_register")


def hclooc_host_unregister(p) -> None:
    _check(lib().hclooc_host_unregister(_ptr(p)), "hclooc_host_unregister")


class HostMatrix:
    """A rows x cols FP64 row-major matrix in pinned host memory (leading dimension ld >= cols),
    allocated with hclooc_host_alloc; `.array` is a numpy view of the whole rows x ld buffer and
    `.view` of the logical rows x cols part."""

    def __init__(self, rows: int, cols: int, ld: int | None = None):
        self.rows, self.cols, self.ld = rows, cols, (cols if ld is None else ld)
        assert self.ld >= cols
        self.nbytes = max(1, rows * self.ld) * 8
        # Pinning large buffers fails now and then with cudaErrorOperatingSystem on the B200 boxes when another CUDA process
        # has just exited (the driver still tearing its mappings down); the library retries for ~12 s, this convenience class
        # three more times, 5 s apart (HCLOOC_PIN_RETRIES overrides; 0 = fail at once), and says so on stderr.
        import os
        retries = int(os.environ.get("HCLOOC_PIN_RETRIES", "3"))
        for attempt in range(retries + 1):
            try:
                self.ptr = hclooc_host_alloc(self.nbytes)
                break
            except HclError:
                if attempt == retries or self.nbytes < (64 << 20):
                    raise
                import gc
                import sys
                import time
                print(f"HostMatrix: pinning {self.nbytes >> 20} MiB failed, retry {attempt + 1} of {retries} in 5 s", file=sys.stderr)
                gc.collect()
                time.sleep(5)
        buf = (ctypes.c_double * max(1, rows * self.ld)).from_address(self.ptr)
        self.array = np.frombuffer(buf, dtype=np.float64)[: rows * self.ld].reshape(rows, self.ld)
        self.view = self.array[:, :cols]

    def free(self):
        if self.ptr:
            self.array = self.view = None
            hclooc_host_free(self.ptr)
            self.ptr = 0

    def __del__(self):
        try:
            self.free()
        except Exception:
            pass


# ------------------------------------------------------------------ planner / schedule
def hclooc_plan(M, N, K, beta_nonzero, alpha_zero, device_budget_bytes) -> Plan:
    p = Plan()
    _check(lib().hclooc_plan(M, N, K, int(bool(beta_nonzero)), int(bool(alpha_zero)), device_budget_bytes, byref(p)), "hclooc_plan")
    return p


def hclooc_plan_ex(M, N, K, beta_nonzero, alpha_zero, device_budget_bytes, operands_on_device) -> Plan:
    p = Plan()
    _check(lib().hclooc_plan_ex(M, N, K, int(bool(beta_nonzero)), int(bool(alpha_zero)), device_budget_bytes,
                                int(operands_on_device), byref(p)), "hclooc_plan_ex")
    return p


def hclooc_plan_trans(M, N, K, beta_nonzero, alpha_zero, device_budget_bytes, operands_on_device, transa, transb) -> Plan:
    p = Plan()
    _check(lib().hclooc_plan_trans(M, N, K, int(bool(beta_nonzero)), int(bool(alpha_zero)), device_budget_bytes,
                                   int(operands_on_device), int(transa), int(transb), byref(p)), "hclooc_plan_trans")
    return p


def hclooc_shard_rows(M, world, rank, align=128):
    """(row0, rows) of the band of C (and A) that process `rank` of `world` owns."""
    r0, n = c_int64(), c_int64()
    _check(lib().hclooc_shard_rows(M, world, rank, align, byref(r0), byref(n)), "hclooc_shard_rows")
    return r0.value, n.value


def hclMatrixPartitioner(M, N, K, budget_elements):
    h, w = c_int64(), c_int64()
    _check(lib().hclMatrixPartitioner(M, N, K, budget_elements, byref(h), byref(w)), "hclMatrixPartitioner")
    return h.value, w.value


def hclooc_schedule(plan: Plan, n_compute: int = 8) -> np.ndarray:
    n = c_size_t()
    _check(lib().hclooc_schedule(byref(plan), n_compute, None, 0, byref(n)), "hclooc_schedule")
    ops = np.zeros(n.value, dtype=OP_DTYPE)
    assert OP_DTYPE.itemsize == 96
    _check(lib().hclooc_schedule(byref(plan), n_compute, ops.ctypes.data if n.value else None, n.value, byref(n)), "hclooc_schedule")
    return ops


# ------------------------------------------------------------------ context and the operation
def hclooc_ctx_create(device=0, d_workspace=None, workspace_bytes=0, stream_h2d=None, stream_d2h=None, compute_streams=None) -> int:
    ctx = c_void_p()
    n = len(compute_streams) if compute_streams else 0
    arr = (c_void_p * n)(*[_ptr(s) for s in compute_streams]) if n else None
    _check(lib().hclooc_ctx_create(byref(ctx), device, _ptr(d_workspace), workspace_bytes, _ptr(stream_h2d),
                                   _ptr(stream_d2h), arr, n), "hclooc_ctx_create")
    return ctx.value


def hclooc_ctx_destroy(ctx) -> None:
    _check(lib().hclooc_ctx_destroy(ctx), "hclooc_ctx_destroy")


TRACE_DTYPE = np.dtype([("kind", "<i4"), ("stream", "<i4"), ("step", "<i8"), ("bytes", "<u8"), ("flops", "<f8"),
                        ("t_start_ms", "<f8"), ("t_end_ms", "<f8")], align=True)


def hclooc_ctx_set_trace(ctx, enable: bool) -> None:
    _check(lib().hclooc_ctx_set_trace(ctx, int(bool(enable))), "hclooc_ctx_set_trace")


def hclooc_ctx_set_direct(ctx, mode: int) -> None:
    _check(lib().hclooc_ctx_set_direct(ctx, int(mode)), "hclooc_ctx_set_direct")


def hclooc_calibrate_link(ctx=None):
    """(h2d, d2h, duplex) in GB/s as measured on this box; the planner's cost model uses them from now on."""
    a, b, c = c_double(), c_double(), c_double()
    _check(lib().hclooc_calibrate_link(ctx, byref(a), byref(b), byref(c)), "hclooc_calibrate_link")
    return a.value, b.value, c.value


def hclooc_ctx_set_debug(ctx, jitter_seed: int, poison) -> None:
    _check(lib().hclooc_ctx_set_debug(ctx, int(jitter_seed), int(poison)), "hclooc_ctx_set_debug")


def hclooc_ctx_get_trace(ctx) -> np.ndarray:
    n = c_size_t()
    _check(lib().hclooc_ctx_get_trace(ctx, None, 0, byref(n)), "hclooc_ctx_get_trace")
    recs = np.zeros(n.value, dtype=TRACE_DTYPE)
    assert TRACE_DTYPE.itemsize == 48
    if n.value:
        _check(lib().hclooc_ctx_get_trace(ctx, recs.ctypes.data, n.value, byref(n)), "hclooc_ctx_get_trace")
    return recs


def hclooc_plan_resident(M, N, K, beta_nonzero, device_budget_bytes, t_slice_model_s=0.0) -> ResidentPlan:
    """The resident schedule's shape for a call whose matrices fit the budget (include/hclooc.h); .applies says whether hclooc_dgemm takes it."""
    out = ResidentPlan()
    _check(lib().hclooc_plan_resident(M, N, K, int(bool(beta_nonzero)), device_budget_bytes, float(t_slice_model_s), byref(out)), "hclooc_plan_resident")
    return out


def hclooc_resident_schedule(plan: ResidentPlan, M, N, K, beta_nonzero, n_compute=8) -> np.ndarray:
    """The operations hclooc_dgemm enqueues for the resident schedule, in host issue order (OP_DTYPE records)."""
    n = c_size_t()
    _check(lib().hclooc_resident_schedule(byref(plan), M, N, K, int(bool(beta_nonzero)), n_compute, None, 0, byref(n)), "hclooc_resident_schedule")
    ops = np.zeros(n.value, dtype=OP_DTYPE)
    _check(lib().hclooc_resident_schedule(byref(plan), M, N, K, int(bool(beta_nonzero)), n_compute, ops.ctypes.data if n.value else None, n.value, byref(n)),
           "hclooc_resident_schedule")
    return ops


def hclooc_dgemm(M, N, K, alpha, A, lda, B, ldb, beta, C, ldc, device_budget_bytes) -> None:
    _check(lib().hclooc_dgemm(M, N, K, alpha, _ptr(A), lda, _ptr(B), ldb, beta, _ptr(C), ldc, device_budget_bytes), "hclooc_dgemm")


def hclooc_dgemm_ex(ctx, M, N, K, alpha, A, lda, B, ldb, beta, C, ldc, device_budget_bytes, want_stats=True):
    st = Stats()
    _check(lib().hclooc_dgemm_ex(ctx, M, N, K, alpha, _ptr(A), lda, _ptr(B), ldb, beta, _ptr(C), ldc,
                                 device_budget_bytes, byref(st) if want_stats else None), "hclooc_dgemm_ex")
    return st if want_stats else None


def hclooc_dgemm_t(ctx, transa, transb, M, N, K, alpha, A, lda, B, ldb, beta, C, ldc, device_budget_bytes, want_stats=True):
    """C = alpha*op(A)*op(B) + beta*C; transa / transb: HCL_OP_N (0) or HCL_OP_T (1)."""
    st = Stats()
    _check(lib().hclooc_dgemm_t(ctx, int(transa), int(transb), M, N, K, alpha, _ptr(A), lda, _ptr(B), ldb, beta, _ptr(C), ldc,
                                device_budget_bytes, byref(st) if want_stats else None), "hclooc_dgemm_t")
    return st if want_stats else None


def hclooc_dsyrk(ctx, uplo, trans, N, K, alpha, A, lda, beta, C, ldc, device_budget_bytes, want_stats=True):
    """C = alpha*A*A^T + beta*C (trans = HCL_OP_N) or alpha*A^T*A + beta*C (HCL_OP_T) on the `uplo` triangle of C."""
    st = Stats()
    _check(lib().hclooc_dsyrk(ctx, int(uplo), int(trans), N, K, alpha, _ptr(A), lda, beta, _ptr(C), ldc,
                              device_budget_bytes, byref(st) if want_stats else None), "hclooc_dsyrk")
    return st if want_stats else None


def hclooc_dsyr2k(ctx, uplo, trans, N, K, alpha, A, lda, B, ldb, beta, C, ldc, device_budget_bytes, want_stats=True):
    """C = alpha*A*B^T + alpha*B*A^T + beta*C (trans = HCL_OP_N; the transposed forms for HCL_OP_T) on the `uplo` triangle."""
    st = Stats()
    _check(lib().hclooc_dsyr2k(ctx, int(uplo), int(trans), N, K, alpha, _ptr(A), lda, _ptr(B), ldb, beta, _ptr(C), ldc,
                               device_budget_bytes, byref(st) if want_stats else None), "hclooc_dsyr2k")
    return st if want_stats else None


def hclooc_dtrsm_plan(M, N, device_budget_bytes, library_owned=True):
    """(NB, chunk, resident, device_bytes) of hclooc_dtrsm under a budget; host arithmetic only."""
    nb, ch, res, by = c_int64(), c_int64(), c_int(), c_uint64()
    _check(lib().hclooc_dtrsm_plan(M, N, device_budget_bytes, int(bool(library_owned)), byref(nb), byref(ch), byref(res), byref(by)),
           "hclooc_dtrsm_plan")
    return nb.value, ch.value, res.value, by.value


def hclooc_dtrsm(ctx, uplo, trans, diag, M, N, alpha, A, lda, B, ldb, device_budget_bytes, want_stats=True):
    """Solve op(T) X = alpha*B in place (X overwrites B); T = the `uplo` triangle of the M x M matrix A, diag: HCL_DIAG_*."""
    st = Stats()
    _check(lib().hclooc_dtrsm(ctx, int(uplo), int(trans), int(diag), M, N, alpha, _ptr(A), lda, _ptr(B), ldb,
                              device_budget_bytes, byref(st) if want_stats else None), "hclooc_dtrsm")
    return st if want_stats else None


def hclooc_dtrsm_side(ctx, side, uplo, trans, diag, M, N, alpha, A, lda, B, ldb, device_budget_bytes, want_stats=True):
    st = Stats()
    _check(lib().hclooc_dtrsm_side(ctx, side, uplo, trans, diag, M, N, alpha, _ptr(A), lda, _ptr(B), ldb, device_budget_bytes,
                                   byref(st) if want_stats else None), "hclooc_dtrsm_side")
    return st if want_stats else None


def hclooc_dtrmm(ctx, side, uplo, trans, diag, M, N, alpha, A, lda, B, ldb, device_budget_bytes):
    st = Stats()
    _check(lib().hclooc_dtrmm(ctx, side, uplo, trans, diag, M, N, alpha, _ptr(A), lda, _ptr(B), ldb, device_budget_bytes, byref(st)), "hclooc_dtrmm")
    return st


def hclooc_dsymm(ctx, side, uplo, M, N, alpha, A, lda, B, ldb, beta, C, ldc, device_budget_bytes):
    st = Stats()
    _check(lib().hclooc_dsymm(ctx, side, uplo, M, N, alpha, _ptr(A), lda, _ptr(B), ldb, beta, _ptr(C), ldc, device_budget_bytes, byref(st)), "hclooc_dsymm")
    return st


def hclooc_dpotrf(ctx, uplo, N, A, lda, device_budget_bytes):
    """Returns (info, stats)."""
    st, info = Stats(), c_int64(0)
    _check(lib().hclooc_dpotrf(ctx, uplo, N, _ptr(A), lda, device_budget_bytes, byref(info), byref(st)), "hclooc_dpotrf")
    return int(info.value), st


def hclooc_dpotrf_plan(N, device_budget_bytes):
    """(NB, panel_bytes)."""
    nb, pb = c_int64(), ctypes.c_uint64()
    _check(lib().hclooc_dpotrf_plan(N, device_budget_bytes, byref(nb), byref(pb)), "hclooc_dpotrf_plan")
    return int(nb.value), int(pb.value)


def hclooc_dgetrf(ctx, M, N, A, lda, device_budget_bytes):
    """Returns (ipiv, info, stats): ipiv = numpy int64 array of min(M, N) 0-based rows."""
    import numpy as np
    st, info = Stats(), c_int64(0)
    ipiv = np.zeros(max(min(M, N), 1), dtype=np.int64)
    _check(lib().hclooc_dgetrf(ctx, M, N, _ptr(A), lda, ipiv.ctypes.data, device_budget_bytes, byref(info), byref(st)), "hclooc_dgetrf")
    return ipiv[:min(M, N)], int(info.value), st


def hclooc_dgetrf_plan(M, N, device_budget_bytes):
    """(NB, reserved_bytes)."""
    nb, rb = c_int64(), ctypes.c_uint64()
    _check(lib().hclooc_dgetrf_plan(M, N, device_budget_bytes, byref(nb), byref(rb)), "hclooc_dgetrf_plan")
    return int(nb.value), int(rb.value)


def hclDgetrf(M, N, dA, lda, stream=None):
    """In-core LU of a device matrix; returns (ipiv, info).  Synchronous."""
    import numpy as np
    info = c_int64(0)
    ipiv = np.zeros(max(min(M, N), 1), dtype=np.int64)
    _check(lib().hclDgetrf(M, N, _ptr(dA), lda, ipiv.ctypes.data, byref(info), _ptr(stream)), "hclDgetrf")
    return ipiv[:min(M, N)], int(info.value)


def hclooc_dgemm_nsteps(ctx, M, N, K, alpha, A, lda, B, ldb, beta, C, ldc, device_budget_bytes, nsteps, step):
    """One call of an nsteps sequence; returns (next step, Stats)."""
    st, sp = Stats(), c_int(step)
    _check(lib().hclooc_dgemm_nsteps(ctx, M, N, K, alpha, _ptr(A), lda, _ptr(B), ldb, beta, _ptr(C), ldc,
                                     device_budget_bytes, nsteps, byref(sp), byref(st)), "hclooc_dgemm_nsteps")
    return sp.value, st


def hclooc_dgemm_fig2(M, N, K, alpha, A, lda, B, ldb, beta, C, ldc, device_budget_bytes, want_stats=True):
    """The paper's Figure 2 pipeline over the hcl* runtime calls (two streams, five event families)."""
    st = Stats()
    _check(lib().hclooc_dgemm_fig2(M, N, K, alpha, _ptr(A), lda, _ptr(B), ldb, beta, _ptr(C), ldc,
                                   device_budget_bytes, byref(st) if want_stats else None), "hclooc_dgemm_fig2")
    return st if want_stats else None


# ------------------------------------------------------------------ the runtime the paper abstracts
def hclMalloc(nbytes: int) -> int:
    p = c_void_p()
    _check(lib().hclMalloc(byref(p), nbytes), "hclMalloc")
    return p.value or 0


def hclFree(dptr) -> None:
    _check(lib().hclFree(_ptr(dptr)), "hclFree")


def hclGetMemSize(device: int = 0) -> int:
    n = c_size_t()
    _check(lib().hclGetMemSize(device, byref(n)), "hclGetMemSize")
    return n.value


def hclStreamCreate() -> int:
    s = c_void_p()
    _check(lib().hclStreamCreate(byref(s)), "hclStreamCreate")
    return s.value


def hclStreamDestroy(s) -> None:
    _check(lib().hclStreamDestroy(_ptr(s)), "hclStreamDestroy")


def hclEventDestroy(e) -> None:
    _check(lib().hclEventDestroy(e), "hclEventDestroy")


def hclMemcpy(dst, src, nbytes, direction) -> None:
    _check(lib().hclMemcpy(_ptr(dst), _ptr(src), nbytes, direction), "hclMemcpy")


def _ev(want_event, event):
    if event is not None:
        return c_void_p(event)
    return c_void_p() if want_event else None


def hclMemcpyAsync(dst, src, nbytes, direction, stream, want_event=False, event=None):
    """Returns the event handle (int) tied to this call when want_event or event is given, else None."""
    ev = _ev(want_event, event)
    _check(lib().hclMemcpyAsync(_ptr(dst), _ptr(src), nbytes, direction, _ptr(stream), byref(ev) if ev is not None else None), "hclMemcpyAsync")
    return ev.value if ev is not None else None


def hclMemcpy2DAsync(dst, dpitch, src, spitch, width_bytes, rows, direction, stream, want_event=False, event=None):
    ev = _ev(want_event, event)
    _check(lib().hclMemcpy2DAsync(_ptr(dst), dpitch, _ptr(src), spitch, width_bytes, rows, direction, _ptr(stream),
                                  byref(ev) if ev is not None else None), "hclMemcpy2DAsync")
    return ev.value if ev is not None else None


def hclDgemmAsyncEx(M, N, K, alpha, dA, lda, dB, ldb, beta, dC, ldc, stream=None, want_event=False, event=None, variant=0):
    ev = _ev(want_event, event)
    _check(lib().hclDgemmAsyncEx(M, N, K, alpha, _ptr(dA), lda, _ptr(dB), ldb, beta, _ptr(dC), ldc, _ptr(stream),
                                 byref(ev) if ev is not None else None, variant), "hclDgemmAsyncEx")
    return ev.value if ev is not None else None


def hclDgemmAsyncT(transa, transb, M, N, K, alpha, dA, lda, dB, ldb, beta, dC, ldc, stream=None, want_event=False, event=None, variant=0):
    ev = _ev(want_event, event)
    _check(lib().hclDgemmAsyncT(int(transa), int(transb), M, N, K, alpha, _ptr(dA), lda, _ptr(dB), ldb, beta, _ptr(dC), ldc, _ptr(stream),
                                byref(ev) if ev is not None else None, variant), "hclDgemmAsyncT")
    return ev.value if ev is not None else None


def hclDgemmAsync(M, N, K, alpha, dA, lda, dB, ldb, beta, dC, ldc, stream=None, want_event=False, event=None):
    ev = _ev(want_event, event)
    _check(lib().hclDgemmAsync(M, N, K, alpha, _ptr(dA), lda, _ptr(dB), ldb, beta, _ptr(dC), ldc, _ptr(stream),
                               byref(ev) if ev is not None else None), "hclDgemmAsync")
    return ev.value if ev is not None else None


def hclDgemmNoAlloc(M, N, K, alpha, dA, lda, dB, ldb, beta, dC, ldc, stream=None):
    """The in-core DGEMM that allocates nothing (include/hclooc.h): scratch in a static device array shared by every call."""
    _check(lib().hclDgemmNoAlloc(M, N, K, alpha, _ptr(dA), lda, _ptr(dB), ldb, beta, _ptr(dC), ldc, _ptr(stream)), "hclDgemmNoAlloc")


def hclDgemmNoAllocScratchBytes():
    return int(lib().hclDgemmNoAllocScratchBytes())


def hclDtrsmAsync(side, uplo, trans, diag, M, N, alpha, dA, lda, dB, ldb, stream=None, want_event=False, event=None):
    ev = _ev(want_event, event)
    _check(lib().hclDtrsmAsync(side, uplo, trans, diag, M, N, alpha, _ptr(dA), lda, _ptr(dB), ldb, _ptr(stream), byref(ev) if ev is not None else None), "hclDtrsmAsync")
    return ev.value if ev is not None else None


def hclDpotrfAsync(uplo, N, dA, lda, d_info, stream=None, want_event=False, event=None):
    ev = _ev(want_event, event)
    _check(lib().hclDpotrfAsync(uplo, N, _ptr(dA), lda, _ptr(d_info), _ptr(stream), byref(ev) if ev is not None else None), "hclDpotrfAsync")
    return ev.value if ev is not None else None


def hclWaitEvent(stream, event) -> None:
    _check(lib().hclWaitEvent(_ptr(stream), event), "hclWaitEvent")


def hclStreamSynchronize(stream=None) -> None:
    _check(lib().hclStreamSynchronize(_ptr(stream)), "hclStreamSynchronize")


def hclDeviceSynchronize(device: int = 0) -> None:
    _check(lib().hclDeviceSynchronize(device), "hclDeviceSynchronize")


def hclooc_strerror(status: int) -> str:
    return lib().hclooc_strerror(status).decode()


def hclooc_last_cuda_error() -> int:
    return lib().hclooc_last_cuda_error()


def hclooc_probe_fp64(kind: int = 0, ctas_per_sm: int = 4, seconds: float = 1.0) -> float:
    """Measured FP64 rate (TFLOP/s) of register-resident DMMA (kind 0) or DFMA (kind 1) chains on the current device."""
    out = c_double(0.0)
    _check(lib().hclooc_probe_fp64(kind, ctas_per_sm, seconds, byref(out)), "hclooc_probe_fp64")
    return out.value


def hclooc_version() -> str:
    return lib().hclooc_version().decode()
