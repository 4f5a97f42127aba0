"""paper_1901_09266_b200 — B200-native SPGD/NNLS hot path of Ma & Qian (arXiv 1901.09266).

Thin ctypes binding over the C ABI of ``include/dode.h`` (argument marshalling only: every step
of the path runs in the library's CUDA kernels).  PyTorch supplies device memory and streams.
There is no CPU fallback: if ``libdode.so`` is missing or fails to load, every call raises.
``paper_1901_09266_b200.synth`` (seeded input generators) does not need the library.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
SO_PATH = os.path.join(_HERE, "libdode.so")

DODE_OK, DODE_EINVAL, DODE_ENOMEM, DODE_ECUDA = 0, -1, -2, -3
DODE_DENSE, DODE_CSR = 0, 1

DODE_OPT_TC_MIN_B, DODE_OPT_LANES, DODE_OPT_TC_KSPLIT, DODE_OPT_PDL, DODE_OPT_TC_BSTAGES, DODE_OPT_TC_PAIR = 0, 1, 2, 3, 4, 5

EXPORTS = ["dode_create", "dode_set_option", "dode_reserve", "dode_spgd_step", "dode_spgd_step_host", "dode_adagrad_step", "dode_adagrad_reset", "dode_join", "dode_dar_build", "dode_assignment_build", "dode_assignment_build_csr", "dode_objective", "dode_r2", "dode_get_q", "dode_set_q",
           "dode_apply", "dode_apply_t", "dode_lipschitz", "dode_timing_enable", "dode_timing_read", "dode_probe_fp32_peak", "dode_visit_static", "dode_launch_count", "dode_last_path", "dode_sync",
           "dode_destroy", "dode_last_error"]


class DodeError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"dode error {code}: {msg}")
        self.code = code


class dode_dims(C.Structure):
    _fields_ = [(k, C.c_int32) for k in ("N", "L", "T", "H", "C", "D", "storage")]


class dode_dar(C.Structure):
    _fields_ = [("dense", C.c_void_p), ("blk_off", C.c_void_p), ("row_ptr", C.c_void_p),
                ("col_idx", C.c_void_p), ("val", C.c_void_p), ("nnz", C.c_int64)]


_lib = None


def lib():
    """Loads libdode.so (never builds, never falls back)."""
    global _lib
    if _lib is None:
        if not os.path.exists(SO_PATH):
            raise ImportError(f"{SO_PATH} is missing: run `python -c 'import __graft_entry__ as g; g.build()'` "
                              "(there is no CPU fallback)")
        L = C.CDLL(SO_PATH)
        vp, i32, f32 = C.c_void_p, C.c_int32, C.c_float
        L.dode_create.argtypes = [C.POINTER(vp), C.POINTER(dode_dims), C.POINTER(dode_dar), vp, vp, f32, vp]
        L.dode_spgd_step.argtypes = [vp, vp, i32, f32]
        L.dode_spgd_step_host.argtypes = [vp, vp, i32, f32, vp, vp]
        L.dode_adagrad_step.argtypes = [vp, vp, i32, f32, f32, vp]
        L.dode_adagrad_reset.argtypes = [vp]
        L.dode_join.argtypes = [vp]
        L.dode_set_option.argtypes = [vp, i32, i32]
        L.dode_reserve.argtypes = [vp, i32]
        L.dode_dar_build.argtypes = [i32, i32, i32, i32, vp, vp, vp, vp, C.c_double, vp, vp]
        L.dode_assignment_build.argtypes = [i32, i32, i32, i32, vp, vp, vp, vp, vp, C.c_double, C.c_double, vp, vp]
        L.dode_assignment_build_csr.argtypes = [i32, i32, i32, i32, vp, vp, vp, vp, vp, C.c_double, C.c_double,
                                                vp, vp, vp, vp, C.c_int64, vp, vp]
        L.dode_objective.argtypes = [vp, vp, i32, vp, vp]
        L.dode_get_q.argtypes = [vp, i32, vp, i32]
        L.dode_set_q.argtypes = [vp, i32, vp, i32]
        L.dode_r2.argtypes = [vp, vp, i32, vp, vp]
        L.dode_apply.argtypes = [vp, i32, vp, vp]
        L.dode_apply_t.argtypes = [vp, i32, vp, vp]
        L.dode_lipschitz.argtypes = [vp, i32, i32, vp]
        L.dode_timing_enable.argtypes = [vp, i32]
        L.dode_timing_read.argtypes = [vp, i32, vp, vp, i32]
        L.dode_probe_fp32_peak.argtypes = [i32, vp, vp]
        L.dode_visit_static.argtypes = [i32, i32, i32, i32, vp, vp, vp, f32, vp]
        L.dode_launch_count.argtypes = [vp]
        L.dode_launch_count.restype = C.c_int64
        L.dode_last_path.argtypes = [vp]
        L.dode_last_path.restype = C.c_char_p
        L.dode_sync.argtypes = [vp]
        L.dode_destroy.argtypes = [vp]
        L.dode_destroy.restype = None
        L.dode_last_error.argtypes = [vp]
        L.dode_last_error.restype = C.c_char_p
        _lib = L
    return _lib


def _chk(h, rc: int):
    if rc != 0:
        raise DodeError(rc, lib().dode_last_error(h).decode())


def _days(days) -> np.ndarray:
    return np.ascontiguousarray(days, dtype=np.int32)


# Shapes of the ctx (binding-side argument validation only) and host tensors that asynchronous calls still use:
# keyed by the handle's address; released by the next synchronising call.
_shape = {}
_keep = {}


def _key(h) -> int:
    return int(h.value) if isinstance(h, C.c_void_p) else int(h)


def _release(h) -> None:
    _keep.pop(_key(h), None)


def _host(t, shape, what):
    import torch
    if not (isinstance(t, torch.Tensor) and not t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()
            and tuple(t.shape) == tuple(shape)):
        raise TypeError(f"{what} must be a contiguous CPU float32 tensor of shape {tuple(shape)}")
    return C.c_void_p(t.data_ptr())


def _any(t, shape, what):
    import torch
    if not (isinstance(t, torch.Tensor) and t.dtype == torch.float32 and t.is_contiguous() and tuple(t.shape) == tuple(shape)):
        raise TypeError(f"{what} must be a contiguous float32 tensor of shape {tuple(shape)}")
    return C.c_void_p(t.data_ptr())


def _dev(t, dtype, what):
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.is_contiguous() and t.dtype == dtype):
        raise TypeError(f"{what} must be a contiguous CUDA tensor of {dtype}")
    return C.c_void_p(t.data_ptr())


def dode_create(N: int, L: int, T: int, H: int, Cn: int, D: int, labels, x, q0: float = 1.0, *,
                dense=None, csr=None, stream: Optional[int] = None):
    """a0.  ``dense``: CUDA fp32 [C][T][H+1][L][N]; or ``csr``: object with CUDA tensors blk_off (int64),
    row_ptr (int32), col_idx (int32), val (fp32).  ``labels``: host int32 [D].  ``x``: CUDA fp32 [D][T][L].
    ``stream``: raw cudaStream_t (default: torch's current stream).  Returns an opaque handle."""
    import torch
    if (dense is None) == (csr is None):
        raise ValueError("give exactly one of dense= or csr=")
    dar = dode_dar()
    if dense is not None:
        if tuple(dense.shape) != (Cn, T, H + 1, L, N):
            raise ValueError(f"dense R has shape {tuple(dense.shape)}, expected {(Cn, T, H + 1, L, N)}")
        dar.dense = _dev(dense, torch.float32, "dense").value
        storage = DODE_DENSE
    else:
        dar.blk_off = _dev(csr.blk_off, torch.int64, "blk_off").value
        dar.row_ptr = _dev(csr.row_ptr, torch.int32, "row_ptr").value
        dar.col_idx = _dev(csr.col_idx, torch.int32, "col_idx").value
        dar.val = _dev(csr.val, torch.float32, "val").value
        dar.nnz = int(csr.val.numel())
        storage = DODE_CSR
    if tuple(x.shape) != (D, T, L):
        raise ValueError(f"x has shape {tuple(x.shape)}, expected {(D, T, L)}")
    lab = np.ascontiguousarray(labels, dtype=np.int32)
    if lab.shape != (D,):
        raise ValueError("labels must have D entries")
    dims = dode_dims(N, L, T, H, Cn, D, storage)
    if stream is None:
        stream = torch.cuda.current_stream().cuda_stream
    h = C.c_void_p()
    rc = lib().dode_create(C.byref(h), C.byref(dims), C.byref(dar), lab.ctypes.data, _dev(x, torch.float32, "x"),
                           C.c_float(q0), C.c_void_p(stream))
    if rc != 0:
        raise DodeError(rc, lib().dode_last_error(None).decode())
    _shape[_key(h)] = (N, L, T, H, Cn, D)
    return h


def dode_set_option(h, option: int, value: int) -> None:
    """Kernel-selection options of this ctx (DODE_OPT_*; include/dode.h).  Results stay valid for every value."""
    _chk(h, lib().dode_set_option(h, int(option), int(value)))


def dode_reserve(h, max_days: int) -> None:
    """Pre-allocates dode_spgd_step's scratch for minibatches of up to ``max_days`` days.  Synchronises."""
    _chk(h, lib().dode_reserve(h, int(max_days)))
    _release(h)


def dode_spgd_step(h, days, eta: float) -> None:
    """a1-a4: one SPGD iteration on ``days`` (host ints, distinct, one cluster).  Asynchronous."""
    d = _days(days)
    _chk(h, lib().dode_spgd_step(h, d.ctypes.data, d.size, C.c_float(eta)))


def dode_dar_build(N: int, L: int, T: int, H: int, path_ptr, path_links, link_len, speed, dt: float, R_out) -> None:
    """NEXT-4: DAR blocks [T][H+1][L][N] of one day from link speeds (Eq. 17-18).  All tensors on the
    GPU: path_ptr/path_links int32, link_len [L] and speed [T][L] float32, R_out float32 (overwritten).  Asynchronous."""
    import torch
    for t, dt_ in ((path_ptr, torch.int32), (path_links, torch.int32), (link_len, torch.float32), (speed, torch.float32),
                   (R_out, torch.float32)):
        assert t.is_cuda and t.dtype == dt_ and t.is_contiguous()
    assert path_ptr.numel() == N + 1 and link_len.numel() == L and speed.shape == (T, L) and R_out.numel() == T * (H + 1) * L * N
    rc = lib().dode_dar_build(N, L, T, H, C.c_void_p(path_ptr.data_ptr()), C.c_void_p(path_links.data_ptr()),
                              C.c_void_p(link_len.data_ptr()), C.c_void_p(speed.data_ptr()), C.c_double(dt),
                              C.c_void_p(R_out.data_ptr()), C.c_void_p(torch.cuda.current_stream().cuda_stream))
    if rc != DODE_OK:
        raise DodeError(rc, lib().dode_last_error(None).decode())


STATIC_SCRATCH_FLOATS = 1 << 18          # include/dode.h: DODE_STATIC_SCRATCH_FLOATS


def dode_visit_static(R, q, x, eta: float) -> None:
    """One visit of one day with NO allocation (include/dode.h: dode_visit_static): R [T][H+1][L][N], q [T][N] (updated in
    place), x [T][L], float32 CUDA tensors; the residual lives in the library's static device array, so T*L must not
    exceed STATIC_SCRATCH_FLOATS (DodeError otherwise).  Runs on torch's current stream; asynchronous."""
    import torch
    for t in (R, q, x):
        assert t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()
    T, H1, L, N = R.shape
    assert q.shape == (T, N) and x.shape == (T, L)
    rc = lib().dode_visit_static(N, L, T, H1 - 1, C.c_void_p(R.data_ptr()), C.c_void_p(q.data_ptr()),
                                 C.c_void_p(x.data_ptr()), C.c_float(eta), C.c_void_p(torch.cuda.current_stream().cuda_stream))
    if rc != DODE_OK:
        raise DodeError(rc, lib().dode_last_error(None).decode())


def dode_assignment_build(N: int, L: int, T: int, H: int, od_ptr, path_ptr, path_links, link_len, speed, dt: float,
                          theta: float, R_out) -> None:
    """NEXT-4 with route choice: B = delta*rho*p [T][H+1][L][N] of one pattern, several paths per OD, Logit shares
    (Eq. 37, 41).  All tensors on the GPU (int32 / float32); R_out is overwritten.  Asynchronous."""
    import torch
    for t, dt_ in ((od_ptr, torch.int32), (path_ptr, torch.int32), (path_links, torch.int32), (link_len, torch.float32),
                   (speed, torch.float32), (R_out, torch.float32)):
        assert t.is_cuda and t.dtype == dt_ and t.is_contiguous()
    assert od_ptr.numel() == N + 1 and link_len.numel() == L and speed.shape == (T, L) and R_out.numel() == T * (H + 1) * L * N
    rc = lib().dode_assignment_build(N, L, T, H, C.c_void_p(od_ptr.data_ptr()), C.c_void_p(path_ptr.data_ptr()),
                                     C.c_void_p(path_links.data_ptr()), C.c_void_p(link_len.data_ptr()),
                                     C.c_void_p(speed.data_ptr()), C.c_double(dt), C.c_double(theta),
                                     C.c_void_p(R_out.data_ptr()), C.c_void_p(torch.cuda.current_stream().cuda_stream))
    if rc != DODE_OK:
        raise DodeError(rc, lib().dode_last_error(None).decode())


def dode_assignment_build_csr(N: int, L: int, T: int, H: int, od_ptr, path_ptr, path_links, link_len, speed, dt: float,
                              theta: float = 0.0):
    """NEXT-4 for large networks: the operator of one pattern in the boundary CSR format.  ``od_ptr`` None = one path per
    OD (dode_dar_build's operator).  All inputs on the GPU (int32 / float32).  Returns an object with CUDA tensors
    blk_off (int64 [T*(H+1)+1]), row_ptr (int32 [T*(H+1)][L+1]), col_idx (int32 [nnz]), val (float32 [nnz]) — what
    dode_create(csr=...) takes for a one-cluster problem.  Synchronises."""
    import torch
    from types import SimpleNamespace
    for t, dt_ in ((path_ptr, torch.int32), (path_links, torch.int32), (link_len, torch.float32), (speed, torch.float32)):
        assert t.is_cuda and t.dtype == dt_ and t.is_contiguous()
    assert link_len.numel() == L and speed.shape == (T, L)
    odp = None
    if od_ptr is not None:
        assert od_ptr.is_cuda and od_ptr.dtype == torch.int32 and od_ptr.numel() == N + 1
        odp = C.c_void_p(od_ptr.data_ptr())
    dev = speed.device
    blk_off = torch.empty(T * (H + 1) + 1, dtype=torch.int64, device=dev)
    row_ptr = torch.empty((T * (H + 1), L + 1), dtype=torch.int32, device=dev)
    stream = C.c_void_p(torch.cuda.current_stream().cuda_stream)
    nnz = C.c_int64()

    def call(col, val, cap):
        return lib().dode_assignment_build_csr(
            N, L, T, H, odp, C.c_void_p(path_ptr.data_ptr()), C.c_void_p(path_links.data_ptr()),
            C.c_void_p(link_len.data_ptr()), C.c_void_p(speed.data_ptr()), C.c_double(dt), C.c_double(theta),
            C.c_void_p(blk_off.data_ptr()), C.c_void_p(row_ptr.data_ptr()),
            None if col is None else C.c_void_p(col.data_ptr()), None if val is None else C.c_void_p(val.data_ptr()),
            C.c_int64(cap), C.byref(nnz), stream)

    rc = call(None, None, 0)                       # sizing call
    if rc not in (DODE_OK, DODE_ENOMEM):
        raise DodeError(rc, lib().dode_last_error(None).decode())
    cap = max(1, nnz.value)
    col = torch.empty(cap, dtype=torch.int32, device=dev)
    val = torch.empty(cap, dtype=torch.float32, device=dev)
    rc = call(col, val, cap)
    if rc != DODE_OK:
        raise DodeError(rc, lib().dode_last_error(None).decode())
    return SimpleNamespace(blk_off=blk_off, row_ptr=row_ptr, col_idx=col[:nnz.value], val=val[:nnz.value], nnz=nnz.value)


def dode_join(h) -> None:
    """Makes the ctx stream wait for every step issued so far (asynchronous)."""
    _chk(h, lib().dode_join(h))


def dode_adagrad_step(h, days, eta: float, eps: float = 1e-10, row_mask=None) -> None:
    """NEXT-1: Alg. 1 as printed — row-chunk residual mask + Adagrad + projection.  ``row_mask``:
    CUDA uint8 tensor [n][T][L] by position in ``days`` (non-zero = row in the chunk) or None.  Asynchronous."""
    d = _days(days)
    mp = None
    if row_mask is not None:
        N, L, T = _shape[_key(h)][:3]
        if not (row_mask.is_cuda and row_mask.element_size() == 1 and row_mask.is_contiguous()
                and row_mask.numel() == d.size * T * L):
            raise TypeError(f"row_mask must be a contiguous CUDA uint8 tensor with {d.size}*{T}*{L} entries")
        mp = C.c_void_p(row_mask.data_ptr())
    _chk(h, lib().dode_adagrad_step(h, d.ctypes.data, d.size, C.c_float(eta), C.c_float(eps), mp))


def dode_adagrad_reset(h) -> None:
    _chk(h, lib().dode_adagrad_reset(h))


def dode_spgd_step_host(h, days, eta: float, x_host, q_host) -> None:
    """Streaming step: uploads the days' counts from ``x_host`` ([n][T][L] CPU float32 tensor, pinned for
    asynchronous copies), steps, and downloads their q into ``q_host`` ([n][T][N] CPU float32 tensor).
    ASYNCHRONOUS: the copies and kernels are only queued.  ``q_host`` is defined, and ``x_host`` may be changed, only
    after the next synchronising call (dode_sync, dode_objective, dode_r2, dode_get_q, dode_set_q, dode_lipschitz,
    dode_timing_read, dode_reserve, dode_destroy); this binding keeps both tensors alive until then."""
    d = _days(days)
    N, L, T = _shape[_key(h)][:3]
    xp = _host(x_host, (d.size, T, L), "x_host")
    qp = _host(q_host, (d.size, T, N), "q_host")
    _keep.setdefault(_key(h), []).append((x_host, q_host))
    _chk(h, lib().dode_spgd_step_host(h, d.ctypes.data, d.size, C.c_float(eta), xp, qp))


def dode_objective(h, days):
    """a5: returns (per_day float64 array, total) for the listed days (any mix of clusters)."""
    d = _days(days)
    per = np.empty(d.size, np.float64)
    tot = C.c_double()
    _chk(h, lib().dode_objective(h, d.ctypes.data, d.size, per.ctypes.data, C.byref(tot)))
    _release(h)
    return per, tot.value


def dode_r2(h, days):
    """Step 6: returns (per-day R2 as a float64 array, their mean) for the listed days."""
    d = _days(days)
    per = np.empty(d.size, np.float64)
    mean = C.c_double()
    _chk(h, lib().dode_r2(h, d.ctypes.data, d.size, per.ctypes.data, C.byref(mean)))
    _release(h)
    return per, mean.value


def dode_get_q(h, day: int, out) -> None:
    """Copies day's q ([T][N], Table 2 order) into ``out`` (CPU or CUDA float32 tensor [T][N], contiguous)."""
    N, L, T = _shape[_key(h)][:3]
    _chk(h, lib().dode_get_q(h, day, _any(out, (T, N), "out"), 1 if out.is_cuda else 0))
    _release(h)


def dode_set_q(h, day: int, src) -> None:
    """Overwrites day's q from ``src`` (CPU or CUDA float32 tensor [T][N], contiguous)."""
    N, L, T = _shape[_key(h)][:3]
    _chk(h, lib().dode_set_q(h, day, _any(src, (T, N), "src"), 1 if src.is_cuda else 0))
    _release(h)


def dode_apply(h, c: int, u, v) -> None:
    """v = rho_c u   (u CUDA fp32 [T][N], v CUDA fp32 [T][L])."""
    import torch
    _chk(h, lib().dode_apply(h, c, _dev(u, torch.float32, "u"), _dev(v, torch.float32, "v")))


def dode_apply_t(h, c: int, v, u) -> None:
    """u = rho_c^T v."""
    import torch
    _chk(h, lib().dode_apply_t(h, c, _dev(v, torch.float32, "v"), _dev(u, torch.float32, "u")))


def dode_lipschitz(h, c: int, iters: int = 50) -> float:
    """a7: L_c ~ lambda_max(rho_c^T rho_c) by power iteration through the production kernels."""
    out = C.c_double()
    _chk(h, lib().dode_lipschitz(h, c, iters, C.byref(out)))
    _release(h)
    return out.value


def dode_timing_enable(h, on: bool) -> None:
    _chk(h, lib().dode_timing_enable(h, 1 if on else 0))


def dode_timing_read(h, kind: int, reset: bool = False):
    """(total device ms, launches) of kind 0 = forward, 1 = gradient+update."""
    ms, cnt = C.c_double(), C.c_int64()
    _chk(h, lib().dode_timing_read(h, kind, C.byref(ms), C.byref(cnt), 1 if reset else 0))
    _release(h)
    return ms.value, cnt.value


def dode_probe_fp32_peak(reps: int = 5) -> float:
    """Measured FP32 FFMA rate of the current device in TFLOP/s (a measurement helper, not on the SPGD path)."""
    import torch
    out = C.c_double()
    rc = lib().dode_probe_fp32_peak(int(reps), C.byref(out), C.c_void_p(torch.cuda.current_stream().cuda_stream))
    if rc != DODE_OK:
        raise DodeError(rc, lib().dode_last_error(None).decode())
    return out.value


def dode_launch_count(h) -> int:
    return int(lib().dode_launch_count(h))


def dode_last_path(h) -> str:
    return lib().dode_last_path(h).decode()


def dode_sync(h) -> None:
    _chk(h, lib().dode_sync(h))
    _release(h)


def dode_destroy(h) -> None:
    lib().dode_destroy(h)
    _release(h)
    _shape.pop(_key(h), None)


def dode_last_error(h) -> str:
    return lib().dode_last_error(h).decode()
