"""ORACLE — test infrastructure, not the product (see dode_oracle.cpp's header).

ctypes wrapper around ``oracle/dode_oracle.cpp`` (built by ``build_oracle()``, also
called from ``__graft_entry__.build()``).  Imports nothing from the CUDA package.
Arrays are numpy, fp32 storage, C-contiguous; notation follows PAPER.md Table 2
 and Alg. 1.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "dode_oracle.cpp")
_SO = os.path.join(_HERE, "liboracle.so")
_lib = None


def build_oracle(force: bool = False) -> str:
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-pthread", "-o", _SO, _SRC])
    return _SO


def _f(a):  # float32 C-contiguous view
    a = np.ascontiguousarray(a, dtype=np.float32)
    return a, a.ctypes.data_as(C.POINTER(C.c_float))


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build_oracle())
        _lib.oracle_objective_day.restype = C.c_double
        _lib.oracle_objective_day_mt.restype = C.c_double
        _lib.oracle_r2_day.restype = C.c_double
        _lib.oracle_objective_day_csr.restype = C.c_double
        _lib.oracle_power_iteration.restype = C.c_double
    return _lib


def _dims(Rc):
    T, H1, L, N = Rc.shape
    return N, L, T, H1 - 1


def forward_residual(Rc: np.ndarray, q: np.ndarray, x: np.ndarray) -> np.ndarray:
    """O2a.  Rc [T][H+1][L][N], q [T][N], x [T][L] -> r [T][L] fp32."""
    N, L, T, H = _dims(Rc)
    Rc, pR = _f(Rc); q, pq = _f(q); x, px = _f(x)
    assert q.shape == (T, N) and x.shape == (T, L)
    r = np.empty((T, L), np.float32)
    lib().oracle_forward_residual(N, L, T, H, pR, pq, px, r.ctypes.data_as(C.POINTER(C.c_float)))
    return r


def gradient(Rc: np.ndarray, r: np.ndarray) -> np.ndarray:
    """O2b.  g [T][N] float64 = rho_c^T r."""
    N, L, T, H = _dims(Rc)
    Rc, pR = _f(Rc); r, pr = _f(r)
    assert r.shape == (T, L)
    g = np.empty((T, N), np.float64)
    lib().oracle_gradient(N, L, T, H, pR, pr, g.ctypes.data_as(C.POINTER(C.c_double)))
    return g


def visit(Rc: np.ndarray, q: np.ndarray, x: np.ndarray, eta: float) -> np.ndarray:
    """One SPGD visit (O2a-c); returns the new q (fp32 [T][N])."""
    N, L, T, H = _dims(Rc)
    Rc, pR = _f(Rc); x, px = _f(x)
    q = np.array(q, dtype=np.float32, order="C", copy=True)
    lib().oracle_visit(N, L, T, H, pR, q.ctypes.data_as(C.POINTER(C.c_float)), px, C.c_float(eta))
    return q


def objective_day(Rc: np.ndarray, q: np.ndarray, x: np.ndarray, threads: int = 1) -> float:
    """O3 for one day: sum of squared residuals, no 1/2 (Eq. 42).  threads > 1: the forward rows are
    computed by several threads and summed in the same order (same value, pin P18)."""
    N, L, T, H = _dims(Rc)
    Rc, pR = _f(Rc); q, pq = _f(q); x, px = _f(x)
    if threads > 1:
        return float(lib().oracle_objective_day_mt(N, L, T, H, pR, pq, px, int(threads)))
    return float(lib().oracle_objective_day(N, L, T, H, pR, pq, px))


def visit_adagrad(Rc: np.ndarray, q: np.ndarray, G: np.ndarray, x: np.ndarray, mask, eta: float, eps: float = 1e-10):
    """O6 (NEXT-1): one row-chunk Adagrad iteration of Alg. 1; returns (new q, new G).
    mask: uint8 [T][L] (rows of the chunk) or None for every row."""
    N, L, T, H = _dims(Rc)
    Rc, pR = _f(Rc); x, px = _f(x)
    q = np.array(q, dtype=np.float32, order="C", copy=True)
    G = np.array(G, dtype=np.float32, order="C", copy=True)
    pm = None
    if mask is not None:
        mask = np.ascontiguousarray(mask, dtype=np.uint8)
        assert mask.shape == (T, L)
        pm = mask.ctypes.data_as(C.c_void_p)
    lib().oracle_visit_adagrad(N, L, T, H, pR, q.ctypes.data_as(C.c_void_p), G.ctypes.data_as(C.c_void_p), px, pm,
                               C.c_float(eta), C.c_float(eps))
    return q, G


def r2_day(Rc: np.ndarray, q: np.ndarray, x: np.ndarray) -> float:
    """O5: coefficient of determination of the fitted counts of one day (Step 6; reading A17)."""
    N, L, T, H = _dims(Rc)
    Rc, pR = _f(Rc); q, pq = _f(q); x, px = _f(x)
    return float(lib().oracle_r2_day(N, L, T, H, pR, pq, px))


def power_iteration(Rc: np.ndarray, iters: int = 50) -> float:
    """O4: L_c ~ lambda_max(rho_c^T rho_c)."""
    N, L, T, H = _dims(Rc)
    Rc, pR = _f(Rc)
    return float(lib().oracle_power_iteration(N, L, T, H, pR, iters))


def run_schedule(R: np.ndarray, labels: np.ndarray, x: np.ndarray, q: np.ndarray,
                 sched: Sequence, etas: Sequence[float], day_mask: Optional[np.ndarray] = None) -> np.ndarray:
    """Replays ``sched`` = [(cluster, int32 days), ...] with per-iteration step ``etas``.
    R [C][T][H+1][L][N]; x [D][T][L]; q [D][T][N] (copied).  Returns the final q."""
    Cn, T, H1, L, N = R.shape
    D = x.shape[0]
    R, pR = _f(R); x, px = _f(x)
    q = np.array(q, dtype=np.float32, order="C", copy=True)
    labels = np.ascontiguousarray(labels, dtype=np.int32)
    days = np.ascontiguousarray(np.concatenate([np.asarray(d, np.int32) for _, d in sched])
                                if len(sched) else np.zeros(0, np.int32))
    ptr = np.zeros(len(sched) + 1, np.int64)
    ptr[1:] = np.cumsum([len(d) for _, d in sched])
    eta = np.ascontiguousarray(etas, dtype=np.float32)
    assert len(eta) == len(sched)
    mask = None if day_mask is None else np.ascontiguousarray(day_mask, dtype=np.uint8)
    lib().oracle_run_schedule(
        N, L, T, H1 - 1, Cn, D, pR, labels.ctypes.data_as(C.POINTER(C.c_int32)), px,
        q.ctypes.data_as(C.POINTER(C.c_float)), days.ctypes.data_as(C.POINTER(C.c_int32)),
        ptr.ctypes.data_as(C.POINTER(C.c_int64)), eta.ctypes.data_as(C.POINTER(C.c_float)),
        len(sched), None if mask is None else mask.ctypes.data_as(C.POINTER(C.c_uint8)))
    return q


def visit_csr(N: int, L: int, T: int, H: int, blk_off, row_ptr, col_idx, val, q, x, eta: float) -> np.ndarray:
    """a6: one visit with R_c as CSR per (s,h) block (see dode_oracle.cpp)."""
    blk_off = np.ascontiguousarray(blk_off, np.int64); row_ptr = np.ascontiguousarray(row_ptr, np.int32)
    col_idx = np.ascontiguousarray(col_idx, np.int32); val, pv = _f(val); x, px = _f(x)
    q = np.array(q, dtype=np.float32, order="C", copy=True)
    lib().oracle_visit_csr(N, L, T, H, blk_off.ctypes.data_as(C.POINTER(C.c_int64)),
                           row_ptr.ctypes.data_as(C.POINTER(C.c_int32)),
                           col_idx.ctypes.data_as(C.POINTER(C.c_int32)), pv,
                           q.ctypes.data_as(C.POINTER(C.c_float)), px, C.c_float(eta))
    return q


def replay_day(Rc: np.ndarray, q: np.ndarray, x: np.ndarray, eta: float, visits: int, checkpoints: Sequence[int],
               threads: int = 1, budget_s: float = 0.0, csr=None):
    """``visits`` consecutive visits of one day (exactly ``visit`` / ``visit_csr`` repeated; pin P18), the output rows of
    each pass split over ``threads`` threads.  Returns (q after each checkpoint visit count reached, visits done): the
    replay stops early once ``budget_s`` seconds have passed.  ``csr`` = (N, L, T, H, blk_off, row_ptr, col_idx, val)
    replays through the CSR loops instead (then ``Rc`` is ignored)."""
    ck = np.ascontiguousarray(sorted(int(c) for c in checkpoints), dtype=np.int32)
    assert ck.size == 0 or (ck[0] >= 1 and ck[-1] <= visits)
    x, px = _f(x)
    q = np.array(q, dtype=np.float32, order="C", copy=True)
    out = np.empty((ck.size,) + q.shape, np.float32)
    pq, po, pc = q.ctypes.data_as(C.c_void_p), out.ctypes.data_as(C.c_void_p), ck.ctypes.data_as(C.c_void_p)
    if csr is None:
        N, L, T, H = _dims(Rc)
        Rc, pR = _f(Rc)
        done = lib().oracle_replay_day(N, L, T, H, pR, pq, px, C.c_float(eta), int(visits), pc, int(ck.size), po,
                                       int(threads), C.c_double(budget_s))
    else:
        N, L, T, H, blk_off, row_ptr, col_idx, val = csr
        blk_off = np.ascontiguousarray(blk_off, np.int64); row_ptr = np.ascontiguousarray(row_ptr, np.int32)
        col_idx = np.ascontiguousarray(col_idx, np.int32); val, pv = _f(val)
        done = lib().oracle_replay_day_csr(N, L, T, H, blk_off.ctypes.data_as(C.c_void_p), row_ptr.ctypes.data_as(C.c_void_p),
                                           col_idx.ctypes.data_as(C.c_void_p), pv, pq, px, C.c_float(eta), int(visits),
                                           pc, int(ck.size), po, int(threads), C.c_double(budget_s))
    reached = [int(c) for c in ck if c <= done]
    return {c: out[i] for i, c in enumerate(reached)}, int(done)


def objective_day_csr(N: int, L: int, T: int, H: int, blk_off, row_ptr, col_idx, val, q, x) -> float:
    blk_off = np.ascontiguousarray(blk_off, np.int64); row_ptr = np.ascontiguousarray(row_ptr, np.int32)
    col_idx = np.ascontiguousarray(col_idx, np.int32); val, pv = _f(val); x, px = _f(x); q, pq = _f(q)
    return float(lib().oracle_objective_day_csr(
        N, L, T, H, blk_off.ctypes.data_as(C.POINTER(C.c_int64)), row_ptr.ctypes.data_as(C.POINTER(C.c_int32)),
        col_idx.ctypes.data_as(C.POINTER(C.c_int32)), pv, pq, px))


def dar_build(N: int, L: int, T: int, H: int, path_ptr, path_links, length, speed, dt: float) -> np.ndarray:
    """O7 (NEXT-4): DAR blocks [T][H+1][L][N] of one day from link speeds (Eq. 17-18, Example 3)."""
    path_ptr = np.ascontiguousarray(path_ptr, dtype=np.int32); path_links = np.ascontiguousarray(path_links, dtype=np.int32)
    length = np.ascontiguousarray(length, dtype=np.float32); speed = np.ascontiguousarray(speed, dtype=np.float32)
    assert path_ptr.shape == (N + 1,) and length.shape == (L,) and speed.shape == (T, L)
    R = np.empty((T, H + 1, L, N), np.float32)
    lib().oracle_dar_build(N, L, T, H, path_ptr.ctypes.data_as(C.c_void_p), path_links.ctypes.data_as(C.c_void_p),
                           length.ctypes.data_as(C.c_void_p), speed.ctypes.data_as(C.c_void_p), C.c_double(dt),
                           R.ctypes.data_as(C.c_void_p))
    return R


def assignment_build(N: int, L: int, T: int, H: int, od_ptr, path_ptr, path_links, length, speed, dt: float,
                     theta: float) -> np.ndarray:
    """O8 (NEXT-4): B = delta * rho * p of one pattern, several paths per OD, Logit shares (Eq. 37, 41)."""
    od_ptr = np.ascontiguousarray(od_ptr, dtype=np.int32); path_ptr = np.ascontiguousarray(path_ptr, dtype=np.int32)
    path_links = np.ascontiguousarray(path_links, dtype=np.int32)
    length = np.ascontiguousarray(length, dtype=np.float32); speed = np.ascontiguousarray(speed, dtype=np.float32)
    assert od_ptr.shape == (N + 1,) and path_ptr.shape == (od_ptr[-1] + 1,) and length.shape == (L,) and speed.shape == (T, L)
    R = np.empty((T, H + 1, L, N), np.float32)
    vp = lambda a: a.ctypes.data_as(C.c_void_p)
    lib().oracle_assignment_build(N, L, T, H, vp(od_ptr), vp(path_ptr), vp(path_links), vp(length), vp(speed),
                                  C.c_double(dt), C.c_double(theta), vp(R))
    return R
