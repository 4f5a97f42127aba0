"""dode_visit_static (include/dode.h): the allocation-free entry point — one visit of one day with the residual in the
library's file-scope device array instead of a cudaMalloc'ed panel.  Collected LAST on purpose (the suite runs with
pytest -x).  The file passes alone in a fresh process and after the other tests: it owns its ctx, and the static
array is overwritten before it is read on every call.

Checked here: its q equals the existing path's (dode_create + dode_spgd_step with one day, the FFMA column-dot
kernels) within the tolerance the other parity tests use, on two calls in a row on the same day and then on another
day (stale scratch of the previous call in place); the oracle's visit beside it; free device memory does not move
across calls; sizes beyond the static array are rejected with a clear error and nothing launched."""
import numpy as np
import pytest
import torch

import paper_1901_09266_b200 as P
from paper_1901_09266_b200 import synth
from tests import harness as hz

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


@pytest.mark.parametrize("shape", [dict(N=70, L=45, T=24, H=5), dict(N=203, L=131, T=60, H=7), dict(N=33, L=9, T=7, H=6)])
def test_visit_static_matches_the_step_path_twice_in_a_row(shape):
    cfg = synth.Config("no_alloc", C=2, D=6, b=1, K=4, kmin=3, kmax=12, **shape)
    p = hz.make_problem(cfg)
    etas = hz.oracle_etas(p, 30)
    g = hz.GpuSolver(p)                                   # existing path: ctx with its own (allocated) panels
    Rd = p.R.to(DEV)
    xd = p.x.to(DEV)
    from oracle import oracle
    for d in (0, 1, 4):                                   # days of both clusters; each call reuses the same static array
        c = int(p.labels[d])
        q = torch.ones((cfg.T, cfg.N), dtype=torch.float32, device=DEV)
        want = np.ones((cfg.T, cfg.N), np.float32)
        for call in (1, 2):                               # two calls in a row on the same day
            P.dode_visit_static(Rd[c], q, xd[d], float(etas[c]))
            P.dode_spgd_step(g.h, [d], float(etas[c]))
            P.dode_sync(g.h)
            assert P.dode_last_path(g.h).startswith("ffma")
            torch.cuda.synchronize()
            got = q.cpu().numpy()
            hz.assert_q_close(got, g.q([d])[0], f"dode_visit_static vs dode_spgd_step, day {d}, call {call}")
            want = oracle.visit(p.R[c].numpy(), want, p.x[d].numpy(), float(etas[c]))
            hz.assert_q_close(got, want, f"dode_visit_static vs oracle, day {d}, call {call}")
    g.close()


def test_visit_static_allocates_nothing_and_runs_on_a_side_stream():
    cfg = synth.Config("no_alloc_mem", N=64, L=40, T=32, H=4, C=1, D=2, b=1, K=2, kmin=3, kmax=12)
    p = hz.make_problem(cfg)
    Rd, xd = p.R.to(DEV), p.x.to(DEV)
    q = torch.ones((cfg.T, cfg.N), dtype=torch.float32, device=DEV)
    q_ref = q.clone()
    side = torch.cuda.Stream(device=DEV)
    P.dode_visit_static(Rd[0], q_ref, xd[0], 1e-3)        # first call on this device: looks up the array's address
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info(0)
    with torch.cuda.stream(side):
        for _ in range(3):
            P.dode_visit_static(Rd[0], q, xd[0], 1e-3)
    side.synchronize()
    free1, _ = torch.cuda.mem_get_info(0)
    assert free1 == free0, f"free device memory moved by {free0 - free1} bytes across dode_visit_static calls"
    for _ in range(2):
        P.dode_visit_static(Rd[0], q_ref, xd[0], 1e-3)
    torch.cuda.synchronize()
    assert torch.equal(q, q_ref)                          # same kernels, same order: bit-identical on any stream


def test_visit_static_rejects_sizes_beyond_the_static_array():
    T, L = 513, 512                                       # T*L = 262656 > DODE_STATIC_SCRATCH_FLOATS = 262144
    assert T * L > P.STATIC_SCRATCH_FLOATS
    R = torch.zeros((T, 1, L, 1), dtype=torch.float32, device=DEV)
    q = torch.ones((T, 1), dtype=torch.float32, device=DEV)
    x = torch.zeros((T, L), dtype=torch.float32, device=DEV)
    with pytest.raises(P.DodeError) as e:
        P.dode_visit_static(R, q, x, 0.1)
    assert e.value.code == P.DODE_EINVAL and "static scratch" in str(e.value) and "262656" in str(e.value)
    torch.cuda.synchronize()
    assert bool((q == 1).all())                           # nothing was launched
    with pytest.raises(P.DodeError):
        P.dode_visit_static(R[:8], q[:8], x[:8], 0.0)     # eta must be > 0
    P.dode_visit_static(R[:512], q[:512], x[:512], 0.1)   # exactly the maximum (512*512) is accepted
    torch.cuda.synchronize()
    assert bool((q[:512] == 1).all())                     # R = 0: g = 0, q unchanged
