"""NEXT-4: DAR construction from link speeds on the GPU (dode_dar_build) against the oracle's O7
(pinned by P16), and the built operator carried through the SPGD path."""
import numpy as np
import pytest
import torch

import paper_1901_09266_b200 as P
from paper_1901_09266_b200 import synth
from tests import harness as hz

pytestmark = pytest.mark.gpu
DT = 300.0


def _build_both(cfg, c=0):
    from oracle import oracle
    ptr, links, length = synth.network(cfg)
    v = synth.speeds(cfg, c)
    want = oracle.dar_build(cfg.N, cfg.L, cfg.T, cfg.H, ptr.numpy(), links.numpy(), length.numpy(), v.numpy(), DT)
    R = torch.full((cfg.T, cfg.H + 1, cfg.L, cfg.N), 7.0, device="cuda")          # stale contents must be overwritten
    P.dode_dar_build(cfg.N, cfg.L, cfg.T, cfg.H, ptr.cuda(), links.cuda(), length.cuda(), v.cuda(), DT, R)
    torch.cuda.synchronize()
    return R.cpu().numpy(), want


@pytest.mark.parametrize("shape", [(61, 37, 50, 5), (4, 6, 288, 6), (60, 120, 288, 12), (300, 90, 24, 30), (7, 5, 3, 0)])
def test_dar_build_matches_oracle(shape):
    N, L, T, H = shape
    cfg = synth.Config("dar", N=N, L=L, T=T, H=H, C=2, D=4, b=2, K=1, kmin=2, kmax=min(20, L))
    for c in range(cfg.C):
        got, want = _build_both(cfg, c)
        # same support (which (s, h, l, n) entries exist is an integer decision; both sides take it in double)
        np.testing.assert_array_equal(got != 0, want != 0)
        np.testing.assert_allclose(got, want, rtol=0, atol=1e-6)
        assert (got >= 0).all() and got.max() <= 1.0 + 1e-6


def test_example3_on_gpu():
    """The hand-worked Example 3 instance (tests/golden/example3_three_link_dar.txt) through the kernel."""
    T, H, L, N = 6, 4, 3, 1
    length = torch.tensor([1000.0, 1500.0, 800.0])
    speed = torch.full((T, L), 8.0)
    speed[0, 0], speed[0, 1], speed[1, 0], speed[1, 1] = 5.0, 10.0, 4.0, 3.75
    R = torch.empty((T, H + 1, L, N), device="cuda")
    P.dode_dar_build(N, L, T, H, torch.tensor([0, 3], dtype=torch.int32).cuda(), torch.tensor([0, 1, 2], dtype=torch.int32).cuda(),
                     length.cuda(), speed.cuda(), DT, R)
    got = R.cpu().numpy()[0, :, :, 0]
    want = np.zeros((H + 1, L))
    want[0, 0] = 1.0
    want[0, 1], want[1, 1] = 100 / 350, 250 / 350
    want[1, 2], want[2, 2], want[3, 2] = 250 / 600, 300 / 600, 50 / 600
    np.testing.assert_allclose(got, want, atol=1e-7)


def test_fifo_violation_on_gpu():
    """The hand-worked FIFO-violation instance (tests/golden/fifo_violation_two_link.txt; reading A20) through the dense
    kernel and the CSR builder."""
    from tests.test_oracle_pins import _fifo_violation_instance
    T, H, L, N, dt, pp, pl, length, speed, want = _fifo_violation_instance()
    tp, tl, tn, ts = (torch.from_numpy(a).cuda() for a in (pp, pl, length, speed))
    R = torch.empty((T, H + 1, L, N), device="cuda")
    P.dode_dar_build(N, L, T, H, tp, tl, tn, ts, dt, R)
    np.testing.assert_allclose(R.cpu().numpy()[:2, :, :, 0], want[:2], atol=1e-7)
    from oracle import oracle
    _csr_equal(P.dode_assignment_build_csr(N, L, T, H, None, tp, tl, tn, ts, dt),
               oracle.dar_build(N, L, T, H, pp, pl, length, speed, dt), 1e-7)


def test_built_operator_through_the_spgd_path():
    """Step 1 -> Step 5 on the GPU: operators built by dode_dar_build for two patterns feed dode_create directly; the
    SPGD iterates equal the oracle's on the oracle-built operators."""
    from oracle import oracle
    cfg = synth.Config("dar_e2e", N=40, L=30, T=36, H=6, C=2, D=24, b=8, K=10, kmin=3, kmax=8)
    ptr, links, length = synth.network(cfg)
    Rg = torch.empty((cfg.C, cfg.T, cfg.H + 1, cfg.L, cfg.N), device="cuda")
    Ro = np.empty((cfg.C, cfg.T, cfg.H + 1, cfg.L, cfg.N), np.float32)
    for c in range(cfg.C):
        v = synth.speeds(cfg, c)
        P.dode_dar_build(cfg.N, cfg.L, cfg.T, cfg.H, ptr.cuda(), links.cuda(), length.cuda(), v.cuda(), DT, Rg[c])
        Ro[c] = oracle.dar_build(cfg.N, cfg.L, cfg.T, cfg.H, ptr.numpy(), links.numpy(), length.numpy(), v.numpy(), DT)
    lab = synth.labels(cfg)
    x = synth.counts(cfg, torch.from_numpy(Ro), synth.q_true(cfg), lab)
    p = hz.Problem(cfg, torch.from_numpy(Ro), lab.numpy(), x, synth.q_true(cfg))
    sched = synth.schedule(cfg, p.labels)
    etas = hz.oracle_etas(p)
    h = P.dode_create(cfg.N, cfg.L, cfg.T, cfg.H, cfg.C, cfg.D, p.labels, x.cuda(), 1.0, dense=Rg)
    for c, days in sched:
        P.dode_spgd_step(h, days, float(etas[c]))
    P.dode_sync(h)
    out = torch.empty((cfg.D, cfg.T, cfg.N))
    for d in range(cfg.D):
        P.dode_get_q(h, d, out[d])
    hz.assert_q_close(out.numpy(), hz.oracle_run(p, sched, etas), "dar_e2e")
    P.dode_destroy(h)


@pytest.mark.parametrize("shape,theta", [((61, 37, 50, 5), 0.01), ((60, 120, 96, 12), 0.002), ((9, 12, 20, 8), 0.0)])
def test_assignment_build_multipath_logit_matches_oracle(shape, theta):
    """B = delta*rho*p with 1-3 paths per OD and Logit shares (Eq. 37, 41) against the oracle's O8 (pin P17)."""
    from oracle import oracle
    N, L, T, H = shape
    cfg = synth.Config("asg", N=N, L=L, T=T, H=H, C=2, D=4, b=2, K=1, kmin=2, kmax=min(12, L))
    od, pp, pl, length = synth.network_multipath(cfg, 3)
    assert int(od[-1]) > N                                           # some OD has more than one path
    for c in range(cfg.C):
        v = synth.speeds(cfg, c)
        want = oracle.assignment_build(N, L, T, H, od.numpy(), pp.numpy(), pl.numpy(), length.numpy(), v.numpy(), DT, theta)
        R = torch.full((T, H + 1, L, N), 3.0, device="cuda")
        P.dode_assignment_build(N, L, T, H, od.cuda(), pp.cuda(), pl.cuda(), length.cuda(), v.cuda(), DT, theta, R)
        got = R.cpu().numpy()
        np.testing.assert_array_equal(got != 0, want != 0)
        np.testing.assert_allclose(got, want, rtol=0, atol=2e-6)
    # one path per OD through the multi-path entry point == dode_dar_build
    ptr, links, length1 = synth.network(cfg)
    ident = torch.arange(N + 1, dtype=torch.int32)
    Ra = torch.empty((T, H + 1, L, N), device="cuda"); Rb = torch.empty_like(Ra)
    v = synth.speeds(cfg, 0).cuda()
    P.dode_assignment_build(N, L, T, H, ident.cuda(), ptr.cuda(), links.cuda(), length1.cuda(), v, DT, theta, Ra)
    P.dode_dar_build(N, L, T, H, ptr.cuda(), links.cuda(), length1.cuda(), v, DT, Rb)
    np.testing.assert_allclose(Ra.cpu().numpy(), Rb.cpu().numpy(), rtol=0, atol=1e-7)


def _csr_equal(got, want_dense, atol):
    """got: CSR namespace from dode_assignment_build_csr (one cluster); want_dense: [T][H+1][L][N] numpy."""
    want = synth.dense_to_csr(torch.from_numpy(want_dense[None]))
    np.testing.assert_array_equal(got.blk_off.cpu().numpy(), want.blk_off.numpy())
    np.testing.assert_array_equal(got.row_ptr.cpu().numpy(), want.row_ptr.numpy())
    np.testing.assert_array_equal(got.col_idx.cpu().numpy(), want.col_idx.numpy())      # identical support, ascending columns
    np.testing.assert_allclose(got.val.cpu().numpy(), want.val.numpy(), rtol=0, atol=atol)


@pytest.mark.parametrize("shape,paths,theta", [((61, 37, 50, 5), 1, 0.0), ((61, 37, 50, 5), 3, 0.01), ((60, 120, 96, 12), 3, 0.002),
                                               ((7, 5, 3, 0), 1, 0.0), ((300, 90, 24, 30), 2, 0.01)])
def test_assignment_build_csr_matches_oracle(shape, paths, theta):
    """CSR output: the oracle's dense O7 / O8 operator converted to the boundary CSR format must
    equal the kernel's arrays — offsets, row pointers and column indices exactly, values to 2e-6 (merged multi-path shares
    are summed in another order).  An operator built this way feeds dode_create(csr=...) directly."""
    from oracle import oracle
    N, L, T, H = shape
    cfg = synth.Config("asg_csr", N=N, L=L, T=T, H=H, C=1, D=6, b=3, K=6, kmin=2, kmax=min(12, L), label_mode="zero")
    v = synth.speeds(cfg, 0)
    if paths == 1:
        ptr, links, length = synth.network(cfg)
        want = oracle.dar_build(N, L, T, H, ptr.numpy(), links.numpy(), length.numpy(), v.numpy(), DT)
        got = P.dode_assignment_build_csr(N, L, T, H, None, ptr.cuda(), links.cuda(), length.cuda(), v.cuda(), DT)
    else:
        od, ptr, links, length = synth.network_multipath(cfg, paths)
        want = oracle.assignment_build(N, L, T, H, od.numpy(), ptr.numpy(), links.numpy(), length.numpy(), v.numpy(), DT, theta)
        got = P.dode_assignment_build_csr(N, L, T, H, od.cuda(), ptr.cuda(), links.cuda(), length.cuda(), v.cuda(), DT, theta)
    assert got.nnz == int((want != 0).sum())
    _csr_equal(got, want, 2e-6)
    # Step 1 -> Step 5 without ever forming the dense slab on the GPU
    lab = synth.labels(cfg)
    Ro = torch.from_numpy(want[None])
    x = synth.counts(cfg, Ro, synth.q_true(cfg), lab)
    p = hz.Problem(cfg, Ro, lab.numpy(), x, synth.q_true(cfg))
    sched = synth.schedule(cfg, p.labels)
    etas = hz.oracle_etas(p)
    h = P.dode_create(N, L, T, H, 1, cfg.D, p.labels, x.cuda(), 1.0, csr=got)
    for c, days in sched:
        P.dode_spgd_step(h, days, float(etas[c]))
    out = torch.empty((cfg.D, T, N))
    for d in range(cfg.D):
        P.dode_get_q(h, d, out[d])
    hz.assert_q_close(out.numpy(), hz.oracle_run(p, sched, etas), "csr-built operator")
    P.dode_destroy(h)


def test_per_day_operators_undo_reading_d3():
    """the paper builds the DAR matrix PER DAY from that day's speeds; north_star
    shares one operator per cluster.  The per-day flow is the same library with C = D: one operator per day built from
    its own speed table, every day its own cluster, minibatches of one day — iterates equal the oracle's."""
    from oracle import oracle
    cfg = synth.Config("per_day", N=30, L=24, T=36, H=6, C=10, D=10, b=1, K=40, kmin=3, kmax=8)
    ptr, links, length = synth.network(cfg)
    Rg = torch.empty((cfg.D, cfg.T, cfg.H + 1, cfg.L, cfg.N), device="cuda")
    Ro = np.empty((cfg.D, cfg.T, cfg.H + 1, cfg.L, cfg.N), np.float32)
    for d in range(cfg.D):
        v = synth.speeds(cfg, d)                                   # a speed table of its own for every day
        P.dode_dar_build(cfg.N, cfg.L, cfg.T, cfg.H, ptr.cuda(), links.cuda(), length.cuda(), v.cuda(), DT, Rg[d])
        Ro[d] = oracle.dar_build(cfg.N, cfg.L, cfg.T, cfg.H, ptr.numpy(), links.numpy(), length.numpy(), v.numpy(), DT)
    assert np.abs(Ro[0] - Ro[1]).max() > 1e-3                      # the days' operators do differ
    lab = torch.arange(cfg.D, dtype=torch.int32)
    x = synth.counts(cfg, torch.from_numpy(Ro), synth.q_true(cfg), lab)
    p = hz.Problem(cfg, torch.from_numpy(Ro), lab.numpy(), x, synth.q_true(cfg))
    sched = synth.schedule(cfg, p.labels)
    assert all(len(days) == 1 for _, days in sched)
    etas = hz.oracle_etas(p)
    h = P.dode_create(cfg.N, cfg.L, cfg.T, cfg.H, cfg.D, cfg.D, p.labels, x.cuda(), 1.0, dense=Rg)
    for c, days in sched:
        P.dode_spgd_step(h, days, float(etas[c]))
    out = torch.empty((cfg.D, cfg.T, cfg.N))
    for d in range(cfg.D):
        P.dode_get_q(h, d, out[d])
    hz.assert_q_close(out.numpy(), hz.oracle_run(p, sched, etas), "per-day operators")
    P.dode_destroy(h)
