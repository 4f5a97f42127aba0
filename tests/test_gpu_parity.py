"""GPU-vs-oracle parity through the C ABI: identical iterates after K steps from the same
q0, eta and schedule, |q_gpu - q_cpu| <= 1e-3 max(1,|q_cpu|), objective relative error <= 1e-4."""
import numpy as np
import pytest
import torch

from paper_1901_09266_b200 import synth
from tests import harness as hz

pytestmark = pytest.mark.gpu

TOL_OBJ = 1e-4


def _oracle():
    from oracle import oracle
    return oracle


def _objective_cpu(p, q, days):
    o = _oracle()
    return np.array([o.objective_day(p.R[p.labels[d]].numpy(), q[i], p.x[d].numpy()) for i, d in enumerate(days)])


def _run_both(cfg, K=None, b=None, sample=None, csr=False, sparse_gen=False, tc_min_b=None, ksplit=None, pair=None):
    p = hz.make_problem_sparse(cfg) if sparse_gen else hz.make_problem(cfg)
    sched = synth.schedule(cfg, p.labels, K=K, b=b)
    etas = hz.oracle_etas(p)
    g = hz.GpuSolver(p, csr=csr, tc_min_b=tc_min_b)
    if ksplit is not None:
        g.P.dode_set_option(g.h, g.P.DODE_OPT_TC_KSPLIT, ksplit)
    if pair is not None:
        g.P.dode_set_option(g.h, g.P.DODE_OPT_TC_PAIR, pair)
    g.run(sched, etas)
    days = list(range(cfg.D)) if sample is None else list(sample)
    q_gpu = g.q(days)
    q_cpu = hz.oracle_run(p, sched, etas, sample)[days]
    hz.assert_q_close(q_gpu, q_cpu, cfg.name)
    # a5: library objective at the GPU's own q vs the oracle's O3 at the same q
    f_gpu, tot = g.P.dode_objective(g.h, days)
    f_cpu = _objective_cpu(p, q_gpu, days)
    np.testing.assert_allclose(f_gpu, f_cpu, rtol=TOL_OBJ)
    assert abs(tot - f_cpu.sum()) <= TOL_OBJ * f_cpu.sum()
    # and the two sides' objectives at their own iterates
    np.testing.assert_allclose(f_gpu, _objective_cpu(p, q_cpu, days), rtol=TOL_OBJ)
    path = g.P.dode_last_path(g.h)
    launches = g.P.dode_launch_count(g.h)
    g.close()
    assert launches >= 2 * len(sched)
    return path


def test_config0_tiny_full():
    """BASELINE.json configs[0] exactly: N=4 L=6 T=288 H=6 D=14, b=4, 500 iterations, all days compared."""
    path = _run_both(synth.CONFIGS["tiny"])
    assert "ffma" in path


def test_tiny12_sub_instance():
    _run_both(synth.CONFIGS["tiny12"])


@pytest.mark.parametrize("b", [1, 2, 3, 5, 8, 11, 20, 37])
def test_ragged_shapes_and_minibatch_widths_ffma(b):
    """FFMA kernels only (tensor path off): N, L not multiples of 4/8 (padding paths), every BT specialisation,
    ragged last chunks, pad days."""
    cfg = synth.Config("ragged", N=61, L=37, T=50, H=5, C=3, D=90, b=b, K=24, kmin=3, kmax=9)
    assert "ffma" in _run_both(cfg, tc_min_b=0)


@pytest.mark.parametrize("b", [8, 11, 16, 20, 37, 64])
def test_ragged_shapes_tensor_core_path(b):
    """tcgen05 3xTF32 path: ragged N/L (zero-filled K tails, partial M tiles), pad days, ragged chunks
    (chunks of fewer than 8 days fall back to the FFMA kernels inside the same run)."""
    cfg = synth.Config("ragged", N=61, L=37, T=50, H=5, C=3, D=200, b=b, K=24, kmin=3, kmax=9)
    _run_both(cfg, sample=[0, 1, 50, 99, 150, 199])


def test_tensor_core_path_multi_tile():
    """Several 128-row tiles in both passes (L=300, N=270), K tails, H >= 1 lags, 2 CTAs per SM."""
    cfg = synth.Config("tc_tiles", N=270, L=300, T=24, H=4, C=2, D=80, b=24, K=8, kmin=5, kmax=20)
    assert "tcgen05" in _run_both(cfg, sample=[0, 11, 40, 79])


def test_corridor_shape_reduced_T():
    """configs[1]'s blocks (N=60, L=120, H=12, C=4, b=32) on a shorter day so the oracle finishes in seconds;
    spans several row tiles (L=120 -> 4 warps-tiles) and two b-tiles of 16."""
    cfg = synth.CONFIGS["corridor"].replace(name="corridor_T72", T=72, D=96, K=16)
    _run_both(cfg, sample=[0, 7, 33, 64, 95])


def test_wide_blocks_several_column_tiles():
    """N4 > 32 (several CTAs along n in the gradient kernel) and L > 32 (several CTAs along l in the forward)."""
    cfg = synth.Config("wide", N=300, L=150, T=20, H=4, C=2, D=24, b=8, K=10, kmin=5, kmax=20)
    _run_both(cfg, sample=[1, 5, 12, 23])


@pytest.mark.parametrize("T,H", [(1, 0), (7, 0), (3, 5), (6, 6)])
def test_degenerate_time_axis(T, H):
    """T=1/H=0 (Fig. 12's plain NNLS), H=0 (no lag), H >= T (band wider than the day)."""
    cfg = synth.Config("degenerate", N=9, L=11, T=T, H=H, C=2, D=10, b=4, K=20, kmin=2, kmax=5)
    _run_both(cfg)


def test_invalid_day_lists_leave_state_untouched():
    cfg = synth.Config("inv", N=8, L=8, T=6, H=2, C=2, D=12, b=4, K=4, kmin=2, kmax=4)
    p = hz.make_problem(cfg)
    g = hz.GpuSolver(p)
    P = g.P
    before = g.q()
    c0 = [int(d) for d in np.nonzero(p.labels == 0)[0]]
    c1 = [int(d) for d in np.nonzero(p.labels == 1)[0]]
    for bad in ([c0[0], c0[0]], [c0[0], c1[0]], [-1], [cfg.D], []):
        with pytest.raises(P.DodeError) as e:
            P.dode_spgd_step(g.h, bad, 0.1)
        assert e.value.code == P.DODE_EINVAL
        assert P.dode_last_error(g.h) != ""
    np.testing.assert_array_equal(g.q(), before)
    g.close()


def test_apply_adjoint_and_lipschitz():
    """<rho u, v> = <u, rho^T v> through the production kernels; dode_apply against the oracle's forward;
    a7 against the oracle's O4."""
    o = _oracle()
    cfg = synth.Config("adj", N=45, L=70, T=30, H=6, C=2, D=4, b=2, K=2, kmin=3, kmax=12)
    p = hz.make_problem(cfg)
    g = hz.GpuSolver(p)
    P = g.P
    gen = torch.Generator().manual_seed(5)
    for c in range(cfg.C):
        u = torch.randn(cfg.T, cfg.N, generator=gen)
        v = torch.randn(cfg.T, cfg.L, generator=gen)
        ru = torch.empty(cfg.T, cfg.L, device="cuda")
        rtv = torch.empty(cfg.T, cfg.N, device="cuda")
        P.dode_apply(g.h, c, u.cuda(), ru)
        P.dode_apply_t(g.h, c, v.cuda(), rtv)
        P.dode_sync(g.h)
        lhs = float((ru.cpu().double() * v.double()).sum())
        rhs = float((u.double() * rtv.cpu().double()).sum())
        assert abs(lhs - rhs) <= 1e-4 * max(1.0, abs(lhs))
        ref = o.forward_residual(p.R[c].numpy(), u.numpy(), np.zeros((cfg.T, cfg.L), np.float32))
        np.testing.assert_allclose(ru.cpu().numpy(), ref, rtol=1e-4, atol=1e-4)
        np.testing.assert_allclose(rtv.cpu().numpy(), o.gradient(p.R[c].numpy(), v.numpy()), rtol=1e-4, atol=1e-4)
        L_gpu = P.dode_lipschitz(g.h, c, 50)
        L_cpu = o.power_iteration(p.R[c].numpy(), 50)
        assert abs(L_gpu - L_cpu) <= 1e-4 * L_cpu
    g.close()


def test_get_set_q_and_host_step():
    cfg = synth.Config("io", N=10, L=14, T=12, H=3, C=1, D=6, b=3, K=3, kmin=2, kmax=5, label_mode="zero")
    p = hz.make_problem(cfg)
    etas = hz.oracle_etas(p)
    g1, g2 = hz.GpuSolver(p), hz.GpuSolver(p, q0=0.0)
    P = g1.P
    # set_q/get_q round trip (host and device buffers)
    src = torch.rand(cfg.T, cfg.N)
    P.dode_set_q(g2.h, 2, src)
    back = torch.empty(cfg.T, cfg.N, device="cuda")
    P.dode_get_q(g2.h, 2, back)
    np.testing.assert_array_equal(back.cpu().numpy(), src.numpy())
    for d in range(cfg.D):
        P.dode_set_q(g2.h, d, torch.ones(cfg.T, cfg.N))
    # streaming step == resident step
    days = [4, 1, 3]
    P.dode_spgd_step(g1.h, days, float(etas[0]))
    xh = p.x[days].contiguous().pin_memory()
    qh = torch.empty(len(days), cfg.T, cfg.N).pin_memory()
    P.dode_spgd_step_host(g2.h, days, float(etas[0]), xh, qh)
    P.dode_sync(g2.h)                      # the streaming step is asynchronous: q_host is defined after a sync
    np.testing.assert_array_equal(qh.numpy(), g1.q(days))
    np.testing.assert_array_equal(g2.q(), g1.q())
    # a pipelined sequence of streaming calls — consecutive calls that share a day, disjoint calls, a repeat two calls
    # later — equals the same sequence of resident steps, and every call's download is that call's state
    seq = [[0, 1, 2], [2, 3], [4, 5], [0, 5], [1], [0, 1, 2, 3, 4, 5], [3]]
    bufs = []
    for days in seq:
        P.dode_spgd_step(g1.h, days, float(etas[0]))
        want = g1.q(days).copy()
        xh = p.x[days].contiguous().pin_memory()
        qh = torch.empty(len(days), cfg.T, cfg.N).pin_memory()
        P.dode_spgd_step_host(g2.h, days, float(etas[0]), xh, qh)
        bufs.append((xh, qh, want))
    P.dode_sync(g2.h)
    for xh, qh, want in bufs:
        np.testing.assert_array_equal(qh.numpy(), want)
    np.testing.assert_array_equal(g2.q(), g1.q())
    g1.close(); g2.close()


def test_streaming_and_plain_steps_interleaved():
    """Streaming steps (helper streams for the scatter into x and the gather of q) interleaved with plain steps on the
    same days, minibatches wide enough for the tensor path and its two lanes: same iterates as plain steps only, and
    every download is its call's state."""
    cfg = synth.Config("mix", N=24, L=20, T=16, H=4, C=1, D=24, b=12, K=3, kmin=2, kmax=6, label_mode="zero")
    p = hz.make_problem(cfg)
    etas = hz.oracle_etas(p)
    g1, g2 = hz.GpuSolver(p), hz.GpuSolver(p)
    P = g1.P
    A, B, Cc = list(range(0, 12)), list(range(12, 24)), list(range(6, 18))
    seq = [("host", A), ("plain", A), ("host", B), ("host", Cc), ("plain", Cc), ("plain", A), ("host", A), ("host", B),
           ("plain", B), ("host", Cc)]
    bufs = []
    for rep in range(3):
        for kind, days in seq:
            P.dode_spgd_step(g1.h, days, float(etas[0]))
            if kind == "plain":
                P.dode_spgd_step(g2.h, days, float(etas[0]))
                continue
            want = g1.q(days).copy()
            xh = p.x[days].contiguous().pin_memory()
            qh = torch.empty(len(days), cfg.T, cfg.N).pin_memory()
            P.dode_spgd_step_host(g2.h, days, float(etas[0]), xh, qh)
            bufs.append((xh, qh, want))
    P.dode_sync(g2.h)
    for xh, qh, want in bufs:
        np.testing.assert_array_equal(qh.numpy(), want)
    np.testing.assert_array_equal(g2.q(), g1.q())
    g1.close(); g2.close()


def test_batch_composition_invariance_on_gpu():
    """P10 on the GPU: the same visits as b=1 steps give the same iterate to rounding."""
    cfg = synth.Config("sep", N=24, L=20, T=16, H=4, C=2, D=20, b=7, K=12, kmin=2, kmax=6)
    p = hz.make_problem(cfg)
    etas = hz.oracle_etas(p)
    sched = synth.schedule(cfg, p.labels)
    single = [(c, np.array([d], np.int32)) for c, days in sched for d in days]
    g1, g2 = hz.GpuSolver(p), hz.GpuSolver(p)
    g1.run(sched, etas)
    g2.run(single, etas)
    hz.assert_q_close(g1.q(), g2.q(), "batch composition")
    g1.close(); g2.close()


@pytest.mark.parametrize("b", [1, 5, 33, 70, 130])
def test_csr_path_on_dense_blocks(b):
    """P13 through the GPU: the same operator given as CSR gives the oracle's iterates (bp = 32/64/128 and a
    minibatch larger than one CSR launch)."""
    cfg = synth.Config("csr_ragged", N=61, L=37, T=30, H=5, C=2, D=280, b=b, K=8, kmin=3, kmax=9)
    path = _run_both(cfg, csr=True, sample=[0, 3, 100, 279])
    assert path.startswith("csr_")


@pytest.mark.parametrize("b", [20, 100])
def test_csr_wide_link_ranges_and_ragged_time_axis(b):
    """Paths that cover hundreds of links (every gradient row block gathers from a 390-link range) at two panel widths;
    T = 37 leaves a ragged last block of departure intervals and a ragged forward time pair."""
    cfg = synth.Config("csr_wide", N=24, L=400, T=37, H=3, C=1, D=2 * b, b=b, K=4, kmin=340, kmax=390, label_mode="zero")
    path = _run_both(cfg, csr=True, sample=[0, 1, b, 2 * b - 1])
    assert path.startswith("csr_")


def test_csr_path_on_generated_sparse_instance():
    """configs[4]'s structure at small size (G7 windowed lags, heavy-tailed demand, calendar factors)."""
    cfg = synth.Config("sparse_small", N=400, L=90, T=40, H=10, C=3, D=60, b=24, K=10, kmin=6, kmax=20,
                       base_mu=1.0, base_sigma=1.2, modulated=True, sparse=True)
    p = hz.make_problem_sparse(cfg)
    # the oracle's own CSR loop agrees with its dense loop on this instance (one visit)
    o = _oracle()
    csr = synth.dense_to_csr(p.R)
    nb = cfg.T * (cfg.H + 1)
    c = int(p.labels[7])
    eta = hz.oracle_etas(p)[c]
    q0 = np.ones((cfg.T, cfg.N), np.float32)
    bo = csr.blk_off.numpy()[c * nb:(c + 1) * nb + 1]
    qa = o.visit_csr(cfg.N, cfg.L, cfg.T, cfg.H, bo, csr.row_ptr.numpy()[c * nb:(c + 1) * nb], csr.col_idx.numpy(),
                     csr.val.numpy(), q0, p.x[7].numpy(), eta)
    np.testing.assert_allclose(qa, o.visit(p.R[c].numpy(), q0, p.x[7].numpy(), eta), rtol=1e-6, atol=1e-6)
    _run_both(cfg, csr=True, sparse_gen=True, sample=[0, 7, 31, 59])


def test_csr_apply_adjoint():
    cfg = synth.Config("csr_adj", N=45, L=70, T=12, H=4, C=1, D=2, b=2, K=2, kmin=3, kmax=12, label_mode="zero")
    p = hz.make_problem(cfg)
    g = hz.GpuSolver(p, csr=True)
    P, o = g.P, _oracle()
    gen = torch.Generator().manual_seed(6)
    u, v = torch.randn(cfg.T, cfg.N, generator=gen), torch.randn(cfg.T, cfg.L, generator=gen)
    ru, rtv = torch.empty(cfg.T, cfg.L, device="cuda"), torch.empty(cfg.T, cfg.N, device="cuda")
    P.dode_apply(g.h, 0, u.cuda(), ru)
    P.dode_apply_t(g.h, 0, v.cuda(), rtv)
    P.dode_sync(g.h)
    np.testing.assert_allclose(ru.cpu().numpy(), o.forward_residual(p.R[0].numpy(), u.numpy(), np.zeros((cfg.T, cfg.L), np.float32)), rtol=1e-4, atol=1e-4)
    np.testing.assert_allclose(rtv.cpu().numpy(), o.gradient(p.R[0].numpy(), v.numpy()), rtol=1e-4, atol=1e-4)
    assert abs(P.dode_lipschitz(g.h, 0, 40) - o.power_iteration(p.R[0].numpy(), 40)) <= 1e-4 * o.power_iteration(p.R[0].numpy(), 40)
    g.close()


def test_r2_quality_check_matches_oracle():
    """NEXT-3 / Step 6: per-day R2 through the library equals the oracle's O5 on the library's own q,
    on the FFMA, tensor-core and CSR forward kernels."""
    o = _oracle()
    cfg = synth.Config("r2", N=37, L=53, T=30, H=5, C=2, D=24, b=12, K=6, kmin=3, kmax=9)
    p = hz.make_problem(cfg)
    sched = synth.schedule(cfg, p.labels)
    etas = hz.oracle_etas(p)
    for csr in (False, True):
        g = hz.GpuSolver(p, csr=csr)
        g.run(sched, etas)
        days = list(range(cfg.D))
        per, mean = g.P.dode_r2(g.h, days)
        q = g.q()
        want = np.array([o.r2_day(p.R[int(p.labels[d])].numpy(), q[d], p.x[d].numpy()) for d in days])
        np.testing.assert_allclose(per, want, rtol=0, atol=1e-5)
        assert abs(mean - want.mean()) < 1e-5
        assert per.max() <= 1.0 + 1e-6
        g.close()


def test_overlapped_steps_keep_day_order_and_join_orders_caller_work():
    """Plain steps alternate on two internal streams (include/dode.h, dode_spgd_step): steps that share days must still
    run in call order, steps on disjoint days may overlap, other library calls interleave correctly, and dode_join makes
    the ctx stream wait for every step issued before it."""
    cfg = synth.Config("lanes", N=70, L=90, T=20, H=3, C=1, D=64, b=16, K=1, kmin=3, kmax=9, label_mode="zero")
    p = hz.make_problem(cfg)
    etas = hz.oracle_etas(p)
    A, B, Cc = list(range(0, 16)), list(range(16, 32)), list(range(8, 24))      # Cc overlaps both A and B
    seq = [A, B, A, A, Cc, B, Cc, A, B, list(range(32, 48)), Cc, list(range(40, 56)), A]
    sched = [(0, np.array(d, np.int32)) for d in seq]
    g = hz.GpuSolver(p)
    P = g.P
    for i, (c, days) in enumerate(sched):
        P.dode_spgd_step(g.h, days, float(etas[c]))
        if i == 5:
            P.dode_objective(g.h, [0, 20])             # a synchronising call in the middle of the overlapped sequence
        if i == 8:
            P.dode_adagrad_reset(g.h)                  # a ctx-stream call that must not disturb the lanes
    assert "tcgen05" in P.dode_last_path(g.h)
    # dode_join: an event recorded on the ctx stream afterwards completes only after all steps; reading q straight from
    # a device-side copy issued on that stream must then see the final state
    P.dode_join(g.h)
    ev = torch.cuda.Event()
    ev.record()
    ev.synchronize()
    q_gpu = g.q()
    q_cpu = hz.oracle_run(p, sched, etas)
    hz.assert_q_close(q_gpu, q_cpu, "lanes")
    g.close()


@pytest.mark.parametrize("T,H,N,L,b", [(1, 0, 600, 520, 16), (2, 1, 300, 600, 40), (3, 4, 260, 200, 8)])
def test_short_time_axis_split_k(T, H, N, L, b):
    """Time axes too short to fill the machine (the Fig. 12 shape, T = 1): the tensor path splits K over several CTAs
    per tile and finishes each pass in splitk_epilogue."""
    cfg = synth.Config("splitk", N=N, L=L, T=T, H=H, C=2, D=4 * b, b=b, K=6, kmin=5, kmax=20)
    _run_both(cfg)          # (the last chunk of the schedule may be a ragged one below 8 days, i.e. an FFMA step)


@pytest.mark.parametrize("ks", [2, 5])
def test_forced_split_k_on_ragged_shapes(ks):
    """Forced split counts on ragged shapes: K ranges that are empty near the day boundary, partial tiles, pad days; the
    Adagrad variant goes through the same epilogue kernel."""
    cfg = synth.Config("ragged", N=61, L=137, T=20, H=5, C=2, D=80, b=20, K=12, kmin=3, kmax=9)
    _run_both(cfg, sample=[0, 1, 40, 79], ksplit=ks)


@pytest.mark.parametrize("pair", [0, 1, 2])
@pytest.mark.parametrize("N,L,T,H,D,b", [(300, 200, 80, 3, 130, 130), (300, 200, 48, 3, 512, 256), (100, 384, 60, 5, 330, 165),
                                         (520, 70, 90, 12, 128, 128), (130, 260, 100, 2, 192, 96),
                                         (40, 300, 200, 0, 100, 100), (33, 257, 160, 2, 129, 129)])
def test_cta_pair_kernel(N, L, T, H, D, b, pair):
    """Minibatches wider than 64 days on the CTA-pair kernel (tcgen05.mma.cta_group::2, kernels_tc2.cuh): even and odd
    tile counts (the odd last tile on the single-CTA kernel, or paired with an idle CTA), a single tile (no pair at
    all), half tiles, one and two day groups of 96 / 128 days, ragged day counts, K ranges shorter than the ring (H = 0); DODE_OPT_TC_PAIR = 0 runs the same
    shapes on the single-CTA kernels."""
    cfg = synth.Config("pair", N=N, L=L, T=T, H=H, C=1, D=D, b=b, K=4, kmin=3, kmax=9, label_mode="zero")
    sample = sorted({0, 1, b // 2 - 1, b // 2, b - 1, D // 2, D - 1})
    path = _run_both(cfg, sample=sample, pair=pair)
    assert ("_pair" in path) == (pair != 0), path


def test_minibatch_larger_than_one_launch():
    """A minibatch of more than 256 days is split into several launches inside one dode_spgd_step (days are independent
    units); the sub-batches alternate on the internal streams."""
    cfg = synth.Config("wide_b", N=30, L=40, T=12, H=3, C=1, D=640, b=300, K=5, kmin=3, kmax=9, label_mode="zero")
    assert "tcgen05" in _run_both(cfg, sample=[0, 1, 255, 256, 299, 300, 639])


def test_options_and_reserve_keep_results():
    """dode_set_option / dode_reserve (include/dode.h): every option value gives the oracle's iterates; unknown options
    and out-of-range values are DODE_EINVAL and change nothing; after dode_reserve(b) the steps allocate nothing (the
    launch count grows by exactly the kernels of the steps and device memory does not move)."""
    cfg = synth.Config("opts", N=70, L=90, T=20, H=3, C=2, D=96, b=24, K=10, kmin=3, kmax=9)
    p = hz.make_problem(cfg)
    sched = synth.schedule(cfg, p.labels)
    etas = hz.oracle_etas(p)
    want = hz.oracle_run(p, sched, etas)
    for opts in ({}, {"LANES": 0}, {"PDL": 0}, {"LANES": 0, "PDL": 0, "TC_KSPLIT": 3}, {"TC_MIN_B": 0}, {"TC_MIN_B": 100},
                 {"TC_BSTAGES": 2}, {"TC_BSTAGES": 5, "TC_KSPLIT": 2}, {"TC_BSTAGES": 8}, {"TC_PAIR": 0}, {"TC_PAIR": 2}):
        g0 = hz.GpuSolver(p)                           # a throw-away pass first: the CUDA runtime loads kernel modules
        for k, v in opts.items():                      # lazily, which moves device memory at a kernel's first launch
            g0.P.dode_set_option(g0.h, getattr(g0.P, "DODE_OPT_" + k), v)
        g0.run(sched, etas)
        g0.close()
        g = hz.GpuSolver(p)
        P = g.P
        for k, v in opts.items():
            P.dode_set_option(g.h, getattr(P, "DODE_OPT_" + k), v)
        for bad in ((99, 1), (P.DODE_OPT_LANES, 2), (P.DODE_OPT_TC_KSPLIT, 33), (P.DODE_OPT_TC_MIN_B, -1), (P.DODE_OPT_PDL, -1),
                    (P.DODE_OPT_TC_BSTAGES, 1), (P.DODE_OPT_TC_BSTAGES, 9), (P.DODE_OPT_TC_PAIR, 3), (P.DODE_OPT_TC_PAIR, -1)):
            with pytest.raises(P.DodeError) as e:
                P.dode_set_option(g.h, *bad)
            assert e.value.code == P.DODE_EINVAL
        P.dode_reserve(g.h, cfg.b)
        free0 = torch.cuda.mem_get_info()[0]
        g.run(sched, etas)
        assert torch.cuda.mem_get_info()[0] == free0, "a step allocated device memory after dode_reserve"
        path = P.dode_last_path(g.h)
        assert ("ffma" in path) == (opts.get("TC_MIN_B") in (0, 100)), (opts, path)
        hz.assert_q_close(g.q(), want, f"options {opts}")
        g.close()
