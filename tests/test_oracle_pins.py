"""Pins of the CPU oracle against what the paper and the mathematics fix.
None of these touch the CUDA path.  Each test names the mistake it would catch."""
import os

import numpy as np
import pytest
import scipy.optimize
import torch

from oracle import oracle
from paper_1901_09266_b200 import synth
from tests.nnls_active_set import nnls_lawson_hanson

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def assemble_dense(Rc: np.ndarray) -> np.ndarray:
    """Table 2: entry [(h2-1)|A|+a, (h1-1)|K|+k] of the (T*L) x (T*N) matrix,
    block (h2,h1) = R[h1][h2-h1]; no block beyond the day.  0-based here."""
    T, H1, L, N = Rc.shape
    B = np.zeros((T * L, T * N), np.float64)
    for h1 in range(T):
        for lag in range(H1):
            h2 = h1 + lag
            if h2 < T:
                B[h2 * L:(h2 + 1) * L, h1 * N:(h1 + 1) * N] = Rc[h1, lag]
    return B


@pytest.fixture(scope="module")
def tiny12():
    cfg = synth.CONFIGS["tiny12"]
    R = synth.dar_dense(cfg)
    lab = synth.labels(cfg)
    qt = synth.q_true(cfg)
    x = synth.counts(cfg, R, qt, lab, noise=True)
    x0 = synth.counts(cfg, R, qt, lab, noise=False)
    return cfg, R.numpy(), lab.numpy(), qt.numpy(), x.numpy(), x0.numpy()


def converge(Rc, x_day, eta, iters, q0=None):
    T, H1, L, N = Rc.shape
    q = np.ones((1, T, N), np.float32) if q0 is None else q0.reshape(1, T, N)
    sched = [(0, np.array([0], np.int32))] * iters
    return oracle.run_schedule(Rc[None], np.zeros(1, np.int32), x_day[None], q, sched, [eta] * iters)[0]


def test_p7_generator_invariants(tiny12):
    """Eq. 17-18: lag fractions of a covered (s,l,n) sum to 1, others are 0, all >= 0."""
    cfg, R, *_ = tiny12
    mask = synth.incidence_mask(cfg).numpy()
    tot = R[0].sum(axis=1)                      # [T][L][N]
    assert (R >= 0).all()
    np.testing.assert_allclose(tot[:, mask], 1.0, atol=1e-5)
    assert (tot[:, ~mask] == 0).all()
    k = mask.sum(axis=0)
    assert k.min() >= cfg.kmin and k.max() <= cfg.kmax


def test_p12_dense_assembly(tiny12):
    """Operator indexing: O2a/O2b equal the plain mat-vec with Table 2's assembled matrix."""
    cfg, R, lab, qt, x, _ = tiny12
    Rc = R[0]
    B = assemble_dense(Rc)
    rng = np.random.default_rng(1)
    q = rng.random((cfg.T, cfg.N)).astype(np.float32) * 30
    r = oracle.forward_residual(Rc, q, x[3])
    ref = B @ q.reshape(-1).astype(np.float64) - x[3].reshape(-1)
    np.testing.assert_allclose(r.reshape(-1), ref, rtol=1e-6, atol=1e-5)
    g = oracle.gradient(Rc, r)
    np.testing.assert_allclose(g.reshape(-1), B.T @ r.reshape(-1).astype(np.float64), rtol=1e-12, atol=1e-9)
    assert abs(oracle.objective_day(Rc, q, x[3]) - float(ref @ ref)) <= 1e-10 * float(ref @ ref)


def test_p12_dense_assembly_full_tiny():
    """Same on config 0 itself (T=288): catches a wrong truncation at either end of the day."""
    cfg = synth.CONFIGS["tiny"]
    Rc = synth.dar_dense(cfg).numpy()[0]
    B = assemble_dense(Rc)
    rng = np.random.default_rng(2)
    q = rng.random((cfg.T, cfg.N)).astype(np.float32)
    x = rng.random((cfg.T, cfg.L)).astype(np.float32)
    r = oracle.forward_residual(Rc, q, x)
    np.testing.assert_allclose(r.reshape(-1), B @ q.reshape(-1).astype(np.float64) - x.reshape(-1), atol=1e-6)
    np.testing.assert_allclose(oracle.gradient(Rc, r).reshape(-1), B.T @ r.reshape(-1).astype(np.float64), atol=1e-9)


def test_p6_example1_two_link():
    """PAPER.md:114-124 Example 1: x1(t)=f(t), x2(t+dt)=f(t), x2(t0)=0 — pins lag direction, day-boundary
    truncation (A5), the gradient factor convention (A1) and the projection."""
    rows = {}
    for line in open(os.path.join(GOLD, "example1_two_link.txt")):
        if line.startswith("#") or ":" not in line:
            continue
        k, v = line.split(":")
        rows[k.strip()] = np.array(v.split(), np.float32)
    f1, x1, x2 = rows["f1"], rows["x1"], rows["x2"]
    T = len(f1)
    Rc = np.zeros((T, 2, 2, 1), np.float32)      # N=1, L=2, H=1
    Rc[:, 0, 0, 0] = 1.0                          # lag 0 -> link 1
    Rc[:, 1, 1, 0] = 1.0                          # lag 1 -> link 2
    fwd = oracle.forward_residual(Rc, f1.reshape(T, 1), np.zeros((T, 2), np.float32))
    np.testing.assert_array_equal(fwd[:, 0], x1)
    np.testing.assert_array_equal(fwd[:, 1], x2)
    # rho^T rho = diag(2,...,2,1) => L = 2, eta = 1/2: one step lands on (x1[s]+x2[s+1])/2, last entry halves its error.
    assert abs(oracle.power_iteration(Rc, 200) - 2.0) < 1e-6
    x = np.stack([x1, x2], axis=1)
    q0 = np.array([7, 0, 2, 30, 1, 4], np.float32).reshape(T, 1)
    q1 = oracle.visit(Rc, q0, x, 0.5)
    expect = np.maximum(0, np.append((x1[:-1] + x2[1:]) / 2, (q0[-1, 0] + x1[-1]) / 2))
    np.testing.assert_allclose(q1[:, 0], expect, rtol=1e-7)
    # projection: a target that is negative must clamp to exactly 0
    xneg = x.copy(); xneg[2, 0] = -50.0
    assert oracle.visit(Rc, q0, xneg, 0.5)[2, 0] == 0.0


def test_p5_degenerate_closed_form():
    """T=1, H=0 reduces to textbook projected gradient; with the constraint inactive
    q_k - q* = (I - eta B^T B)^k (q_0 - q*)."""
    B = np.array([[2.0, 0.5, 0.1], [0.3, 1.5, 0.2], [0.1, 0.4, 1.0]], np.float32)
    qstar = np.array([4.0, 5.0, 6.0])
    y = (B.astype(np.float64) @ qstar).astype(np.float32)
    Rc = B.reshape(1, 1, 3, 3)
    eta = 0.15
    q = np.array([[5.0, 4.0, 7.0]], np.float32)
    M = np.eye(3) - eta * B.astype(np.float64).T @ B.astype(np.float64)
    qs64 = np.linalg.solve(B.astype(np.float64), y.astype(np.float64))
    e0 = q[0].astype(np.float64) - qs64
    for k in range(1, 21):
        q = oracle.visit(Rc, q, y.reshape(1, 3), eta)
        np.testing.assert_allclose(q[0], qs64 + np.linalg.matrix_power(M, k) @ e0, rtol=2e-6)


def test_p8_adjoint(tiny12):
    """<rho u, v> = <u, rho^T v>: the transpose loop is the adjoint of the forward loop, truncation included."""
    cfg, R, *_ = tiny12
    rng = np.random.default_rng(3)
    for Rc in (R[0], synth.dar_dense(synth.CONFIGS["tiny"]).numpy()[0][:40]):
        T, H1, L, N = Rc.shape
        u = rng.standard_normal((T, N)).astype(np.float32)
        v = rng.standard_normal((T, L)).astype(np.float32)
        ru = oracle.forward_residual(Rc, u, np.zeros((T, L), np.float32)).astype(np.float64)
        rtv = oracle.gradient(Rc, v)
        lhs, rhs = float((ru * v).sum()), float((u.astype(np.float64) * rtv).sum())
        assert abs(lhs - rhs) <= 1e-5 * max(1.0, abs(lhs))


def test_p3_finite_differences(tiny12):
    """d f / d q = 2 g (reading A1): f is quadratic, so central differences are exact up to rounding."""
    cfg, R, lab, qt, x, _ = tiny12
    Rc = R[0]
    rng = np.random.default_rng(4)
    q = (rng.random((cfg.T, cfg.N)) * 40).astype(np.float32)
    g = oracle.gradient(Rc, oracle.forward_residual(Rc, q, x[0]))
    delta = 0.5
    for (s, n) in [(0, 0), (3, 2), (7, 1), (11, 3), (5, 0)]:
        qp, qm = q.copy(), q.copy()
        qp[s, n] += delta
        qm[s, n] -= delta
        fd = (oracle.objective_day(Rc, qp, x[0]) - oracle.objective_day(Rc, qm, x[0])) / (2 * delta)
        assert abs(fd - 2 * g[s, n]) <= 1e-5 * max(1.0, abs(fd))


def _eta(Rc):
    return np.float32(1.0 / oracle.power_iteration(Rc, 50))


def test_power_iteration_matches_eigensolver(tiny12):
    """O4 against numpy's symmetric eigensolver on the assembled Gram matrix."""
    cfg, R, *_ = tiny12
    B = assemble_dense(R[0])
    lam = np.linalg.eigvalsh(B.T @ B)[-1]
    est = oracle.power_iteration(R[0], 50)
    assert est <= lam * (1 + 1e-12) and est >= 0.98 * lam
    assert abs(oracle.power_iteration(R[0], 3000) - lam) <= 1e-6 * lam


def test_p1_p2_active_set_and_kkt(tiny12):
    """T=12 sub-instance (48 unknowns, 72 equations): the oracle iterated to convergence equals the
    Lawson-Hanson solve (own implementation and scipy's), and satisfies KKT."""
    cfg, R, lab, qt, x, _ = tiny12
    Rc = R[0]
    B = assemble_dense(Rc)
    np.linalg.cholesky(B.T @ B)                       # Gram matrix must be PD (generator contract, G2)
    ev = np.linalg.eigvalsh(B.T @ B)
    assert ev[-1] / ev[0] < 1e4                       # synth.TINY_REDRAW was chosen for this
    eta = _eta(Rc)
    for day in (0, 5):
        y = x[day].reshape(-1).astype(np.float64)
        q_lh = nnls_lawson_hanson(B, y)
        q_sp, _ = scipy.optimize.nnls(B, y, maxiter=10000)
        np.testing.assert_allclose(q_lh, q_sp, atol=1e-8)
        q = converge(Rc, x[day], eta, 60000)
        g = oracle.gradient(Rc, oracle.forward_residual(Rc, q, x[day]))
        eps = 1e-4 * np.abs(B.T @ y).max()             # A14
        assert (g[q == 0] >= -eps).all()
        assert (np.abs(g[q > 0]) <= eps).all()
        f_or = oracle.objective_day(Rc, q, x[day])
        f_lh = float(np.sum((B @ q_lh - y) ** 2))
        assert f_or >= f_lh * (1 - 1e-9) and f_or <= f_lh * (1 + 1e-6)
        np.testing.assert_allclose(q.reshape(-1), q_lh, atol=5e-3, rtol=1e-4)


def test_p4_planted_recovery(tiny12):
    """Fig. 12 protocol: x = rho q_true noiseless => f -> 0 and q -> q_true (full column rank)."""
    cfg, R, lab, qt, _, x0 = tiny12
    Rc = R[0]
    q = converge(Rc, x0[2], _eta(Rc), 200000)
    f0 = oracle.objective_day(Rc, np.ones_like(qt[2]), x0[2])
    assert oracle.objective_day(Rc, q, x0[2]) <= 1e-8 * f0
    np.testing.assert_allclose(q, qt[2], rtol=5e-3, atol=5e-3)


def test_p9_monotone_descent(tiny12):
    """Projected gradient with eta <= 1/L never increases the objective."""
    cfg, R, lab, qt, x, _ = tiny12
    Rc = R[0]
    eta = _eta(Rc)
    q = np.ones((cfg.T, cfg.N), np.float32)
    f = oracle.objective_day(Rc, q, x[1])
    for _ in range(200):
        q = oracle.visit(Rc, q, x[1], eta)
        f2 = oracle.objective_day(Rc, q, x[1])
        assert f2 <= f * (1 + 1e-7)
        f = f2


def test_p10_separability_and_schedule(tiny12):
    """A day's iterate depends only on its visit count: minibatch composition, and a day mask, change nothing."""
    cfg, R, lab, qt, x, _ = tiny12
    eta = _eta(R[0])
    sched = synth.schedule(cfg, lab, K=60)
    for c, days in sched:
        assert len(set(days.tolist())) == len(days) <= cfg.b and all(lab[d] == c for d in days)
    q0 = np.ones((cfg.D, cfg.T, cfg.N), np.float32)
    qa = oracle.run_schedule(R, lab, x, q0, sched, [eta] * len(sched))
    single = [(c, np.array([d], np.int32)) for c, days in sched for d in days]      # b = 1, same visits
    qb = oracle.run_schedule(R, lab, x, q0, single, [eta] * len(single))
    np.testing.assert_array_equal(qa, qb)
    mask = np.zeros(cfg.D, np.uint8); mask[[2, 9]] = 1
    qc = oracle.run_schedule(R, lab, x, q0, sched, [eta] * len(sched), day_mask=mask)
    np.testing.assert_array_equal(qc[[2, 9]], qa[[2, 9]])
    np.testing.assert_array_equal(qc[0], q0[0])
    visits = np.bincount(np.concatenate([d for _, d in sched]), minlength=cfg.D)
    q5 = q0[5]
    for _ in range(visits[5]):
        q5 = oracle.visit(R[0], q5, x[5], eta)
    np.testing.assert_array_equal(q5, qa[5])


def test_p10b_schedule_with_several_clusters_and_a_step_per_iteration():
    """oracle_run_schedule picks the operator by the DAY's label and the step by the ITERATION (dode_oracle.cpp: `R +
    Rc_sz * labels[day]`, `sched_eta[k]`).  Pinned against replays that use nothing but oracle.visit with R[labels[d]]
    and eta[k], bit for bit, on C = 3 clusters whose operators differ and with a different step in every iteration: a
    wrong cluster stride, an operator picked by the chunk's position, or a step indexed by day fail it."""
    cfg = synth.Config("p10b", N=5, L=7, T=9, H=3, C=3, D=17, b=3, K=40, kmin=2, kmax=4)
    R = synth.dar_dense(cfg).numpy()
    lab = synth.labels(cfg).numpy()
    assert len(set(lab.tolist())) == 3 and not np.array_equal(R[0], R[1]) and not np.array_equal(R[1], R[2])
    x = synth.counts(cfg, torch.from_numpy(R), synth.q_true(cfg), torch.from_numpy(lab)).numpy()
    sched = synth.schedule(cfg, lab)
    base = [_eta(R[c]) for c in range(cfg.C)]
    etas = [np.float32(base[c] * (0.35 + 0.6 * ((7 * k) % 11) / 11.0)) for k, (c, _) in enumerate(sched)]
    assert len(set(float(e) for e in etas)) > 20
    q0 = (1.0 + np.random.default_rng(3).random((cfg.D, cfg.T, cfg.N))).astype(np.float32)
    got = oracle.run_schedule(R, lab, x, q0, sched, etas)
    want = q0.copy()
    for k, (c, days) in enumerate(sched):
        for d in days:
            assert lab[d] == c
            want[d] = oracle.visit(R[lab[d]], want[d], x[d], float(etas[k]))
    np.testing.assert_array_equal(got, want)
    assert not np.array_equal(got, q0)
    # and the mistakes it is meant to catch do change the result on this instance
    wrong = q0.copy()
    for k, (c, days) in enumerate(sched):
        for d in days:
            wrong[d] = oracle.visit(R[(lab[d] + 1) % cfg.C], wrong[d], x[d], float(etas[k]))
    assert np.abs(wrong - want).max() > 1e-3


@pytest.mark.parametrize("threads", [1, 3, 8])
def test_p18_day_replay_equals_repeated_visits(tiny12, threads):
    """oracle_replay_day / oracle_replay_day_csr (the full-K replays of the GPU parity tests): the output rows of each
    pass go to several threads, every output element is accumulated in the same order — so any thread count, dense or
    CSR, must reproduce repeated oracle_visit / oracle_visit_csr BIT FOR BIT at every checkpoint."""
    cfg, R, lab, qt, x, _ = tiny12
    eta = _eta(R[0])
    q0 = (1.0 + np.random.default_rng(8).random((cfg.T, cfg.N))).astype(np.float32)
    ck = [1, 2, 5, 11, 12]
    got, done = oracle.replay_day(R[0], q0, x[6], eta, 12, ck, threads=threads)
    assert done == 12 and sorted(got) == ck
    q = q0
    for v in range(1, 13):
        q = oracle.visit(R[0], q, x[6], eta)
        if v in got:
            np.testing.assert_array_equal(got[v], q)
    assert (q == 0).any() and (q > 0).any()          # the projection is active on this instance
    assert oracle.objective_day(R[0], q, x[6], threads=threads) == oracle.objective_day(R[0], q, x[6])
    csr = synth.dense_to_csr(torch.from_numpy(R))
    arrs = (cfg.N, cfg.L, cfg.T, cfg.H, csr.blk_off.numpy(), csr.row_ptr.numpy(), csr.col_idx.numpy(), csr.val.numpy())
    got, done = oracle.replay_day(None, q0, x[6], eta, 7, [3, 7], threads=threads, csr=arrs)
    q = q0
    for v in range(1, 8):
        q = oracle.visit_csr(*arrs, q, x[6], eta)
        if v in got:
            np.testing.assert_array_equal(got[v], q)
    assert done == 7 and sorted(got) == [3, 7]
    # a spent time budget stops the replay between visits and reports how far it got
    got, done = oracle.replay_day(R[0], q0, x[6], eta, 100000, [1, 100000], threads=threads, budget_s=0.05)
    assert 1 <= done < 100000 and sorted(got) == [1]


def test_schedule_epoch_structure():
    """A8: per epoch every day appears exactly once; chunks are same-cluster, <= b, ragged tails kept."""
    cfg = synth.CONFIGS["corridor"]
    lab = synth.labels(cfg).numpy()
    ep = synth.one_epoch(cfg, lab)
    alld = np.concatenate([d for _, d in ep])
    assert sorted(alld.tolist()) == list(range(cfg.D))
    assert len(ep) == sum(-(-int((lab == c).sum()) // cfg.b) for c in range(cfg.C))
    s1, s2 = synth.schedule(cfg, lab, K=37), synth.schedule(cfg, lab, K=37)
    assert all(a[0] == b[0] and (a[1] == b[1]).all() for a, b in zip(s1, s2)) and len(s1) == 37
    full = synth.schedule(cfg, lab, K=20, full_only=True)
    assert all(len(d) == cfg.b for _, d in full)


def test_p13_dense_vs_csr(tiny12):
    """a6: the CSR visit equals the dense visit on the same operator."""
    cfg, R, lab, qt, x, _ = tiny12
    csr = synth.dense_to_csr(torch.from_numpy(R))
    assert csr.nnz == int((R != 0).sum())
    eta = _eta(R[0])
    q = np.ones((cfg.T, cfg.N), np.float32)
    qd, qs = q, q
    for _ in range(5):
        qd = oracle.visit(R[0], qd, x[4], eta)
        qs = oracle.visit_csr(cfg.N, cfg.L, cfg.T, cfg.H, csr.blk_off.numpy(), csr.row_ptr.numpy(),
                              csr.col_idx.numpy(), csr.val.numpy(), qs, x[4], eta)
    np.testing.assert_allclose(qs, qd, rtol=1e-6, atol=1e-6)
    fd = oracle.objective_day(R[0], qd, x[4])
    fs = oracle.objective_day_csr(cfg.N, cfg.L, cfg.T, cfg.H, csr.blk_off.numpy(), csr.row_ptr.numpy(),
                                  csr.col_idx.numpy(), csr.val.numpy(), qd, x[4])
    assert abs(fd - fs) <= 1e-12 * fd


def test_p14_r2_closed_forms(tiny12):
    """O5 (Step 6; reading A17): R2 = 1 - SS_res / SS_tot with the observed counts as reference.
    Pinned by cases with a closed form: a perfect fit gives exactly 1; q = 0 gives 1 - sum x^2 / sum (x - mean)^2;
    and the general case equals the textbook formula evaluated with the Table-2 assembled matrix."""
    cfg, R, lab, qt, x, xclean = tiny12
    o = oracle
    Rc = R[0]
    d = 3
    # perfect fit on the noiseless counts (x0 is rho q_true rounded to fp32, hence the tolerance)
    assert abs(o.r2_day(Rc, qt[d], xclean[d]) - 1.0) < 1e-9
    # q = 0: the residual is -x
    xd = x[d].astype(np.float64)
    want0 = 1.0 - (xd ** 2).sum() / ((xd - xd.mean()) ** 2).sum()
    assert abs(o.r2_day(Rc, np.zeros((cfg.T, cfg.N), np.float32), x[d]) - want0) < 1e-12
    # general q: dense assembly (P12's matrix) + numpy
    A = assemble_dense(Rc)
    q = (np.random.default_rng(5).random((cfg.T, cfg.N)) * 30).astype(np.float32)
    fit = A @ q.reshape(-1).astype(np.float64)
    want = 1.0 - ((xd.reshape(-1) - fit) ** 2).sum() / ((xd - xd.mean()) ** 2).sum()
    assert abs(o.r2_day(Rc, q, x[d]) - want) < 1e-10
    # a better fit scores higher: a few SPGD visits raise R2 from the q0 = 1 start
    eta = _eta(Rc)
    q1 = np.ones((cfg.T, cfg.N), np.float32)
    r2_a = o.r2_day(Rc, q1, x[d])
    for _ in range(20):
        q1 = o.visit(Rc, q1, x[d], eta)
    assert o.r2_day(Rc, q1, x[d]) > r2_a


def test_p15_row_chunk_adagrad_against_torch(tiny12):
    """O6 / NEXT-1 (Alg. 1 as printed): row-chunk minibatches + Adagrad + projection.  The paper's
    implementation is PyTorch, so the pin is torch.optim.Adagrad itself on the Table-2 assembled matrix: the same
    permuted row chunks, g = B_o^T(B_o x - y_o), optimizer step, clamp — in float64."""
    import torch
    cfg, R, lab, qt, x, _ = tiny12
    Rc = R[0]
    d = 2
    A = torch.from_numpy(assemble_dense(Rc))                       # (T*L) x (T*N), float64
    y = torch.from_numpy(x[d].astype(np.float64).reshape(-1))
    rows = cfg.T * cfg.L
    rng = np.random.default_rng(11)
    eta, eps, bs = 0.5, 1e-10, 29                                  # 72 rows -> chunks of 29, 29, 14 (ragged tail)
    p = torch.nn.Parameter(torch.ones(cfg.T * cfg.N, dtype=torch.float64))
    opt = torch.optim.Adagrad([p], lr=eta, eps=eps, initial_accumulator_value=0.0, lr_decay=0.0)
    q = np.ones((cfg.T, cfg.N), np.float32)
    G = np.zeros((cfg.T, cfg.N), np.float32)
    for epoch in range(6):
        perm = rng.permutation(rows)
        for c0 in range(0, rows, bs):
            chunk = perm[c0:c0 + bs]
            mask = np.zeros(rows, np.uint8); mask[chunk] = 1
            Bo, yo = A[chunk], y[chunk]
            with torch.no_grad():
                p.grad = Bo.T @ (Bo @ p - yo)                      # Alg. 1 line 9: no factor 2 (reading A1)
            opt.step()
            with torch.no_grad():
                p.clamp_(min=0.0)                                  # line 11
            q, G = oracle.visit_adagrad(Rc, q, G, x[d], mask.reshape(cfg.T, cfg.L), eta, eps)
    want = p.detach().numpy().reshape(cfg.T, cfg.N)
    np.testing.assert_allclose(q, want, rtol=2e-4, atol=2e-4)
    # mask = None is the full-batch step
    qa, Ga = oracle.visit_adagrad(Rc, q, G, x[d], None, eta, eps)
    qb, Gb = oracle.visit_adagrad(Rc, q, G, x[d], np.ones((cfg.T, cfg.L), np.uint8), eta, eps)
    np.testing.assert_array_equal(qa, qb); np.testing.assert_array_equal(Ga, Gb)


# ---- P16: DAR construction from speeds (O7, NEXT-4) -----------------------------------------------------------------
def _example3_instance():
    T, H, L, N, dt = 6, 4, 3, 1, 300.0
    length = np.array([1000.0, 1500.0, 800.0], np.float32)
    speed = np.full((T, L), 8.0, np.float32)
    speed[0, 0], speed[0, 1] = 5.0, 10.0
    speed[1, 0], speed[1, 1] = 4.0, 3.75
    return T, H, L, N, dt, np.array([0, 3], np.int32), np.array([0, 1, 2], np.int32), length, speed


def test_p16_dar_example3_worked_by_hand():
    """Example 3 (Eq. 19-28) with numbers fixed in tests/golden/example3_three_link_dar.txt."""
    T, H, L, N, dt, pp, pl, length, speed = _example3_instance()
    R = oracle.dar_build(N, L, T, H, pp, pl, length, speed, dt)
    want = np.zeros((H + 1, L))
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "example3_three_link_dar.txt")):
        if line.startswith("#") or not line.strip():
            continue
        l, h2, v = line.split()
        want[int(h2), int(l)] = float(v)
    np.testing.assert_allclose(R[0, :, :, 0], want, rtol=0, atol=1e-7)


def _fifo_violation_instance():
    T, H, L, N, dt = 4, 3, 2, 1, 300.0
    length = np.array([3000.0, 600.0], np.float32)
    speed = np.full((T, L), 10.0, np.float32)
    speed[0, 0] = 5.0
    speed[1:, 0] = 30.0
    want = np.zeros((T, H + 1, L))
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "fifo_violation_two_link.txt")):
        if line.startswith("#") or not line.strip():
            continue
        s_, l, h2, v = line.split()
        want[int(s_), int(h2) - int(s_), int(l)] = float(v)
    return T, H, L, N, dt, np.array([0, 2], np.int32), np.array([0, 1], np.int32), length, speed, want


def test_p16_dar_fifo_violation_worked_by_hand():
    """The `a2 <= a1` branch of O7 (reading A20): when a speed jump lets the trailing trajectory overtake the leading one,
    the whole flow goes to the interval of the LEADING arrival (tests/golden/fifo_violation_two_link.txt, worked by hand),
    and the next departure interval is an ordinary window again."""
    T, H, L, N, dt, pp, pl, length, speed, want = _fifo_violation_instance()
    R = oracle.dar_build(N, L, T, H, pp, pl, length, speed, dt)
    np.testing.assert_allclose(R[:2, :, :, 0], want[:2], rtol=0, atol=1e-7)
    # the multi-path builder with one path takes the same branch
    R8 = oracle.assignment_build(N, L, T, H, np.array([0, 1], np.int32), pp, pl, length, speed, dt, 0.01)
    np.testing.assert_array_equal(R8, R)


def test_p16_dar_constant_speed_closed_form_and_row_sums():
    """Constant speeds: link j is reached after c_j = sum of travel times, so the flow of interval s arrives in intervals
    s + floor(c_j/dt) and the next one with shares 1 - frac and frac (Eq. 17); every covered (s, l, n) sums to 1 over
    h2 (Eq. 18) unless truncated at the day end / at lag H."""
    T, H, L, N, dt = 12, 5, 7, 3, 300.0
    rng = np.random.default_rng(4)
    length = rng.uniform(500, 3000, L).astype(np.float32)
    v = rng.uniform(5, 30, L).astype(np.float32)
    speed = np.tile(v, (T, 1))
    paths = [[0, 1, 2, 3], [2, 3, 4, 5, 6], [6]]
    pp = np.cumsum([0] + [len(p) for p in paths]).astype(np.int32)
    pl = np.concatenate(paths).astype(np.int32)
    R = oracle.dar_build(N, L, T, H, pp, pl, length, speed, dt)
    for n, path in enumerate(paths):
        c = 0.0
        for l in path:
            hh, fr = int(c // dt), (c / dt) % 1.0
            for s in range(T):
                exp = np.zeros(H + 2)
                if hh <= H: exp[hh] = 1.0 - fr
                if hh + 1 <= H + 1: exp[hh + 1] = fr
                exp = exp[:H + 1].copy()
                exp[max(0, T - s):] = 0.0                       # arrival intervals beyond the day are dropped
                np.testing.assert_allclose(R[s, :, l, n], exp, atol=2e-6)
            c += float(length[l]) / float(v[l])
        off = [l for l in range(L) if l not in path]
        assert not R[:, :, off, n].any()
    assert (R >= 0).all()


def test_p16_dar_conserves_vehicles_through_the_forward_operator():
    """Time-varying speeds, H large enough and departures early enough that nothing is truncated: each covered (s, l, n)
    sums to 1 over the lags, so every vehicle of q is counted exactly once on every link of its path by O2a."""
    T, H, L, N, dt = 40, 12, 9, 4, 300.0
    rng = np.random.default_rng(9)
    length = rng.uniform(800, 2500, L).astype(np.float32)
    speed = rng.uniform(6, 25, (T, L)).astype(np.float32)
    paths = [[0, 1, 2, 3, 4], [3, 4, 5], [5, 6, 7, 8], [1, 2]]
    pp = np.cumsum([0] + [len(p) for p in paths]).astype(np.int32)
    pl = np.concatenate(paths).astype(np.int32)
    R = oracle.dar_build(N, L, T, H, pp, pl, length, speed, dt)
    for n, path in enumerate(paths):
        np.testing.assert_allclose(R[:T - H - 1, :, path, n].sum(axis=1), 1.0, atol=1e-6)
    q = np.zeros((T, N), np.float32)
    q[:T - H - 1] = rng.uniform(1, 50, (T - H - 1, N)).astype(np.float32)
    x = oracle.forward_residual(R, q, np.zeros((T, L), np.float32))
    for l in range(L):
        users = [n for n, path in enumerate(paths) if l in path]
        np.testing.assert_allclose(x[:, l].sum(), q[:, users].sum(), rtol=1e-5)


# ---- P17: assignment matrix with several paths per OD and Logit shares (O8, NEXT-4) ---------------------------------
def test_p17_single_path_reduces_to_dar_and_logit_closed_form():
    T, H, L, N, dt = 30, 10, 8, 2, 300.0
    rng = np.random.default_rng(12)
    length = rng.uniform(800, 2500, L).astype(np.float32)
    speed = rng.uniform(6, 25, (T, L)).astype(np.float32)
    # (a) one path per OD: p = 1 and O8 == O7 (Eq. 41 with p = 1)
    paths = [[0, 1, 2, 3], [4, 5, 6]]
    pp = np.cumsum([0] + [len(p) for p in paths]).astype(np.int32)
    pl = np.concatenate(paths).astype(np.int32)
    R7 = oracle.dar_build(N, L, T, H, pp, pl, length, speed, dt)
    R8 = oracle.assignment_build(N, L, T, H, np.array([0, 1, 2], np.int32), pp, pl, length, speed, dt, 0.01)
    np.testing.assert_array_equal(R7, R8)
    # (b) one OD, two link-disjoint paths: the first links carry the route shares themselves, which follow the binary
    #     Logit closed form p_1 = 1 / (1 + exp(-theta (c_2 - c_1))) with the travel times recomputed here (Eq. 37)
    paths = [[0, 1, 2], [4, 5, 6, 7]]
    pp = np.cumsum([0] + [len(p) for p in paths]).astype(np.int32)
    pl = np.concatenate(paths).astype(np.int32)
    theta = 0.01
    R = oracle.assignment_build(1, L, T, H, np.array([0, 2], np.int32), pp, pl, length, speed, dt, theta)
    for s in range(T):
        c = []
        for path in paths:
            t = s * dt
            for l in path:
                t += float(length[l]) / float(speed[min(T - 1, int(t // dt)), l])
            c.append(t - s * dt)
        p1 = 1.0 / (1.0 + np.exp(-theta * (c[1] - c[0])))
        assert abs(R[s, 0, 0, 0] - p1) < 1e-6 and abs(R[s, 0, 4, 0] - (1 - p1)) < 1e-6
    # (c) theta = 0: equal shares; a huge theta: all flow on the faster path
    R0 = oracle.assignment_build(1, L, T, H, np.array([0, 2], np.int32), pp, pl, length, speed, dt, 0.0)
    np.testing.assert_allclose(R0[:, 0, 0, 0], 0.5); np.testing.assert_allclose(R0[:, 0, 4, 0], 0.5)
    Rinf = oracle.assignment_build(1, L, T, H, np.array([0, 2], np.int32), pp, pl, length, speed, dt, 50.0)
    assert set(np.unique(np.round(Rinf[:, 0, 0, 0], 6))) <= {0.0, 1.0}
    # (d) two paths sharing a link: the shared link's shares add up (Eq. 40 sums over k), conservation holds on it
    paths = [[0, 1, 2], [3, 1, 5]]
    pp = np.cumsum([0] + [len(p) for p in paths]).astype(np.int32)
    pl = np.concatenate(paths).astype(np.int32)
    Rs = oracle.assignment_build(1, L, T, H, np.array([0, 2], np.int32), pp, pl, length, speed, dt, theta)
    np.testing.assert_allclose(Rs[:T - H - 1, :, 1, 0].sum(axis=1), 1.0, atol=1e-6)
    np.testing.assert_allclose(Rs[:T - H - 1, 0, 0, 0] + Rs[:T - H - 1, 0, 3, 0], 1.0, atol=1e-6)
