"""Parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (same b, same kernels, inputs
generated on the device by the same synth calls).  The oracle cannot replay whole epochs of configs 2-4, so — days
being independent units (pin P10) — it replays every visit of a few SAMPLED days one by one and those
days' final q and objective are compared; config 1 is also compared on ALL days after one epoch."""
import numpy as np
import pytest
import torch

import paper_1901_09266_b200 as P
from paper_1901_09266_b200 import synth
from tests import harness as hz

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


def _oracle():
    from oracle import oracle
    oracle.build_oracle()
    return oracle


def _check(q_gpu, q_cpu, f_gpu, f_cpu, what):
    worst = hz.assert_q_close(q_gpu, q_cpu, what)
    rel = abs(f_gpu - f_cpu) / max(abs(f_cpu), 1e-30)
    assert rel <= 1e-4, f"{what}: objective relative error {rel:.3e}"
    return worst


def _get_q(h, cfg, day):
    out = torch.empty((cfg.T, cfg.N), dtype=torch.float32)
    P.dode_get_q(h, int(day), out)
    return out.numpy()


def _dense_setup(cfg):
    dev = torch.device(DEV)
    lab = synth.labels(cfg).numpy()
    R = synth.dar_dense(cfg, device=dev)
    x = synth.counts(cfg, R, synth.q_true(cfg, dev), torch.from_numpy(lab))
    torch.cuda.empty_cache()
    h = P.dode_create(cfg.N, cfg.L, cfg.T, cfg.H, cfg.C, cfg.D, lab, x, 1.0, dense=R)
    etas = np.array([np.float32(1.0 / P.dode_lipschitz(h, c, 30)) for c in range(cfg.C)], np.float32)   # a7: a plain number for both sides
    return h, lab, R, x, etas


def _replay(o, Rc_host, x_days, sched, etas, sample, T, N):
    """Oracle replay of the sampled days' visits only."""
    q = {int(d): np.ones((T, N), np.float32) for d in sample}
    for c, days in sched:
        for d in days:
            if int(d) in q:
                q[int(d)] = o.visit(Rc_host[c], q[int(d)], x_days[int(d)], float(etas[c]))
    return q


def test_config1_corridor_full_all_days_then_sampled():
    cfg = synth.CONFIGS["corridor"]
    o = _oracle()
    h, lab, R, x, etas = _dense_setup(cfg)
    Rh = {c: R[c].cpu().numpy() for c in range(cfg.C)}
    xh = x.cpu().numpy()
    del R
    epochs = 4
    rng = synth._Counter(cfg.seed, synth.S_SCHED)
    sched = []
    per_epoch = []
    for _ in range(epochs):
        ep = synth.epoch_chunks(np.asarray(lab, np.int64), cfg.b, rng)
        per_epoch.append(len(ep))
        sched += ep
    # epoch 1: every day, element by element
    for c, days in sched[: per_epoch[0]]:
        P.dode_spgd_step(h, days, float(etas[c]))
    P.dode_sync(h)
    assert P.dode_last_path(h).startswith("tcgen05")
    q_cpu = _replay(o, Rh, xh, sched[: per_epoch[0]], etas, range(cfg.D), cfg.T, cfg.N)
    worst = 0.0
    for d in range(cfg.D):
        worst = max(worst, hz.assert_q_close(_get_q(h, cfg, d), q_cpu[d], f"corridor epoch 1 day {d}"))
    # remaining epochs: sampled days, with the objective
    for c, days in sched[per_epoch[0]:]:
        P.dode_spgd_step(h, days, float(etas[c]))
    P.dode_sync(h)
    sample = [0, 17, 101, 200, 364]
    q_cpu = _replay(o, Rh, xh, sched, etas, sample, cfg.T, cfg.N)
    per_day, _ = P.dode_objective(h, sample)
    for i, d in enumerate(sample):
        f_cpu = o.objective_day(Rh[int(lab[d])], q_cpu[d], xh[d])
        _check(_get_q(h, cfg, d), q_cpu[d], per_day[i], f_cpu, f"corridor {epochs} epochs day {d}")
    P.dode_destroy(h)


def test_config2_multiyear_full_sampled_days():
    cfg = synth.CONFIGS["multiyear"]
    o = _oracle()
    h, lab, R, x, etas = _dense_setup(cfg)
    rng = synth._Counter(cfg.seed, synth.S_SCHED)
    sched = []
    for _ in range(2):
        sched += synth.epoch_chunks(np.asarray(lab, np.int64), cfg.b, rng)
    c0, first = sched[0]
    sample = [int(first[0]), int(first[len(first) // 2]), int(first[-1])]
    Rh = {c0: R[c0].cpu().numpy()}
    xh = {d: x[d].cpu().numpy() for d in sample}
    del R
    for c, days in sched:
        P.dode_spgd_step(h, days, float(etas[c]))
    P.dode_sync(h)
    assert P.dode_last_path(h).startswith("tcgen05")
    q_cpu = _replay(o, Rh, xh, [(c, d) for c, d in sched if c == c0], etas, sample, cfg.T, cfg.N)
    per_day, _ = P.dode_objective(h, sample)
    for i, d in enumerate(sample):
        _check(_get_q(h, cfg, d), q_cpu[d], per_day[i], o.objective_day(Rh[c0], q_cpu[d], xh[d]), f"multiyear day {d}")
    P.dode_destroy(h)


def test_config3_large_dense_minibatch_sweep_sampled_days():
    cfg = synth.CONFIGS["large_dense"]
    o = _oracle()
    h, lab, R, x, etas = _dense_setup(cfg)
    c0 = int(lab[0])
    days_c0 = np.nonzero(lab == c0)[0].astype(np.int32)
    sample = [int(days_c0[0]), int(days_c0[5])]
    Rh = {c0: R[c0].cpu().numpy()}
    xh = {d: x[d].cpu().numpy() for d in sample}
    del R
    torch.cuda.empty_cache()
    ones = torch.ones((cfg.T, cfg.N), dtype=torch.float32)
    # oracle: two visits of each sampled day from q0 = 1 (G8: every b starts from a fresh q0)
    sched2 = [(c0, np.array(sample, np.int32))] * 2
    q_cpu = _replay(o, Rh, xh, sched2, etas, sample, cfg.T, cfg.N)
    f_cpu = {d: o.objective_day(Rh[c0], q_cpu[d], xh[d]) for d in sample}
    for b in (1, 8, 64, 256):
        paths = set()
        for d in days_c0[: max(b, 8)]:
            P.dode_set_q(h, int(d), ones)
        if b == 1:
            lists = [np.array([d], np.int32) for d in sample]
        else:
            lists = [days_c0[:b]]                      # contains both sampled days (positions 0 and 5)
        for _ in range(2):
            for days in lists:
                P.dode_spgd_step(h, days, float(etas[c0]))
                paths.add(P.dode_last_path(h))
        P.dode_sync(h)
        assert all(p.startswith("ffma" if b < 8 else "tcgen05") for p in paths), paths
        per_day, _ = P.dode_objective(h, sample)
        for i, d in enumerate(sample):
            _check(_get_q(h, cfg, d), q_cpu[d], per_day[i], f_cpu[d], f"large_dense b={b} day {d}")
    P.dode_destroy(h)


def test_config4_large_sparse_full_sampled_days():
    cfg = synth.CONFIGS["large_sparse"]
    o = _oracle()
    dev = torch.device(DEV)
    lab = synth.labels(cfg).numpy()
    csr, x = synth.sparse_problem(cfg, dev)
    torch.cuda.empty_cache()
    h = P.dode_create(cfg.N, cfg.L, cfg.T, cfg.H, cfg.C, cfg.D, lab, x, 1.0, csr=csr)
    c0 = int(lab[0])
    eta = np.float32(1.0 / P.dode_lipschitz(h, c0, 20))
    days_c0 = np.nonzero(lab == c0)[0].astype(np.int32)
    days = days_c0[: cfg.b]
    sample = [int(days[0]), int(days[-1])]
    nb = cfg.T * (cfg.H + 1)
    bo = csr.blk_off[c0 * nb:(c0 + 1) * nb + 1].cpu().numpy()
    k0, k1 = int(bo[0]), int(bo[-1])
    rp = csr.row_ptr[c0 * nb:(c0 + 1) * nb].cpu().numpy()
    ci, va = csr.col_idx[k0:k1].cpu().numpy(), csr.val[k0:k1].cpu().numpy()
    bo = bo - k0
    xh = {d: x[d].cpu().numpy() for d in sample}
    del csr
    for _ in range(2):
        P.dode_spgd_step(h, days, float(eta))
    P.dode_sync(h)
    assert P.dode_last_path(h).startswith("csr_")
    per_day, _ = P.dode_objective(h, sample)
    for i, d in enumerate(sample):
        q = np.ones((cfg.T, cfg.N), np.float32)
        for _ in range(2):
            q = o.visit_csr(cfg.N, cfg.L, cfg.T, cfg.H, bo, rp, ci, va, q, xh[d], float(eta))
        f_cpu = o.objective_day_csr(cfg.N, cfg.L, cfg.T, cfg.H, bo, rp, ci, va, q, xh[d])
        _check(_get_q(h, cfg, d), q, per_day[i], f_cpu, f"large_sparse day {d}")
    P.dode_destroy(h)
