"""NEXT-1: Alg. 1 as the paper prints it — row-chunk minibatches + Adagrad +
projection — through dode_adagrad_step on all three kernel families, against the oracle's O6 (pinned by P15)."""
import numpy as np
import pytest
import torch

from paper_1901_09266_b200 import synth
from tests import harness as hz

pytestmark = pytest.mark.gpu

ETA, EPS = 0.5, 1e-10


def _row_chunks(rng, rows, bs):
    """Alg. 1 lines 5-7: permute the row range, cut it into chunks of bs (ragged tail kept)."""
    perm = rng.permutation(rows)
    return [perm[i:i + bs] for i in range(0, rows, bs)]


def _run(cfg, csr=False, sparse_gen=False, tc_min_b=None, bs_frac=0.3, full_batch_every=4):
    from oracle import oracle
    p = hz.make_problem_sparse(cfg) if sparse_gen else hz.make_problem(cfg)
    sched = synth.schedule(cfg, p.labels)
    rows = cfg.T * cfg.L
    bs = max(1, int(rows * bs_frac))
    rng = np.random.default_rng(5)
    g = hz.GpuSolver(p, csr=csr, tc_min_b=tc_min_b)
    P = g.P
    q = np.ones((cfg.D, cfg.T, cfg.N), np.float32)
    G = np.zeros_like(q)
    visited = set()
    for it, (c, days) in enumerate(sched):
        Rc = p.R[c].numpy()
        if full_batch_every and it % full_batch_every == full_batch_every - 1:
            masks, mdev = [None] * len(days), None                  # NULL mask = every row
        else:
            m = np.zeros((len(days), rows), np.uint8)
            for i in range(len(days)):                               # each day draws its own chunk of its own system
                ch = _row_chunks(rng, rows, bs)
                m[i, ch[int(rng.integers(len(ch)))]] = 1
            masks = list(m.reshape(len(days), cfg.T, cfg.L))
            mdev = torch.from_numpy(m).cuda()
        P.dode_adagrad_step(g.h, days, ETA, EPS, mdev)
        for i, d in enumerate(days):
            q[d], G[d] = oracle.visit_adagrad(Rc, q[d], G[d], p.x[d].numpy(), masks[i], ETA, EPS)
            visited.add(int(d))
    P.dode_sync(g.h)
    days = sorted(visited)
    hz.assert_q_close(g.q(days), q[days], cfg.name)
    path = P.dode_last_path(g.h)
    # reset: the accumulator is zero again, so one more step equals an oracle step from G = 0
    P.dode_adagrad_reset(g.h)
    c, dl = sched[0]
    P.dode_adagrad_step(g.h, dl, ETA, EPS, None)
    want = np.stack([oracle.visit_adagrad(p.R[c].numpy(), q[d], np.zeros_like(G[d]), p.x[d].numpy(), None, ETA, EPS)[0]
                     for d in dl])
    hz.assert_q_close(g.q(dl), want, cfg.name + " after reset")
    with pytest.raises(Exception):
        P.dode_adagrad_step(g.h, dl, ETA, 0.0, None)                 # eps must be positive
    g.close()
    return path


@pytest.mark.parametrize("b", [1, 3, 5])
def test_adagrad_row_chunks_ffma(b):
    cfg = synth.Config("ada_ffma", N=61, L=37, T=50, H=5, C=2, D=30, b=b, K=30, kmin=3, kmax=9)
    assert "ffma" in _run(cfg, tc_min_b=0)


@pytest.mark.parametrize("b", [16, 37])
def test_adagrad_row_chunks_tensor_core(b):
    cfg = synth.Config("ada_tc", N=150, L=140, T=30, H=4, C=2, D=120, b=b, K=16, kmin=3, kmax=12)
    assert "tcgen05" in _run(cfg)


def test_adagrad_row_chunks_cta_pair_kernel():
    """The Adagrad / row-mask epilogues of the CTA-pair kernel (minibatch wider than 64 days, an odd tile count)."""
    cfg = synth.Config("ada_pair", N=300, L=150, T=60, H=3, C=1, D=192, b=96, K=6, kmin=3, kmax=12, label_mode="zero")
    assert "tcgen05_pair" in _run(cfg)


@pytest.mark.parametrize("b", [5, 40])
def test_adagrad_row_chunks_csr(b):
    cfg = synth.Config("ada_csr", N=80, L=50, T=40, H=6, C=2, D=90, b=b, K=12, kmin=4, kmax=10)
    assert "csr" in _run(cfg, csr=True)


def test_adagrad_paper_chunk_size_on_tiny():
    """BASELINE.json configs[0] shape with the paper's proportions: chunks of a third of a day's 1728 rows, 60 iterations."""
    cfg = synth.CONFIGS["tiny"].replace(K=60)
    _run(cfg, bs_frac=1.0 / 3.0)
