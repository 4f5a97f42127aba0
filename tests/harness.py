"""Shared test harness: builds one seeded problem and runs it through the oracle and/or the CUDA library.
Every input array is generated once (synth) and the same bytes go to both sides."""
from __future__ import annotations

import dataclasses
from typing import List, Optional, Sequence, Tuple

import numpy as np
import torch

from paper_1901_09266_b200 import synth


@dataclasses.dataclass
class Problem:
    cfg: synth.Config
    R: torch.Tensor          # CPU fp32 [C][T][H+1][L][N]
    labels: np.ndarray       # int32 [D]
    x: torch.Tensor          # CPU fp32 [D][T][L]
    q_true: torch.Tensor     # CPU fp32 [D][T][N]


def make_problem(cfg: synth.Config, noise: bool = True) -> Problem:
    R = synth.dar_dense(cfg)
    lab = synth.labels(cfg)
    qt = synth.q_true(cfg)
    x = synth.counts(cfg, R, qt, lab, noise=noise)
    return Problem(cfg, R, lab.numpy(), x, qt)


def make_problem_sparse(cfg: synth.Config) -> Problem:
    """G7 sparse instance (small): generated as CSR, densified for the oracle's dense loops."""
    csr, x = synth.sparse_problem(cfg)
    return Problem(cfg, synth.csr_to_dense(cfg, csr), synth.labels(cfg).numpy(), x, synth.q_true(cfg))


def oracle_etas(p: Problem, iters: int = 50) -> np.ndarray:
    """eta_c = (float) 1 / L_c with L_c from the oracle's power iteration (O4)."""
    from oracle import oracle
    return np.array([np.float32(1.0 / oracle.power_iteration(p.R[c].numpy(), iters)) for c in range(p.cfg.C)],
                    np.float32)


def oracle_run(p: Problem, sched, etas: np.ndarray, sample_days: Optional[Sequence[int]] = None) -> np.ndarray:
    from oracle import oracle
    cfg = p.cfg
    q0 = np.ones((cfg.D, cfg.T, cfg.N), np.float32)
    mask = None
    if sample_days is not None:
        mask = np.zeros(cfg.D, np.uint8)
        mask[list(sample_days)] = 1
    return oracle.run_schedule(p.R.numpy(), p.labels, p.x.numpy(), q0, sched, [etas[c] for c, _ in sched], mask)


class GpuSolver:
    """Owns one dode ctx on cuda:0 for a Problem."""

    def __init__(self, p: Problem, csr: bool = False, q0: float = 1.0, tc_min_b: Optional[int] = None):
        import paper_1901_09266_b200 as P
        self.P, self.p = P, p
        cfg = p.cfg
        dev = torch.device("cuda:0")
        xd = p.x.to(dev)
        if csr:
            cs = synth.dense_to_csr(p.R).to(dev)
            self.h = P.dode_create(cfg.N, cfg.L, cfg.T, cfg.H, cfg.C, cfg.D, p.labels, xd, q0, csr=cs)
        else:
            Rd = p.R.to(dev)
            self.h = P.dode_create(cfg.N, cfg.L, cfg.T, cfg.H, cfg.C, cfg.D, p.labels, xd, q0, dense=Rd)
        # the library keeps no caller pointer: dropping Rd / xd here is part of the contract under test
        if tc_min_b is not None:
            P.dode_set_option(self.h, P.DODE_OPT_TC_MIN_B, tc_min_b)

    def run(self, sched, etas):
        for c, days in sched:
            self.P.dode_spgd_step(self.h, days, float(etas[c]))
        self.P.dode_sync(self.h)

    def q(self, days: Optional[Sequence[int]] = None) -> np.ndarray:
        cfg = self.p.cfg
        days = range(cfg.D) if days is None else days
        out = torch.empty((len(days), cfg.T, cfg.N), dtype=torch.float32)
        for i, d in enumerate(days):
            self.P.dode_get_q(self.h, int(d), out[i])
        return out.numpy()

    def close(self):
        if self.h is not None:
            self.P.dode_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def assert_q_close(q_gpu: np.ndarray, q_cpu: np.ndarray, what: str = ""):
    """north_star tolerance: |q_gpu - q_cpu| <= 1e-3 * max(1, |q_cpu|) per element."""
    err = np.abs(q_gpu.astype(np.float64) - q_cpu.astype(np.float64)) / np.maximum(1.0, np.abs(q_cpu))
    worst = float(err.max()) if err.size else 0.0
    assert worst <= 1e-3, f"{what}: max scaled |dq| = {worst:.3e} at {np.unravel_index(err.argmax(), err.shape)}"
    return worst
