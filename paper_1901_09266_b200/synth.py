"""Seeded synthetic inputs for the DODE SPGD hot path.

This module holds *input generators only*: the DAR blocks, cluster labels,
planted demand, observed counts and the minibatch schedule.  It contains none
of the method's arithmetic (no residual, gradient, projection or step-size
code) and is the only module shared by the oracle tests and the CUDA tests:
every array is generated ONCE and the same bytes are handed to both sides
(G1: transcendentals differ by ulps between libm and CUDA, so inputs are never
regenerated independently).

The inputs stand in for the paper's Sacramento I-5/SR-99 2014-2016 data
(PeMS counts, NPMRDS speeds), which are not available;
shapes follow BASELINE.json's five configs (T = 288 five-minute intervals,
PAPER.md:474; D = 1096 days = 3 years).

All generators take a ``device`` so that the large configs can be produced on
the GPU with plain torch ops; the integer hash is bit-identical everywhere,
the floating-point post-processing is not, hence "generate once".
"""
from __future__ import annotations

import dataclasses
import math
import warnings
from typing import List, Optional, Tuple

import numpy as np
import torch

MASTER_SEED = 20190129  # the paper's arXiv date; arbitrary

# stream ids (one per generated array)
S_INC_K, S_INC_START, S_DAR, S_BASE, S_DAYF, S_NOISE, S_LABEL, S_RELABEL = range(1, 9)
S_SCHED, S_TAU, S_WIN, S_SPFRAC, S_PROBE = range(9, 14)
S_LEN, S_VFREE, S_CONG, S_VNOISE, S_NPATH = range(14, 19)

_MASK64 = (1 << 64) - 1


def _i64(v: int) -> int:
    """Two's-complement view of an unsigned 64-bit constant (torch has no uint64 math)."""
    v &= _MASK64
    return v - (1 << 64) if v >= (1 << 63) else v


_K_GOLD = _i64(0x9E3779B97F4A7C15)
_K_M1 = _i64(0xBF58476D1CE4E5B9)
_K_M2 = _i64(0x94D049BB133111EB)
_K_SEED = _i64(0xD1342543DE82EF95)
_K_STREAM = _i64(0xA0761D6478BD642F)


def _lsr(z: torch.Tensor, k: int) -> torch.Tensor:
    """Logical shift right on int64 (torch's >> is arithmetic)."""
    return (z >> k) & ((1 << (64 - k)) - 1)


def mix64(seed: int, stream: int, idx: torch.Tensor) -> torch.Tensor:
    """Counter-based integer mixer (G1): splitmix64 finaliser of
    seed*K_SEED + stream*K_STREAM + idx, all modulo 2^64.  ``idx`` is int64."""
    base = _i64((seed * 0xD1342543DE82EF95 + stream * 0xA0761D6478BD642F) & _MASK64)
    z = idx + base
    z = z + _K_GOLD
    z = (z ^ _lsr(z, 30)) * _K_M1
    z = (z ^ _lsr(z, 27)) * _K_M2
    z = z ^ _lsr(z, 31)
    return z


def mix64_int(seed: int, stream: int, idx: int) -> int:
    """Pure-Python twin of :func:`mix64` for scalar draws (schedule, redraw counters)."""
    z = (seed * 0xD1342543DE82EF95 + stream * 0xA0761D6478BD642F + idx) & _MASK64
    z = (z + 0x9E3779B97F4A7C15) & _MASK64
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _MASK64
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _MASK64
    return z ^ (z >> 31)


def uniform01(seed: int, stream: int, idx: torch.Tensor, dtype=torch.float32) -> torch.Tensor:
    """u in (0, 1]: (top 24 bits + 1) / 2^24, exact in fp32 (G1)."""
    k = _lsr(mix64(seed, stream, idx), 40) + 1
    return k.to(dtype) * (1.0 / 16777216.0)


def randint(seed: int, stream: int, idx: torch.Tensor, lo: int, hi: int) -> torch.Tensor:
    """Integer in [lo, hi] (inclusive) from the top 32 bits (multiply-shift, no modulo bias to speak of)."""
    k = _lsr(mix64(seed, stream, idx), 32)
    return lo + ((k * (hi - lo + 1)) >> 32)


def normal(seed: int, stream: int, idx: torch.Tensor, dtype=torch.float32) -> torch.Tensor:
    """Box-Muller on two decorrelated counters (2*idx, 2*idx+1)."""
    u1 = uniform01(seed, stream, idx * 2, torch.float64)
    u2 = uniform01(seed, stream, idx * 2 + 1, torch.float64)
    z = torch.sqrt(-2.0 * torch.log(u1)) * torch.cos(2.0 * math.pi * u2)
    return z.to(dtype)


@dataclasses.dataclass(frozen=True)
class Config:
    """One workload of BASELINE.json:configs (notation: SURVEY §8)."""
    name: str
    N: int            # OD pairs
    L: int            # observed links
    T: int            # intervals per day (288 = 24 h of 5 min)
    H: int            # max lag
    C: int            # clusters (traffic patterns)
    D: int            # days
    b: int            # minibatch (days)
    K: int            # SPGD iterations
    kmin: int         # links per OD path (G2)
    kmax: int
    base_mu: float = 3.0
    base_sigma: float = 0.5
    modulated: bool = False   # weekly + seasonal day factors (G4, cfg 2 & 4)
    label_mode: str = "uniform"  # "zero" | "uniform" | "calendar" (G6)
    sparse: bool = False      # G7 windowed lags, CSR storage
    fig12: bool = False       # NEXT-2: the paper's efficiency experiment: random dense B, x >= 0, y = Bx
    seed: int = MASTER_SEED

    @property
    def nb(self) -> int:
        """Valid (s,h) blocks per cluster: s+h < T (PAPER.md:333 truncation)."""
        return self.T * (self.H + 1) - self.H * (self.H + 1) // 2

    def replace(self, **kw) -> "Config":
        return dataclasses.replace(self, **kw)


CONFIGS = {
    "tiny": Config("tiny", N=4, L=6, T=288, H=6, C=1, D=14, b=4, K=500, kmin=2, kmax=4,
                   label_mode="zero"),
    "tiny12": Config("tiny12", N=4, L=6, T=12, H=6, C=1, D=14, b=4, K=500, kmin=2, kmax=4,
                     label_mode="zero"),
    "corridor": Config("corridor", N=60, L=120, T=288, H=12, C=4, D=365, b=32, K=2000,
                       kmin=5, kmax=20),
    "multiyear": Config("multiyear", N=200, L=400, T=288, H=18, C=8, D=1096, b=64, K=5000,
                        kmin=5, kmax=20, modulated=True, label_mode="calendar"),
    "large_dense": Config("large_dense", N=1000, L=800, T=288, H=12, C=2, D=1096, b=8, K=1000,
                          kmin=5, kmax=20),
    "large_sparse": Config("large_sparse", N=20000, L=5000, T=288, H=24, C=4, D=1096, b=128,
                           K=1000, kmin=10, kmax=40, base_mu=1.0, base_sigma=1.2,
                           modulated=True, sparse=True),
}
# NEXT-2: "random generate a matrix B in R^{n x n}, x in (R+)^n, compute y = Bx and solve NNLS(B, y)",
# n from 100 to 6000.  Here: T = 1, H = 0, L = N = n, one cluster, D right-hand sides solved together (b = D).
CONFIGS["fig12"] = Config("fig12", N=6000, L=6000, T=1, H=0, C=1, D=64, b=64, K=200, kmin=1, kmax=1,
                          label_mode="zero", fig12=True)
CONFIG_ORDER = ["tiny", "corridor", "multiyear", "large_dense", "large_sparse"]


# --------------------------------------------------------------------------
# G2: path/link incidence (PAPER.md:107 delta^{ka}_{rs}; a corridor path is a
# contiguous run of links)
# --------------------------------------------------------------------------
TINY_REDRAW = 34  # N=4/L=6 instances: smallest redraw whose T=12 Gram matrix has cond < 1e4 (PD; tests check it) so P1/P4 converge


def incidence(cfg: Config, device="cpu", redraw: Optional[int] = None) -> Tuple[torch.Tensor, torch.Tensor]:
    """Returns (start[N], k[N]) int64: OD n covers links start..start+k-1."""
    if redraw is None:
        redraw = TINY_REDRAW if cfg.N == 4 and cfg.L == 6 else 0
    n = torch.arange(cfg.N, dtype=torch.int64, device=device) + redraw * cfg.N
    k = randint(cfg.seed, S_INC_K, n, cfg.kmin, min(cfg.kmax, cfg.L))
    u = _lsr(mix64(cfg.seed, S_INC_START, n), 32)
    start = (u * (cfg.L - k + 1)) >> 32
    return start, k


def incidence_mask(cfg: Config, device="cpu", redraw: Optional[int] = None) -> torch.Tensor:
    """Boolean [L][N]: True where OD n's path passes link l."""
    start, k = incidence(cfg, device, redraw)
    l = torch.arange(cfg.L, dtype=torch.int64, device=device)[:, None]
    return (l >= start[None, :]) & (l < (start + k)[None, :])


# --------------------------------------------------------------------------
# G3: dense DAR blocks R[c][s][h][l][n] (Eq. 17-18: for one
# (path, link, departure interval) the lag fractions sum to 1)
# --------------------------------------------------------------------------
def dar_dense(cfg: Config, device="cpu", s_chunk: int = 16, redraw: Optional[int] = None,
              out: Optional[torch.Tensor] = None) -> torch.Tensor:
    """fp32 [C][T][H+1][L][N]; flat Dirichlet over h on covered (l, n), 0 elsewhere.
    Blocks with s+h >= T are generated too (they are simply unused, A13)."""
    C, T, H1, L, N = cfg.C, cfg.T, cfg.H + 1, cfg.L, cfg.N
    if out is None:
        out = torch.empty((C, T, H1, L, N), dtype=torch.float32, device=device)
    if cfg.fig12:                                  # a random dense matrix, entries U[0,1)
        flat = out.view(-1)
        step = 1 << 24
        for i0 in range(0, flat.numel(), step):
            idx = torch.arange(i0, min(flat.numel(), i0 + step), dtype=torch.int64, device=device)
            flat[i0:i0 + idx.numel()] = uniform01(cfg.seed, S_DAR, idx)
        return out
    mask = incidence_mask(cfg, device, redraw)
    blk = H1 * L * N
    for c in range(C):
        for s0 in range(0, T, s_chunk):
            s1 = min(T, s0 + s_chunk)
            base = (c * T + s0) * blk
            idx = torch.arange(base, base + (s1 - s0) * blk, dtype=torch.int64, device=device)
            e = -torch.log(uniform01(cfg.seed, S_DAR, idx)).view(s1 - s0, H1, L, N)
            e = e * mask
            tot = e.sum(dim=1, keepdim=True)
            out[c, s0:s1] = e / torch.where(tot > 0, tot, torch.ones_like(tot))
    return out


# --------------------------------------------------------------------------
# G9 (NEXT-4): network and speeds for the DAR construction (stand-in for the NPMRDS 5-minute probe speeds of 43 TMCs,
# PAPER.md:484-486).  Paths are the G2 link runs in travel order; link lengths U[0.5, 3] km; speed = free-flow
# U[24, 31] m/s reduced in the two weekday peaks (the G4 profile) by a per-link, per-pattern congestion factor
# U[0, 0.7], times (1 + 2 % noise).
# --------------------------------------------------------------------------
def network(cfg: Config, device="cpu"):
    """(path_ptr int32 [N+1], path_links int32, link_len fp32 [L]) for dode_dar_build / the oracle's O7."""
    start, k = incidence(cfg, device)
    ptr = torch.zeros(cfg.N + 1, dtype=torch.int64, device=device)
    ptr[1:] = torch.cumsum(k, 0)
    j = torch.arange(int(ptr[-1]), dtype=torch.int64, device=device)
    owner = torch.searchsorted(ptr[1:].contiguous(), j, right=True)
    links = start[owner] + (j - ptr[owner])
    l = torch.arange(cfg.L, dtype=torch.int64, device=device)
    length = 500.0 + 2500.0 * uniform01(cfg.seed, S_LEN, l)
    return ptr.to(torch.int32), links.to(torch.int32), length.to(torch.float32)


def network_multipath(cfg: Config, kpaths: int = 3, device="cpu"):
    """(od_ptr int32 [N+1], path_ptr int32 [P+1], path_links int32, link_len fp32 [L]): OD n has 1..kpaths paths; path 0
    is its G2 link run, the others are link runs drawn independently with the same rule (a stand-in for the path set
    that "needs to be generated prior to the estimation framework")."""
    n = torch.arange(cfg.N, dtype=torch.int64, device=device)
    cnt = randint(cfg.seed, S_NPATH, n, 1, kpaths)
    od_ptr = torch.zeros(cfg.N + 1, dtype=torch.int64, device=device)
    od_ptr[1:] = torch.cumsum(cnt, 0)
    P = int(od_ptr[-1])
    pid = torch.arange(P, dtype=torch.int64, device=device)
    owner = torch.searchsorted(od_ptr[1:].contiguous(), pid, right=True)
    alt = pid - od_ptr[owner]                                   # 0 = the OD's G2 path
    key = owner + alt * cfg.N                                   # distinct draw per (OD, alternative); alt 0 == G2's index
    k = randint(cfg.seed, S_INC_K, key, cfg.kmin, min(cfg.kmax, cfg.L))
    u = _lsr(mix64(cfg.seed, S_INC_START, key), 32)
    start = (u * (cfg.L - k + 1)) >> 32
    path_ptr = torch.zeros(P + 1, dtype=torch.int64, device=device)
    path_ptr[1:] = torch.cumsum(k, 0)
    j = torch.arange(int(path_ptr[-1]), dtype=torch.int64, device=device)
    po = torch.searchsorted(path_ptr[1:].contiguous(), j, right=True)
    links = start[po] + (j - path_ptr[po])
    l = torch.arange(cfg.L, dtype=torch.int64, device=device)
    length = 500.0 + 2500.0 * uniform01(cfg.seed, S_LEN, l)
    return od_ptr.to(torch.int32), path_ptr.to(torch.int32), links.to(torch.int32), length.to(torch.float32)


def speeds(cfg: Config, c: int = 0, device="cpu") -> torch.Tensor:
    """fp32 [T][L] link speeds (m/s) of traffic pattern c."""
    l = torch.arange(cfg.L, dtype=torch.int64, device=device)
    vfree = 24.0 + 7.0 * uniform01(cfg.seed, S_VFREE, l, torch.float64)
    cong = 0.7 * uniform01(cfg.seed, S_CONG, l + c * cfg.L, torch.float64)
    peak = (profile(cfg.T, device) - 0.1).clamp(0.0, 1.0)
    idx = torch.arange(cfg.T * cfg.L, dtype=torch.int64, device=device) + c * cfg.T * cfg.L
    noise = 1.0 + 0.02 * normal(cfg.seed, S_VNOISE, idx, torch.float64).view(cfg.T, cfg.L)
    v = vfree[None, :] * (1.0 - cong[None, :] * peak[:, None]) * noise
    return v.clamp(min=1.0).to(torch.float32)


# --------------------------------------------------------------------------
# G4: planted demand q_true[d][s][n]  (two weekday peaks PAPER.md:587, lower
# Dec/Jan demand PAPER.md:601)
# --------------------------------------------------------------------------
def profile(T: int, device="cpu") -> torch.Tensor:
    s = torch.arange(T, dtype=torch.float64, device=device) * (288.0 / T)
    return 0.1 + torch.exp(-(s - 93.0) ** 2 / (2 * 15.0 ** 2)) + 0.9 * torch.exp(-(s - 207.0) ** 2 / (2 * 18.0 ** 2))


def day_factor(cfg: Config, device="cpu") -> torch.Tensor:
    d = torch.arange(cfg.D, dtype=torch.int64, device=device)
    f = 0.8 + 0.4 * uniform01(cfg.seed, S_DAYF, d, torch.float64)
    if cfg.modulated:
        weekday = (d + 2) % 7                      # day 0 = Wednesday, Monday = 0
        f = f * torch.where(weekday >= 5, 0.75, 1.0)
        doy = torch.remainder(d.to(torch.float64), 365.25)
        f = f * (1.0 + 0.08 * torch.cos(2 * math.pi * (doy - 200.0) / 365.25))
    return f


def q_true(cfg: Config, device="cpu", dtype=torch.float32) -> torch.Tensor:
    """[D][T][N] = base_n * profile(s) * dayfactor_d."""
    if cfg.fig12:                                  # x in (R+)^n, one vector per right-hand side
        idx = torch.arange(cfg.D * cfg.T * cfg.N, dtype=torch.int64, device=device)
        return uniform01(cfg.seed, S_BASE, idx, torch.float64).view(cfg.D, cfg.T, cfg.N).to(dtype)
    n = torch.arange(cfg.N, dtype=torch.int64, device=device)
    base = torch.exp(cfg.base_mu + cfg.base_sigma * normal(cfg.seed, S_BASE, n, torch.float64))
    q = day_factor(cfg, device)[:, None, None] * profile(cfg.T, device)[None, :, None] * base[None, None, :]
    return q.to(dtype)


# --------------------------------------------------------------------------
# G6: cluster labels (stand-in for t-SNE + k-means)
# --------------------------------------------------------------------------
def labels(cfg: Config) -> torch.Tensor:
    """int32 [D] on the CPU (labels are host data at the boundary)."""
    d = torch.arange(cfg.D, dtype=torch.int64)
    if cfg.label_mode == "zero" or cfg.C == 1:
        lab = torch.zeros(cfg.D, dtype=torch.int64)
    elif cfg.label_mode == "uniform":
        lab = randint(cfg.seed, S_LABEL, d, 0, cfg.C - 1)
    elif cfg.label_mode == "calendar":
        assert cfg.C == 8
        weekend = ((d + 2) % 7 >= 5).to(torch.int64)
        doy = torch.remainder(d.to(torch.float64), 365.25)
        quarter = torch.clamp((doy / 91.3125).floor().to(torch.int64), 0, 3)
        lab = 4 * weekend + quarter
        re = uniform01(cfg.seed, S_RELABEL, d, torch.float64) <= 0.10
        lab = torch.where(re, randint(cfg.seed, S_LABEL, d, 0, cfg.C - 1), lab)
    else:
        raise ValueError(cfg.label_mode)
    return lab.to(torch.int32)


# --------------------------------------------------------------------------
# G5: observed counts x[d][t][l] (data synthesis, not the solver: a batched
# library matmul per lag, independent of both the oracle and the CUDA path)
# --------------------------------------------------------------------------
def counts(cfg: Config, R: torch.Tensor, qt: torch.Tensor, lab: torch.Tensor, noise: bool = True,
           acc_dtype=None) -> torch.Tensor:
    """x_d = rho_{c(d)} q_true,d (+ N(0,(0.05 x)^2), clipped at 0) -> fp32 [D][T][L]."""
    dev = R.device
    if acc_dtype is None:
        acc_dtype = torch.float64 if dev.type == "cpu" else torch.float32
    T, H = cfg.T, cfg.H
    x = torch.zeros((cfg.D, T, cfg.L), dtype=acc_dtype, device=dev)
    lab_d = lab.to(dev)
    for c in range(cfg.C):
        days = torch.nonzero(lab_d == c).flatten()
        if days.numel() == 0:
            continue
        qc = qt[days].to(acc_dtype).transpose(0, 1)                 # [T][Dc][N]
        xc = torch.zeros((T, days.numel(), cfg.L), dtype=acc_dtype, device=dev)
        for h in range(min(H, T - 1) + 1):
            blk = R[c, :T - h, h].to(acc_dtype).transpose(1, 2)     # [T-h][N][L]
            xc[h:] += torch.bmm(qc[:T - h], blk)
        x[days] = xc.transpose(0, 1)
    if noise:
        idx = torch.arange(x.numel(), dtype=torch.int64, device=dev).view(x.shape)
        x = x + 0.05 * x * normal(cfg.seed, S_NOISE, idx, acc_dtype)
        x = torch.clamp(x, min=0.0)
    return x.to(torch.float32)


# --------------------------------------------------------------------------
# A8: minibatch schedule (permute, chunk, all chunks each
# epoch) re-scoped to days of one cluster.  Integer-only.
# --------------------------------------------------------------------------
class _Counter:
    def __init__(self, seed: int, stream: int):
        self.seed, self.stream, self.i = seed, stream, 0

    def below(self, n: int) -> int:
        v = mix64_int(self.seed, self.stream, self.i)
        self.i += 1
        return ((v >> 32) * n) >> 32


def epoch_chunks(lab: np.ndarray, b: int, rng: _Counter, full_only: bool = False) -> List[Tuple[int, np.ndarray]]:
    D = len(lab)
    perm = list(range(D))
    for i in range(D - 1, 0, -1):                    # Fisher-Yates
        j = rng.below(i + 1)
        perm[i], perm[j] = perm[j], perm[i]
    chunks: List[Tuple[int, np.ndarray]] = []
    for c in sorted(set(int(v) for v in lab)):
        days = [d for d in perm if lab[d] == c]      # stable split by cluster
        for i in range(0, len(days), b):
            ch = days[i:i + b]
            if full_only and len(ch) < b:
                continue
            chunks.append((c, np.asarray(ch, dtype=np.int32)))
    for i in range(len(chunks) - 1, 0, -1):          # shuffle the chunk list
        j = rng.below(i + 1)
        chunks[i], chunks[j] = chunks[j], chunks[i]
    return chunks


def schedule(cfg: Config, lab, K: Optional[int] = None, b: Optional[int] = None,
             full_only: bool = False) -> List[Tuple[int, np.ndarray]]:
    """Exactly K iterations, each (cluster, int32 day list of <= b distinct same-cluster days)."""
    K = cfg.K if K is None else K
    b = cfg.b if b is None else b
    lab = np.asarray(lab, dtype=np.int64)
    rng = _Counter(cfg.seed, S_SCHED)
    out: List[Tuple[int, np.ndarray]] = []
    while len(out) < K:
        ch = epoch_chunks(lab, b, rng, full_only)
        if not ch:
            raise ValueError("no chunk of the requested size exists")
        out.extend(ch)
    return out[:K]


def one_epoch(cfg: Config, lab, b: Optional[int] = None) -> List[Tuple[int, np.ndarray]]:
    """One epoch: every day receives exactly one step (sum_c ceil(D_c / b) iterations)."""
    b = cfg.b if b is None else b
    return epoch_chunks(np.asarray(lab, dtype=np.int64), b, _Counter(cfg.seed, S_SCHED))


# --------------------------------------------------------------------------
# CSR view of the DAR blocks (boundary format for storage = CSR; a format
# conversion of generated input, no solver arithmetic)
# --------------------------------------------------------------------------
@dataclasses.dataclass
class CsrDar:
    """Per (c,s,h) block CSR (rows = links, cols = OD pairs), blocks concatenated in [c][s][h] order.
    blk_off int64 [C*T*(H+1)+1]: first nnz of each block; row_ptr int32 [C*T*(H+1)][L+1] relative to
    the block start; col_idx int32 [nnz]; val fp32 [nnz]."""
    blk_off: torch.Tensor
    row_ptr: torch.Tensor
    col_idx: torch.Tensor
    val: torch.Tensor

    @property
    def nnz(self) -> int:
        return int(self.val.numel())

    def to(self, device) -> "CsrDar":
        return CsrDar(self.blk_off.to(device), self.row_ptr.to(device), self.col_idx.to(device), self.val.to(device))


def dense_to_csr(R: torch.Tensor) -> CsrDar:
    """[C][T][H+1][L][N] dense -> CsrDar keeping exactly the non-zero entries."""
    Cn, T, H1, L, N = R.shape
    nzmask = R != 0
    per_row = nzmask.sum(dim=-1).to(torch.int64)                      # [C][T][H1][L]
    per_blk = per_row.sum(dim=-1).flatten()
    blk_off = torch.zeros(per_blk.numel() + 1, dtype=torch.int64, device=R.device)
    blk_off[1:] = torch.cumsum(per_blk, 0)
    row_ptr = torch.zeros((Cn * T * H1, L + 1), dtype=torch.int64, device=R.device)
    row_ptr[:, 1:] = torch.cumsum(per_row.view(-1, L), 1)
    idx = torch.nonzero(nzmask.view(-1, N))                           # row-major => CSR order
    return CsrDar(blk_off, row_ptr.to(torch.int32).contiguous(), idx[:, 1].to(torch.int32).contiguous(),
                  R[nzmask].contiguous())


# --------------------------------------------------------------------------
# G7: sparse DAR for large networks (cfg 4), generated directly in the boundary CSR format.
# Example 3: departures of one interval reach a link spread over a few ADJACENT
# arrival intervals, later the further downstream the link is.  Link at position j of OD n's path gets
# lag offset h0 = min(floor(j*tau), H-w+1) (tau ~ U(0.3,0.9) intervals per link, per cluster and OD) and a
# window of w ~ U{2,3,4} lags with flat-Dirichlet fractions (redrawn per departure interval s).
# --------------------------------------------------------------------------
def sparse_pattern(cfg: Config, c: int, device="cpu"):
    """Sorted (h, l, n) pattern of cluster c (identical for every s) plus the (n,j) group id of each entry."""
    start, k = incidence(cfg, device)
    n_all = torch.arange(cfg.N, dtype=torch.int64, device=device)
    tau = 0.3 + 0.6 * uniform01(cfg.seed, S_TAU, c * cfg.N + n_all, torch.float64)
    kmax = int(k.max())
    j = torch.arange(kmax, dtype=torch.int64, device=device)[None, :].expand(cfg.N, kmax)
    valid = j < k[:, None]
    nn = n_all[:, None].expand(cfg.N, kmax)[valid]
    jj = j[valid]
    gid = torch.arange(nn.numel(), dtype=torch.int64, device=device)          # one group per (n, j)
    w = randint(cfg.seed, S_WIN, (c * cfg.N + nn) * 64 + jj, 2, 4).clamp(max=cfg.H + 1)
    h0 = torch.minimum((jj.to(torch.float64) * tau[nn]).floor().to(torch.int64), cfg.H - w + 1)
    ll = start[nn] + jj
    wmax = int(w.max())
    i = torch.arange(wmax, dtype=torch.int64, device=device)[None, :].expand(nn.numel(), wmax)
    vi = i < w[:, None]
    eh = (h0[:, None] + i)[vi]
    el = ll[:, None].expand(-1, wmax)[vi]
    en = nn[:, None].expand(-1, wmax)[vi]
    eg = gid[:, None].expand(-1, wmax)[vi]
    ei = i[vi]
    order = torch.argsort((eh * cfg.L + el) * cfg.N + en)
    return eh[order], el[order], en[order], eg[order], ei[order], int(gid.numel())


def dar_sparse(cfg: Config, device="cpu", s_chunk: int = 8) -> CsrDar:
    """CsrDar in [c][s][h] block order; same sparsity pattern for every s of a cluster, values per s."""
    T, H1, L = cfg.T, cfg.H + 1, cfg.L
    cols, vals, rps, blk_counts = [], [], [], []
    for c in range(cfg.C):
        eh, el, en, eg, ei, G = sparse_pattern(cfg, c, device)
        P = eh.numel()
        per_row = torch.zeros(H1 * L, dtype=torch.int64, device=device)
        per_row.index_add_(0, eh * L + el, torch.ones(P, dtype=torch.int64, device=device))
        rp = torch.zeros((H1, L + 1), dtype=torch.int64, device=device)
        rp[:, 1:] = torch.cumsum(per_row.view(H1, L), 1)
        per_blk = rp[:, -1]
        col32 = en.to(torch.int32)
        rps.append(rp.to(torch.int32).repeat(T, 1, 1))                          # [T][H1][L+1]
        blk_counts.append(per_blk.repeat(T))
        for s0 in range(0, T, s_chunk):
            s1 = min(T, s0 + s_chunk)
            S = s1 - s0
            sidx = torch.arange(s0, s1, dtype=torch.int64, device=device)[:, None]
            hidx = ((c * T + sidx) * G + eg[None, :]) * 4 + ei[None, :]
            e = -torch.log(uniform01(cfg.seed, S_SPFRAC, hidx))                 # [S][P]
            tot = torch.zeros((S, G), dtype=torch.float32, device=device)
            tot.index_add_(1, eg, e)
            vals.append((e / tot[:, eg]).reshape(-1))
            cols.append(col32.repeat(S))
    per_blk_all = torch.cat(blk_counts)
    blk_off = torch.zeros(per_blk_all.numel() + 1, dtype=torch.int64, device=device)
    blk_off[1:] = torch.cumsum(per_blk_all, 0)
    return CsrDar(blk_off, torch.cat(rps).view(-1, L + 1).contiguous(), torch.cat(cols), torch.cat(vals))


def counts_sparse(cfg: Config, csr: CsrDar, qt: torch.Tensor, lab: torch.Tensor, noise: bool = True) -> torch.Tensor:
    """x_d = rho_{c(d)} q_true,d (+ noise) with library sparse matmuls per (cluster, s) — data synthesis only."""
    dev = csr.val.device
    T, H1, L, N = cfg.T, cfg.H + 1, cfg.L, cfg.N
    acc_dtype = torch.float64 if dev.type == "cpu" else torch.float32
    x = torch.zeros((cfg.D, T + cfg.H, L), dtype=acc_dtype, device=dev)
    lab_d = lab.to(dev)
    for c in range(cfg.C):
        days = torch.nonzero(lab_d == c).flatten()
        if days.numel() == 0:
            continue
        xc = torch.zeros((T + cfg.H, L, days.numel()), dtype=acc_dtype, device=dev)
        for s in range(T):
            b0 = (c * T + s) * H1
            k0, k1 = int(csr.blk_off[b0]), int(csr.blk_off[b0 + H1])
            # rows of the stacked [(H+1)*L] x N matrix of departure interval s
            rp = csr.row_ptr[b0:b0 + H1].to(torch.int64)
            base = (csr.blk_off[b0:b0 + H1] - k0)[:, None]
            crow = torch.cat([(rp[:, :-1] + base).reshape(-1), torch.tensor([k1 - k0], device=dev)])
            with warnings.catch_warnings():
                warnings.simplefilter("ignore")
                A = torch.sparse_csr_tensor(crow, csr.col_idx[k0:k1].to(torch.int64), csr.val[k0:k1].to(acc_dtype),
                                            size=(H1 * L, N))
            xc[s:s + H1] += (A @ qt[days, s].to(acc_dtype).T).view(H1, L, -1)
        x[days] = xc.permute(2, 0, 1)
    x = x[:, :T].contiguous()                       # arrivals after the day are dropped
    if noise:
        idx = torch.arange(x.numel(), dtype=torch.int64, device=dev).view(x.shape)
        x = torch.clamp(x + 0.05 * x * normal(cfg.seed, S_NOISE, idx, acc_dtype), min=0.0)
    return x.to(torch.float32)


def sparse_problem(cfg: Config, device="cpu"):
    """(CsrDar, x) for a sparse config, both on ``device``."""
    csr = dar_sparse(cfg, device)
    x = counts_sparse(cfg, csr, q_true(cfg, device), labels(cfg))
    return csr, x


def csr_to_dense(cfg: Config, csr: CsrDar) -> torch.Tensor:
    """[C][T][H+1][L][N] dense copy of a CsrDar (small test instances only)."""
    R = torch.zeros((cfg.C * cfg.T * (cfg.H + 1), cfg.L, cfg.N), dtype=torch.float32)
    bo, rp, ci, va = csr.blk_off.cpu(), csr.row_ptr.cpu().to(torch.int64), csr.col_idx.cpu().to(torch.int64), csr.val.cpu()
    for b in range(R.shape[0]):
        k0 = int(bo[b])
        cnt = rp[b, 1:] - rp[b, :-1]
        rows = torch.repeat_interleave(torch.arange(cfg.L), cnt)
        k1 = k0 + int(rp[b, -1])
        R[b, rows, ci[k0:k1]] = va[k0:k1]
    return R.view(cfg.C, cfg.T, cfg.H + 1, cfg.L, cfg.N)
