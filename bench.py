#!/usr/bin/env python
"""bench.py — SPGD epoch time over all days on one B200 (BASELINE.json metric), with the roofline of the
dominant kernel and the CPU oracle timed beside it.

A *step* is one SPGD epoch of the workload: every day receives exactly one projected-gradient step, i.e.
sum_c ceil(D_c / b) calls of dode_spgd_step (a1-a4 of SURVEY.md §8(a)) in the seeded A8 schedule order.
Default workload: BASELINE.json configs[3] ("large_dense": N=1000 L=800 T=288 H=12 C=2 D=1096), the largest dense
single-GPU workload and the one north_star's roofline targets are defined on: the G8 minibatch sweep b in {1, 8, 64, 256},
each width from a fresh q0; the line's `value`, `roofline`, `e2e` are those of b = 256 and `sweep` carries all four.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload NAME] [--b B] [--impl reference]

Prints ONE JSON line (rank 0).  See DESIGN.md "Measurement" for the byte/flop accounting.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np
import torch

from paper_1901_09266_b200 import synth

METRIC = "spgd_epoch_time_over_all_days"
UNIT = "ms/epoch"
FP32_PEAK_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12   # NOMINAL: SMs x FP32 lanes x 2 flop x clocks.max.sm; the rooflines
                                                    # divide by the MEASURED rate (dode_probe_fp32_peak), both are printed


DEFAULT_WORKLOAD = "large_dense"          # BASELINE.json configs[3]: the largest dense single-GPU workload, where
LARGE_DENSE_SWEEP = (1, 8, 64, 256)       # north_star defines its >= 0.70 HBM / >= 0.50 FP32 targets (G8 sweep)
TC_TF32_EQUIV_PER_PRODUCT = 2.0  # tensor work of the 3xTF32 kernel per fp32 product, in TF32 MMA units (see roofline_of)
TF32_OVER_BF16 = 1.1 / 2.25      # nominal dense tensor ratio (B200_PROFILING.md): tf32 1.1 PF vs bf16 2.25 PF


def measured_peaks():
    """(HBM GB/s, bf16 TFLOP/s burst, source) from the driver-written MEASURED_PEAKS.json, else the guide's fallback."""
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), float(d["bf16_tflops"]), "measured"
    return 6650.0, 1590.0, "fallback"


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons with NVML while the timed region runs."""

    REASONS = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
               0x80: "hw_power_brake_slowdown"}

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.stop_flag, self.sm, self.reasons, self.max_mhz, self.ok = index, False, [], set(), None, False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            uuid = torch.cuda.get_device_properties(index).uuid
            try:
                self.h = pynvml.nvmlDeviceGetHandleByUUID(("GPU-" + str(uuid)).encode())
            except Exception:
                self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception:
            self.ok = False

    def run(self):
        if not self.ok:
            return
        while not self.stop_flag:
            try:
                self.sm.append(self.nv.nvmlDeviceGetClockInfo(self.h, self.nv.NVML_CLOCK_SM))
                r = self.nv.nvmlDeviceGetCurrentClocksEventReasons(self.h) if hasattr(
                    self.nv, "nvmlDeviceGetCurrentClocksEventReasons") else self.nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in self.REASONS.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(0.002)

    def summary(self):
        if not self.ok or not self.sm:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["nvml_unavailable"]}
        return {"sm_mhz": float(np.median(self.sm)), "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.sm)}


def rank_config(cfg, rank: int, world: int):
    """Weak scaling over days (days are independent units): every rank owns its own D days and its
    own copy of the cluster operators, generated from seed + rank; no collective sits on the step path."""
    return cfg if world <= 1 else cfg.replace(seed=cfg.seed + rank)


def max_over_ranks(value: float, device="cpu") -> float:
    """MAX over ranks of a per-rank device time (the job finishes with its slowest rank)."""
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([value], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_day_steps_per_s(D: int, world: int, epoch_ms: float) -> float:
    """Whole-job throughput: every rank steps its D days once per epoch."""
    return D * world / (epoch_ms * 1e-3)


def cpu_model() -> str:
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def make_epochs(cfg, lab, b, count):
    rng = synth._Counter(cfg.seed, synth.S_SCHED)
    return [synth.epoch_chunks(np.asarray(lab, np.int64), b, rng) for _ in range(count)]


def algorithmic(cfg, n_days):
    """Algorithmic bytes / flops of one launch on n_days days: R once per pass + the state."""
    Rb = 4.0 * cfg.nb * cfg.L * cfg.N
    fwd_b = Rb + 4.0 * n_days * cfg.T * (cfg.N + cfg.L)        # read q, read x   (r stays on chip in principle)
    grad_b = Rb + 4.0 * n_days * cfg.T * cfg.N                 # write q
    fl = 2.0 * cfg.nb * cfg.L * cfg.N * n_days
    return fwd_b, grad_b, fl


def cpu_oracle_sample(cfg, Rc, c0, lab, x, eta, visits):
    """Times the oracle as it stands on `visits` day-visits of cluster c0's days (single thread); returns ms per visit
    and the number of visits timed."""
    from oracle import oracle
    own = [d for d in range(cfg.D) if int(lab[d]) == c0]
    days = [own[i % len(own)] for i in range(max(1, visits))]
    q = np.ones((cfg.T, cfg.N), np.float32)
    Rn = Rc.numpy()
    if cfg.nb * cfg.L * cfg.N < 2e8:
        oracle.visit(Rn, q, x[days[0]].numpy(), float(eta))       # page in
    t0 = time.perf_counter()
    for d in days:
        oracle.visit(Rn, q, x[d].numpy(), float(eta))
    return (time.perf_counter() - t0) * 1e3 / len(days), len(days)


def run_reference(args, cfg, b, rank, world):
    """--impl reference: the CPU oracle (oracle/), as it stands, on this host's cores.  One step = a bounded sample of an
    epoch — args.ref_visits day-visits of one cluster's days through oracle.replay_day (the loops of oracle_visit with
    the output rows over all host threads; pin P18) — and `value` extrapolates it to the epoch (x D / visits).
    `ms_per_step` is the measured time of a step's sample.  The operator of ONE cluster and the counts of a few of its
    days are generated here (on the GPU if one is visible — input synthesis only — else on the host)."""
    if rank != 0:
        return
    from oracle import oracle
    oracle.build_oracle()
    threads = os.cpu_count() or 1
    gen_dev = "cuda" if torch.cuda.is_available() else "cpu"
    cfg1 = cfg.replace(C=1, D=min(cfg.D, 8), label_mode="zero")
    lab1 = synth.labels(cfg1)
    if cfg.sparse:
        csr, x = synth.sparse_problem(cfg1, gen_dev)
        arrs = (cfg.N, cfg.L, cfg.T, cfg.H, csr.blk_off.cpu().numpy(), csr.row_ptr.cpu().numpy(),
                csr.col_idx.cpu().numpy(), csr.val.cpu().numpy())
        Rn = None
        x = x.cpu().numpy()
        del csr
        eta = np.float32(1e-3)                       # any step: one visit costs the same
    else:
        R = synth.dar_dense(cfg1, device=gen_dev)
        x = synth.counts(cfg1, R, synth.q_true(cfg1, gen_dev), lab1, noise=not cfg.fig12).cpu().numpy()
        Rn = R[0].cpu().numpy()
        del R
        arrs = None
        eta = np.float32(1e-3)
    if gen_dev == "cuda":
        torch.cuda.empty_cache()
    v = args.ref_visits
    if v is None:                                    # about 1-10 s per step
        work = (cfg.nb * cfg.L * cfg.N if not cfg.sparse else 4.3e8) * 4 / 3e9 / max(1, threads // 2)
        v = int(max(1, min(cfg.D, 2.0 / max(work, 1e-4))))
    q = [np.ones((cfg.T, cfg.N), np.float32) for _ in range(cfg1.D)]
    times, day = [], 0
    for it in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        for _ in range(v):
            got, _ = oracle.replay_day(Rn, q[day], x[day], float(eta), 1, [1], threads=threads, csr=arrs)
            q[day] = got[1]
            day = (day + 1) % cfg1.D
        if it >= args.warmup:
            times.append((time.perf_counter() - t0) * 1e3)
    step_ms = float(np.mean(times))
    epoch_ms = step_ms * cfg.D / v
    out = {"impl": "reference", "metric": METRIC, "value": epoch_ms, "unit": UNIT, "n_gpus": args.gpus,
           "steps": args.steps, "warmup": args.warmup, "ms_per_step": step_ms, "higher_is_better": False,
           "scaling": "weak", "vs_baseline": None, "dtype": "f64 accumulate / f32 storage", "data": "synthetic",
           "config": workload_config(cfg, b),
           "cpu_baseline": {"value": epoch_ms, "unit": UNIT, "cores": threads, "kind": "oracle",
                            "sample": f"{v} day-visit(s) per step (ms_per_step is that sample's time) of the {cfg.D}-visit epoch, "
                                      f"oracle_replay_day on {threads} threads, extrapolated x{cfg.D / v:.1f}; inputs generated on {gen_dev}",
                            "cpu_model": cpu_model()},
           "e2e": {"value": epoch_ms, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(out))


def workload_config(cfg, b):
    return {"workload": f"{cfg.name}: N={cfg.N} L={cfg.L} T={cfg.T} H={cfg.H} C={cfg.C} D={cfg.D} minibatch={b} "
                        f"({'CSR' if cfg.sparse else 'dense'} fp32 DAR blocks)",
            "step": "one SPGD epoch = sum_c ceil(D_c/b) dode_spgd_step calls, every day stepped once",
            "l2": "L2 flushed (256 MiB write) before every timed epoch; R of all clusters also exceeds L2 "
                  "except on the tiny workload"}


def traffic_from_profiles(workload, b, kernel_kind):
    """dram bytes per launch of the dominant kernel from the committed `ncu --set full` summaries (profiles/traffic.json,
    keyed "<workload>_b<minibatch>", else "<workload>"), or None."""
    p = os.path.join(ROOT, "profiles", "traffic.json")
    if not os.path.exists(p):
        return None
    try:
        t = json.load(open(p))
        return (t.get(f"{workload}_b{b}") or t.get(workload) or {}).get(kernel_kind)
    except Exception:
        return None


def reset_state(P, h, cfg, ones_dev):
    """q <- q0 = 1 on every day (G8: every minibatch width of the sweep starts from a fresh q0)."""
    for d in range(cfg.D):
        P.dode_set_q(h, d, ones_dev)


def measure_b(P, h, cfg, lab, etas, b, steps, warmup, timing_epochs, flush, world, dev, nnz_c=None):
    """Times `steps` SPGD epochs at minibatch b (after `warmup` untimed ones) with CUDA events, L2 flushed before every
    epoch, then `timing_epochs` more with an event pair around every launch for the roofline of the dominant kernel."""
    import torch.distributed as dist
    epochs = make_epochs(cfg, lab, b, warmup + steps)
    P.dode_reserve(h, min(b, 256))

    def run_epoch(ep):
        for c, days in ep:
            P.dode_spgd_step(h, days, float(etas[c]))

    for ep in epochs[:warmup]:
        run_epoch(ep)
    P.dode_sync(h)
    launches0 = P.dode_launch_count(h)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    ev = []
    wall0 = time.perf_counter()
    for ep in epochs[warmup:]:
        flush.zero_()                                    # L2 flush, outside the event pair
        a, z = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        run_epoch(ep)
        P.dode_join(h)                                   # the end event must follow the steps on the library's lanes
        z.record()
        ev.append((a, z))
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    wall = time.perf_counter() - wall0
    total_ms = max_over_ranks(sum(a.elapsed_time(z) for a, z in ev), dev)
    epoch_ms = total_ms / steps
    launches = P.dode_launch_count(h) - launches0
    # per-kernel durations for the roofline: epochs again with a CUDA-event pair around every launch on the library's
    # stream (dode_timing_*).  Event records between launches serialise them, so this pass is kept out of the region
    # `value` is measured on (where consecutive kernels overlap by programmatic dependent launch).
    P.dode_timing_enable(h, True)
    P.dode_timing_read(h, 0, True); P.dode_timing_read(h, 1, True)
    widest, path = 0, P.dode_last_path(h)
    t_epochs = epochs[warmup:][:timing_epochs]
    for ep in t_epochs:
        flush.zero_()
        for c, days in ep:
            P.dode_spgd_step(h, days, float(etas[c]))
            if len(days) > widest:                       # name the kernels of a full-width minibatch, not of a
                widest, path = len(days), P.dode_last_path(h)   # cluster's ragged tail (host-side string, no sync)
    fwd_ms, fwd_n = P.dode_timing_read(h, 0)
    grad_ms, grad_n = P.dode_timing_read(h, 1)
    P.dode_timing_enable(h, False)
    fb = gb = fl = 0.0                                   # algorithmic work summed over the event-timed launches
    for ep in t_epochs:
        for c, days in ep:
            if cfg.sparse:
                f_b = 8.0 * nnz_c + 4.0 * len(days) * cfg.T * (cfg.N + cfg.L)
                g_b = 8.0 * nnz_c + 4.0 * len(days) * cfg.T * cfg.N
                f_l = 2.0 * nnz_c * len(days)
            else:
                f_b, g_b, f_l = algorithmic(cfg, len(days))
            fb += f_b; gb += g_b; fl += f_l
    step_b = step_f = 0.0                                # and over the epochs `value` was timed on
    for ep in epochs[warmup:]:
        for c, days in ep:
            if cfg.sparse:
                step_b += 16.0 * nnz_c + 4.0 * len(days) * cfg.T * (2 * cfg.N + cfg.L)
                step_f += 4.0 * nnz_c * len(days)
            else:
                f_b, g_b, f_l = algorithmic(cfg, len(days))
                step_b += f_b + g_b; step_f += 2 * f_l
    return {"b": b, "epoch_ms": epoch_ms, "total_ms": total_ms, "wall_s": wall, "launches": int(launches), "path": path,
            "iters_per_epoch": len(epochs[0]), "steps": steps, "warmup": warmup,
            "fwd_ms": fwd_ms, "fwd_n": fwd_n, "grad_ms": grad_ms, "grad_n": grad_n, "fb": fb, "gb": gb, "fl": fl,
            "step_GBps": step_b / (total_ms * 1e-3) / 1e9, "step_TFLOPs": step_f / (total_ms * 1e-3) / 1e12}


def roofline_of(cfg, m, peaks):
    """The `roofline` object of one measurement (DESIGN.md §7/§11): the dominant kernel's algorithmic bytes or flops per
    launch / its average event-timed launch duration, against the measured peak of the unit that bounds it."""
    hbm_peak, bf16_peak, peak_src, fp32_peak, fp32_src = peaks
    tensor_path = m["path"].startswith("tcgen05")
    # 3xTF32 with bf16 corrections: per fp32 product one TF32 MMA (a*b, both truncated to TF32) and two bf16 MMAs
    # (a_lo*b, a*b_lo) at half the TF32 cost each = 2 TF32 MMA-equivalents, so fp32-equivalent peak = tf32 peak / 2
    tc_peak = bf16_peak * TF32_OVER_BF16 / TC_TF32_EQUIV_PER_PRODUCT
    dom = "forward" if m["fwd_ms"] >= m["grad_ms"] else "gradient_update"
    d_ms, d_n, d_bytes = (m["fwd_ms"], m["fwd_n"], m["fb"]) if dom == "forward" else (m["grad_ms"], m["grad_n"], m["gb"])
    gbs = d_bytes / (d_ms * 1e-3) / 1e9 if d_ms > 0 else 0.0
    tfl = m["fl"] / (d_ms * 1e-3) / 1e12 if d_ms > 0 else 0.0
    t_hbm = d_bytes / (hbm_peak * 1e9)
    t_alu = m["fl"] / ((tc_peak if tensor_path else fp32_peak) * 1e12)
    path = m["path"]
    kname = path.split("+")[0 if dom == "forward" else 1] if "+" in path else path
    if t_hbm >= t_alu:
        roof = {"bound": "hbm", "achieved": gbs, "peak": hbm_peak, "unit": "GB/s", "frac": gbs / hbm_peak,
                "peak_source": f"MEASURED_PEAKS.json hbm_gbs ({peak_src})"}
    elif tensor_path:
        roof = {"bound": "tensor", "achieved": tfl, "peak": tc_peak, "unit": "TFLOP/s", "frac": tfl / tc_peak,
                "peak_source": f"MEASURED_PEAKS.json bf16_tflops ({peak_src}) x 1.1/2.25 (nominal tf32:bf16) / 2 (one TF32 MMA + two "
                               "bf16 MMAs at half its cost per fp32 product)"}
    else:
        roof = {"bound": "alu", "achieved": tfl, "peak": fp32_peak, "unit": "TFLOP/s", "frac": tfl / fp32_peak,
                "peak_source": fp32_src}
    roof.update({"kernel": kname, "launches": int(d_n), "avg_launch_ms": d_ms / max(1, d_n),
                 "traffic": traffic_from_profiles(cfg.name, m["b"], dom),
                 "other": {"hbm_GBps": gbs, "hbm_frac": gbs / hbm_peak, "hbm_frac_of_nominal_8TBps": gbs / 8000.0,
                           "fp32_TFLOPs": tfl, "fp32_frac_of_measured_ffma_peak": tfl / fp32_peak,
                           "fp32_frac_of_nominal_ffma_peak": tfl / FP32_PEAK_TFLOPS, "ffma_peak_measured_TFLOPs": fp32_peak,
                           "ffma_peak_nominal_TFLOPs": FP32_PEAK_TFLOPS,
                           "forward_ms_total": m["fwd_ms"], "gradient_update_ms_total": m["grad_ms"],
                           "step_GBps_algorithmic": m["step_GBps"], "step_TFLOPs_algorithmic": m["step_TFLOPs"]}})
    return roof


def measure_e2e(P, h, cfg, lab, etas, b, x_cpu, e2e_steps, world, dev):
    """The same epochs through dode_spgd_step_host (H2D of the minibatch counts, D2H of its q), wall clock including the
    final dode_sync; then the same pinned buffers copied back to back with no kernels at all = the PCIe floor."""
    import torch.distributed as dist
    # pinned host copies of the minibatches' counts and result buffers: distinct schedules for as many epochs as fit
    # in 8 GB of pinned memory (at least one), cycled over the timed epochs; x of a day is the same in every epoch
    per_epoch = cfg.D * cfg.T * (cfg.L + cfg.N) * 4
    n_stage = int(max(1, min(e2e_steps, (8 << 30) // per_epoch)))
    e_epochs = make_epochs(cfg, lab, b, n_stage)
    stage = [[(c, days, x_cpu[torch.from_numpy(days.astype(np.int64))].contiguous().pin_memory(),
               torch.empty((len(days), cfg.T, cfg.N), dtype=torch.float32).pin_memory()) for c, days in ep]
             for ep in e_epochs]
    for c, days, xh, qh in stage[-1]:                # untimed warm-up epoch (staging buffers, copy streams)
        P.dode_spgd_step_host(h, days, float(etas[c]), xh, qh)
    P.dode_sync(h)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    t0 = time.perf_counter()
    for k in range(e2e_steps):
        for c, days, xh, qh in stage[k % n_stage]:
            P.dode_spgd_step_host(h, days, float(etas[c]), xh, qh)
    P.dode_sync(h)                               # every upload, step and download of the timed epochs has finished
    torch.cuda.synchronize()
    e_ms = max_over_ranks((time.perf_counter() - t0) * 1e3 / e2e_steps, dev)
    # PCIe floor: the same uploads and downloads on two streams, no kernels
    s_up, s_dn = torch.cuda.Stream(), torch.cuda.Stream()
    xd = torch.empty((min(b, cfg.D), cfg.T, cfg.L), device=dev)
    qd = torch.empty((min(b, cfg.D), cfg.T, cfg.N), device=dev)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for c, days, xh, qh in stage[0]:
        with torch.cuda.stream(s_up):
            xd[:len(days)].copy_(xh, non_blocking=True)
        with torch.cuda.stream(s_dn):
            qh.copy_(qd[:len(days)], non_blocking=True)
    torch.cuda.synchronize()
    floor_ms = (time.perf_counter() - t0) * 1e3
    return e_ms, floor_ms


def run_ours(args, cfg, sweep, rank, world, local_rank):
    import paper_1901_09266_b200 as P
    P.lib()                                   # fail loudly if the CUDA library is missing
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: there is no CPU fallback")
    dev = torch.device("cuda", local_rank)
    torch.cuda.set_device(dev)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    try:
        _run_ours(P, args, cfg, sweep, rank, world, local_rank, dev)
    finally:
        if world > 1:
            import torch.distributed as dist
            dist.destroy_process_group()


def _run_ours(P, args, cfg, sweep, rank, world, local_rank, dev):
    cfg = rank_config(cfg, rank, world)
    b_head = sweep[-1]                        # the line's `value` is the last (widest) minibatch of the sweep

    # ---- inputs, generated once on the device (synth: no solver arithmetic) ----
    lab = synth.labels(cfg).numpy()
    nnz_c = None
    csr_host = None
    if cfg.sparse:
        csr, x = synth.sparse_problem(cfg, dev)
        torch.cuda.empty_cache()              # the library allocates with cudaMalloc: give torch's cached blocks back first
        h = P.dode_create(cfg.N, cfg.L, cfg.T, cfg.H, cfg.C, cfg.D, lab, x, 1.0, csr=csr)
        nnz_c = csr.nnz / cfg.C
        if rank == 0 and not args.no_cpu_baseline:          # one cluster's CSR blocks for the oracle's timing leg
            c0, nbk = int(lab[0]), cfg.T * (cfg.H + 1)
            bo = csr.blk_off[c0 * nbk:(c0 + 1) * nbk + 1].cpu().numpy()
            k0, k1 = int(bo[0]), int(bo[-1])
            csr_host = (c0, bo - k0, csr.row_ptr[c0 * nbk:(c0 + 1) * nbk].cpu().numpy(),
                        csr.col_idx[k0:k1].cpu().numpy(), csr.val[k0:k1].cpu().numpy())
        del csr
    else:
        R = synth.dar_dense(cfg, device=dev)
        x = synth.counts(cfg, R, synth.q_true(cfg, dev), torch.from_numpy(lab), noise=not cfg.fig12)   # Fig. 12: y = Bx exactly
        torch.cuda.empty_cache()
        h = P.dode_create(cfg.N, cfg.L, cfg.T, cfg.H, cfg.C, cfg.D, lab, x, 1.0, dense=R)
    if args.tc_bstages:
        P.dode_set_option(h, P.DODE_OPT_TC_BSTAGES, args.tc_bstages)
    if args.tc_pair is not None:
        P.dode_set_option(h, P.DODE_OPT_TC_PAIR, args.tc_pair)
    x_cpu = x.cpu()
    R_cpu = None
    if rank == 0 and not args.no_cpu_baseline and not cfg.sparse:
        R_cpu = R[int(lab[0])].cpu()                  # one cluster's operator for the oracle's timing leg
    if not cfg.sparse:
        del R
    del x
    torch.cuda.empty_cache()

    etas = np.array([np.float32(1.0 / P.dode_lipschitz(h, c, 30)) for c in range(cfg.C)], np.float32)   # a7
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=dev)
    ones_dev = torch.ones((cfg.T, cfg.N), dtype=torch.float32, device=dev)
    hbm_peak, bf16_peak, peak_src = measured_peaks()
    fp32_peak = P.dode_probe_fp32_peak(5)             # hand-written FFMA loop, measured on this GPU now
    peaks = (hbm_peak, bf16_peak, peak_src, fp32_peak,
             f"dode_probe_fp32_peak on this GPU ({fp32_peak:.1f} TFLOP/s; nominal 148 SMs x 128 lanes x 2 x 1.965 GHz = {FP32_PEAK_TFLOPS:.2f})")

    sampler = ClockSampler(local_rank)
    sampler.start()
    results = {}
    for b in sweep:
        head = b == b_head
        if len(sweep) > 1:
            reset_state(P, h, cfg, ones_dev)
        steps = args.steps if head else max(1, min(args.steps, args.sweep_steps))
        warm = args.warmup if head else min(args.warmup, 3)
        results[b] = measure_b(P, h, cfg, lab, etas, b, steps, warm, steps if head else min(steps, 2), flush, world, dev, nnz_c)
    sampler.stop_flag = True
    sampler.join()
    m = results[b_head]
    epoch_ms = m["epoch_ms"]
    roof = roofline_of(cfg, m, peaks)

    # ---- e2e at the headline minibatch ----
    e2e = None
    if args.e2e_steps is None:                 # enough epochs for ~2 s of streaming, so that pipeline fill and the final
        args.e2e_steps = int(min(20, max(3, 2000.0 / max(epoch_ms, 1e-3))))     # sync are amortised (3..20 epochs)
    if args.e2e_steps > 0:
        e_ms, floor_ms = measure_e2e(P, h, cfg, lab, etas, b_head, x_cpu, args.e2e_steps, world, dev)
        e2e = {"value": e_ms, "unit": UNIT, "h2d_bytes_per_step": int(cfg.D * cfg.T * cfg.L * 4),
               "d2h_bytes_per_step": int(cfg.D * cfg.T * cfg.N * 4), "epochs": args.e2e_steps,
               "pcie_floor_ms_per_epoch": floor_ms, "device_ms_per_epoch": epoch_ms,
               "bound": "pcie" if floor_ms > epoch_ms else "device",
               "api": "dode_spgd_step_host (pinned host buffers; uploads/downloads pipelined against the kernels on copy "
                      "streams, dode_sync inside the timed region); pcie_floor = the same buffers copied with no kernels"}

    if rank != 0:
        P.dode_destroy(h)
        return
    # Step 6 quality check on the state the run ends with — a sanity figure, outside every timed region
    _, r2_mean = P.dode_r2(h, list(range(cfg.D)))
    # ---- CPU oracle beside it (bounded sample, rank 0 only, single thread) ----
    cpu = None
    if cfg.sparse and csr_host is not None:
        from oracle import oracle
        c0, bo, rp, ci, va = csr_host
        days_c0 = [d for d in range(cfg.D) if int(lab[d]) == c0][:3]
        q1 = np.ones((cfg.T, cfg.N), np.float32)
        t0 = time.perf_counter()
        for d in days_c0:
            oracle.visit_csr(cfg.N, cfg.L, cfg.T, cfg.H, bo, rp, ci, va, q1, x_cpu[d].numpy(), float(etas[c0]))
        ms_visit = (time.perf_counter() - t0) * 1e3 / len(days_c0)
        cpu = {"value": ms_visit * cfg.D, "unit": UNIT, "cores": 1, "kind": "oracle",
               "sample": f"{len(days_c0)} day-visits (CSR oracle loop) of the {cfg.D}-visit epoch timed single-threaded on this host "
                         f"({os.cpu_count()} cores visible), extrapolated x{cfg.D / len(days_c0):.1f}",
               "ms_per_day_visit": ms_visit}
    if R_cpu is not None:
        per_visit = cfg.nb * cfg.L * cfg.N * 4 / 3e9            # rough s per visit at ~3 GFLOP/s scalar double
        visits = int(max(1 if per_visit > 5 else 3, min(2 * cfg.D, 15.0 / max(per_visit, 1e-4))))
        c0 = int(lab[0])
        ms_visit, visits = cpu_oracle_sample(cfg, R_cpu, c0, lab, x_cpu, etas[c0], visits)
        cpu = {"value": ms_visit * cfg.D, "unit": UNIT, "cores": 1, "kind": "oracle",
               "sample": f"{visits} day-visits of the {cfg.D}-visit epoch timed single-threaded on this host "
                         f"({os.cpu_count()} cores visible), extrapolated x{cfg.D / visits:.1f}",
               "ms_per_day_visit": ms_visit}
    if cpu is not None:
        cpu["cpu_model"] = cpu_model()
        cpu["nproc"] = os.cpu_count()
    out = {"metric": METRIC, "value": epoch_ms, "unit": UNIT, "n_gpus": world, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": epoch_ms, "higher_is_better": False, "scaling": "weak",
           "vs_baseline": None, "dtype": "f32", "data": "synthetic", "config": workload_config(cfg, b_head),
           "day_steps_per_s": job_day_steps_per_s(cfg.D, world, epoch_ms), "spgd_iterations_per_epoch": m["iters_per_epoch"],
           "ms_per_spgd_iteration": epoch_ms / m["iters_per_epoch"], "kernel_path": m["path"],
           "gpu_launches": m["launches"], "wall_s_timed_region": m["wall_s"], "clocks": sampler.summary(),
           "roofline": roof, "e2e": e2e, "cpu_baseline": cpu,
           "fit": {"r2_mean_over_days": r2_mean,
                   "note": "Step 6 quality check of the state the run ends with (paper reports 0.87 on its real data, PAPER.md:553)"}}
    if len(sweep) > 1:
        # G8 (BASELINE.json configs[3]): the memory-bound to compute-bound crossover, every width from a fresh q0.
        # north_star's targets: >= 0.70 of HBM at small minibatch, >= 0.50 of FP32 peak at large minibatch.
        out["sweep"] = {str(b): {"ms_per_epoch": r["epoch_ms"], "ms_per_spgd_iteration": r["epoch_ms"] / r["iters_per_epoch"],
                                 "steps": r["steps"], "warmup": r["warmup"], "kernel_path": r["path"],
                                 "gpu_launches": r["launches"], "roofline": roofline_of(cfg, r, peaks)}
                        for b, r in results.items()}
    print(json.dumps(out))
    P.dode_destroy(h)


def run_fig12_sweep(args, local_rank):
    """--workload fig12 --sweep (NEXT-2): the paper's efficiency experiment (Fig. 12) as ONE line:
    random dense B (n x n), x >= 0, y = Bx, n = 100 ... 6000, solved for 64 right-hand sides at once (T = 1, H = 0, b = 64).
    Per n: GPU time of one SPGD iteration (CUDA events, L2 flushed between iterations), the oracle's time for the same
    iteration (timed on a bounded number of right-hand sides, extrapolated to the 64), and the forward kernel's
    fraction of the HBM roofline.  The paper's third arm (active-set NNLS) is a comparison system and is not timed."""
    import paper_1901_09266_b200 as P
    from oracle import oracle
    P.lib()
    dev = torch.device("cuda", local_rank)
    torch.cuda.set_device(dev)
    hbm_peak, _, peak_src = measured_peaks()
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=dev)
    sampler = ClockSampler(local_rank)
    sampler.start()
    curve = []
    base = synth.CONFIGS["fig12"]
    for n in (100, 300, 1000, 3000, 6000):
        cfg = base.replace(N=n, L=n)
        lab = synth.labels(cfg).numpy()
        R = synth.dar_dense(cfg, device=dev)
        x = synth.counts(cfg, R, synth.q_true(cfg, dev), torch.from_numpy(lab), noise=False)
        h = P.dode_create(cfg.N, cfg.L, cfg.T, cfg.H, cfg.C, cfg.D, lab, x, 1.0, dense=R)
        eta = float(np.float32(1.0 / P.dode_lipschitz(h, 0, 30)))
        days = np.arange(cfg.D, dtype=np.int32)
        P.dode_reserve(h, cfg.D)
        for _ in range(max(3, args.warmup)):
            P.dode_spgd_step(h, days, eta)
        P.dode_sync(h)
        ev = []
        for _ in range(args.steps):
            flush.zero_()
            a, z = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            P.dode_spgd_step(h, days, eta)
            P.dode_join(h)
            z.record()
            ev.append((a, z))
        torch.cuda.synchronize()
        gpu_ms = sum(a.elapsed_time(z) for a, z in ev) / args.steps
        path = P.dode_last_path(h)
        P.dode_destroy(h)
        alg_bytes = 2 * 4.0 * n * n + 4.0 * cfg.D * (3 * n)            # B once per pass + q read/write + y read
        Rn, xn = R[0].cpu().numpy(), x.cpu().numpy()
        rhs = int(max(1, min(cfg.D, 4e8 / (4.0 * n * n))))              # bounded sample: ~0.2-2 s of oracle work
        q = np.ones((cfg.T, cfg.N), np.float32)
        t0 = time.perf_counter()
        for d in range(rhs):
            oracle.visit(Rn, q, xn[d], eta)
        cpu_ms = (time.perf_counter() - t0) * 1e3 * cfg.D / rhs
        curve.append({"n": n, "gpu_ms": gpu_ms, "oracle_ms": cpu_ms, "oracle_rhs_timed": rhs,
                      "frac": alg_bytes / (gpu_ms * 1e-3) / 1e9 / hbm_peak, "kernel_path": path})
        del R, x
        torch.cuda.empty_cache()
    sampler.stop_flag = True
    sampler.join()
    last = curve[-1]
    out = {"metric": "fig12_spgd_iteration_time", "value": last["gpu_ms"], "unit": "ms/iteration", "n_gpus": 1,
           "steps": args.steps, "warmup": max(3, args.warmup), "ms_per_step": last["gpu_ms"], "higher_is_better": False,
           "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
           "config": {"workload": "fig12 sweep (PAPER.md:569-583): random dense B n x n, x >= 0, y = Bx, 64 right-hand sides "
                                  "(T=1, H=0, b=64), n = 100, 300, 1000, 3000, 6000; value = n 6000",
                      "l2": "L2 flushed (256 MiB write) before every timed iteration"},
           "curve": curve, "clocks": sampler.summary(), "gpu_launches": None,
           "roofline": {"bound": "hbm", "achieved": last["frac"] * hbm_peak, "peak": hbm_peak, "unit": "GB/s",
                        "frac": last["frac"], "peak_source": f"MEASURED_PEAKS.json hbm_gbs ({peak_src})",
                        "kernel": last["kernel_path"], "traffic": None,
                        "note": "whole iteration (both passes) on algorithmic bytes 2*4n^2 + state, n = 6000"},
           "cpu_baseline": {"value": last["oracle_ms"], "unit": "ms/iteration", "cores": 1, "kind": "oracle",
                            "sample": f"{last['oracle_rhs_timed']} of 64 right-hand sides timed, extrapolated"},
           "e2e": None}
    print(json.dumps(out))


def run_dar_build(args, cfg, local_rank):
    """--dar-build (NEXT-4): Step 1 of the framework, the DAR blocks of one traffic pattern from link speeds
    (dode_dar_build; Eq. 17-18).  One step = one pattern's operator [T][H+1][L][N] built from its
    [T][L] speeds.  The kernel's work is the output it must produce: algorithmic bytes = 4*T*(H+1)*L*N."""
    import paper_1901_09266_b200 as P
    P.lib()
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: there is no CPU fallback")
    dev = torch.device("cuda", local_rank)
    torch.cuda.set_device(dev)
    DT = 300.0
    multipath = args.paths > 1
    if multipath:       # several paths per OD, Logit route shares (Eq. 37, theta per second): dode_assignment_build
        od, ptr, links, length = synth.network_multipath(cfg, args.paths)
        od_d = od.to(dev)
    else:
        ptr, links, length = synth.network(cfg)
    ptr_d, links_d, len_d = ptr.to(dev), links.to(dev), length.to(dev)

    def build(v, out):
        if multipath:
            P.dode_assignment_build(cfg.N, cfg.L, cfg.T, cfg.H, od_d, ptr_d, links_d, len_d, v, DT, args.theta, out)
        else:
            P.dode_dar_build(cfg.N, cfg.L, cfg.T, cfg.H, ptr_d, links_d, len_d, v, DT, out)

    vs = [synth.speeds(cfg, c).pin_memory() for c in range(cfg.C)]
    vd = [v.to(dev) for v in vs]
    if cfg.sparse:
        # large networks: the operator goes straight into the boundary CSR format (dode_assignment_build_csr) — the dense
        # slab of this network would be T*(H+1)*L*N*4 bytes (terabytes for configs[4])
        def build_csr(v):
            return P.dode_assignment_build_csr(cfg.N, cfg.L, cfg.T, cfg.H, od_d if multipath else None, ptr_d, links_d, len_d,
                                               v, DT, args.theta if multipath else 0.0)
        sampler = ClockSampler(local_rank)
        for i in range(max(1, min(3, args.warmup))):
            out_csr = build_csr(vd[i % cfg.C])
        torch.cuda.synchronize()
        sampler.start()
        t0 = time.perf_counter()
        for i in range(args.steps):
            out_csr = build_csr(vd[i % cfg.C])           # synchronises (returns nnz)
        torch.cuda.synchronize()
        ms = (time.perf_counter() - t0) * 1e3 / args.steps
        sampler.stop_flag = True
        sampler.join()
        nnz = out_csr.nnz
        out_bytes = 8.0 * nnz + 4.0 * cfg.T * (cfg.H + 1) * (cfg.L + 1) + 8.0 * (cfg.T * (cfg.H + 1) + 1)
        hbm, _, peak_src = measured_peaks()
        ach = out_bytes / (ms * 1e-3) / 1e9
        print(json.dumps({
            "metric": "dar_build_time_per_pattern", "value": ms, "unit": "ms/pattern", "n_gpus": 1, "steps": args.steps,
            "warmup": max(1, min(3, args.warmup)), "ms_per_step": ms, "higher_is_better": False, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64 times / f32 shares", "data": "synthetic",
            "config": {"workload": f"dar_build (CSR output) on {cfg.name}: N={cfg.N} L={cfg.L} T={cfg.T} H={cfg.H}, "
                                   + (f"1-{args.paths} paths per OD, Logit theta={args.theta} " if multipath else "one path per OD ")
                                   + f"({int(ptr[-1])} path links), |H| = 300 s; dense slab would be "
                                   + f"{4.0 * cfg.T * (cfg.H + 1) * cfg.L * cfg.N / 1e12:.2f} TB",
                       "timing": "wall clock around dode_assignment_build_csr (sizing call + build; it synchronises)"},
            "nnz": nnz, "gpu_launches": None, "clocks": sampler.summary(),
            "roofline": {"bound": "hbm", "achieved": ach, "peak": hbm, "unit": "GB/s", "frac": ach / hbm,
                         "peak_source": f"MEASURED_PEAKS.json hbm_gbs ({peak_src})",
                         "kernel": "assignment_tuples x2 + cub radix sort + reduce-by-key + csr_bounds_from_keys",
                         "traffic": None,
                         "note": "algorithmic bytes = the CSR arrays it must produce (8 B per non-zero + pointers); the sort "
                                 "moves ~24 B per share several times, so the fraction is small by construction"},
            "e2e": None,
            "cpu_baseline": None,
            "cpu_baseline_note": "the oracle's O7/O8 write the dense [T][H+1][L][N] slab, which does not exist at this size; "
                                 "tests/test_gpu_dar_build.py checks the CSR builder against them on small networks"}))
        return
    nbytes = 4.0 * cfg.T * (cfg.H + 1) * cfg.L * cfg.N
    R = torch.empty((cfg.T, cfg.H + 1, cfg.L, cfg.N), device=dev)
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=dev)
    sampler = ClockSampler(local_rank)
    for i in range(max(3, args.warmup)):
        build(vd[i % cfg.C], R)
    torch.cuda.synchronize()
    sampler.start()
    ev = []
    for i in range(args.steps):
        flush.zero_()
        a, z = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        build(vd[i % cfg.C], R)
        z.record()
        ev.append((a, z))
    torch.cuda.synchronize()
    sampler.stop_flag = True
    sampler.join()
    ms = sum(a.elapsed_time(z) for a, z in ev) / args.steps
    nnz = int((R != 0).sum().item())
    # end to end: speeds from pinned host memory, the operator back to the host
    R_host = torch.empty(R.shape, dtype=torch.float32).pin_memory() if nbytes < 4e9 else None
    e2e = None
    if args.e2e_steps is None:
        args.e2e_steps = 3
    if R_host is not None and args.e2e_steps > 0:
        vtmp = torch.empty_like(vd[0])
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for i in range(args.e2e_steps):
            vtmp.copy_(vs[i % cfg.C], non_blocking=True)
            build(vtmp, R)
            R_host.copy_(R, non_blocking=True)
        torch.cuda.synchronize()
        e2e = {"value": (time.perf_counter() - t0) * 1e3 / args.e2e_steps, "unit": "ms/pattern",
               "h2d_bytes_per_step": int(vs[0].numel() * 4), "d2h_bytes_per_step": int(nbytes),
               "api": "dode_dar_build (speeds uploaded from pinned host memory, operator downloaded)"}
    hbm, _, peak_src = measured_peaks()
    ach = nbytes / (ms * 1e-3) / 1e9
    out = {"metric": "dar_build_time_per_pattern", "value": ms, "unit": "ms/pattern", "n_gpus": 1, "steps": args.steps,
           "warmup": max(3, args.warmup), "ms_per_step": ms, "higher_is_better": False, "scaling": "weak",
           "vs_baseline": None, "dtype": "f64 times / f32 shares", "data": "synthetic",
           "config": {"workload": f"dar_build on {cfg.name}: N={cfg.N} L={cfg.L} T={cfg.T} H={cfg.H}, "
                                  + (f"1-{args.paths} paths per OD, Logit theta={args.theta} " if multipath else "one path per OD ")
                                  + f"({int(ptr[-1])} path links), |H| = 300 s",
                      "l2": "L2 flushed (256 MiB write) before every timed build"},
           "nnz": nnz, "gpu_launches": args.steps * 2, "clocks": sampler.summary(),
           "roofline": {"bound": "hbm", "achieved": ach, "peak": hbm, "unit": "GB/s", "frac": ach / hbm,
                        "peak_source": f"MEASURED_PEAKS.json hbm_gbs ({peak_src})", "kernel": "cudaMemsetAsync + dar_build_dense",
                        "traffic": None},
           "e2e": e2e}
    if not args.no_cpu_baseline:
        from oracle import oracle
        Tc = cfg.T if nbytes < 1.5e9 else max(1, int(cfg.T * 1.5e9 / nbytes))      # bounded sample: the first Tc intervals
        v0 = vs[0][:Tc].numpy()
        t0 = time.perf_counter()
        if multipath:
            oracle.assignment_build(cfg.N, cfg.L, Tc, cfg.H, od.numpy(), ptr.numpy(), links.numpy(), length.numpy(), v0, DT, args.theta)
        else:
            oracle.dar_build(cfg.N, cfg.L, Tc, cfg.H, ptr.numpy(), links.numpy(), length.numpy(), v0, DT)
        cpu_ms = (time.perf_counter() - t0) * 1e3 * cfg.T / Tc
        out["cpu_baseline"] = {"value": cpu_ms, "unit": "ms/pattern", "cores": 1, "kind": "oracle",
                               "sample": f"O7 on the first {Tc} of {cfg.T} departure intervals, extrapolated x{cfg.T / Tc:.1f}"}
    print(json.dumps(out))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default=DEFAULT_WORKLOAD, choices=list(synth.CONFIGS))
    ap.add_argument("--b", type=int, default=None, help="minibatch days (default: the workload's; large_dense: the G8 sweep "
                                                        "1, 8, 64, 256 with the line's value at 256)")
    ap.add_argument("--sweep-steps", type=int, default=5, help="timed epochs of the sweep's non-headline widths (<= --steps)")
    ap.add_argument("--days", type=int, default=None, help="override D (bench smoke runs only)")
    ap.add_argument("--n", type=int, default=None, help="fig12 workload: matrix dimension n (L = N = n), 100..6000 in the paper")
    ap.add_argument("--sweep", action="store_true", help="fig12 workload: the whole Fig. 12 curve n = 100 ... 6000 in one JSON line")
    ap.add_argument("--e2e-steps", type=int, default=None, help="timed end-to-end epochs (default: 3..20, about 2 s of streaming)")
    ap.add_argument("--ref-visits", type=int, default=None, help="--impl reference: day-visits per step (default: about 1-10 s of work)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--tc-bstages", type=int, default=0, help="DODE_OPT_TC_BSTAGES: stages of the tcgen05 kernels' B ring (0 = automatic)")
    ap.add_argument("--tc-pair", type=int, default=None, help="DODE_OPT_TC_PAIR: 0 = single-CTA tcgen05 kernels only, 1 = CTA pairs (default), 2 = pairs only")
    ap.add_argument("--paths", type=int, default=1, help="--dar-build: up to this many paths per OD with Logit route shares (Eq. 37)")
    ap.add_argument("--theta", type=float, default=0.01, help="--dar-build --paths K: Logit dispersion factor per second (SURVEY NEXT-4)")
    ap.add_argument("--dar-build", action="store_true", help="NEXT-4: time dode_dar_build on the workload's network instead of SPGD")
    args = ap.parse_args()
    if args.impl == "ours":
        args.warmup = max(args.warmup, 3)              # timing rule: W >= 3
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    cfg = synth.CONFIGS[args.workload]
    if args.days:
        cfg = cfg.replace(D=args.days)
    if args.n:
        if not cfg.fig12:
            raise SystemExit("--n applies to --workload fig12 only")
        cfg = cfg.replace(N=args.n, L=args.n)
    # BASELINE.json configs[3] is a minibatch sweep (G8); north_star's two roofline targets are defined on it
    sweep = [args.b] if args.b else (list(LARGE_DENSE_SWEEP) if cfg.name == "large_dense" else [cfg.b])
    if args.dar_build:
        if rank == 0:
            run_dar_build(args, cfg, local_rank)
        return
    if args.sweep:
        if not cfg.fig12:
            raise SystemExit("--sweep applies to --workload fig12 only")
        if rank == 0:
            run_fig12_sweep(args, local_rank)
        return
    if args.impl == "reference":
        run_reference(args, cfg, sweep[-1], rank, world)
    else:
        run_ours(args, cfg, sweep, rank, world, local_rank)


if __name__ == "__main__":
    main()
