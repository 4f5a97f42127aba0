"""N>1 path of bench.py on CPU: two gloo ranks (world_size 2).  The SPGD path shards by days with no data-path
collective; what is multi-rank is the sharding rule, the max-over-ranks timing and the
whole-job aggregate — covered here without a GPU."""
import os
import socket
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out_dir: str):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    from paper_1901_09266_b200 import synth
    cfg = bench.rank_config(synth.CONFIGS["tiny12"], rank, world)
    lab = synth.labels(cfg).numpy()
    qt = synth.q_true(cfg).numpy()
    epochs = bench.make_epochs(cfg, lab, cfg.b, 2)
    # every rank steps each of ITS days exactly once per epoch
    for ep in epochs:
        seen = np.sort(np.concatenate([d for _, d in ep]))
        assert np.array_equal(seen, np.arange(cfg.D))
    # shards are different data (seed + rank), same shape
    gathered = [torch.zeros(qt.shape, dtype=torch.float32) for _ in range(world)]
    dist.all_gather(gathered, torch.from_numpy(qt))
    assert gathered[0].shape == gathered[1].shape
    assert not torch.equal(gathered[0], gathered[1])
    # timing: max over ranks; throughput: whole job
    my_ms = 1.0 + rank          # rank 1 is the slow one
    job_ms = bench.max_over_ranks(my_ms)
    assert job_ms == float(world)
    thr = bench.job_day_steps_per_s(cfg.D, world, job_ms)
    assert abs(thr - cfg.D * world / (world * 1e-3)) < 1e-6
    dist.barrier()
    with open(os.path.join(out_dir, f"ok{rank}"), "w") as f:
        f.write("ok")
    dist.destroy_process_group()


def test_two_gloo_ranks_shard_days_and_reduce_timing(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    assert all((tmp_path / f"ok{r}").exists() for r in range(world))


def test_single_rank_helpers_are_identity():
    import bench
    from paper_1901_09266_b200 import synth
    cfg = synth.CONFIGS["tiny"]
    assert bench.rank_config(cfg, 0, 1) is cfg
    assert bench.max_over_ranks(3.5) == 3.5
