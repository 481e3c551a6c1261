"""Host logic of the N > 1 path, run with world_size-2 gloo on CPU.

Ranks own contiguous ranges of the global event index, the only exchange is one
all_reduce(sum) of the three reduction outputs.  The per-rank arithmetic here is the oracle's
(this is a test; the product's kernels need a GPU): what is checked is that sharding by
`workloads.shard_range` + one all_reduce reproduces the single-process result, and that
bench.py's `--impl reference` arm prints on rank 0 only.
"""
import json
import os
import socket
import subprocess
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_0908_4403_b200 import workloads

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_shard_range_partitions_the_index_space():
    for n_events in (0, 1, 7, 64, 1000003):
        for world in (1, 2, 3, 8):
            nxt, total = 0, 0
            for r in range(world):
                first, count = workloads.shard_range(n_events, r, world)
                assert first == nxt and count >= 0
                nxt, total = first + count, total + count
            assert total == n_events
            counts = [workloads.shard_range(n_events, r, world)[1] for r in range(world)]
            assert max(counts) - min(counts) <= 1


def _worker(rank, world, port, n_events, out_path):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    os.environ["OMP_NUM_THREADS"] = "2"
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import oracle
    c = workloads.CONFIGS["4gamma"]
    first, count = workloads.shard_range(n_events, rank, world)
    mom, w = oracle.gen_events(c["seed"], c["n"], count, mode=c["mode"], a=c["a"], b=c["b"], y_max=c["y_max"],
                               apply_cuts=True, first_event=first)
    a2 = oracle.amp2(mom)
    out3 = torch.from_numpy(oracle.xsec_reduce(a2, w, c["n"]))
    dist.all_reduce(out3)                       # the path's one exchange step
    gathered = [None] * world
    dist.all_gather_object(gathered, (first, mom, w))
    if rank == 0:
        gathered.sort(key=lambda t: t[0])
        np.savez(out_path, out3=out3.numpy(), mom=np.concatenate([g[1] for g in gathered]),
                 w=np.concatenate([g[2] for g in gathered]))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_shards_and_allreduce_reproduce_the_single_process_result(tmp_path):
    import oracle
    n_events = 1001                             # odd: ragged shards (501 + 500)
    out_path = str(tmp_path / "w2.npz")
    mp.spawn(_worker, args=(2, _free_port(), n_events, out_path), nprocs=2, join=True)
    got = np.load(out_path)
    c = workloads.CONFIGS["4gamma"]
    mom, w = oracle.gen_events(c["seed"], c["n"], n_events, mode=c["mode"], a=c["a"], b=c["b"],
                               y_max=c["y_max"], apply_cuts=True)
    assert np.array_equal(got["mom"], mom) and np.array_equal(got["w"], w)     # global Philox counters
    ref3 = oracle.xsec_reduce(oracle.amp2(mom), w, c["n"])
    assert got["out3"][2] == ref3[2]
    np.testing.assert_allclose(got["out3"][:2], ref3[:2], rtol=1e-13)


def test_reference_arm_prints_on_rank_zero_only():
    env = dict(os.environ, OMP_NUM_THREADS="2")
    lines = {}
    for rank in (0, 1):
        env.update(RANK=str(rank), WORLD_SIZE="2", LOCAL_RANK=str(rank))
        res = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                              "--steps", "1", "--warmup", "0", "--config", "2gamma"], env=env, capture_output=True,
                             text=True, timeout=300)
        assert res.returncode == 0, res.stderr
        lines[rank] = res.stdout.strip()
    assert lines[1] == ""
    rec = json.loads(lines[0])
    assert rec["impl"] == "reference" and rec["unit"] == "events/s" and rec["value"] > 0
    assert rec["cpu_baseline"]["kind"] == "oracle" and rec["e2e"]["h2d_bytes_per_step"] == 0
