"""N > 1 logic of bench.py on CPU (world size 2, gloo): replicas only, no data-path collective.

The dedispersion path does not shard: every rank processes its own beam, the only
communication is the barrier and the MAX over ranks of the device time.  These tests run that host
logic with the `gloo` backend; the kernels themselves are covered by the `-m gpu` tests.
"""
import os
import socket
import subprocess
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank),
                      WORLD_SIZE=str(world), LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    import workloads

    # the timing rule: every rank reports the MAX over ranks
    local_ms = 10.0 + 5.0 * rank
    got = bench.reduce_max(local_ms, dist, "cpu")
    assert got == 10.0 + 5.0 * (world - 1)

    # replicas: same geometry, different seeded beam per rank
    cfg = workloads.get_config("tiny")
    x = workloads.make_filterbank(cfg, seed=bench.replica_seed(cfg, rank), nsamp=2048)
    assert x.shape == (2048, cfg["nchan"])
    digest = torch.tensor([float(x.to(torch.float64).sum())], dtype=torch.float64)
    gathered = [torch.zeros_like(digest) for _ in range(world)]
    dist.all_gather(gathered, digest)
    sums = [float(g.item()) for g in gathered]
    assert len(set(sums)) == world, "every rank must dedisperse its own beam"

    # whole-job value = units of all ranks / max-over-ranks time
    units = 1000.0
    value = world * units / (got * 1e-3)
    np.save(os.path.join(out_dir, f"value_{rank}.npy"), np.array([value]))
    dist.barrier()
    dist.destroy_process_group()


def test_world_size_2_gloo_replica_logic(tmp_path):
    world = 2
    port = _free_port()
    mp.spawn(_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    vals = [float(np.load(tmp_path / f"value_{r}.npy")[0]) for r in range(world)]
    assert vals[0] == vals[1] == world * 1000.0 / 15e-3


def _shard_worker(rank, world, port, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank),
                      WORLD_SIZE=str(world), LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    import workloads

    # DM-sharded run (bench.py --shard dm): ONE beam, generated on rank 0 and broadcast; disjoint DM slices
    cfg = workloads.get_config("tiny")
    x = (workloads.make_filterbank(cfg, nsamp=1024) if rank == 0
         else torch.zeros((1024, cfg["nchan"]), dtype=torch.uint8))
    dist.broadcast(x, src=0)
    ref = workloads.make_filterbank(cfg, nsamp=1024)
    assert torch.equal(x, ref), "every rank dedisperses the same beam"
    dms = workloads.plan_args(cfg)["dm_list"]
    mine, off = bench.dm_shard(dms, rank, world)
    np.save(os.path.join(out_dir, f"dms_{rank}.npy"), np.concatenate([[off], mine]))
    dist.barrier()
    dist.destroy_process_group()


def test_world_size_2_gloo_dm_sharding(tmp_path):
    world = 2
    mp.spawn(_shard_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    import workloads
    dms = workloads.plan_args(workloads.get_config("tiny"))["dm_list"]
    parts = [np.load(tmp_path / f"dms_{r}.npy") for r in range(world)]
    assert [int(p[0]) for p in parts] == [0, len(dms) // 2]
    np.testing.assert_array_equal(np.concatenate([p[1:] for p in parts]), dms)     # disjoint, complete, in order


def test_dm_shard_covers_the_list_for_any_world_size():
    import bench
    dms = np.arange(0.0, 1024.0)
    for world in (1, 2, 3, 4, 8):
        got = [bench.dm_shard(dms, r, world) for r in range(world)]
        np.testing.assert_array_equal(np.concatenate([g[0] for g in got]), dms)
        assert [g[1] for g in got] == [(1024 * r) // world for r in range(world)]
        assert max(len(g[0]) for g in got) - min(len(g[0]) for g in got) <= 1


def test_reduce_max_single_process_is_identity():
    import bench
    assert bench.reduce_max(3.25) == 3.25


def test_reference_arm_prints_only_on_rank_zero():
    """bench.py --impl reference under torchrun: ranks != 0 exit 0 without work or output."""
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1", MASTER_ADDR="127.0.0.1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""
