"""Multi-rank host logic of bench.py on CPU (gloo, world_size 2).  The hot path does not shard
(BASELINE.json north_star: one GPU, no sharding or collectives; replicas only), so the
only multi-rank logic is: barrier, MAX of the per-rank device time, whole-job value = all ranks' units /
slowest rank's time; `--impl reference` runs on rank 0 only."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms_local = 10.0 + 5.0 * rank                      # rank 1 is the slow replica
    dist.barrier()
    ms_max = bench.max_over_ranks(ms_local, dist, torch.device("cpu"))
    value = bench.whole_job_value(1000.0, 4, ms_max, dist.get_world_size())
    out[rank] = (ms_max, value)
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_and_whole_job_value_world2():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    with ctx.Manager() as m:
        out = m.dict()
        port = 29500 + os.getpid() % 1000
        procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
        for p in procs:
            p.start()
        for p in procs:
            p.join(120)
            assert p.exitcode == 0
        res = dict(out)
    # both ranks see the slowest replica's time; 2 replicas x 1000 units x 4 steps / 15 ms
    for r in (0, 1):
        assert res[r][0] == 15.0
        assert abs(res[r][1] - 2 * 1000.0 * 4 / 15e-3) < 1e-6


def test_single_rank_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.5, None, None) == 3.5
    assert bench.whole_job_value(10.0, 2, 4.0, 1) == 10.0 * 2 / 4e-3


def test_reference_arm_runs_on_rank0_only():
    """Under torchrun the oracle arm prints on rank 0; other ranks exit 0 without work or output."""
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], capture_output=True, text=True, env=env, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""


@pytest.mark.parametrize("workload", ["hmf_1e4"])
def test_reference_arm_line_rank0(workload):
    env = dict(os.environ, RANK="0", WORLD_SIZE="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", workload,
                        "--steps", "1", "--warmup", "0"], capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0, r.stderr
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["value"] > 0 and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["unit"] == "particle-steps/s"


# ---- sharding plumbing: bounds and the two collectives, gloo world 2 on CPU -------------

def test_shard_bounds_cover_every_particle_once():
    sys.path.insert(0, ROOT)
    from paper_1212_0262_b200.sharded import shard_bounds
    for n, w in ((10, 2), (10, 3), (7, 7), (1_048_576, 8), (50_000_000, 8), (5, 2)):
        b = shard_bounds(n, w)
        assert b[0][0] == 0 and sum(k for _, k in b) == n
        for (i0, k), (j0, _) in zip(b[:-1], b[1:]):
            assert i0 + k == j0
        assert max(k for _, k in b) - min(k for _, k in b) <= 1


def _coll_worker(rank, world, port, out):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    from paper_1212_0262_b200.sharded import TorchDistCollectives, shard_bounds
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    coll = TorchDistCollectives(dist, rank, world)
    # HMF exchange: each rank's (sum cos, sum sin), summed in place
    t = torch.tensor([1.0 + rank, 10.0 * (rank + 1)], dtype=torch.float64)
    coll.all_reduce_sum_(t)
    res = {"sum": t.tolist()}
    # pair-model exchange: packed 16-byte elements, equal shards (n = 6) and unequal shards (n = 7)
    for n in (6, 7):
        bounds = shard_bounds(n, world)
        whole = torch.zeros(n * 16, dtype=torch.uint8)
        i0, k = bounds[rank]
        whole[i0 * 16:(i0 + k) * 16] = rank + 1
        coll.all_gather_inplace_(whole, [(b * 16, (b + m) * 16) for b, m in bounds])
        res[f"gather{n}"] = whole.view(-1, 16)[:, 0].tolist()
    out[rank] = res
    dist.barrier()
    dist.destroy_process_group()


def test_sharding_collectives_gloo_world2():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    with ctx.Manager() as m:
        out = m.dict()
        port = 29500 + (os.getpid() + 7) % 1000
        procs = [ctx.Process(target=_coll_worker, args=(r, 2, port, out)) for r in range(2)]
        for p in procs:
            p.start()
        for p in procs:
            p.join(120)
            assert p.exitcode == 0
        res = dict(out)
    for r in (0, 1):
        assert res[r]["sum"] == [3.0, 30.0]
        assert res[r]["gather6"] == [1, 1, 1, 2, 2, 2]
        assert res[r]["gather7"] == [1, 1, 1, 2, 2, 2, 2]


# ---- bench.py --sharded: host logic (plan, strong-scaling value, max over ranks), gloo world 2 on CPU ----------------

def _sharded_bench_worker(rank, world, port, out):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    from paper_1212_0262_b200 import inputs
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    res = {}
    for key in ("grav2d_1m", "hmf_5e7"):
        w = inputs.WORKLOADS[key]
        plan = bench.sharded_plan(w, world, rank)
        ms_local = 100.0 + 50.0 * rank                       # rank 1 is the slow shard
        ms_max = bench.max_over_ranks(ms_local, dist, torch.device("cpu"))
        res[key] = (plan, ms_max, bench.strong_scaling_value(plan["units_per_step"], 5, ms_max))
    out[rank] = res
    dist.barrier()
    dist.destroy_process_group()


def test_sharded_bench_host_logic_gloo_world2():
    """Strong scaling: ONE problem split over the ranks; value = its units / the slowest rank's time (not summed over
    ranks, unlike the replicas line); the shards tile the particles; the exchange per substage is 16 N bytes
    (all-gather) or 16 bytes (all-reduce)."""
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    with ctx.Manager() as m:
        out = m.dict()
        port = 29500 + (os.getpid() + 13) % 1000
        procs = [ctx.Process(target=_sharded_bench_worker, args=(r, 2, port, out)) for r in range(2)]
        for p in procs:
            p.start()
        for p in procs:
            p.join(120)
            assert p.exitcode == 0
        res = dict(out)
    for key, N, units in (("grav2d_1m", 1_048_576, 3.0 * 1_048_576.0 ** 2), ("hmf_5e7", 50_000_000, 5e7)):
        p0, p1 = res[0][key][0], res[1][key][0]
        assert p0["i0"] == 0 and p0["i0"] + p0["n_local"] == p1["i0"] and p1["i0"] + p1["n_local"] == N
        assert p0["units_per_step"] == units == p1["units_per_step"]
        for r in (0, 1):
            assert res[r][key][1] == 150.0
            assert abs(res[r][key][2] - units * 5 / 0.150) <= 1e-6 * units
    assert res[0]["grav2d_1m"][0]["exchange"] == {"collective": "all_gather", "bytes_per_substage": 16 * 1_048_576}
    assert res[0]["hmf_5e7"][0]["exchange"] == {"collective": "all_reduce", "bytes_per_substage": 16}
    assert res[1]["grav2d_1m"][0]["rows_x_columns"] == [524_288, 1_048_576]
