"""Host-side logic of bench.py on CPU: the replica sharding and the max/sum-over-ranks reductions run under
torch.distributed with the gloo backend, world_size 2 (the N>1 launch path of the bench without a GPU)."""
import os
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)
import bench  # noqa: E402


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        assert bench.dist_env() == (rank, rank, world)
        ids = bench.shard_queries(rank, world, 8)
        t = [10.0 + rank, 3.0 - rank]
        mx = bench.reduce_max(t)
        sm = bench.reduce_sum([float(len(ids))])
        q.put((rank, ids, mx, sm))
    finally:
        dist.destroy_process_group()


def test_replica_sharding_and_reductions_gloo_world2():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + (os.getpid() % 2000)
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, ids0, mx0, sm0), (r1, ids1, mx1, sm1) = res
    assert ids0 == list(range(0, 8)) and ids1 == list(range(8, 16))  # disjoint seeds, same count per replica
    assert mx0 == mx1 == [11.0, 3.0]
    assert sm0 == sm1 == [16.0]


def test_single_process_reductions_are_identity():
    assert bench.reduce_max([1.5, 2.5]) == [1.5, 2.5]
    assert bench.reduce_sum([4.0]) == [4.0]


def test_bytes_model():
    # Jacobi-CG (r = 0) and deflated: the default kernel adds one n x r pass (8 n r bytes), the literal
    # recurrence two (16 n r, the count of SURVEY.md 8(d))
    a = bench.algorithmic_bytes_per_iter(nnz=1000, N=200, n=150, r=0)
    b = bench.algorithmic_bytes_per_iter(nnz=1000, N=200, n=150, r=8)
    c = bench.algorithmic_bytes_per_iter(nnz=1000, N=200, n=150, r=8, tall_passes=2)
    assert a == (24 * 1000 + 17 * 200) * (150 / 200) + 112 * 150
    assert b - a == 8 * 150 * 8
    assert c - a == 16 * 150 * 8
    # at n = N the model is round 1's: both matrices once, t on all rows, the mask, 14 vector passes, one tall pass
    assert bench.algorithmic_bytes_per_iter(nnz=1000, N=200, n=200, r=8) == 24 * 1000 + 17 * 200 + 112 * 200 + 8 * 200 * 8


def test_reference_arm_runs_on_cpu(capsys):
    # the oracle arm on a tiny twin: prints one JSON line with impl = reference
    import json

    assert bench.main(["--impl", "reference", "--twin", "c2_48", "--steps", "1", "--warmup", "0", "--cpu-budget", "1"]) == 0
    line = capsys.readouterr().out.strip().splitlines()[-1]
    d = json.loads(line)
    assert d["impl"] == "reference" and d["unit"] == "s/query" and d["higher_is_better"] is False
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["cpu_baseline"]["kind"] == "oracle"
    assert d["cpu_baseline"]["cores"] >= 1 and "OpenMP threads" in d["cpu_baseline"]["sample"]


def test_default_workload_is_the_largest_config():
    # the driver runs plain `python bench.py --gpus 1 --steps K --warmup W`: that line must be on config 5
    import argparse

    ns = argparse.Namespace(pdas_cap=0, twin=None)
    assert bench.build_parser().parse_args([]).config == 5

    class W:  # noqa: N801 - stand-in with the two fields pdas_cap_for reads
        config, pdas_cap = 2, 100

    assert bench.pdas_cap_for(ns, W) == 400  # the paper's raised cap
    W.config = 5
    assert bench.pdas_cap_for(ns, W) == 100
    ns.pdas_cap = 37
    assert bench.pdas_cap_for(ns, W) == 37


def test_query_ok_needs_outer_inner_and_kkt():
    ok = dict(status=0, worst_inner_status=0, kkt=[1e-12] * 5)
    assert bench.query_ok(ok)
    assert not bench.query_ok(dict(ok, status=-7))
    assert not bench.query_ok(dict(ok, worst_inner_status=-6))
    assert not bench.query_ok(dict(ok, kkt=[0, 0, 0, 2e-8, 0]))
