"""N>1 rank plumbing of bench.py on CPU (world_size 2, gloo): barrier, max-over-ranks timing, per-rank seeds and the
whole-job aggregate.  The path shards over independent sequences with no data-path collective, so
this is all the multi-process logic there is; the kernels are covered by the -m gpu tests."""
from __future__ import annotations

import os
import socket
import time

import torch
import torch.multiprocessing as mp


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out_dir: str):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    import bench
    from paper_2606_24957_b200 import synth
    d = bench.Dist()
    assert d.on and d.rank == rank and d.world == world
    d.init("gloo")
    try:
        # max over ranks
        assert d.max_float(10.0 + rank, "cpu") == 10.0 + (world - 1)
        # the timed region is bracketed by barriers and reports the slowest rank
        delay = 0.02 * (rank + 1)
        ms = bench.time_steps(lambda: time.sleep(delay), steps=3, warmup=1, dist=d, device="cpu",
                              timer=bench.HostTimer())
        slowest = 1e3 * 0.02 * world
        assert slowest * 0.95 <= ms < slowest * 3, (ms, slowest)
        # every rank draws its own batch of the same workload
        cfg = bench.rank_seed(synth.config_tiny(), rank)
        inp = synth.make_layer(cfg, 0, "cpu")
        torch.save({"q": inp.q, "ms": ms, "seed": cfg.seed}, os.path.join(out_dir, f"r{rank}.pt"))
        agg = bench.aggregate(100.0, cfg, world)
        assert agg["global_batch"] == cfg.batch * world
        assert abs(agg["sequences_per_s"] - cfg.batch * world / 100e-6) < 1e-6
    finally:
        d.finish()


def test_two_ranks_gloo(tmp_path):
    world, port = 2, _free_port()
    mp.spawn(_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    r0, r1 = (torch.load(tmp_path / f"r{r}.pt") for r in range(world))
    assert r0["ms"] == r1["ms"]                                   # all ranks agree on the max
    assert r0["seed"] != r1["seed"] and not torch.equal(r0["q"], r1["q"])
    from paper_2606_24957_b200 import synth
    assert r0["seed"] == synth.config_tiny().seed                   # rank 0 keeps the workload's base seed


def test_single_process_is_a_noop():
    for k in ("RANK", "LOCAL_RANK", "WORLD_SIZE"):
        os.environ.pop(k, None)
    import bench
    d = bench.Dist()
    assert not d.on
    d.init("gloo")
    d.barrier()
    assert d.max_float(3.5, "cpu") == 3.5
    d.finish()


def test_reference_arm_runs_only_on_rank0(monkeypatch, capsys):
    import bench

    class A:
        gpus, steps, warmup, batch, ctx, layers, packed = 2, 1, 0, 1, 256, 1, False

    d = bench.Dist()
    d.rank, d.world, d.on = 1, 2, True
    bench.run_reference(A, d)                                     # non-zero rank: no work, no output
    assert capsys.readouterr().out == ""


def test_gpus_flag_without_launcher_spawns_the_ranks():
    """`python bench.py --gpus 2` with no WORLD_SIZE in the environment must start two ranks itself (never print
    n_gpus = 2 from one process): checked on the reference arm, which needs no GPU -- rank 0 prints the one line and
    reports the world it ran in, rank 1 exits quietly."""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "LOCAL_RANK", "WORLD_SIZE", "MASTER_PORT")}
    r = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--impl", "reference", "--gpus", "2", "--batch",
                        "1", "--ctx", "256", "--layers", "1", "--steps", "1", "--warmup", "0"],
                       capture_output=True, text=True, env=env, cwd=root, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [json.loads(l) for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    assert lines[0]["impl"] == "reference" and lines[0]["n_gpus"] == 2
    assert lines[0]["run"]["world"] == 2 and "self-spawned" in lines[0]["run"]["launcher"]
