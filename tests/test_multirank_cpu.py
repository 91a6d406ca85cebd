"""World-size-2 test of bench.py's multi-rank host logic on CPU (gloo).  The hot path has no exchange step (DESIGN.md
"Multi-GPU": independent replicas), so the N > 1 path consists of: per-rank problem selection (rank 0 = the seeded
config, other ranks the same shapes with their own shifts), a barrier, the MAX-reduction of the measured time and
the whole-job aggregate.  No GPU and no kernel is involved here."""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        probs = bench.rank_problems(1, rank)
        ev = bench.evals_of(probs)
        # every rank holds independent problems of the same shape
        sig = torch.tensor([float(probs[0]["shifts"][0, 0]), float(probs[0]["params"][0]), ev], dtype=torch.float64)
        gathered = [torch.zeros(3, dtype=torch.float64) for _ in range(world)]
        dist.all_gather(gathered, sig)
        dist.barrier()
        # max-over-ranks timing: rank r pretends to have needed (1 + r) ms
        t = torch.tensor([1e-3 * (1 + rank)], dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        value = bench.aggregate([ev] * world, float(t.item()))
        if rank == 0:
            out.put({"gathered": [g.tolist() for g in gathered], "tmax": float(t.item()), "value": value, "ev": ev})
    finally:
        dist.destroy_process_group()


def test_two_ranks_gloo():
    world = 2
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    res = out.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    g = res["gathered"]
    assert g[0][2] == g[1][2] == res["ev"] == 1048573 * 32          # same shape on every rank (weak scaling)
    assert g[0][1] == g[1][1]                                        # same integrand parameters
    assert g[0][0] != g[1][0]                                        # rank-specific shifts: independent problems
    assert res["tmax"] == pytest.approx(2e-3)                        # the slowest rank defines the time
    assert res["value"] == pytest.approx(2 * res["ev"] / 2e-3)       # whole-job throughput: all ranks' evaluations / max time


def test_rank0_gets_exactly_the_seeded_config():
    import bench
    from paper_1811_11720_b200 import synth
    a, b = bench.rank_problems(2, 0)[0], synth.config(2)[0]
    assert np.array_equal(a["shifts"], b["shifts"]) and np.array_equal(a["params"], b["params"]) and np.array_equal(a["z"], b["z"])
    c = bench.rank_problems(2, 3)[0]
    assert c["shifts"].shape == b["shifts"].shape and not np.array_equal(c["shifts"], b["shifts"])
    assert np.all((c["shifts"] >= 0) & (c["shifts"] < 1))


def test_gpus_flag_spawns_its_own_ranks(monkeypatch):
    """`python bench.py --gpus N` outside torchrun starts N ranks of itself on 127.0.0.1 (--gpus was ignored
    without torchrun); under torchrun a mismatching --gpus is an error."""
    import subprocess
    import sys
    import bench
    seen = {}
    monkeypatch.setattr(subprocess, "call", lambda cmd: seen.setdefault("cmd", cmd) and 0)
    monkeypatch.delenv("WORLD_SIZE", raising=False)
    monkeypatch.setattr(sys, "argv", ["bench.py", "--gpus", "4", "--steps", "2", "--warmup", "3"])
    with pytest.raises(SystemExit) as ex:
        bench.main()
    assert ex.value.code == 0
    cmd = seen["cmd"]
    assert cmd[1:4] == ["-m", "torch.distributed.run", "--nnodes=1"] and "--nproc-per-node=4" in cmd
    assert cmd[cmd.index("--master-addr") + 1] == "127.0.0.1"
    assert cmd[-6:] == ["--gpus", "4", "--steps", "2", "--warmup", "3"] and cmd[-7].endswith("bench.py")
    monkeypatch.setenv("WORLD_SIZE", "2")
    with pytest.raises(SystemExit) as ex:
        bench.main()
    assert "WORLD_SIZE" in str(ex.value.code)


def test_oracle_sample_keeps_the_cores_busy_and_is_bounded():
    """the bounded sample of the oracle legs: about 1/64 of the evaluations, never fewer than 128 chunks of 2^16 indices per
    problem unless the lattice is smaller, whole problems for a batch"""
    import bench
    from paper_1811_11720_b200 import synth
    for c in (1, 2, 3, 4):
        probs = synth.config(c)
        smp = bench.oracle_sample(probs, bench.ORACLE_SAMPLE_DIV)
        done = sum(k * p["m"] for p, k in smp)
        assert done <= bench.evals_of(probs)
        if c == 3:
            assert len(smp) == 4 and all(k == p["n"] for p, k in smp)
        else:
            assert smp[0][1] == min(probs[0]["n"], max(-(-probs[0]["n"] // 64), 128 * 65536))
