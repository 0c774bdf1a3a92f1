"""The N > 1 path of bench.py is "independent replicas": no data-path collective, one
all-reduce(MAX) of the timed totals, rank 0 prints.  World-size-2 gloo processes on CPU cover that host logic."""
import json
import os
import socket
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = textwrap.dedent("""
    import json, os, sys
    sys.path.insert(0, %r)
    import torch
    import torch.distributed as dist
    import bench
    from paper_2103_03348_b200 import synth
    rank, world, local = bench.dist_env()
    dist.init_process_group("gloo")
    # each replica times its own work: pretend rank r needed (10 + 5 r) ms for 4 steps and (20 - 3 r) ms end to end
    total, e2e = bench.max_over_ranks(dist, [10.0 + 5.0 * rank, 20.0 - 3.0 * rank], torch.device("cpu"))
    seed = bench.replica_seed(7, rank)
    ev = synth.make_events(50, seed)
    out = {"rank": rank, "world": world, "total": total, "e2e": e2e, "seed": seed, "t0": float(ev.t[0]),
           "value": bench.whole_job_value(world, 4, total)}
    gathered = [None] * world
    dist.all_gather_object(gathered, out)
    if rank == 0:
        print(json.dumps(gathered), flush=True)
    dist.destroy_process_group()
""") % ROOT


def free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_two_replicas_max_over_ranks_and_seeds(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    port = free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), GLOO_SOCKET_IFNAME="lo")
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=180) for p in procs]
    assert all(p.returncode == 0 for p in procs), outs
    assert outs[1][0].strip() == ""                       # only rank 0 prints
    res = json.loads(outs[0][0].strip().splitlines()[-1])
    assert [r["rank"] for r in res] == [0, 1] and all(r["world"] == 2 for r in res)
    # MAX over ranks: slowest device-resident total is rank 1's (15 ms), slowest end-to-end is rank 0's (20 ms)
    assert all(r["total"] == 15.0 and r["e2e"] == 20.0 for r in res)
    assert all(abs(r["value"] - 2 * 4 / 15e-3) < 1e-9 for r in res)     # whole-job evaluations/s
    assert res[0]["seed"] == 7 and res[1]["seed"] == 8 and res[0]["t0"] != res[1]["t0"]


SHARD_WORKER = textwrap.dedent("""
    import json, os, sys
    sys.path.insert(0, %r)
    sys.path.insert(0, os.path.join(%r, "tests"))
    import numpy as np
    import torch
    import torch.distributed as dist
    import oracle
    import paper_2103_03348_b200 as hp
    from paper_2103_03348_b200 import synth
    from shard_stub import StubShardContext
    rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
    dist.init_process_group("gloo")
    ev = synth.small_random(700, seed=5, ties=True, duplicates=True)
    ev.x *= 6.0
    ev.t *= 15.0
    f = lambda a: torch.from_numpy(np.ascontiguousarray(a))
    res = []
    for sym in (True, False):
        ctx = StubShardContext(workers_per_rank=5, symmetric=sym)
        r = hp.shard_eval(ctx, dist, rank, world, f(ev.x), f(ev.t), f(ev.theta), ev.params, hp.WANT_LL | hp.WANT_GRAD_THETA)
        ref = oracle.evaluate(ev.x, ev.t, ev.theta, ev.params)
        res.append({"rank": rank, "sym": sym,
                    "lam_err": float(np.max(np.abs(ctx.lam - ref.lam) / ref.lam)),
                    "ll_err": abs(r.ll.item() - ref.integral - ref.ll) / abs(ref.ll),
                    "grad_err": float(np.max(np.abs(r.grad_theta.numpy() - ref.grad_theta)) / np.max(np.abs(ref.grad_theta))),
                    "lam_sum": float(ctx.lam.sum())})
    gathered = [None] * world
    dist.all_gather_object(gathered, res)
    if rank == 0:
        print(json.dumps(gathered), flush=True)
    dist.destroy_process_group()
""") % (ROOT, ROOT)


def test_two_ranks_shard_one_evaluation(tmp_path):
    """paper_2103_03348_b200.shard_eval (the orchestration the GPU path uses: phase, all-gather, phase, ...) over gloo with
    two processes.  The phases are a numpy stand-in (tests/shard_stub.py) that evaluates exactly the pieces of the pair
    space hawkes_plan_segments gives each rank, so the test covers the cut, the exchange and the rank-ordered sums: the
    assembled lambda, ell and d ell/d theta must be the oracle's, identically on both ranks."""
    script = tmp_path / "shard_worker.py"
    script.write_text(SHARD_WORKER)
    port = free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), GLOO_SOCKET_IFNAME="lo")
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=300) for p in procs]
    assert all(p.returncode == 0 for p in procs), outs
    res = json.loads(outs[0][0].strip().splitlines()[-1])
    for a, b in zip(res[0], res[1]):                       # per pass-1 form: rank 0's and rank 1's record
        assert a["rank"] == 0 and b["rank"] == 1 and a["sym"] == b["sym"]
        for r in (a, b):
            assert r["lam_err"] < 1e-12 and r["ll_err"] < 1e-13 and r["grad_err"] < 1e-12, r
        assert a["lam_sum"] == b["lam_sum"]                # replicated: the same bits on both ranks


def test_single_process_helpers():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(None, [1.5, 2.5], None) == [1.5, 2.5]
    assert bench.replica_seed(3, 0) == 3
    assert abs(bench.whole_job_value(1, 50, 62.5) - 800.0) < 1e-12
