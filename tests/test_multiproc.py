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


def test_single_process_helpers():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(None, [1.5, 2.5], None) == [1.5, 2.5]
    assert bench.replica_seed(3, 0) == 3
    assert abs(bench.whole_job_value(1, 50, 62.5) - 800.0) < 1e-12
