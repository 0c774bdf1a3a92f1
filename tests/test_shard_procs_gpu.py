"""The sharded evaluation (hawkes_shard_* through hp.shard_eval) as REAL processes
with the REAL kernels: two ranks, each with its own process, CUDA context and HawkesContext, exchanging their partial sums
between the phases with a torch.distributed all-gather.

 - test_two_processes_one_gpu: both ranks share the one GPU of the test box.  NCCL refuses two ranks on one device and
   gloo has no CUDA all-gather, so a test-side adapter stages `all_gather_into_tensor` through host memory; everything
   else is the code path a multi-GPU job runs.  The ranks' kernels never wait on one another (only the hosts do, in the
   gather), so sharing the GPU costs overlap, not correctness.
 - test_two_processes_two_gpus_nccl: the same worker over NCCL, one GPU per rank; skipped with fewer than two GPUs.

Checked: every output against the oracle (tests/parity.py tolerance), the same bits on both ranks, and the same bits as the
in-process emulation of tests/test_shard_gpu.py (ranks one after the other, a context each)."""
import os
import socket
import subprocess
import sys
import textwrap

import numpy as np
import pytest

import oracle
from paper_2103_03348_b200 import synth
from parity import check, scales

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
THREADS = max(1, min(os.cpu_count() or 1, 64))

WORKER = textwrap.dedent("""
    import os, sys
    sys.path.insert(0, %r)
    import numpy as np
    import torch
    import torch.distributed as dist
    import paper_2103_03348_b200 as hp
    from paper_2103_03348_b200 import synth

    backend, out_dir = sys.argv[1], sys.argv[2]
    rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
    torch.cuda.set_device(int(os.environ["LOCAL_RANK"]) if backend == "nccl" else 0)
    dist.init_process_group(backend)

    class HostStagedGather:
        '''all_gather_into_tensor of CUDA tensors over a CPU-only backend: device -> host, gather, host -> device.'''
        def all_gather_into_tensor(self, out, part):
            h = part.cpu()
            allh = torch.empty(world * h.numel(), dtype=h.dtype)
            dist.all_gather_into_tensor(allh, h)
            out.copy_(allh)

    comm = dist if backend == "nccl" else HostStagedGather()
    want = hp.WANT_GRAD
    for name, ev in (("config1", synth.config(1)), ("ragged", synth.small_random(1281, 4, dim=2, ties=True, duplicates=True))):
        if name == "ragged":
            ev.x *= np.sqrt(ev.n / 16.0)
            ev.t *= ev.n / 40.0
        f = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
        x, t, th = f(ev.x), f(ev.t), f(ev.theta)
        ctx = hp.HawkesContext(ev.n, ev.dim, torch.cuda.current_device())
        r = hp.shard_eval(ctx, comm, rank, world, x, t, th, ev.params, want)
        st = ctx.last_status()
        lam = ctx.get_lambda(ev.n)
        torch.cuda.synchronize()
        res = {"status": st, "lam": lam.cpu().numpy(), "ll": r.ll.cpu().numpy(), "grad_theta": r.grad_theta.cpu().numpy(),
               "grad_hyper": r.grad_hyper.cpu().numpy()}
        if rank == 0:
            # the in-process emulation: the same ranks one after the other, a context each, concatenation for the gather
            ctxs = [hp.HawkesContext(ev.n, ev.dim, torch.cuda.current_device()) for _ in range(world)]
            mk = lambda *s: torch.empty(*s, dtype=torch.float64, device="cuda")
            parts, parts2 = mk(world, ctx.shard_part_doubles(ev.n, want, 1)), mk(world, ctx.shard_part_doubles(ev.n, want, 2))
            o = ctxs[0].new_outputs(ev.n, want)
            for k, c in enumerate(ctxs):
                c.shard_pass1(x, t, th, ev.params, want, k, world, parts[k])
            for c in ctxs:
                c.shard_reduce1(ev.n, ev.params, want, world, parts, o)
            for k, c in enumerate(ctxs):
                c.shard_pass2(ev.n, ev.params, want, k, world, parts2[k])
            ctxs[0].shard_finish(ev.n, ev.params, want, world, parts2, o)
            torch.cuda.synchronize()
            res.update(emu_ll=o.ll.cpu().numpy(), emu_grad_theta=o.grad_theta.cpu().numpy(), emu_grad_hyper=o.grad_hyper.cpu().numpy())
        np.savez(os.path.join(out_dir, f"{name}_rank{rank}.npz"), **res)
    dist.barrier()
    dist.destroy_process_group()
""") % ROOT


def free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def run_two_ranks(tmp_path, backend):
    script = tmp_path / "shard_proc_worker.py"
    script.write_text(WORKER)
    port = free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), GLOO_SOCKET_IFNAME="lo")
        procs.append(subprocess.Popen([sys.executable, str(script), backend, str(tmp_path)], env=env,
                                      stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    try:
        outs = [p.communicate(timeout=600) for p in procs]
    finally:
        for p in procs:
            if p.poll() is None:
                p.kill()
    assert all(p.returncode == 0 for p in procs), outs
    for name, ev in (("config1", synth.config(1)), ("ragged", synth.small_random(1281, 4, dim=2, ties=True, duplicates=True))):
        if name == "ragged":
            ev.x *= np.sqrt(ev.n / 16.0)
            ev.t *= ev.n / 40.0
        ref = oracle.evaluate(ev.x, ev.t, ev.theta, ev.params, row_d1=True, threads=THREADS)
        s = scales(ev, ref)
        r0, r1 = (np.load(tmp_path / f"{name}_rank{k}.npz") for k in range(2))
        assert int(r0["status"]) == int(r1["status"]) == ref.status == 0
        check("lambda", r0["lam"], ref.lam)
        check("ll", r0["ll"][0], ref.ll, s["ll"])
        check("grad_theta", r0["grad_theta"], ref.grad_theta, s["grad_theta"])
        check("grad_hyper", r0["grad_hyper"], ref.grad_hyper, s["grad_hyper"])
        for f in ("lam", "ll", "grad_theta", "grad_hyper"):
            assert np.array_equal(r0[f], r1[f]), (name, f)                 # replicated: the same bits on both ranks
        for f in ("ll", "grad_theta", "grad_hyper"):
            assert np.array_equal(r0[f], r0["emu_" + f]), (name, f)        # ... and as the one-process emulation


def test_two_processes_one_gpu(tmp_path):
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    run_two_ranks(tmp_path, "gloo")


def test_two_processes_two_gpus_nccl(tmp_path):
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs (one per rank); the one-GPU box runs test_two_processes_one_gpu instead")
    run_two_ranks(tmp_path, "nccl")
