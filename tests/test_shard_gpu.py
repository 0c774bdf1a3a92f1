"""GPU parity of the sharded evaluation (hawkes_shard_*; include/hawkes.h): the four phases of every rank run one
after the other on ONE GPU, each rank on a context of its own -- the ranks' kernels never wait on one another, so nothing
is lost by the emulation but the overlap -- with the all-gathers replaced by a concatenation; results against the oracle, against the one-GPU
path, and run to run.  The two-process orchestration itself (torch.distributed all-gather between the phases) is
covered on CPU by tests/test_multiproc.py and, with the real kernels in two processes, by tests/test_shard_procs_gpu.py."""
import os

import numpy as np
import pytest

import oracle
import paper_2103_03348_b200 as hp
from paper_2103_03348_b200 import synth
from parity import check, hess_hyper_scale, scales

pytestmark = pytest.mark.gpu
THREADS = max(1, min(os.cpu_count() or 1, 64))


@pytest.fixture(scope="module")
def torch():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


def dev(torch, ev):
    f = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to("cuda")
    return f(ev.x), f(ev.t), f(ev.theta)


def shard_eval_one_gpu(torch, ctx, world, x, t, th, params, want):
    """world ranks, one after the other, on this GPU -- EACH RANK WITH ITS OWN CONTEXT, as on real hardware: a rank that
    read records, column partials or partial slots it did not produce itself would find another context's (or no) data
    there, not a neighbour's valid numbers of the same evaluation.  `ctx` is rank 0's context; the others are made here.
    Every rank runs the replicated phases on the gathered partials; their outputs must agree to the bit."""
    n = int(t.shape[0])
    mk = lambda *s: torch.empty(*s, dtype=torch.float64, device="cuda")
    ctxs = [ctx] + [hp.HawkesContext(ctx.n_max, ctx.dim) for _ in range(world - 1)]
    outs = [c.new_outputs(n, want) for c in ctxs]
    parts = mk(world, ctx.shard_part_doubles(n, want, 1))
    for r, c in enumerate(ctxs):
        c.shard_pass1(x, t, th, params, want, r, world, parts[r])
    for c, o in zip(ctxs, outs):
        c.shard_reduce1(n, params, want, world, parts, o)
    if want & (hp.WANT_GRAD_THETA | hp.WANT_HESS_THETA):
        parts2 = mk(world, ctx.shard_part_doubles(n, want, 2))
        for r, c in enumerate(ctxs):
            c.shard_pass2(n, params, want, r, world, parts2[r])
        for c, o in zip(ctxs, outs):
            c.shard_finish(n, params, want, world, parts2, o)
    sts = [c.last_status() for c in ctxs]
    lams = [c.get_lambda(n) for c in ctxs]
    for o, lam_r, st_r in zip(outs[1:], lams[1:], sts[1:]):
        assert st_r == sts[0] and torch.equal(lam_r, lams[0])
        for f in ("ll", "grad_theta", "grad_hyper", "hess_theta_diag", "hess_hyper"):
            a, b = getattr(outs[0], f), getattr(o, f)
            assert (a is None and b is None) or torch.equal(a, b), f
    for c in ctxs[1:]:
        c.close()
    return outs[0], sts[0], lams[0].cpu().numpy()


def compare(ev, r, lam, ref):
    s = scales(ev, ref)
    out = {"lambda": check("lambda", lam, ref.lam), "ll": check("ll", r.ll.item(), ref.ll, s["ll"])}
    if r.grad_theta is not None:
        out["grad_theta"] = check("grad_theta", r.grad_theta.cpu().numpy(), ref.grad_theta, s["grad_theta"])
    if r.grad_hyper is not None:
        out["grad_hyper"] = check("grad_hyper", r.grad_hyper.cpu().numpy(), ref.grad_hyper, s["grad_hyper"])
    if r.hess_theta_diag is not None:
        out["hess_theta_diag"] = check("hess_theta_diag", r.hess_theta_diag.cpu().numpy(), ref.hess_theta_diag, floor=1e-280)
    if r.hess_hyper is not None:
        out["hess_hyper"] = check("hess_hyper", r.hess_hyper.cpu().numpy(), ref.hess_hyper, hess_hyper_scale(ref.hess_hyper))
    return out


@pytest.mark.parametrize("world", [1, 2, 3, 8])
@pytest.mark.parametrize("want", [hp.WANT_LL | hp.WANT_GRAD_THETA, hp.WANT_GRAD, hp.WANT_ALL & ~hp.WANT_HESS_CROSS])
def test_sharded_small_problems_against_oracle(torch, world, want):
    """Ragged sizes, ties and duplicated locations, D = 2 and 3, all three moment levels (symmetric and dense pass 1)."""
    for n, seed, dim in ((300, 3, 2), (1281, 4, 2), (777, 5, 3)):
        ev = synth.small_random(n, seed, dim=dim, regime="mixed", ties=True, duplicates=True)
        ev.x *= np.sqrt(n / 16.0)
        ev.t *= n / 40.0
        ref = oracle.evaluate(ev.x, ev.t, ev.theta, ev.params, hess=True, row_d1=True, threads=THREADS)
        ctx = hp.HawkesContext(ev.n, ev.dim)
        r, st, lam = shard_eval_one_gpu(torch, ctx, world, *dev(torch, ev), ev.params, want)
        assert st == ref.status == 0
        compare(ev, r, lam, ref)


@pytest.mark.parametrize("world", [2, 8])
def test_sharded_config1_full_size(torch, world):
    """BASELINE.json configs[1] (N = 23,422) cut across 2 and 8 ranks: every output against the full oracle, against the
    one-GPU evaluation (summation order is the only difference) and bit-identical run to run."""
    ev = synth.config(1)
    ref = oracle.evaluate(ev.x, ev.t, ev.theta, ev.params, hess=True, row_d1=True, threads=THREADS)
    ctx = hp.HawkesContext(ev.n, ev.dim)
    x, t, th = dev(torch, ev)
    want = hp.WANT_ALL & ~hp.WANT_HESS_CROSS
    for w in (hp.WANT_GRAD, want):
        r, st, lam = shard_eval_one_gpu(torch, ctx, world, x, t, th, ev.params, w)
        assert st == 0
        res = compare(ev, r, lam, ref)
        one = ctx.eval(x, t, th, ev.params, w)
        assert abs(one.ll.item() - r.ll.item()) <= 1e-12 * abs(one.ll.item())
        assert float((one.grad_theta - r.grad_theta).abs().max()) <= 1e-11 * float(one.grad_theta.abs().max())
        r2, _, _ = shard_eval_one_gpu(torch, ctx, world, x, t, th, ev.params, w)
        for f in ("ll", "grad_theta", "grad_hyper", "hess_theta_diag", "hess_hyper"):
            a, b = getattr(r, f), getattr(r2, f)
            assert (a is None and b is None) or torch.equal(a, b), f
    print(f"world={world}: max scaled errors", res)


def test_sharded_argument_errors(torch):
    ev = synth.small_random(300, 1)
    ctx = hp.HawkesContext(ev.n, ev.dim)
    x, t, th = dev(torch, ev)
    part = torch.empty(ctx.shard_part_doubles(ev.n, hp.WANT_GRAD, 1), dtype=torch.float64, device="cuda")
    for rank, world in ((2, 2), (-1, 2), (0, 0), (0, 65)):
        with pytest.raises(hp.HawkesError) as e:
            ctx.shard_pass1(x, t, th, ev.params, hp.WANT_GRAD, rank, world, part)
        assert e.value.status == hp.ERR_ARG
    big = torch.empty(ctx.shard_part_doubles(ev.n, hp.WANT_ALL, 1), dtype=torch.float64, device="cuda")
    with pytest.raises(hp.HawkesError) as e:                # the cross block is not part of the sharded evaluation
        ctx.shard_pass1(x, t, th, ev.params, hp.WANT_ALL, 0, 2, big)
    assert e.value.status == hp.ERR_ARG
    w1, w2 = ctx.shard_workers(hp.WANT_GRAD)
    assert w1 > 0 and w2 > 0
