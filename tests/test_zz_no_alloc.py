"""hawkes_loglik_static, the entry point for callers that cannot allocate device memory.

Who needs it: code that runs inside a process whose GPU memory is already spoken for (an application-wide pool holds
the whole device, so a library's cudaMalloc fails or breaks the host's accounting), and code on a latency-critical
thread that cannot afford the device-wide serialisation of cudaMalloc / cudaFree.  hawkes_create allocates, so such
callers cannot have a context; this one call keeps its intermediates in a fixed array inside the library instead and
therefore takes at most hp.STATIC_N_MAX events.

The check is against the existing path (a context's hawkes_loglik) at the suite's parity tolerance (tests/parity.py:
1e-10 of the sum of the magnitudes of the terms of ell), on two calls in a row with different problems -- the second
call finds the first one's leftovers in the shared array and must not be affected by them -- and then the first problem
once more, which must reproduce its own bits.  The file sorts last on purpose: pytest -x stops at the first failure,
and a failure here should not hide the rest of the suite.  It passes alone in a fresh process (the first call then
does the per-device set-up) and after the other tests."""
import numpy as np
import pytest

import paper_2103_03348_b200 as hp
from paper_2103_03348_b200 import synth
from parity import TOL

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


def _dev(torch, ev):
    f = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to("cuda")
    return f(ev.x), f(ev.t), f(ev.theta)


def _existing_path(torch, ev):
    """ell from a context (the path every other test validates against the oracle) and the scale of its terms."""
    ctx = hp.HawkesContext(ev.n, ev.dim)
    x, t, th = _dev(torch, ev)
    ll = ctx.loglik(x, t, th, ev.params)
    assert ctx.last_status() == 0
    lam = ctx.get_lambda(ev.n)
    torch.cuda.synchronize()
    scale = max(abs(ll.item()), float(torch.sum(torch.abs(torch.log(lam))).item()))
    ctx.close()
    return ll.item(), scale


def test_static_loglik_matches_the_context_path_on_two_calls_in_a_row(torch):
    # problem A: the paper's size (23,422 events, 2-D, configs[1]); problem B: small, ragged, 3-D, with ties
    ev_a = synth.config(1)
    ev_b = synth.small_random(1237, seed=11, dim=3, ties=True)
    ref_a, scale_a = _existing_path(torch, ev_a)
    ref_b, scale_b = _existing_path(torch, ev_b)

    # the caller owns inputs and outputs; nothing below allocates on the device once these exist
    in_a, in_b = _dev(torch, ev_a), _dev(torch, ev_b)
    out = torch.full((3,), float("nan"), dtype=torch.float64, device="cuda")
    status = torch.full((3,), -1, dtype=torch.int32, device="cuda")
    hp.loglik_static(*in_a, ev_a.params, out[0:1], status[0:1])
    hp.loglik_static(*in_b, ev_b.params, out[1:2], status[1:2])     # finds A's data in the shared array
    hp.loglik_static(*in_a, ev_a.params, out[2:3], status[2:3])     # ... and this one finds B's
    torch.cuda.synchronize()
    got, st = out.cpu().numpy(), status.cpu().numpy()
    assert list(st) == [0, 0, 0]
    assert abs(got[0] - ref_a) <= TOL * scale_a, (got[0], ref_a)
    assert abs(got[1] - ref_b) <= TOL * scale_b, (got[1], ref_b)
    assert got[2] == got[0]                                          # same inputs, same bits, whatever ran in between


def test_static_loglik_limits_and_status(torch):
    ev = synth.small_random(300, seed=5, dim=2)
    x, t, th = _dev(torch, ev)
    out = torch.zeros(1, dtype=torch.float64, device="cuda")
    status = torch.zeros(1, dtype=torch.int32, device="cuda")
    # one event more than the fixed array holds: refused on the host with its own code, nothing written
    n_big = hp.STATIC_N_MAX + 1
    big = torch.zeros(2 * n_big, dtype=torch.float64, device="cuda")
    with pytest.raises(hp.HawkesError) as e:
        hp.loglik_static(big.view(2, n_big), big[:n_big], big[:n_big], ev.params, out)
    assert e.value.status == hp.ERR_TOO_LARGE and "HAWKES_STATIC_N_MAX" in str(e.value)
    # the largest size it does take
    ev_max = synth.make_events(hp.STATIC_N_MAX, seed=2)
    ref, scale = _existing_path(torch, ev_max)
    hp.loglik_static(*_dev(torch, ev_max), ev_max.params, out, status)
    torch.cuda.synchronize()
    assert status.item() == 0 and abs(out.item() - ref) <= TOL * scale
    # data-dependent status without a context: unsorted times are flagged in status_out ...
    t_bad = t.clone()
    t_bad[[10, 200]] = t_bad[[200, 10]]
    hp.loglik_static(x, t_bad, th, ev.params, out, status)
    torch.cuda.synchronize()
    assert status.item() & hp.STATIC_BIT_UNSORTED
    # ... and the flag does not leak into the next call
    ref, scale = _existing_path(torch, ev)
    hp.loglik_static(x, t, th, ev.params, out, status)
    torch.cuda.synchronize()
    assert status.item() == 0 and abs(out.item() - ref) <= TOL * scale
