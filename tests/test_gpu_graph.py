"""The hot path under CUDA graph capture: afqmc_local_energy allocates nothing, copies nothing to the host and never
synchronises (include/afqmc.h), so K1 -> K2 (per spin) -> K3 can be captured once and replayed -- the way to run the
launch-bound small configurations (tiny: five launches for 57 us of work).  Replays must reproduce the direct call bit for
bit, also after the walkers have changed in place."""
import numpy as np
import pytest
import torch

from gen import make_inputs
from tests.test_gpu_parity import _le

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("name,nw", [("tiny", 4), ("small", 16)])
def test_local_energy_replayed_from_a_cuda_graph_is_bit_identical(name, nw):
    inp = make_inputs(name, n_walkers=nw)
    le = _le(inp)
    wk = torch.from_numpy(inp.walkers_packed()).cuda()
    E = torch.empty(nw, dtype=torch.complex128, device="cuda")
    lo = torch.empty_like(E)
    le.local_energy(wk, nw, E, lo)                       # warm-up outside the capture (module loading)
    torch.cuda.synchronize()
    E_direct, lo_direct = E.clone(), lo.clone()

    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):                        # capture on torch's capture stream (the binding passes the current stream)
        le.local_energy(wk, nw, E, lo)
    E.zero_(); lo.zero_()
    graph.replay()
    torch.cuda.synchronize()
    assert torch.equal(E, E_direct) and torch.equal(lo, lo_direct)

    # new walkers in the same buffers: the replay sees them, and agrees with a direct call on them
    perm = torch.arange(nw - 1, -1, -1)
    wk2 = torch.from_numpy(inp.walkers_packed(list(perm.numpy()))).cuda()
    wk.copy_(wk2)
    graph.replay()
    torch.cuda.synchronize()
    E_replay = E.clone()
    E2, _ = le.local_energy(wk2, nw)
    torch.cuda.synchronize()
    assert torch.equal(E_replay, E2)
    assert torch.equal(E_replay, E_direct[perm.cuda()])  # and walker w of the permuted batch is walker nw-1-w of the first

    # timing, for the record (printed with -s): direct launches vs replay
    def timed(fn, reps=200):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        fn(); torch.cuda.synchronize()
        e0.record()
        for _ in range(reps):
            fn()
        e1.record(); torch.cuda.synchronize()
        return e0.elapsed_time(e1) / reps * 1e3
    t_direct = timed(lambda: le.local_energy(wk, nw, E, lo))
    t_graph = timed(graph.replay)
    print(f"{name}: {t_direct:.1f} us per step with direct launches, {t_graph:.1f} us replayed from a CUDA graph")
    le.close()


def test_force_bias_only_and_propagate_replayed_from_cuda_graphs():
    from paper_2209_04015_b200 import sample_fields
    inp = make_inputs("small", n_walkers=9, n_gamma=50)
    nw, dt = inp.n_walkers, 1e-4
    le = _le(inp)
    chol = torch.from_numpy(inp.chol).cuda()
    le.enable_propagation(torch.from_numpy(inp.h1e).cuda(), chol, dt)          # also enables the force-bias path
    wk0 = torch.from_numpy(inp.walkers_packed()).cuda()
    x = sample_fields(5, 0, nw, inp.n_gamma)
    wts = torch.ones(nw, dtype=torch.float64, device="cuda")

    fb = torch.empty((nw, inp.n_gamma), dtype=torch.complex128, device="cuda")
    le.force_bias_only(wk0, nw, fb)
    torch.cuda.synchronize()
    fb_direct = fb.clone()
    g1 = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g1):
        le.force_bias_only(wk0, nw, fb)
    fb.zero_()
    g1.replay()
    torch.cuda.synchronize()
    assert torch.equal(fb, fb_direct)

    wk = wk0.clone()
    w_out, lo_out = torch.empty_like(wts), torch.empty(nw, dtype=torch.complex128, device="cuda")
    le.propagate(wk, nw, x, wts, 6, w_out, lo_out)                              # direct step on a copy
    torch.cuda.synchronize()
    ref = (wk.clone(), w_out.clone(), lo_out.clone())
    g2 = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g2):
        le.propagate(wk, nw, x, wts, 6, w_out, lo_out)
    wk.copy_(wk0); w_out.zero_(); lo_out.zero_()
    g2.replay()
    torch.cuda.synchronize()
    assert torch.equal(wk, ref[0]) and torch.equal(w_out, ref[1]) and torch.equal(lo_out, ref[2])
    le.close()
