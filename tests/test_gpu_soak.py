"""Random-shape soak of the whole boundary against the oracle: for each of a fixed, seeded list of shapes (orbitals,
occupations incl. empty and unequal spins, Cholesky vectors, walkers, real / mixed / complex trial) the energy and
log-overlap of every walker, the force bias (by-product and dedicated GEMM), <S^2>, the host-buffer entry point (bit for bit),
the allocation-free overlaps, and -- for half of the shapes -- one propagation step.  The shapes are drawn, not chosen, so
that tile, strip, chunk and size-class boundaries nobody thought of get hit (a 5-minute run of the same loop over 4 000
shapes was clean when this file was written)."""
import numpy as np
import pytest
import torch

from gen.configs import Inputs
from oracle import afqmc_oracle as orc
from oracle import propagation_oracle as prop
from tests.test_gpu_parity import _custom, _le, assert_parity, gpu_energy

pytestmark = pytest.mark.gpu


def _shapes(seed, count, n_max):
    rng = np.random.default_rng(seed)
    out = []
    while len(out) < count:
        N = int(rng.integers(2, n_max))
        na, nb = int(rng.integers(0, min(N, 64) + 1)), int(rng.integers(0, min(N, 64) + 1))
        if na + nb == 0:
            na = 1
        cx = [False, True, "both"][int(rng.integers(0, 3))]
        if cx and max(na, nb) > 52:                        # documented limit of a complex trial block
            cx = False
        out.append((int(rng.integers(0, 2 ** 31)), N, na, nb, int(rng.integers(1, 40)), int(rng.integers(1, 14)), cx,
                    bool(rng.integers(0, 2)), int(rng.integers(0, 2 ** 31))))
    return out


@pytest.mark.parametrize("block", range(4))
def test_random_shapes_against_the_oracle(block):
    from paper_2209_04015_b200 import log_overlap_static
    for seed, N, na, nb, ng, nw, cx, with_step, aux in _shapes(20250 + block, 50, 75 if block < 3 else 140):
        tag = (seed, N, na, nb, ng, nw, cx)
        inp = _custom(seed, N, na, nb, ng, nw, complex_trial=cx)
        Eo, loo = orc.local_energy_batch(inp, rung="O3")
        le = _le(inp)
        E, lo = gpu_energy(inp, le)
        assert_parity(E, lo, Eo, loo)
        k = aux % nw
        fb, s2 = le.force_bias(nw), le.spin_squared(nw)
        torch.cuda.synchronize()
        ref = orc.force_bias(inp.chol, inp.psi_a, inp.psi_b, inp.phi_a[k], inp.phi_b[k])
        scale = max(np.max(np.abs(ref)), 1e-300)
        assert np.all(np.abs(fb.cpu().numpy()[k] - ref) <= 1e-10 * scale), tag
        s2o = orc.spin_squared(inp.psi_a, inp.psi_b, inp.phi_a[k], inp.phi_b[k])
        assert abs(s2.cpu().numpy()[k] - s2o) <= 1e-9 * max(1.0, abs(s2o)), tag
        Eh, _ = le.local_energy_host(torch.from_numpy(inp.walkers_packed()).pin_memory(), nw)
        assert np.array_equal(Eh.numpy().view(np.float64), E.view(np.float64)), tag
        le.enable_force_bias(torch.from_numpy(inp.chol).cuda())
        fb2 = le.force_bias_only(torch.from_numpy(inp.walkers_packed()).cuda(), nw)
        torch.cuda.synchronize()
        assert np.all(np.abs(fb2.cpu().numpy()[k] - ref) <= 1e-10 * scale), tag
        le.close()
        los = log_overlap_static(torch.from_numpy(inp.trial_packed()).cuda(), torch.from_numpy(inp.walkers_packed()).cuda(), N, na, nb, nw)
        torch.cuda.synchronize()
        assert_parity(E, los.cpu().numpy(), Eo, loo)
        if not with_step:
            continue
        inp2 = Inputs(**{**inp.__dict__, "chol": inp.chol * 0.3})
        rng = np.random.default_rng(aux)
        x, wts = rng.standard_normal((nw, ng)), rng.uniform(0.5, 2.0, nw)
        nrm = max(np.linalg.norm(np.einsum("g,gpq->pq", x[w], inp2.chol), 1) for w in range(nw))
        dt = min(0.01, (3.0 / max(nrm, 1e-12)) ** 2)
        le = _le(inp2)
        le.enable_propagation(torch.from_numpy(inp2.h1e).cuda(), torch.from_numpy(inp2.chol).cuda(), dt)
        wk = torch.from_numpy(inp2.walkers_packed()).cuda()
        w_new, _ = le.propagate(wk, nw, torch.from_numpy(x).cuda(), torch.from_numpy(wts).cuda(), taylor_order=40)
        torch.cuda.synchronize()
        out = wk.cpu().numpy()
        got = {"phi_a": out[: nw * N * na].reshape(nw, N, na)[k], "phi_b": out[nw * N * na:].reshape(nw, N, nb)[k]}
        r = prop.propagate_walker(inp2.h1e, inp2.chol, inp2.psi_a, inp2.psi_b, inp2.phi_a[k], inp2.phi_b[k], wts[k], x[k], dt)
        for key in ("phi_a", "phi_b"):
            if r[key].size:
                assert np.max(np.abs(got[key] - r[key])) <= 1e-10 * np.max(np.abs(r[key])), (tag, key)
        # the weight is exp() of a sum of magnitude ~100 that is itself good to 1e-10 relative
        assert abs(w_new[k].item() - r["weight"]) <= 1e-7 * max(abs(r["weight"]), 1e-300), tag
        le.close()
