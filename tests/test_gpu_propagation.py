"""GPU parity of afqmc_propagate (one hybrid phaseless step, Eq. 6-13) against
oracle/propagation_oracle.py, element by element on the propagated determinants, the shift xbar (Eq. 9), the new
log-overlap (Eq. 8) and the new weight (Eq. 7, 10-12).  Bar: 1e-10 relative (north_star's tolerance)."""
import math

import numpy as np
import pytest
import torch

from gen import make_inputs
from gen.configs import Inputs
from oracle import afqmc_oracle as orc
from oracle import propagation_oracle as prop
from tests.test_gpu_parity import _custom, _le

pytestmark = pytest.mark.gpu
RTOL = 1e-10


def _fields(inp, seed):
    rng = np.random.default_rng(seed)
    return rng.standard_normal((inp.n_walkers, inp.n_gamma)), rng.uniform(0.5, 2.0, inp.n_walkers)


def _converging_dt(inp, x, target=3.0, cap=0.01):
    """A time step for which the Taylor series of exp(A), A = i sqrt(dt) sum (x - xbar)_g L^g, has ||A||_1 <= ~target
    on these synthetic Hamiltonians (their Cholesky vectors are far larger than a molecule's)."""
    nrm = max(np.linalg.norm(np.einsum("g,gpq->pq", x[w], inp.chol), 1) for w in range(inp.n_walkers))
    return min(cap, (target / nrm) ** 2)


def _gpu_step(inp, x, wts, dt, order, le=None, idx=None):
    own = le is None
    if own:
        le = _le(inp)
        le.enable_propagation(torch.from_numpy(inp.h1e).cuda(), torch.from_numpy(inp.chol).cuda(), dt)
    nw = inp.n_walkers if idx is None else len(idx)
    wk = torch.from_numpy(inp.walkers_packed(idx)).cuda()
    xs = torch.from_numpy(np.ascontiguousarray(x if idx is None else x[idx])).cuda()
    ws = torch.from_numpy(np.ascontiguousarray(wts if idx is None else wts[idx])).cuda()
    w_new, lo_new = le.propagate(wk, nw, xs, ws, taylor_order=order)
    xbar = le.propagation_xbar()
    torch.cuda.synchronize()
    out = wk.cpu().numpy()
    na, nb, N = inp.n_alpha, inp.n_beta, inp.N
    phi_a = out[: nw * N * na].reshape(nw, N, na)
    phi_b = out[nw * N * na:].reshape(nw, N, nb)
    res = dict(phi_a=phi_a, phi_b=phi_b, weight=w_new.cpu().numpy(), lo=lo_new.cpu().numpy(), xbar=xbar.cpu().numpy())
    if own:
        le.close()
    return res


def _assert_step(inp, x, wts, dt, got, walkers=None, tol=RTOL):
    walkers = range(inp.n_walkers) if walkers is None else walkers
    for k, w in enumerate(walkers):
        ref = prop.propagate_walker(inp.h1e, inp.chol, inp.psi_a, inp.psi_b, inp.phi_a[w], inp.phi_b[w], wts[w], x[w], dt)
        A1 = np.linalg.norm(prop.hs_potential(inp.chol, dt, x[w] - ref["xbar"]), 1)
        assert A1 < 8.0, f"test set-up: ||A||_1 = {A1} is too large for the Taylor order used"
        assert np.max(np.abs(got["xbar"][k] - ref["xbar"])) <= tol * np.max(np.abs(ref["xbar"])), w
        for key in ("phi_a", "phi_b"):
            if ref[key].size:
                assert np.max(np.abs(got[key][k] - ref[key])) <= tol * np.max(np.abs(ref[key])), (w, key)
        lo = ref["log_ovlp_new"]
        assert abs(got["lo"][k].real - lo.real) <= tol * max(1.0, abs(lo.real)), w
        dphi = abs((got["lo"][k].imag - lo.imag + math.pi) % (2 * math.pi) - math.pi)
        assert dphi <= tol * max(1.0, abs(lo.real)), w
        assert abs(got["weight"][k] - ref["weight"]) <= 10 * tol * max(abs(ref["weight"]), 1e-300), (w, got["weight"][k], ref["weight"])


@pytest.mark.parametrize("name,nw", [("tiny", 4), ("small", 5)])
def test_propagate_matches_oracle_on_the_named_configs(name, nw):
    inp = make_inputs(name, n_walkers=nw)
    x, wts = _fields(inp, 21)
    dt = _converging_dt(inp, x)
    got = _gpu_step(inp, x, wts, dt, order=40)
    _assert_step(inp, x, wts, dt, got)
    assert np.all(got["weight"] >= 0.0)


@pytest.mark.parametrize("N,na,nb,ng,nw,cx", [
    (12, 5, 2, 9, 3, False),       # unequal spins, odd sizes, non-orthonormal walkers
    (9, 4, 0, 7, 5, False),        # no beta electrons, N odd (odd pitches)
    (9, 0, 3, 7, 2, False),        # no alpha electrons
    (33, 13, 11, 70, 7, False),    # ragged strips and k-steps
    (21, 6, 5, 50, 9, "both"),     # complex trial
    (70, 33, 31, 41, 3, False),    # two column groups (2 (n_alpha + n_beta) = 128 > 104 columns)
    (200, 8, 7, 6, 2, False),      # two row tiles in K9 (N > 192)
])
def test_propagate_edge_shapes(N, na, nb, ng, nw, cx):
    inp = _custom(1200 + N, N, na, nb, ng, nw, complex_trial=cx)
    inp = Inputs(**{**inp.__dict__, "chol": inp.chol * 0.3})
    x, wts = _fields(inp, 22)
    dt = _converging_dt(inp, x)
    got = _gpu_step(inp, x, wts, dt, order=40)
    _assert_step(inp, x, wts, dt, got)


@pytest.mark.parametrize("N,na,nb,ng,nw", [
    (12, 3, 2, 6, 160),     # one K9 row tile per walker: 148 walkers fill a round, the other 12 go in the finer-tiled launch
    (170, 4, 3, 5, 80),     # two row tiles per walker (22 strips): 74 walkers in whole rounds, 6 walkers as 4 tiles of 6 strips
])
def test_propagate_batches_larger_than_one_round_of_ctas(N, na, nb, ng, nw):
    """k9_apply runs one CTA per SM; batch items beyond whole rounds of the GPU go in a second launch with row tiles of
    half the height (launch_k9 in csrc/afqmc.cu).  Walkers on both sides of that boundary against the oracle."""
    inp = _custom(1300 + N, N, na, nb, ng, nw)
    inp = Inputs(**{**inp.__dict__, "chol": inp.chol * 0.3})
    x, wts = _fields(inp, 23)
    dt = _converging_dt(inp, x)
    got = _gpu_step(inp, x, wts, dt, order=40)
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    per_item = (((N + 7) // 8) + 19) // 20
    main_items = (per_item * nw // sms) * sms // per_item
    assert 0 < main_items < nw
    idx = sorted({0, main_items - 1, main_items, nw - 1})
    sub = {k: v[idx] for k, v in got.items()}
    _assert_step(inp, x, wts, dt, sub, walkers=idx)


def test_propagate_full_size_in_the_bench_configuration():
    """Cu2O2-scale, all 256 walkers, the time step and Taylor order bench.py times (5e-5, 6): the propagated determinants and
    the shift of sampled walkers -- the first, both sides of k9_apply's whole-rounds boundary (222 of 256 walkers on 148
    SMs) and the last -- against the oracle's matrices with the series truncated at the same order, summed by hand."""
    from tests.test_gpu_parity import _full_inputs
    inp = _full_inputs("cu2o2")
    x, wts = _fields(inp, 24)
    dt, order = 5e-5, 6
    got = _gpu_step(inp, x, wts, dt, order=order)
    E = prop.expm_symmetric(-0.5 * dt * prop.one_body_shift(inp.h1e, inp.chol))
    for w in (0, 221, 222, 255):
        xbar = prop.force_bias_shift(inp.chol, inp.psi_a, inp.psi_b, inp.phi_a[w], inp.phi_b[w], dt)
        assert np.max(np.abs(got["xbar"][w] - xbar)) <= RTOL * np.max(np.abs(xbar)), w
        A = prop.hs_potential(inp.chol, dt, x[w] - xbar)
        series, term = np.eye(inp.N, dtype=np.complex128), np.eye(inp.N, dtype=np.complex128)
        for k in range(1, order + 1):
            term = term @ A / k
            series = series + term
        new = {}
        for key, phi in (("phi_a", inp.phi_a[w]), ("phi_b", inp.phi_b[w])):
            new[key] = ref = E @ (series @ (E @ phi))
            assert np.max(np.abs(got[key][w] - ref)) <= RTOL * np.max(np.abs(ref)), (w, key)
        # overlap ratio and weight (Eq. 7-12) of the same truncated step; these synthetic Cholesky vectors are ~100x a
        # molecule's, so the importance function may overflow exp(): then both sides must say inf
        lo_old = complex(*orc.log_overlap(inp.psi_a, inp.psi_b, inp.phi_a[w], inp.phi_b[w]))
        lo_new = complex(*orc.log_overlap(inp.psi_a, inp.psi_b, new["phi_a"], new["phi_b"]))
        assert abs(got["lo"][w].real - lo_new.real) <= RTOL * max(1.0, abs(lo_new.real)), w
        w_ref = orc.phaseless_weight_update(wts[w], lo_old, lo_new, x[w], xbar)
        if np.isfinite(w_ref):
            assert abs(got["weight"][w] - w_ref) <= 1e-8 * max(abs(w_ref), 1e-300), (w, got["weight"][w], w_ref)
        else:
            assert got["weight"][w] == w_ref, (w, got["weight"][w], w_ref)
    assert not np.any(np.isnan(got["weight"])) and np.all(got["weight"] >= 0.0)


def test_propagate_truncated_series_and_batch_subsets_and_repeatability():
    """(i) a low Taylor order gives exactly the truncated series (checked against the oracle's matrices summed by
    hand), (ii) a subset of walkers on a larger handle, (iii) bit-identical repeats, (iv) zero fields at order 0 reduce
    to the one-body propagator exp(-dt h') with the force-bias shift only in the weights."""
    inp = make_inputs("tiny")
    x, wts = _fields(inp, 23)
    dt = 0.004
    le = _le(inp, max_walkers=7)
    le.enable_propagation(torch.from_numpy(inp.h1e).cuda(), torch.from_numpy(inp.chol).cuda(), dt)
    got3 = _gpu_step(inp, x, wts, dt, order=3, le=le)
    E = prop.expm_symmetric(-0.5 * dt * prop.one_body_shift(inp.h1e, inp.chol))
    for w in range(inp.n_walkers):
        xbar = prop.force_bias_shift(inp.chol, inp.psi_a, inp.psi_b, inp.phi_a[w], inp.phi_b[w], dt)
        A = prop.hs_potential(inp.chol, dt, x[w] - xbar)
        series = np.eye(inp.N) + A + A @ A / 2 + A @ A @ A / 6
        ref = E @ series @ E @ inp.phi_a[w]
        assert np.max(np.abs(got3["phi_a"][w] - ref)) <= RTOL * np.max(np.abs(ref))
    sub = [2, 0]
    got_sub = _gpu_step(inp, x, wts, dt, order=40, le=le, idx=sub)
    _assert_step(inp, x, wts, dt, got_sub, walkers=sub)
    again = _gpu_step(inp, x, wts, dt, order=40, le=le, idx=sub)
    for key in ("phi_a", "phi_b", "weight", "lo", "xbar"):
        assert np.array_equal(np.asarray(got_sub[key]).view(np.float64), np.asarray(again[key]).view(np.float64)), key
    le.close()


def test_propagate_argument_errors():
    from paper_2209_04015_b200 import AfqmcError
    inp = make_inputs("tiny")
    le = _le(inp)
    wk = torch.from_numpy(inp.walkers_packed()).cuda()
    x = torch.zeros((4, inp.n_gamma), dtype=torch.float64, device="cuda")
    w = torch.ones(4, dtype=torch.float64, device="cuda")
    with pytest.raises(AfqmcError, match="afqmc_enable_propagation first"):
        le.propagate(wk, 4, x, w)
    h, c = torch.from_numpy(inp.h1e).cuda(), torch.from_numpy(inp.chol).cuda()
    with pytest.raises(AfqmcError, match="dt must be positive"):
        le.enable_propagation(h, c, 0.0)
    le.enable_propagation(h, c, 0.01)
    with pytest.raises(AfqmcError, match="already enabled"):
        le.enable_propagation(h, c, 0.02)
    with pytest.raises(AfqmcError, match="taylor_order"):
        le.propagate(wk, 4, x, w, taylor_order=65)
    le.close()
