"""GPU parity: the CUDA path (through the C-ABI, via the ctypes binding) against the CPU oracle, element by
element on the same seeded inputs.  Bar (BASELINE.json north_star): relative 1e-10 on each walker's complex
energy and on its log-overlap."""
import json
import math
import os

import numpy as np
import pytest
import torch

from gen import CONFIGS, make_inputs
from gen.configs import Inputs
from oracle import afqmc_oracle as orc

pytestmark = pytest.mark.gpu
RTOL = 1e-10
GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "oracle_energies.json")


_FULL = {}


def _full_inputs(name):
    """Full-size inputs, generated once per session and per config (`large` takes minutes of host time and 6 GB)."""
    if name not in _FULL:
        _FULL[name] = make_inputs(name)
    return _FULL[name]


def _le(inp, max_walkers=None):
    from paper_2209_04015_b200 import LocalEnergy
    dev = "cuda"
    return LocalEnergy(torch.from_numpy(inp.h1e).to(dev), torch.from_numpy(inp.chol).to(dev),
                       torch.from_numpy(inp.trial_packed()).to(dev), inp.N, inp.n_alpha, inp.n_beta, inp.n_gamma,
                       inp.e0, max_walkers or inp.n_walkers)


def gpu_energy(inp, le=None, idx=None):
    own = le is None
    le = le or _le(inp)
    nw = inp.n_walkers if idx is None else len(idx)
    E, lo = le.local_energy(torch.from_numpy(inp.walkers_packed(idx)).cuda(), nw)
    torch.cuda.synchronize()
    E, lo = E.cpu().numpy(), lo.cpu().numpy()
    if own:
        le.close()
    return E, lo


def assert_parity(E, lo, Eo, loo, tol=RTOL):
    E, lo, Eo, loo = map(np.asarray, (E, lo, Eo, loo))
    err = np.abs(E - Eo) / np.abs(Eo)
    assert np.all(err <= tol), f"energy rel err max {err.max():.3e} at walker {err.argmax()}"
    dre = np.abs(lo.real - loo.real) / np.maximum(1.0, np.abs(loo.real))
    assert np.all(dre <= tol), f"log|ovlp| err max {dre.max():.3e}"
    dim = np.abs((lo.imag - loo.imag + math.pi) % (2 * math.pi) - math.pi)
    assert np.all(dim <= tol * np.maximum(1.0, np.abs(loo.real))), f"arg ovlp err max {dim.max():.3e}"
    assert np.all(lo.imag <= math.pi) and np.all(lo.imag > -math.pi)


# ---- small configs: every walker against the definition oracle (O1, stored ERIs) -----------------
@pytest.mark.parametrize("name", ["tiny", "small"])
def test_parity_all_walkers_vs_definition(name):
    inp = make_inputs(name)
    Eo, loo = orc.local_energy_batch(inp, rung="O1")
    E, lo = gpu_energy(inp)
    assert_parity(E, lo, Eo, loo)


# ---- full-size configs, in the launch configuration bench.py times: sampled walkers ----------------
@pytest.mark.parametrize("name", ["medium", "cu2o2", "large"])
def test_parity_full_size_vs_golden(name):
    """All walkers run on the GPU at BASELINE.json's full size; the sampled walkers are compared with oracle
    values stored by tests/golden/make_golden.py (O2 = definition with streamed ERIs, O3 = Cholesky-direct),
    and one walker is recomputed live with O3."""
    with open(GOLDEN) as f:
        gold = json.load(f)[name]
    inp = _full_inputs(name)
    assert (gold["N"], gold["n_gamma"], gold["n_walkers"]) == (inp.N, inp.n_gamma, inp.n_walkers)
    E, lo = gpu_energy(inp)
    assert np.all(np.isfinite(E.view(np.float64))) and np.all(np.isfinite(lo.view(np.float64)))
    for key in ("definition", "O3"):
        if key not in gold:
            continue
        g = gold[key]
        idx = g["walkers"]
        Eo = np.array(g["E_re"]) + 1j * np.array(g["E_im"])
        loo = np.array(g["logabs"]) + 1j * np.array(g["arg"])
        assert_parity(E[idx], lo[idx], Eo, loo)
    w = inp.n_walkers // 2 + 1
    Eo, loo = orc.local_energy_batch(inp, rung="O3", walkers=[w])
    assert_parity(E[[w]], lo[[w]], Eo, loo)


@pytest.mark.parametrize("name", ["medium", "cu2o2", "large"])
def test_parity_every_walker_full_size_vs_listing4(name):
    """Every walker of the full-size launch (not only the sampled ones above) against the paper's half-rotated CPU
    algorithm (oracle/listing4_cpu.py), which tests/test_oracle_pins.py pins to the definition oracle."""
    from oracle.listing4_cpu import HalfRotated, local_energy_listing4
    inp = _full_inputs(name)
    E, lo = gpu_energy(inp)
    hr = HalfRotated(inp.h1e, inp.chol, inp.psi_a, inp.psi_b)
    ref = [local_energy_listing4(hr, inp.e0, inp.phi_a[w], inp.phi_b[w]) for w in range(inp.n_walkers)]
    assert_parity(E, lo, np.array([r[0] for r in ref]), np.array([r[1] for r in ref]))


# ---- edge cases --------------------------------------------------------------------------------------
def _custom(seed, N, na, nb, ng, nw, noise=0.2, complex_trial=False):
    rng = np.random.default_rng(seed)
    a = rng.standard_normal((N, N))
    h = 0.5 * (a + a.T) + np.diag(np.arange(N, dtype=float))
    b = rng.standard_normal((ng, N, N))
    chol = 0.5 * (b + b.transpose(0, 2, 1)) * np.exp(-np.arange(ng) / max(4.0, ng / 3))[:, None, None]
    q, _ = np.linalg.qr(rng.standard_normal((N, N)))
    psi_a = q[:, :na].astype(np.complex128)
    q2, _ = np.linalg.qr(rng.standard_normal((N, N)))
    psi_b = q2[:, :nb].astype(np.complex128)
    if complex_trial:        # orthonormal complex columns: Q factor of a complex Gaussian matrix
        qa, _ = np.linalg.qr(rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N)))
        psi_a = qa[:, :na]
        if complex_trial == "both":
            qb, _ = np.linalg.qr(rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N)))
            psi_b = qb[:, :nb]
    phi_a = psi_a[None] + noise * (rng.standard_normal((nw, N, na)) + 1j * rng.standard_normal((nw, N, na)))
    phi_b = psi_b[None] + noise * (rng.standard_normal((nw, N, nb)) + 1j * rng.standard_normal((nw, N, nb)))
    return Inputs(name="custom", N=N, n_alpha=na, n_beta=nb, n_gamma=ng, e0=-1.25, h1e=h, chol=chol,
                  psi_a=np.ascontiguousarray(psi_a), psi_b=np.ascontiguousarray(psi_b),
                  phi_a=np.ascontiguousarray(phi_a), phi_b=np.ascontiguousarray(phi_b))


@pytest.mark.parametrize("N,na,nb,ng,nw", [
    (12, 5, 2, 9, 3),      # unequal spins, non-orthonormal walkers, odd sizes
    (9, 4, 0, 7, 5),       # no beta electrons
    (9, 0, 3, 7, 2),       # no alpha electrons
    (7, 1, 1, 3, 1),       # one electron per spin, single walker
    (33, 13, 11, 70, 7),   # ragged everything; several row tiles
    (70, 33, 31, 41, 5),   # N not a multiple of 4, large odd n
    (64, 64, 1, 5, 3),     # n = N = AFQMC_MAX_NOCC (theta = psi-independent limit)
])
def test_parity_edge_shapes(N, na, nb, ng, nw):
    inp = _custom(100 + N, N, na, nb, ng, nw)
    Eo, loo = orc.local_energy_batch(inp, rung="O1" if N <= 40 else "O3")
    E, lo = gpu_energy(inp)
    assert_parity(E, lo, Eo, loo)


@pytest.mark.parametrize("N,na,nb,ng,nw,which", [
    (12, 5, 2, 9, 3, "both"),      # complex trial in both spins (4-product path), odd sizes
    (12, 4, 3, 9, 3, True),        # complex alpha block, real beta block
    (33, 13, 11, 70, 7, "both"),   # several row tiles, ragged tails
    (70, 33, 31, 41, 5, "both"),   # 2n = 66 rows per gamma block, n > 32 (two lane chunks)
    (9, 3, 0, 7, 2, True),         # no beta electrons
])
def test_parity_complex_trial(N, na, nb, ng, nw, which):
    """Complex (non-real) trial: Ltilde is complex and T needs four real products (Eq. 21
    with a complex psi).  The oracle is the same definition (it never forms Ltilde)."""
    inp = _custom(300 + N, N, na, nb, ng, nw, complex_trial=which)
    Eo, loo = orc.local_energy_batch(inp, rung="O1" if N <= 40 else "O3")
    E, lo = gpu_energy(inp)
    assert_parity(E, lo, Eo, loo)
    from paper_2209_04015_b200 import LocalEnergy  # noqa: F401  (force-bias check on the complex path too)
    le = _le(inp)
    gpu_energy(inp, le)
    fb = le.force_bias(nw)
    torch.cuda.synchronize()
    ref = orc.force_bias(inp.chol, inp.psi_a, inp.psi_b, inp.phi_a[0], inp.phi_b[0])
    assert np.all(np.abs(fb.cpu().numpy()[0] - ref) <= 1e-10 * np.max(np.abs(ref)))
    le.close()


def _k2_witnesses():
    from tests.k2_instances import WITNESS
    return [pytest.param(k, v, id=f"MT{k[0]}_NT{k[1]}") for k, v in sorted(WITNESS.items())]


@pytest.mark.parametrize("inst,shape", _k2_witnesses())
def test_every_k2_instantiation_against_the_oracle(inst, shape):
    """Every compiled k2_exchange<MT, NT> is launched once (tests/k2_instances.py names a shape the planner maps to
    it) and compared with the oracle on the first, a middle and the last walker."""
    n, cx, N, ng, nw = shape
    inp = _custom(7000 + 100 * inst[0] + inst[1], N, n, 0, ng, nw, complex_trial=bool(cx))
    le = _le(inp)
    info = le.info()
    assert (info["mt"][0], info["nt"][0]) == inst
    E, lo = gpu_energy(inp, le)
    le.close()
    idx = sorted({0, nw // 2, nw - 1})
    Eo, loo = orc.local_energy_batch(inp, rung="O3", walkers=idx)
    assert np.all(np.isfinite(E.view(np.float64)))
    assert_parity(E[idx], lo[idx], Eo, loo)


@pytest.mark.parametrize("cx", [False, True], ids=["real", "complex"])
def test_sweep_over_every_occupation_number(cx):
    """n_sigma = 1 .. 64 (complex trial: .. 52, the documented limit), unequal spins, N just above n, several gamma tiles
    and a ragged walker tile: every walker against the oracle."""
    for n in range(1, 53 if cx else 65):
        nb = (n * 5) // 7
        N = max(n + 2, 9)
        inp = _custom(8000 + n, N, n, nb, 11, 3, complex_trial="both" if cx else False)
        Eo, loo = orc.local_energy_batch(inp, rung="O3")
        E, lo = gpu_energy(inp)
        assert_parity(E, lo, Eo, loo)


def test_unequal_spins_sharing_one_kernel_instantiation():
    """Both spins map to the same K2 template instance with different shared-memory sizes (the opt-in
    attribute is process-global per instantiation, so the smaller spin must not lower the cap for the larger)."""
    from paper_2209_04015_b200 import plan
    p = plan(50, 19, 15, 7, 1)
    assert (p["mt"][0], p["nt"][0]) == (p["mt"][1], p["nt"][1]) and p["k2_smem_bytes"][0] != p["k2_smem_bytes"][1]
    inp = _custom(901, 50, 19, 15, 7, 1)
    Eo, loo = orc.local_energy_batch(inp, rung="O3")
    E, lo = gpu_energy(inp)
    assert_parity(E, lo, Eo, loo)


def test_two_live_handles_of_different_size_used_alternately():
    """Handles are independent (include/afqmc.h): a second, smaller handle created while the first is alive must not
    disturb the first one's launches (shared-memory opt-in, workspaces), and vice versa."""
    big = make_inputs("small", n_walkers=9)
    small = _custom(902, 12, 5, 2, 9, 3)
    le_big = _le(big)
    E_big0, lo_big0 = gpu_energy(big, le_big)
    le_small = _le(small)
    Eo_s, loo_s = orc.local_energy_batch(small, rung="O1")
    Eo_b, loo_b = orc.local_energy_batch(big, rung="O3")
    for _ in range(2):
        E_s, lo_s = gpu_energy(small, le_small)
        assert_parity(E_s, lo_s, Eo_s, loo_s)
        E_b, lo_b = gpu_energy(big, le_big)
        assert_parity(E_b, lo_b, Eo_b, loo_b)
        assert np.array_equal(E_b.view(np.float64), E_big0.view(np.float64))
    le_big.enable_force_bias(torch.from_numpy(big.chol).cuda())
    le_small.enable_force_bias(torch.from_numpy(small.chol).cuda())
    fb_b = le_big.force_bias_only(torch.from_numpy(big.walkers_packed()).cuda(), 9)
    fb_s = le_small.force_bias_only(torch.from_numpy(small.walkers_packed()).cuda(), 3)
    fb_b2 = le_big.force_bias_only(torch.from_numpy(big.walkers_packed()).cuda(), 9)
    torch.cuda.synchronize()
    assert torch.equal(fb_b.view(torch.float64), fb_b2.view(torch.float64))
    ref = orc.force_bias(small.chol, small.psi_a, small.psi_b, small.phi_a[1], small.phi_b[1])
    assert np.all(np.abs(fb_s.cpu().numpy()[1] - ref) <= 1e-10 * np.max(np.abs(ref)))
    le_big.close()
    le_small.close()


def test_two_handles_on_two_streams_running_concurrently():
    """"Use one handle per concurrent stream" (include/afqmc.h): two handles, two non-default streams, launches
    interleaved without any synchronisation in between; each must return exactly what it returns alone."""
    inps = [make_inputs("small", n_walkers=24, n_gamma=60), _custom(77, 33, 13, 11, 40, 19)]
    les = [_le(i) for i in inps]
    wks = [torch.from_numpy(i.walkers_packed()).cuda() for i in inps]
    alone = []
    for le, i, wk in zip(les, inps, wks):
        E, lo = le.local_energy(wk, i.n_walkers)
        torch.cuda.synchronize()
        alone.append((E.clone(), lo.clone()))
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    outs = [[], []]
    for rep in range(6):
        for k in (0, 1):
            with torch.cuda.stream(streams[k]):
                outs[k].append(les[k].local_energy(wks[k], inps[k].n_walkers, stream=streams[k]))
    torch.cuda.synchronize()
    for k in (0, 1):
        for E, lo in outs[k]:
            assert torch.equal(E, alone[k][0]) and torch.equal(lo, alone[k][1])
    for le in les:
        le.close()


def test_outputs_of_the_last_call_are_sized_by_the_library_not_the_caller():
    """force_bias / spin_squared / greens_function write results for the walkers of the LAST call; the
    binding sizes `out` from that and rejects a caller-supplied count or buffer that disagrees."""
    from paper_2209_04015_b200 import AfqmcError
    inp = make_inputs("tiny")
    le = _le(inp)
    with pytest.raises(AfqmcError, match="no preceding"):
        le.spin_squared()
    gpu_energy(inp, le)
    assert le.force_bias().shape == (4, inp.n_gamma) and le.spin_squared().shape == (4,)
    assert le.greens_function(1).shape == (4, inp.N, inp.N)
    with pytest.raises(AfqmcError, match="holds 4 walkers"):
        le.force_bias(2)
    with pytest.raises(AfqmcError, match="shape"):
        le.greens_function(0, out=torch.empty((2, inp.N, inp.N), dtype=torch.complex128, device="cuda"))
    gpu_energy(inp, le, [1, 3])
    assert le.spin_squared().shape == (2,)
    le.close()


def test_fewer_walkers_than_capacity_and_ragged_tail():
    inp = make_inputs("small", n_walkers=13)
    le = _le(inp, max_walkers=64)
    Eo, loo = orc.local_energy_batch(inp, rung="O3")
    for idx in ([0, 1, 2, 3, 4, 5, 6, 7, 8, 9, 10, 11, 12], [3], [12, 5, 7]):
        E, lo = gpu_energy(inp, le, idx)
        assert_parity(E, lo, Eo[idx], loo[idx])
    le.close()


def test_invariance_under_column_mixing_on_gpu():
    inp = make_inputs("small", n_walkers=4)
    rng = np.random.default_rng(8)
    Ca = rng.standard_normal((4, inp.n_alpha, inp.n_alpha)) + 1j * rng.standard_normal((4, inp.n_alpha, inp.n_alpha))
    E0, lo0 = gpu_energy(inp)
    inp2 = Inputs(**{**inp.__dict__, "phi_a": np.ascontiguousarray(inp.phi_a @ Ca)})
    E1, lo1 = gpu_energy(inp2)
    assert np.all(np.abs(E1 - E0) <= 1e-9 * np.abs(E0))
    s, l = np.linalg.slogdet(Ca)
    assert np.all(np.abs(lo1.real - lo0.real - l) < 1e-9)


def test_singular_walker_is_data_not_error():
    inp = make_inputs("tiny")
    phi_a = inp.phi_a.copy()
    phi_a[2] = 0.0           # S = 0 exactly: walker orthogonal to the trial
    inp2 = Inputs(**{**inp.__dict__, "phi_a": phi_a})
    E, lo = gpu_energy(inp2)
    Eo, loo = orc.local_energy_batch(inp, rung="O3")
    assert np.isnan(E[2].real) and np.isnan(E[2].imag) and lo[2].real == -np.inf
    keep = [0, 1, 3]
    assert_parity(E[keep], lo[keep], Eo[keep], loo[keep])


def test_bitwise_determinism():
    inp = make_inputs("small", n_walkers=16)
    le = _le(inp)
    E0, lo0 = gpu_energy(inp, le)
    for _ in range(3):
        E1, lo1 = gpu_energy(inp, le)
        assert np.array_equal(E0.view(np.float64), E1.view(np.float64))
        assert np.array_equal(lo0.view(np.float64), lo1.view(np.float64))
    le.close()


def test_bitwise_determinism_full_size_and_mixed_batches():
    """No compute-sanitizer on this pool, so races in K2's barrier protocol are hunted the slow way: the full-size
    headline launch repeated, with batches of another size interleaved on the same handle, must reproduce bit for bit
    (each batch shape against itself)."""
    inp = make_inputs("cu2o2")
    le = _le(inp)
    w_all = torch.from_numpy(inp.walkers_packed()).cuda()
    E0, lo0 = le.local_energy(w_all, inp.n_walkers)
    E0, lo0 = E0.clone(), lo0.clone()
    sub = [0, 17, 255, 128, 3]
    w_sub = torch.from_numpy(inp.walkers_packed(sub)).cuda()
    Es0 = None
    for rep in range(6):
        Es, _ = le.local_energy(w_sub, len(sub))
        # another batch shape deals the (gamma, walker) blocks to the warps in another order: same walkers, other rounding
        assert torch.all((Es - E0[sub]).abs() <= 1e-13 * E0[sub].abs()), rep
        Es0 = Es.clone() if Es0 is None else Es0
        assert torch.equal(Es.view(torch.float64), Es0.view(torch.float64)), rep
        E1, lo1 = le.local_energy(w_all, inp.n_walkers)
        assert torch.equal(E1.view(torch.float64), E0.view(torch.float64)), rep
        assert torch.equal(lo1.view(torch.float64), lo0.view(torch.float64)), rep
    le.close()


def test_host_entry_point_and_force_bias():
    inp = make_inputs("small", n_walkers=6)
    le = _le(inp)
    E, lo = gpu_energy(inp, le)
    wh = torch.from_numpy(inp.walkers_packed()).pin_memory()
    Eh, loh = le.local_energy_host(wh, 6)
    assert np.array_equal(Eh.numpy().view(np.float64), E.view(np.float64))
    assert np.array_equal(loh.numpy().view(np.float64), lo.view(np.float64))
    fb = le.force_bias(6)
    torch.cuda.synchronize()
    fb = fb.cpu().numpy()
    for w in (0, 5):
        ref = orc.force_bias(inp.chol, inp.psi_a, inp.psi_b, inp.phi_a[w], inp.phi_b[w])
        assert np.all(np.abs(fb[w] - ref) <= 1e-10 * np.max(np.abs(ref)))
    le.close()


@pytest.mark.parametrize("N,na,nb,ng,nw", [
    (20, 5, 4, 23, 67),     # three blocks: first eighth of alpha (rounded up to whole K2 column tiles), rest of alpha, beta; ragged tail
    (20, 0, 4, 23, 40),     # no alpha electrons: the blocks are cut from the beta spin
    (20, 5, 0, 23, 33),     # no beta electrons
    (33, 13, 11, 12, 19),   # two walkers per K2 column tile: block boundaries fall on tile boundaries
])
def test_host_entry_point_in_blocks_is_bit_identical_and_matches_oracle(N, na, nb, ng, nw):
    """afqmc_local_energy_host copies the walkers in up to three blocks and runs K1 + K2 block by block on walker ranges
    (include/afqmc.h): the result must equal afqmc_local_energy bit for bit, and the oracle to 1e-10."""
    inp = _custom(900 + nw, N, na, nb, ng, nw)
    le = _le(inp)
    E, lo = gpu_energy(inp, le)
    wh = torch.from_numpy(inp.walkers_packed()).pin_memory()
    Eh, loh = le.local_energy_host(wh, nw)
    assert np.array_equal(Eh.numpy().view(np.float64), E.view(np.float64))
    assert np.array_equal(loh.numpy().view(np.float64), lo.view(np.float64))
    Eh2, _ = le.local_energy_host(torch.from_numpy(inp.walkers_packed()), nw)            # pageable host memory
    assert np.array_equal(Eh2.numpy().view(np.float64), E.view(np.float64))
    idx = sorted({0, nw // 8, nw // 8 + 1, nw // 2, nw - 1})
    Eo, loo = orc.local_energy_batch(inp, rung="O3", walkers=idx)
    assert_parity(E[idx], lo[idx], Eo, loo)
    fewer = max(1, nw // 3)                                                              # fewer walkers than capacity, host path
    Ef, _ = le.local_energy_host(torch.from_numpy(inp.walkers_packed(list(range(fewer)))).pin_memory(), fewer)
    Ed, _ = gpu_energy(inp, le, idx=list(range(fewer)))
    assert np.array_equal(Ef.numpy().view(np.float64), Ed.view(np.float64))
    le.close()


@pytest.mark.parametrize("case", ["small", "ragged", "complex", "one_spin"])
def test_force_bias_only_matches_oracle_and_energy_path(case):
    """Dedicated force-bias GEMM (afqmc_force_bias_only) against sum_pq G_pq L^gamma_pq from the full Green's
    function (Eq. 19), and against the traces the energy path produces."""
    if case == "small":
        inp = make_inputs("small", n_walkers=70, n_gamma=130)      # two walker tiles (64 + 6), two gamma tiles
    elif case == "ragged":
        inp = _custom(411, 33, 13, 11, 101, 7)
    elif case == "complex":
        inp = _custom(412, 21, 6, 5, 50, 9, complex_trial="both")
    else:
        inp = _custom(413, 10, 4, 0, 9, 3)
    le = _le(inp)
    from paper_2209_04015_b200 import AfqmcError
    w = torch.from_numpy(inp.walkers_packed()).cuda()
    with pytest.raises(AfqmcError, match="afqmc_enable_force_bias"):
        le.force_bias_only(w, inp.n_walkers)
    le.enable_force_bias(torch.from_numpy(inp.chol).cuda())
    fb = le.force_bias_only(w, inp.n_walkers)
    torch.cuda.synchronize()
    fb = fb.cpu().numpy()
    for k in sorted({0, inp.n_walkers // 2, inp.n_walkers - 1}):
        ref = orc.force_bias(inp.chol, inp.psi_a, inp.psi_b, inp.phi_a[k], inp.phi_b[k])
        assert np.all(np.abs(fb[k] - ref) <= 1e-10 * np.max(np.abs(ref))), k
    le.local_energy(w, inp.n_walkers)
    fb2 = le.force_bias(inp.n_walkers)
    torch.cuda.synchronize()
    assert np.all(np.abs(fb2.cpu().numpy() - fb) <= 1e-11 * np.max(np.abs(fb)))
    le.close()


@pytest.mark.parametrize("case", ["small", "uhf", "complex", "polarised", "big_n"])
def test_spin_squared_matches_oracle(case):
    """<S^2> mixed estimator (Eq. 31 / Listing 6) from the half-rotated Green's function against the
    oracle's full-Green's-function einsum."""
    if case == "small":
        inp = make_inputs("small", n_walkers=9, n_gamma=20)            # RHF-style trial: a singlet, s2 = 0
    elif case == "uhf":
        inp = _custom(511, 33, 13, 11, 12, 6)
    elif case == "complex":
        inp = _custom(512, 21, 6, 5, 10, 5, complex_trial="both")
    elif case == "polarised":
        inp = _custom(513, 10, 4, 0, 9, 3)
    else:
        inp = _custom(514, 70, 64, 40, 6, 3)
    le = _le(inp)
    gpu_energy(inp, le)
    s2 = le.spin_squared(inp.n_walkers)
    torch.cuda.synchronize()
    s2 = s2.cpu().numpy()
    ref = np.array([orc.spin_squared(inp.psi_a, inp.psi_b, inp.phi_a[k], inp.phi_b[k]) for k in range(inp.n_walkers)])
    assert np.all(np.abs(s2 - ref) <= 1e-10 * np.maximum(1.0, np.abs(ref))), np.max(np.abs(s2 - ref))
    if case == "small":
        assert np.all(np.abs(s2) < 1e-9)
    le.close()


@pytest.mark.parametrize("case", ["uhf", "complex", "one_spin", "n64"])
def test_full_greens_function_matches_oracle(case):
    """Optional full Green's function (Eq. 22; build_full=True of PAPER.md:412-414) against the oracle's
    phi (psi^dagger phi)^-1 psi^dagger, and the paper's Listing 6 estimator evaluated from it against afqmc_spin_squared."""
    inp = {"uhf": lambda: _custom(611, 33, 13, 11, 6, 4),
           "complex": lambda: _custom(612, 21, 6, 5, 6, 3, complex_trial="both"),
           "one_spin": lambda: _custom(613, 10, 4, 0, 5, 2),
           "n64": lambda: _custom(614, 70, 64, 33, 4, 2)}[case]()
    le = _le(inp)
    gpu_energy(inp, le)
    G = [le.greens_function(s, inp.n_walkers) for s in (0, 1)]
    s2 = le.spin_squared(inp.n_walkers)
    torch.cuda.synchronize()
    for w in range(inp.n_walkers):
        for s, (psi, phi) in enumerate(((inp.psi_a, inp.phi_a[w]), (inp.psi_b, inp.phi_b[w]))):
            ref = orc.greens_function(psi, phi)[0]
            got = G[s][w].cpu().numpy()
            assert np.max(np.abs(got - ref)) <= 1e-10 * max(1.0, np.max(np.abs(ref))), (w, s)
    # Listing 6: two_body = -einsum("zij,zji->z", Ga, Gb)
    ms = 0.5 * (inp.n_alpha - inp.n_beta)
    listing6 = inp.n_beta + ms * (ms + 1) - torch.einsum("zij,zji->z", G[0], G[1])
    assert torch.all((listing6 - s2).abs() <= 1e-10 * torch.clamp(s2.abs(), min=1.0))
    le.close()


def test_phaseless_weight_update_matches_oracle():
    """Eq. 7-12 on the GPU against the oracle, with real log-overlaps and force biases from the library (before / after
    a made-up rotation of the walkers) and phases on both sides of the cos cut-off."""
    from paper_2209_04015_b200 import phaseless_weights
    inp = make_inputs("small", n_walkers=11, n_gamma=37)
    le = _le(inp)
    le.enable_force_bias(torch.from_numpy(inp.chol).cuda())
    w0 = torch.from_numpy(inp.walkers_packed()).cuda()
    xbar = le.force_bias_only(w0, 11).clone()
    _, lo_old = le.local_energy(w0, 11)
    lo_old = lo_old.clone()
    rng = np.random.default_rng(5)
    phase = np.exp(1j * np.linspace(-3.0, 3.0, 11))                 # rotates arg(ovlp) through the cut-off
    phi_a2 = inp.phi_a * (1.0 + 0.05 * rng.standard_normal(inp.phi_a.shape)) * phase[:, None, None]
    inp2 = Inputs(**{**inp.__dict__, "phi_a": np.ascontiguousarray(phi_a2)})
    _, lo_new = le.local_energy(torch.from_numpy(inp2.walkers_packed()).cuda(), 11)
    x = torch.from_numpy(rng.standard_normal((11, 37))).cuda()
    xbar = (xbar * 1e-3).contiguous()                               # keep exp() in range for this synthetic Hamiltonian
    wts = torch.from_numpy(rng.uniform(0.5, 2.0, 11)).cuda()
    got = phaseless_weights(x, xbar, lo_old, lo_new, wts)
    torch.cuda.synchronize()
    ref = np.array([orc.phaseless_weight_update(wts[k].item(), complex(lo_old[k].item()), complex(lo_new[k].item()),
                                                x[k].cpu().numpy(), xbar[k].cpu().numpy()) for k in range(11)])
    got = got.cpu().numpy()
    assert np.all(np.abs(got - ref) <= 1e-10 * np.maximum(np.abs(ref), 1e-300))
    assert np.any(ref == 0.0) and np.any(ref > 0.0)
    le.close()


def test_errors_are_reported():
    from paper_2209_04015_b200 import AfqmcError, LocalEnergy
    inp = make_inputs("tiny")
    dev = "cuda"
    h, c = torch.from_numpy(inp.h1e).to(dev), torch.from_numpy(inp.chol).to(dev)
    t = torch.from_numpy(inp.trial_packed()).to(dev)
    with pytest.raises(AfqmcError, match="non-finite"):
        LocalEnergy(h, c, t * float("nan"), inp.N, 3, 3, inp.n_gamma, 0.0, 4)
    with pytest.raises(AfqmcError, match="out of range"):
        LocalEnergy(h, c, t, inp.N, 3, 3, inp.n_gamma, 0.0, 0)
    le = LocalEnergy(h, c, t, inp.N, 3, 3, inp.n_gamma, 0.0, 2)
    w = torch.from_numpy(inp.walkers_packed()).to(dev)
    with pytest.raises(AfqmcError):
        le.local_energy(w, 4)
    le.close()
