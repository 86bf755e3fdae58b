"""Pins for the CPU oracle: everything here checks ``oracle/`` against something other than itself
(closed forms, brute force, invariances, textbook special cases).  CPU only.  SURVEY.md §8(c) P1-P12."""
import itertools
import math

import numpy as np
import pytest

from gen import CONFIGS, make_inputs
from oracle import afqmc_oracle as orc
from tests.bruteforce import brute_force_local_energy, hartree_fock_energy_mo

RTOL = 1e-11


def rel(a, b):
    return abs(a - b) / max(abs(b), 1e-300)


def random_system(seed, N, na, nb, ng, complex_trial=True, nw=2, noise=0.3):
    rng = np.random.default_rng(seed)
    a = rng.standard_normal((N, N))
    h = 0.5 * (a + a.T)
    b = rng.standard_normal((ng, N, N))
    chol = 0.5 * (b + b.transpose(0, 2, 1)) * np.exp(-np.arange(ng) / 3.0)[:, None, None]

    def orth(n):
        m = rng.standard_normal((N, n)) + (1j * rng.standard_normal((N, n)) if complex_trial else 0)
        q, _ = np.linalg.qr(m)
        return q.astype(np.complex128)
    psi_a, psi_b = orth(na), orth(nb)
    phis_a = np.stack([psi_a + noise * (rng.standard_normal((N, na)) + 1j * rng.standard_normal((N, na)))
                       for _ in range(nw)])
    phis_b = np.stack([psi_b + noise * (rng.standard_normal((N, nb)) + 1j * rng.standard_normal((N, nb)))
                       for _ in range(nw)])
    return h, chol, 0.37, psi_a, psi_b, phis_a, phis_b


@pytest.fixture(scope="module")
def tiny():
    inp = make_inputs("tiny")
    return inp, orc.eri_from_cholesky(inp.chol)


# ---- P1 Hermiticity of the inputs and of the ERIs --------------------------------------------
def test_p1_hermiticity(tiny):
    inp, V = tiny
    assert np.array_equal(inp.h1e, inp.h1e.T)
    assert np.array_equal(inp.chol, inp.chol.transpose(0, 2, 1))
    assert np.allclose(V, V.transpose(1, 0, 2, 3), rtol=0, atol=1e-13)
    assert np.allclose(V, V.transpose(0, 1, 3, 2), rtol=0, atol=1e-13)
    assert np.allclose(V, V.transpose(2, 3, 0, 1), rtol=0, atol=1e-13)
    for name in ("tiny", "small"):
        x = make_inputs(name)
        for psi in (x.psi_a, x.psi_b):
            assert np.allclose(psi.conj().T @ psi, np.eye(psi.shape[1]), atol=1e-12)
        assert np.allclose(np.einsum("wpi,wpj->wij", x.phi_a.conj(), x.phi_a), np.eye(x.n_alpha), atol=1e-12)
        assert x.psi_a.imag.max() == 0.0


# ---- P11 LU / determinant / inverse against Leibniz and LAPACK --------------------------------
def leibniz_det(A):
    n = A.shape[0]
    tot = 0j
    for perm in itertools.permutations(range(n)):
        inv = sum(1 for i in range(n) for j in range(i + 1, n) if perm[i] > perm[j])
        term = (-1) ** inv
        for i in range(n):
            term *= A[i, perm[i]]
        tot += term
    return tot


@pytest.mark.parametrize("n", [1, 2, 3, 4, 5])
def test_p11_det_vs_leibniz(n):
    rng = np.random.default_rng(10 + n)
    A = rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))
    la, arg, Ainv = orc.logdet_and_inverse(A)
    d = leibniz_det(A)
    assert rel(math.exp(la) * complex(math.cos(arg), math.sin(arg)), d) < 1e-12
    assert np.allclose(Ainv @ A, np.eye(n), atol=1e-12)


def test_p11_lu_vs_lapack_and_pivoting():
    rng = np.random.default_rng(5)
    for n in (7, 26, 50):
        A = rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))
        A[0, 0] = 0.0                      # forces a row exchange at the first step
        la, arg, Ainv = orc.logdet_and_inverse(A)
        sign, logabs = np.linalg.slogdet(A)
        assert abs(la - logabs) < 1e-11
        assert abs(orc.wrap_angle(arg - math.atan2(sign.imag, sign.real))) < 1e-11
        assert np.allclose(Ainv, np.linalg.inv(A), rtol=1e-9, atol=1e-11)
    la, arg, _ = orc.logdet_and_inverse(np.zeros((3, 3), dtype=complex))
    assert la == -math.inf


# ---- explicit loops == einsum form (index strings checked by eye in the loop version) ----------
def test_explicit_loops_equal_einsum(tiny):
    inp, V = tiny
    for w in range(2):
        a = orc.local_energy_explicit_loops(inp.h1e, inp.chol, inp.e0, inp.psi_a, inp.psi_b, inp.phi_a[w], inp.phi_b[w])
        b = orc.local_energy_full_eri(inp.h1e, V, inp.e0, inp.psi_a, inp.psi_b, inp.phi_a[w], inp.phi_b[w])
        for k in ("E", "E1", "EC", "EX"):
            assert rel(a[k], b[k]) < 1e-12, k


# ---- P2 closed-form Hartree-Fock energy when phi = psi ----------------------------------------
@pytest.mark.parametrize("complex_trial", [False, True])
def test_p2_hartree_fock_closed_form(complex_trial):
    h, chol, e0, psi_a, psi_b, _, _ = random_system(21, N=8, na=3, nb=2, ng=12, complex_trial=complex_trial)
    V = orc.eri_from_cholesky(chol)
    r = orc.local_energy_full_eri(h, V, e0, psi_a, psi_b, psi_a, psi_b)
    ehf = hartree_fock_energy_mo(h, chol, e0, psi_a, psi_b)
    assert rel(r["E"], ehf) < RTOL
    assert abs(r["logabs"]) < 1e-12 and abs(r["arg"]) < 1e-12
    assert abs(r["E"].imag) < 1e-11 * abs(r["E"])


def test_p2_hartree_fock_tiny_config(tiny):
    inp, V = tiny
    r = orc.local_energy_full_eri(inp.h1e, V, inp.e0, inp.psi_a, inp.psi_b, inp.psi_a, inp.psi_b)
    assert rel(r["E"], hartree_fock_energy_mo(inp.h1e, inp.chol, inp.e0, inp.psi_a, inp.psi_b)) < RTOL


# ---- P3 invariance under phi -> phi C ---------------------------------------------------------
def test_p3_invariance_under_column_mixing(tiny):
    inp, V = tiny
    rng = np.random.default_rng(3)
    for w in range(inp.n_walkers):
        Ca = rng.standard_normal((3, 3)) + 1j * rng.standard_normal((3, 3))
        Cb = rng.standard_normal((3, 3)) + 1j * rng.standard_normal((3, 3))
        r0 = orc.local_energy_full_eri(inp.h1e, V, inp.e0, inp.psi_a, inp.psi_b, inp.phi_a[w], inp.phi_b[w])
        r1 = orc.local_energy_full_eri(inp.h1e, V, inp.e0, inp.psi_a, inp.psi_b, inp.phi_a[w] @ Ca, inp.phi_b[w] @ Cb)
        assert rel(r1["E"], r0["E"]) < 1e-11
        sa, la = np.linalg.slogdet(Ca)
        sb, lb = np.linalg.slogdet(Cb)
        assert abs(r1["logabs"] - r0["logabs"] - la - lb) < 1e-11
        assert abs(orc.wrap_angle(r1["arg"] - r0["arg"] - np.angle(sa) - np.angle(sb))) < 1e-11


# ---- P4 brute force over the full determinant space -------------------------------------------
def test_p4_brute_force_small_complex_unequal_spin():
    h, chol, e0, psi_a, psi_b, phis_a, phis_b = random_system(44, N=5, na=2, nb=1, ng=6, complex_trial=True)
    V = orc.eri_from_cholesky(chol)
    for w in range(2):
        r = orc.local_energy_full_eri(h, V, e0, psi_a, psi_b, phis_a[w], phis_b[w])
        e_bf, ov = brute_force_local_energy(h, chol, e0, psi_a, psi_b, phis_a[w], phis_b[w])
        assert rel(r["E"], e_bf) < RTOL
        assert abs(r["logabs"] - math.log(abs(ov))) < 1e-11
        assert abs(orc.wrap_angle(r["arg"] - np.angle(ov))) < 1e-11


def test_p4_brute_force_tiny_config(tiny):
    """The tiniest config of BASELINE.json: N=10, 3+3 electrons, 120^2 = 14 400 determinants."""
    inp, V = tiny
    w = 1
    r = orc.local_energy_full_eri(inp.h1e, V, inp.e0, inp.psi_a, inp.psi_b, inp.phi_a[w], inp.phi_b[w])
    e_bf, ov = brute_force_local_energy(inp.h1e, inp.chol, inp.e0, inp.psi_a, inp.psi_b, inp.phi_a[w], inp.phi_b[w])
    assert rel(r["E"], e_bf) < RTOL
    assert abs(r["logabs"] - math.log(abs(ov))) < 1e-11
    assert abs(orc.wrap_angle(r["arg"] - np.angle(ov))) < 1e-11


# ---- P5 identity Cholesky vectors: closed form for arbitrary walkers ----------------------------
def test_p5_identity_cholesky_closed_form():
    N, na, nb, ng = 7, 3, 2, 5
    h, _, e0, psi_a, psi_b, phis_a, phis_b = random_system(55, N, na, nb, ng)
    c = np.array([0.7, -0.3, 0.2, 1.1, 0.05])
    chol = c[:, None, None] * np.eye(N)[None]
    mu = 0.83
    V = orc.eri_from_cholesky(chol)
    ne = na + nb
    expect = e0 + mu * ne + 0.5 * np.sum(c * c) * ne * (ne - 1)
    for w in range(2):
        r = orc.local_energy_full_eri(mu * np.eye(N), V, e0, psi_a, psi_b, phis_a[w], phis_b[w])
        assert rel(r["E"], expect) < RTOL


# ---- P6 one electron: two-body energy vanishes -------------------------------------------------
def test_p6_one_electron():
    h, chol, e0, psi_a, psi_b, phis_a, phis_b = random_system(66, N=6, na=1, nb=0, ng=4)
    V = orc.eri_from_cholesky(chol)
    r = orc.local_energy_full_eri(h, V, e0, psi_a, psi_b, phis_a[0], phis_b[0])
    assert abs(r["EC"] + r["EX"]) < 1e-12 * max(1.0, abs(r["EC"]))
    G = np.outer(phis_a[0][:, 0], psi_a[:, 0].conj()).T / (psi_a[:, 0].conj() @ phis_a[0][:, 0])
    assert rel(r["E"], e0 + np.sum(h * G)) < RTOL


# ---- P7 two electrons of opposite spin: pure Coulomb from rank-1 Green's functions -------------
def test_p7_two_electrons_opposite_spin():
    h, chol, e0, psi_a, psi_b, phis_a, phis_b = random_system(77, N=6, na=1, nb=1, ng=4)
    V = orc.eri_from_cholesky(chol)
    r = orc.local_energy_full_eri(h, V, e0, psi_a, psi_b, phis_a[1], phis_b[1])
    Ga = np.outer(psi_a[:, 0].conj(), phis_a[1][:, 0]) / (psi_a[:, 0].conj() @ phis_a[1][:, 0])
    Gb = np.outer(psi_b[:, 0].conj(), phis_b[1][:, 0]) / (psi_b[:, 0].conj() @ phis_b[1][:, 0])
    e2 = np.einsum("prqs,pr,qs->", V, Ga, Gb)
    assert rel(r["EC"] + r["EX"], e2) < RTOL


# ---- P8 conjugation symmetry -------------------------------------------------------------------
def test_p8_conjugation(tiny):
    inp, V = tiny
    w = 2
    r0 = orc.local_energy_full_eri(inp.h1e, V, inp.e0, inp.psi_a, inp.psi_b, inp.phi_a[w], inp.phi_b[w])
    r1 = orc.local_energy_full_eri(inp.h1e, V, inp.e0, inp.psi_a, inp.psi_b, inp.phi_a[w].conj(), inp.phi_b[w].conj())
    assert rel(r1["E"], np.conj(r0["E"])) < RTOL
    assert abs(r1["logabs"] - r0["logabs"]) < 1e-12 and abs(orc.wrap_angle(r1["arg"] + r0["arg"])) < 1e-12
    r2 = orc.local_energy_full_eri(inp.h1e, V, inp.e0, inp.psi_a, inp.psi_b,
                                   inp.phi_a[w].real.astype(complex), inp.phi_b[w].real.astype(complex))
    assert abs(r2["E"].imag) < 1e-12 * abs(r2["E"])


# ---- P9 orbital-rotation covariance ------------------------------------------------------------
def test_p9_orbital_rotation(tiny):
    inp, V = tiny
    rng = np.random.default_rng(9)
    U, _ = np.linalg.qr(rng.standard_normal((inp.N, inp.N)))
    h2 = U.T @ inp.h1e @ U
    chol2 = np.einsum("pa,gpq,qb->gab", U, inp.chol, U)
    V2 = orc.eri_from_cholesky(chol2)
    w = 3
    r0 = orc.local_energy_full_eri(inp.h1e, V, inp.e0, inp.psi_a, inp.psi_b, inp.phi_a[w], inp.phi_b[w])
    r1 = orc.local_energy_full_eri(h2, V2, inp.e0, U.T @ inp.psi_a, U.T @ inp.psi_b, U.T @ inp.phi_a[w], U.T @ inp.phi_b[w])
    assert rel(r1["E"], r0["E"]) < RTOL
    assert abs(r1["logabs"] - r0["logabs"]) < 1e-12


# ---- P10 spin swap -----------------------------------------------------------------------------
def test_p10_spin_swap(tiny):
    inp, V = tiny
    w = 0
    r0 = orc.local_energy_full_eri(inp.h1e, V, inp.e0, inp.psi_a, inp.psi_b, inp.phi_a[w], inp.phi_b[w])
    r1 = orc.local_energy_full_eri(inp.h1e, V, inp.e0, inp.psi_b, inp.psi_a, inp.phi_b[w], inp.phi_a[w])
    assert rel(r1["E"], r0["E"]) < 1e-13


# ---- P12 the memory rungs O2, O3 reproduce O1 walker by walker ---------------------------------
@pytest.mark.parametrize("name,nw", [("tiny", 4), ("small", 6)])
def test_p12_rungs_agree(name, nw):
    inp = make_inputs(name, n_walkers=nw)
    V = orc.eri_from_cholesky(inp.chol)
    o1 = [orc.local_energy_full_eri(inp.h1e, V, inp.e0, inp.psi_a, inp.psi_b, inp.phi_a[w], inp.phi_b[w])
          for w in range(nw)]
    o2 = orc.local_energy_streamed_eri(inp.h1e, inp.chol, inp.e0, inp.psi_a, inp.psi_b, inp.phi_a, inp.phi_b)
    o3 = [orc.local_energy_cholesky(inp.h1e, inp.chol, inp.e0, inp.psi_a, inp.psi_b, inp.phi_a[w], inp.phi_b[w])
          for w in range(nw)]
    for w in range(nw):
        for k in ("E", "E1", "EC", "EX"):
            assert rel(o2[w][k], o1[w][k]) < 1e-12, (w, k)
            assert rel(o3[w][k], o1[w][k]) < 1e-12, (w, k)
        assert o2[w]["logabs"] == o1[w]["logabs"] and o3[w]["arg"] == o1[w]["arg"]


def test_p12_rungs_agree_unequal_spin_complex_trial():
    h, chol, e0, psi_a, psi_b, phis_a, phis_b = random_system(91, N=9, na=4, nb=2, ng=7, complex_trial=True, nw=3)
    V = orc.eri_from_cholesky(chol)
    o2 = orc.local_energy_streamed_eri(h, chol, e0, psi_a, psi_b, phis_a, phis_b)
    for w in range(3):
        o1 = orc.local_energy_full_eri(h, V, e0, psi_a, psi_b, phis_a[w], phis_b[w])
        o3 = orc.local_energy_cholesky(h, chol, e0, psi_a, psi_b, phis_a[w], phis_b[w])
        assert rel(o2[w]["E"], o1["E"]) < 1e-12 and rel(o3["E"], o1["E"]) < 1e-12


def test_batch_front_end(tiny):
    inp, V = tiny
    E, lo = orc.local_energy_batch(inp, rung="O1", V=V)
    E3, lo3 = orc.local_energy_batch(inp, rung="O3", walkers=[1, 3])
    assert np.allclose(E3, E[[1, 3]], rtol=1e-12) and np.allclose(lo3, lo[[1, 3]], rtol=1e-12)


@pytest.mark.parametrize("name,nw", [("tiny", 4), ("small", 3)])
def test_listing4_agrees_with_definition(name, nw):
    """The paper's own half-rotated CPU algorithm (oracle/listing4_cpu.py, baseline B) against the definition oracle."""
    from oracle.listing4_cpu import HalfRotated, local_energy_listing4
    inp = make_inputs(name, n_walkers=nw)
    Eo, loo = orc.local_energy_batch(inp, rung="O1")
    hr = HalfRotated(inp.h1e, inp.chol, inp.psi_a, inp.psi_b)
    for w in range(nw):
        E, lo = local_energy_listing4(hr, inp.e0, inp.phi_a[w], inp.phi_b[w])
        assert rel(E, Eo[w]) < 1e-11
        assert abs(lo.real - loo[w].real) < 1e-10 and abs(np.angle(np.exp(1j * (lo.imag - loo[w].imag)))) < 1e-10


def test_listing4_complex_trial_unequal_spin():
    from oracle.listing4_cpu import HalfRotated, local_energy_listing4
    h1e, chol, e0, psi_a, psi_b, phis_a, phis_b = random_system(77, 9, 4, 2, 11, complex_trial=True)
    V = orc.eri_from_cholesky(chol)
    hr = HalfRotated(h1e, chol, psi_a, psi_b)
    for w in range(len(phis_a)):
        Eo = orc.local_energy_full_eri(h1e, V, e0, psi_a, psi_b, phis_a[w], phis_b[w])["E"]
        E, _ = local_energy_listing4(hr, e0, phis_a[w], phis_b[w])
        assert rel(E, Eo) < 1e-11


@pytest.mark.parametrize("complex_trial", [False, True])
def test_greens_function_index_order_by_operator_application(complex_trial):
    """G_pq = <a+_p a_q> (Eq. 20) element by element from the determinant expansion.  The energy cannot pin the index
    order (h and L are symmetric), and Eq. 22's two members are transposes of each other (DESIGN.md section 3 #16)."""
    from tests.bruteforce import brute_force_greens_function
    h1e, chol, e0, psi_a, psi_b, phis_a, phis_b = random_system(91, 6, 3, 2, 2, complex_trial=complex_trial)
    for spin, (psi, phi) in enumerate(((psi_a, phis_a[0]), (psi_b, phis_b[0]))):
        G = orc.greens_function(psi, phi)[0]
        ref = brute_force_greens_function(psi_a, psi_b, phis_a[0], phis_b[0], spin)
        assert np.max(np.abs(G - ref)) < 1e-12
        assert np.max(np.abs(G - G.T)) > 1e-3          # the case can tell G from its transpose
