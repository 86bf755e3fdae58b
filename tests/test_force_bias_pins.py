"""Pins for ``oracle.force_bias`` (Eq. 19: xbar^gamma = sum_pq G_pq L^gamma_pq), CPU only.
Each check compares it with something it does not compute itself, so that a dropped spin sector, a stray factor, a
real-part-only contraction or a transposed Green's function fails at least one of them."""
import numpy as np
import pytest

from gen import make_inputs
from oracle import afqmc_oracle as orc
from tests.bruteforce import brute_force_greens_function
from tests.test_oracle_pins import random_system


def test_coulomb_energy_is_half_the_squared_force_bias():
    """Eq. 26's Coulomb term 1/2 sum_prqs V_prqs Gtot_pr Gtot_qs with Eq. 3 substituted is 1/2 sum_gamma xbar_gamma^2.
    EC comes from the stored-ERI rung O1 (einsum over V), which never forms sum G L: the complex value, both spin
    sectors and the absence of any extra factor in xbar are fixed by it."""
    for seed, complex_trial in ((3, False), (4, True)):
        h, chol, e0, pa, pb, fa, fb = random_system(seed, 7, 3, 2, 5, complex_trial=complex_trial, nw=3)
        V = orc.eri_from_cholesky(chol)
        for w in range(3):
            xbar = orc.force_bias(chol, pa, pb, fa[w], fb[w])
            ec = orc.local_energy_full_eri(h, V, e0, pa, pb, fa[w], fb[w])["EC"]
            assert xbar.shape == (5,) and np.abs(xbar.imag).max() > 1e-3        # genuinely complex
            assert abs(0.5 * np.sum(xbar * xbar) - ec) <= 1e-12 * abs(ec)


def test_identity_cholesky_closed_form():
    """L^gamma = c_gamma 1  =>  xbar_gamma = c_gamma Tr G = c_gamma (n_alpha + n_beta) for ANY walker (Tr G = N_e)."""
    h, chol, e0, pa, pb, fa, fb = random_system(5, 8, 3, 2, 4, complex_trial=True, nw=2)
    c = np.array([0.7, -1.3, 0.2, 2.0])
    chol = c[:, None, None] * np.eye(8)[None]
    for w in range(2):
        xbar = orc.force_bias(chol, pa, pb, fa[w], fb[w])
        assert np.max(np.abs(xbar - c * 5)) <= 1e-12


@pytest.mark.parametrize("complex_trial", [False, True])
def test_against_brute_force_operator_application(complex_trial):
    """xbar_gamma = sum_pq L^gamma_pq <psi|a+_p a_q|phi>/<psi|phi>, the expectation values taken by applying the
    operators to the determinant expansion (tests/bruteforce.py: no Green's-function formula, no overlap matrix).
    L^gamma is made NON-symmetric here so that contracting with G^T instead of G would fail."""
    h, chol, e0, pa, pb, fa, fb = random_system(6 + int(complex_trial), 5, 2, 1, 3, complex_trial=complex_trial, nw=1)
    rng = np.random.default_rng(77)
    chol = rng.standard_normal((3, 5, 5))
    Ga = brute_force_greens_function(pa, pb, fa[0], fb[0], 0)
    Gb = brute_force_greens_function(pa, pb, fa[0], fb[0], 1)
    ref = np.array([np.sum(chol[g] * (Ga + Gb)) for g in range(3)])
    xbar = orc.force_bias(chol, pa, pb, fa[0], fb[0])
    assert np.max(np.abs(xbar - ref)) <= 1e-11 * np.max(np.abs(ref))
    wrong = np.array([np.sum(chol[g].T * (Ga + Gb)) for g in range(3)])
    assert np.max(np.abs(wrong - ref)) > 1e-3                                   # the pin can tell the two apart


def test_one_spin_sector_empty_and_additivity_over_spins():
    """With no beta electrons only the alpha Green's function contributes; with both, the two sectors add."""
    h, chol, e0, pa, pb, fa, fb = random_system(9, 6, 3, 2, 4, complex_trial=False, nw=1)
    empty_psi, empty_phi = np.zeros((6, 0), dtype=complex), np.zeros((6, 0), dtype=complex)
    xa = orc.force_bias(chol, pa, empty_psi, fa[0], empty_phi)
    xb = orc.force_bias(chol, empty_psi, pb, empty_phi, fb[0])
    xab = orc.force_bias(chol, pa, pb, fa[0], fb[0])
    S = pa.conj().T @ fa[0]
    Ga = (fa[0] @ np.linalg.inv(S) @ pa.conj().T).T                             # LAPACK inverse, not the oracle's LU
    assert np.max(np.abs(xa - np.einsum("gpq,pq->g", chol, Ga))) <= 1e-12 * np.max(np.abs(xa))
    assert np.max(np.abs(xab - (xa + xb))) <= 1e-13 * np.max(np.abs(xab))
    assert np.max(np.abs(xb)) > 1e-3


def test_hartree_fock_limit_is_real_trace_of_mo_cholesky():
    """phi = psi (real trial): G = (psi psi^T), so xbar_gamma = sum_sigma Tr(psi_sigma^T L^gamma psi_sigma), real."""
    inp = make_inputs("tiny", n_walkers=1)
    xbar = orc.force_bias(inp.chol, inp.psi_a, inp.psi_b, inp.psi_a, inp.psi_b)
    ref = sum(np.einsum("pi,gpq,qi->g", p.real, inp.chol, p.real) for p in (inp.psi_a, inp.psi_b))
    assert np.max(np.abs(xbar.imag)) <= 1e-13 and np.max(np.abs(xbar.real - ref)) <= 1e-12 * np.max(np.abs(ref))
