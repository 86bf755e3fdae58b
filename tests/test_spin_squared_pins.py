"""Pins of the oracle's <S^2> mixed estimator (Eq. 31 / Listing 6), none of which re-types its formula:
brute-force operator application over the determinant space, the textbook single-determinant closed form, exact
values for spin eigenfunctions, and invariance under column mixing of the walker."""
import numpy as np
import pytest

from oracle import afqmc_oracle as orc
from tests.bruteforce import brute_force_spin_squared


def _system(seed, N, na, nb, complex_trial=True, noise=0.4):
    rng = np.random.default_rng(seed)
    def orth(n):
        a = rng.standard_normal((N, N)) + (1j * rng.standard_normal((N, N)) if complex_trial else 0)
        return np.ascontiguousarray(np.linalg.qr(a)[0][:, :n].astype(np.complex128))
    psi_a, psi_b = orth(na), orth(nb)
    phi_a = psi_a + noise * (rng.standard_normal((N, na)) + 1j * rng.standard_normal((N, na)))
    phi_b = psi_b + noise * (rng.standard_normal((N, nb)) + 1j * rng.standard_normal((N, nb)))
    return psi_a, psi_b, phi_a, phi_b


@pytest.mark.parametrize("N,na,nb,ct", [(6, 3, 2, True), (5, 2, 2, False), (6, 1, 3, True), (4, 2, 0, True)])
def test_brute_force_operator_application(N, na, nb, ct):
    psi_a, psi_b, phi_a, phi_b = _system(10 + N + na, N, na, nb, ct)
    ref = brute_force_spin_squared(psi_a, psi_b, phi_a, phi_b)
    got = orc.spin_squared(psi_a, psi_b, phi_a, phi_b)
    assert abs(got - ref) <= 1e-11 * max(1.0, abs(ref))


def test_single_determinant_closed_form():
    """phi = psi: <S^2> = M_S (M_S + 1) + N_dn - sum_ij |<psi_up_i|psi_dn_j>|^2 (textbook UHF formula)."""
    psi_a, psi_b, _, _ = _system(3, 9, 4, 3)
    ms = 0.5
    ref = ms * (ms + 1) + 3 - np.sum(np.abs(psi_a.conj().T @ psi_b) ** 2)
    got = orc.spin_squared(psi_a, psi_b, psi_a, psi_b)
    assert abs(got - ref) < 1e-12 and abs(got.imag) < 1e-12


def test_spin_eigenfunctions_give_exact_values():
    """A closed-shell trial (psi_dn = psi_up) is a singlet and a fully polarised one has S = M_S, and S^2 is Hermitian
    and commutes with nothing that matters here: the mixed estimator equals S(S+1) for ANY walker."""
    psi_a, _, phi_a, phi_b = _system(5, 8, 3, 3)
    assert abs(orc.spin_squared(psi_a, psi_a.copy(), phi_a, phi_b)) < 1e-11                      # singlet: 0
    psi_a, psi_b, phi_a, phi_b = _system(6, 7, 4, 0)
    assert abs(orc.spin_squared(psi_a, psi_b, phi_a, phi_b) - 2.0 * 3.0) < 1e-11                 # S = 2: 6


def test_invariance_under_column_mixing():
    psi_a, psi_b, phi_a, phi_b = _system(7, 10, 4, 3)
    rng = np.random.default_rng(1)
    Ca = rng.standard_normal((4, 4)) + 1j * rng.standard_normal((4, 4))
    Cb = rng.standard_normal((3, 3)) + 1j * rng.standard_normal((3, 3))
    a = orc.spin_squared(psi_a, psi_b, phi_a, phi_b)
    b = orc.spin_squared(psi_a, psi_b, phi_a @ Ca, phi_b @ Cb)
    assert abs(a - b) < 1e-10 * max(1.0, abs(a))
