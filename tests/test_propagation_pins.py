"""Pins for ``oracle/propagation_oracle.py`` (one hybrid phaseless step, Eq. 4 and 96-123 Eq. 6-13).
CPU only.  The propagator B(dt, y) is a READING of the paper (it only gives Eq. 4); Eq. 4 itself, evaluated in the
full determinant space with brute-force many-body matrices, is what decides whether the reading is right."""
import math

import numpy as np
import pytest
import scipy.linalg

from oracle import afqmc_oracle as orc
from oracle import propagation_oracle as prop
from tests.bruteforce import (determinant_vector, hamiltonian_matrix, one_body_operator_matrix)
from tests.test_oracle_pins import random_system


def small_system(seed, N=4, na=2, nb=1, ng=2, scale=0.6):
    h, chol, e0, pa, pb, fa, fb = random_system(seed, N, na, nb, ng, complex_trial=False, nw=1, noise=0.3)
    return h, scale * chol, pa, pb, fa[0], fb[0]


def gauss_hermite_normal(npts, dim):
    """Nodes [K, dim] and weights [K] of the tensor Gauss-Hermite rule for the standard normal density p(x)."""
    t, w = np.polynomial.hermite_e.hermegauss(npts)
    w = w / math.sqrt(2.0 * math.pi)
    grids = np.meshgrid(*([t] * dim), indexing="ij")
    wg = np.meshgrid(*([w] * dim), indexing="ij")
    return np.stack([g.ravel() for g in grids], axis=1), np.prod(np.stack([g.ravel() for g in wg], axis=1), axis=1)


def test_thouless_determinant_transforms_like_the_many_body_exponential():
    """exp(sum A_pq a+_p a_q) |phi> = |exp(A) phi>: the oracle's way of applying a one-body propagator (matrix times
    coefficient matrix) against the dense many-body exponential of the operator, complex non-symmetric A."""
    N, na, nb = 4, 2, 1
    rng = np.random.default_rng(1)
    A = 0.3 * (rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N)))
    phi_a = rng.standard_normal((N, na)) + 1j * rng.standard_normal((N, na))
    phi_b = rng.standard_normal((N, nb)) + 1j * rng.standard_normal((N, nb))
    Amb = one_body_operator_matrix(A, N, na, nb)
    lhs = scipy.linalg.expm(Amb) @ determinant_vector(phi_a, phi_b, N)
    B = prop.expm_general(A)
    rhs = determinant_vector(B @ phi_a, B @ phi_b, N)
    assert np.max(np.abs(lhs - rhs)) <= 1e-12 * np.max(np.abs(lhs))
    assert np.max(np.abs(B - scipy.linalg.expm(A))) <= 1e-13


def _eq4_error(h, chol, dt, vec, N, na, nb, shift=True, npts=24):
    """|| sum_k w_k |B(dt, x_k) phi>  -  exp(-dt H) |phi> ||  in the determinant space (Gauss-Hermite over p(x))."""
    Hmb = hamiltonian_matrix(h, chol, N, na, nb)
    exact = scipy.linalg.expm(-dt * Hmb) @ determinant_vector(*vec, N)
    xs, ws = gauss_hermite_normal(npts, chol.shape[0])
    h_used = h if shift else h + 0.5 * np.einsum("gpr,grq->pq", chol, chol)     # cancels the oracle's shift
    acc = np.zeros_like(exact)
    for x, w in zip(xs, ws):
        B = prop.hs_propagator_matrix(h_used, chol, dt, x)
        acc += w * determinant_vector(B @ vec[0], B @ vec[1], N)
    return np.linalg.norm(acc - exact) / np.linalg.norm(exact)


def test_eq4_hubbard_stratonovich_reproduces_exp_minus_dt_h_to_second_order():
    """PAPER.md:74-79 (Eq. 4): int dx p(x) B(x) = exp(-dt H) + O(dt^2).  H is the brute-force many-body matrix of
    Eq. 2 (normal ordered, no shift).  The error must fall ~4x when dt halves; with the -1/2 sum L^2 one-body shift
    left out it is O(dt) (falls ~2x) and much larger: the pin fixes the shift, the i sqrt(dt) factor, the symmetric
    split and that both spins are propagated by the same matrix."""
    N, na, nb = 4, 2, 1
    h, chol, pa, pb, fa, fb = small_system(11)
    e1 = _eq4_error(h, chol, 0.04, (fa, fb), N, na, nb)
    e2 = _eq4_error(h, chol, 0.02, (fa, fb), N, na, nb)
    e3 = _eq4_error(h, chol, 0.01, (fa, fb), N, na, nb)
    assert e1 < 5e-3 and 3.3 < e1 / e2 < 4.7 and 3.5 < e2 / e3 < 4.5, (e1, e2, e3)
    b1 = _eq4_error(h, chol, 0.02, (fa, fb), N, na, nb, shift=False)
    b2 = _eq4_error(h, chol, 0.01, (fa, fb), N, na, nb, shift=False)
    assert b2 > 20 * e3 and 1.7 < b1 / b2 < 2.3, (b1, b2)


def test_zero_field_is_the_one_body_propagator_and_zero_one_body_part_inverts():
    h, chol, pa, pb, fa, fb = small_system(12, N=6, na=3, nb=2, ng=3)
    dt = 0.05
    hp = h - 0.5 * sum(L @ L for L in chol)
    assert np.max(np.abs(prop.one_body_shift(h, chol) - hp)) <= 1e-14
    B0 = prop.hs_propagator_matrix(h, chol, dt, np.zeros(3))
    assert np.max(np.abs(B0 - scipy.linalg.expm(-dt * hp))) <= 1e-13 * np.max(np.abs(B0))
    y = np.array([0.3 - 0.2j, -1.1 + 0.4j, 0.5 + 0.0j])
    h0 = 0.5 * sum(L @ L for L in chol)                     # makes h' = 0: B is the pure Hubbard-Stratonovich factor
    Bp, Bm = prop.hs_propagator_matrix(h0, chol, dt, y), prop.hs_propagator_matrix(h0, chol, dt, -y)
    assert np.max(np.abs(Bp @ Bm - np.eye(6))) <= 1e-13
    assert np.max(np.abs(Bp - scipy.linalg.expm(1j * math.sqrt(dt) * np.einsum("g,gpq->pq", y, chol)))) <= 1e-13


def test_shift_invariance_of_the_importance_sampled_integral():
    """Eq. 6-7: int dx p(x) exp(x.xbar - xbar.xbar/2) B(x - xbar) = int dx p(x) B(x) for ANY (complex) xbar: the
    exponent of the importance function and the argument of B belong together."""
    N, na, nb = 4, 1, 1
    h, chol, pa, pb, fa, fb = small_system(13, N=N, na=na, nb=nb, ng=2, scale=0.5)
    dt = 0.05
    xs, ws = gauss_hermite_normal(40, 2)
    xbar = np.array([0.21 - 0.13j, -0.08 + 0.17j])
    plain = np.zeros((N, N), dtype=complex)
    shifted = np.zeros((N, N), dtype=complex)
    for x, w in zip(xs, ws):
        plain += w * prop.hs_propagator_matrix(h, chol, dt, x)
        shifted += w * np.exp(np.sum(x * xbar) - 0.5 * np.sum(xbar * xbar)) * prop.hs_propagator_matrix(h, chol, dt, x - xbar)
    assert np.max(np.abs(plain - shifted)) <= 1e-10 * np.max(np.abs(plain))


def test_force_bias_shift_makes_the_importance_function_stationary():
    """Eq. 9 is the "optimal" force bias: with xbar = -sqrt(dt) <v'>, v' = i v, the x-gradient of
    log I = x.xbar - xbar.xbar/2 + log O(x - xbar) at x = 0 vanishes to leading order, i.e. it is O(dt) while each of
    its two parts is O(sqrt(dt)).  A wrong sign, a missing i or a missing sqrt(dt) leaves an O(sqrt(dt)) gradient."""
    h, chol, pa, pb, fa, fb = small_system(14, N=6, na=3, nb=2, ng=3)

    def grad_log_I(dt, xbar):
        def log_o(x):
            B = prop.hs_propagator_matrix(h, chol, dt, x - xbar)
            la, aa = orc.log_overlap(pa, pb, B @ fa, B @ fb)
            return complex(la, aa)
        g = np.zeros(3, dtype=complex)
        for k in range(3):
            e = np.zeros(3)
            e[k] = 1e-5
            g[k] = (log_o(e) - log_o(-e)) / 2e-5 + xbar[k]
        return g
    for dt in (0.01, 0.0025):
        xbar = prop.force_bias_shift(chol, pa, pb, fa, fb, dt)
        good = np.linalg.norm(grad_log_I(dt, xbar))
        assert good < 12 * dt and good < 0.12 * np.linalg.norm(xbar), (dt, good, np.linalg.norm(xbar))
        for wrong in (-xbar, xbar.conj(), 1j * xbar):
            assert np.linalg.norm(grad_log_I(dt, wrong)) > 5 * good


def test_one_step_against_brute_force_overlaps_and_the_paper_formulas():
    """propagate_walker: phi' = B(x - xbar) phi (Eq. 13); the overlap ratio (Eq. 8) against <psi|phi'>/<psi|phi> from
    the determinant expansions (Cauchy-Binet, no overlap matrix); the weight from Eq. 7, 10-12 typed out here."""
    N, na, nb = 5, 2, 2
    h, chol, pa, pb, fa, fb = small_system(15, N=N, na=na, nb=nb, ng=3)
    dt, w0 = 0.02, 1.7
    x = np.array([0.4, -1.2, 0.7])
    out = prop.propagate_walker(h, chol, pa, pb, fa, fb, w0, x, dt)
    xbar = -1j * math.sqrt(dt) * np.einsum("gpq,pq->g", chol, orc.greens_function(pa, fa)[0] + orc.greens_function(pb, fb)[0])
    assert np.max(np.abs(out["xbar"] - xbar)) <= 1e-14
    B = prop.hs_propagator_matrix(h, chol, dt, x - xbar)
    assert np.max(np.abs(out["phi_a"] - B @ fa)) <= 1e-14 and np.max(np.abs(out["phi_b"] - B @ fb)) <= 1e-14
    c_psi = determinant_vector(pa, pb, N)
    ratio = np.vdot(c_psi, determinant_vector(out["phi_a"], out["phi_b"], N)) / np.vdot(c_psi, determinant_vector(fa, fb, N))
    assert abs(np.exp(out["log_ovlp_new"] - out["log_ovlp_old"]) - ratio) <= 1e-12 * abs(ratio)
    imp = ratio * np.exp(np.sum(x * xbar) - 0.5 * np.sum(xbar * xbar))
    assert abs(out["weight"] - abs(imp) * max(0.0, math.cos(np.angle(ratio))) * w0) <= 1e-12 * out["weight"]
    assert out["weight"] > 0
