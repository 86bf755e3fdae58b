"""CPU ORACLE for one step of the hybrid phaseless propagation (Eq. 4; Eq. 6-13).

TEST INFRASTRUCTURE ONLY, like ``afqmc_oracle.py``: only ``tests/``, ``__graft_entry__.smoke()`` and the CPU-baseline
legs of ``bench.py`` may import it; it shares no code with ``paper_2209_04015_b200/``.

The paper states the propagator only through Eq. 4, ``exp(-dt H) = int dx p(x) B(x) + O(dt^2)`` with p the normal
distribution and B "a one-body propagator coupled to a vector of N_aux auxiliary fields"; it does not write B out.
The reading taken here (rows 17-19) is the standard one that Eq. 2, 3, 4 and 9 force:

  * Eq. 2 is normal ordered.  With v_g = sum_pr L^g_pr a+_p a_r (Eq. 3's vectors as one-body operators),
        1/2 sum_g v_g^2 = 1/2 sum_pqrs (pr|qs) a+_p a+_q a_s a_r + 1/2 sum_pq [sum_g (L^g L^g)_pq] a+_p a_q ,
    so  H = sum_pq h'_pq a+_p a_q + 1/2 sum_g v_g^2   with   h' = h - 1/2 sum_g (L^g)^2            (one_body_shift)
  * Hubbard-Stratonovich with p(x) the standard normal:  exp(-dt v^2 / 2) = int dx p(x) exp(i sqrt(dt) x v), and a
    symmetric Trotter split of the one-body part:
        B(dt, y) = exp(-dt h'/2) exp(i sqrt(dt) sum_g y_g L^g) exp(-dt h'/2)                      (hs_propagator_matrix)
    acting on a determinant by multiplying its coefficient matrix (both spins alike).  No mean-field shift.
  * Eq. 9's operator v' is the one that multiplies sqrt(dt) x in the exponent, v'_g = i v_g, hence
        xbar_g = -sqrt(dt) <v'_g> = -i sqrt(dt) sum_pq G_pq L^g_pq = -i sqrt(dt) * (Eq. 19's force bias).   (force_bias_shift)
All matrix exponentials are evaluated to convergence (the product path truncates its Taylor series at a caller-chosen
order; the truncation error is the caller's to bound, see include/afqmc.h).  float64 / complex128 throughout.

What pins it (tests/test_propagation_pins.py): Eq. 4 itself, in the full determinant space of a small system (Gauss-
Hermite quadrature of p(x) B(x) against exp(-dt H) with H the brute-force many-body matrix of Eq. 2: error O(dt^2),
falling 4x when dt halves, and only O(dt) if the -1/2 sum L^2 shift is left out); Thouless' theorem against the
many-body exponential of the one-body operator; y = 0 and h' = 0 closed forms; the shift invariance that Eq. 6-7
express; the stationarity that makes Eq. 9's xbar "optimal"; and Eq. 8 against brute-force overlaps.
"""
from __future__ import annotations

import math

import numpy as np

from . import afqmc_oracle as orc


def one_body_shift(h1e: np.ndarray, chol: np.ndarray) -> np.ndarray:
    """h' = h - 1/2 sum_g L^g L^g : the one-body operator left over when Eq. 2's normal-ordered two-body term is
    written as 1/2 sum_g v_g^2 (header)."""
    return h1e - 0.5 * np.einsum("gpr,grq->pq", chol, chol)


def expm_symmetric(A: np.ndarray) -> np.ndarray:
    """exp(A) of a real symmetric matrix by eigendecomposition (a library step: numpy.linalg.eigh)."""
    w, U = np.linalg.eigh(A)
    return (U * np.exp(w)[None, :]) @ U.T


def expm_general(A: np.ndarray) -> np.ndarray:
    """exp(A) of a general complex matrix: scaling and squaring around a Taylor series summed to convergence."""
    A = np.asarray(A, dtype=np.complex128)
    n = A.shape[0]
    nrm = np.linalg.norm(A, 1)
    s = max(0, int(math.ceil(math.log2(nrm))) + 1) if nrm > 0.5 else 0
    X = A / (2.0 ** s)
    term = np.eye(n, dtype=np.complex128)
    out = term.copy()
    for k in range(1, 64):
        term = term @ X / k
        out = out + term
        if np.linalg.norm(term, 1) <= 1e-18 * np.linalg.norm(out, 1):
            break
    for _ in range(s):
        out = out @ out
    return out


def hs_potential(chol: np.ndarray, dt: float, y: np.ndarray) -> np.ndarray:
    """A(y) = i sqrt(dt) sum_g y_g L^g  (N x N, complex symmetric): the exponent of the two-body factor of B."""
    return 1j * math.sqrt(dt) * np.einsum("g,gpq->pq", np.asarray(y, dtype=np.complex128), chol)


def hs_propagator_matrix(h1e, chol, dt: float, y) -> np.ndarray:
    """B(dt, y) = exp(-dt h'/2) exp(i sqrt(dt) sum_g y_g L^g) exp(-dt h'/2) as an N x N matrix (header)."""
    E = expm_symmetric(-0.5 * dt * one_body_shift(h1e, chol))
    return E @ expm_general(hs_potential(chol, dt, y)) @ E


def force_bias_shift(chol, psi_a, psi_b, phi_a, phi_b, dt: float) -> np.ndarray:
    """xbar_g = -sqrt(dt) <v'_g> with v'_g = i v_g  (Eq. 9)  = -i sqrt(dt) sum_pq G_pq L^g_pq."""
    return -1j * math.sqrt(dt) * orc.force_bias(chol, psi_a, psi_b, phi_a, phi_b)


def propagate_walker(h1e, chol, psi_a, psi_b, phi_a, phi_b, weight: float, x, dt: float):
    """One hybrid phaseless step of one walker, PAPER.md:96-123 in the paper's order:
        xbar            Eq. 9                              (force_bias_shift)
        phi'  = B(dt, x - xbar) phi     both spins         Eq. 13
        O     = <psi|phi'> / <psi|phi>                     Eq. 8
        I     = O exp(x . xbar - xbar . xbar / 2)          Eq. 7
        w'    = |I| max(0, cos(arg O)) w                   Eq. 10-12
    x: the real auxiliary-field vector drawn by the caller (Eq. 4's p(x)).  Returns dict(phi_a, phi_b, weight, xbar,
    log_ovlp_old, log_ovlp_new) with log-overlaps as complex (log|ovlp|, arg)."""
    x = np.asarray(x, dtype=np.float64)
    xbar = force_bias_shift(chol, psi_a, psi_b, phi_a, phi_b, dt)
    B = hs_propagator_matrix(h1e, chol, dt, x - xbar)
    new_a, new_b = B @ phi_a, B @ phi_b
    lo_old = complex(*orc.log_overlap(psi_a, psi_b, phi_a, phi_b))
    lo_new = complex(*orc.log_overlap(psi_a, psi_b, new_a, new_b))
    w_new = orc.phaseless_weight_update(weight, lo_old, lo_new, x, xbar)
    return dict(phi_a=new_a, phi_b=new_b, weight=w_new, xbar=xbar, log_ovlp_old=lo_old, log_ovlp_new=lo_new)
