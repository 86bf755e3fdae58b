"""The paper's own CPU algorithm for the local energy (half-rotated, "direct"), restated in numpy.

TEST / BASELINE INFRASTRUCTURE ONLY, like ``afqmc_oracle.py`` (only ``tests/`` and the CPU-baseline legs of
``bench.py`` import it; it shares no code with ``paper_2209_04015_b200/``).  It is NOT the parity oracle: it has
the same algebraic structure as the GPU path (half-rotated Cholesky vectors, theta, T), so it serves as a third
opinion and as the fair "same algorithm on the host cores" timing that SURVEY.md 8(d) calls baseline B, next to the
N^4 definition oracle.  It is pinned by agreeing with the definition oracle walker by walker
(tests/test_oracle_pins.py::test_listing4_agrees_with_definition).

Steps, in the paper's order and notation (rchol = half-rotated Cholesky vectors, theta = half-rotated Green's function):
  rchol^gamma = psi^dagger L^gamma          (naux, nocc * nbasis), built once      PAPER.md:179-183 (Eq. 21)
  S = psi^dagger phi, theta = (phi S^-1)^T                                          PAPER.md:199-204 (Listing 2), Eq. 23
  e1 = sum htilde * theta
  xbar^gamma = rchol . theta.ravel()       (the Coulomb traces / force bias)        PAPER.md:195 (Eq. 24)
  per walker: theta_r, theta_i = contiguous copies of theta.T real / imag;
  per gamma:  T = rchol[gamma] . theta_r + 1j * rchol[gamma] . theta_i ;  exx += dot(T.ravel(), T.T.ravel());  exx *= 0.5
                                                                                    PAPER.md:244-278 (Listing 4, as
                                                                                    reconstructed in DESIGN.md section 3)
  E = E0 + e1 + 1/2 sum_gamma xbar_gamma^2 - exx
The loop over gamma of Listing 4 (a Numba-compiled loop in the paper) is one batched ``numpy.matmul`` here.
"""
from __future__ import annotations

import numpy as np


class HalfRotated:
    """rchol and htilde for one trial (built once, "only needs to be constructed once")."""

    def __init__(self, h1e, chol, psi_a, psi_b):
        self.psi = (psi_a, psi_b)
        self.ht = [p.conj().T @ h1e for p in self.psi]                                  # [n][N]
        self.rchol = [np.matmul(p.conj().T[None, :, :], chol) for p in self.psi]       # [naux][n][N]
        self.real = [bool(np.all(p.imag == 0.0)) for p in self.psi]
        for s in range(2):
            if self.real[s]:                                                            # "a real-valued array rchol"
                self.rchol[s] = np.ascontiguousarray(self.rchol[s].real)


def local_energy_listing4(hr: HalfRotated, e0, phi_a, phi_b):
    """(E, log-overlap) of one walker with the paper's half-rotated direct algorithm."""
    e1 = 0.0 + 0.0j
    exx = 0.0 + 0.0j
    logabs, arg = 0.0, 0.0
    naux = hr.rchol[0].shape[0]
    xbar = np.zeros(naux, dtype=np.complex128)
    for s, phi in enumerate((phi_a, phi_b)):
        n = phi.shape[1]
        if n == 0:
            continue
        S = hr.psi[s].conj().T @ phi
        sign, la = np.linalg.slogdet(S)
        logabs += la
        arg += np.angle(sign)
        theta = (phi @ np.linalg.inv(S)).T                                              # [n][N]
        e1 += np.sum(hr.ht[s] * theta)
        rchol = hr.rchol[s]
        xbar += rchol.reshape(naux, -1) @ theta.ravel()
        if hr.real[s]:
            theta_r = np.ascontiguousarray(theta.T.real)                                # Listing 4 lines 13-14
            theta_i = np.ascontiguousarray(theta.T.imag)
            T = rchol @ theta_r + 1.0j * (rchol @ theta_i)                              # [naux][n][n]
        else:
            T = rchol @ theta.T
        exx += np.einsum("gij,gji->", T, T)
    exx *= 0.5
    E = e0 + e1 + 0.5 * np.sum(xbar * xbar) - exx
    arg = (arg + np.pi) % (2.0 * np.pi) - np.pi
    if arg == -np.pi:
        arg = np.pi
    return E, complex(logabs, arg)
