"""Brute-force second-quantised evaluation of <psi|H|phi>/<psi|phi> over the full determinant space.

A pin for the oracle that shares nothing with it: no Green's function, no Wick's theorem, no overlap
matrix.  Both Slater determinants are expanded in occupation-number bitstrings (coefficients are minors),
the Hamiltonian of PAPER.md:68 (Eq. 2),

    H = sum_pq h_pq a+_p a_q + 1/2 sum_pqrs (pr|qs) a+_p a+_q a_s a_r ,   (pr|qs) = sum_g L^g_pr L^g_qs  (Eq. 3)

is applied operator by operator to every bitstring with explicit fermionic signs, and the local energy
is E0 + <psi|H|phi>/<psi|phi> (Eq. 26).  Spin-orbital index = p for alpha, N + p for beta; a determinant
|I> = prod_{P in I ascending} a+_P |0>, so a_P |I> carries (-1)^(number of occupied Q < P).
"""
from itertools import combinations

import numpy as np


def _minor_expansion(phi_a, phi_b, N):
    """bitstrings [D] (int64) and coefficients [D] of |phi> = prod_j phi+_aj prod_k phi+_bk |0>."""
    na, nb = phi_a.shape[1], phi_b.shape[1]
    bits, coef = [], []
    combos_a = list(combinations(range(N), na))
    combos_b = list(combinations(range(N), nb))
    det_a = [np.linalg.det(phi_a[list(I), :]) if na else 1.0 for I in combos_a]
    det_b = [np.linalg.det(phi_b[list(I), :]) if nb else 1.0 for I in combos_b]
    for Ia, da in zip(combos_a, det_a):
        ba = sum(1 << p for p in Ia)
        for Ib, db in zip(combos_b, det_b):
            bb = sum(1 << (N + p) for p in Ib)
            bits.append(ba | bb)
            coef.append(da * db)
    return np.array(bits, dtype=np.int64), np.array(coef, dtype=np.complex128)


def _annihilate(bits, amp, P):
    occ = ((bits >> P) & 1) == 1
    bits, amp = bits[occ], amp[occ]
    sign = 1 - 2 * (np.bitwise_count(bits & ((1 << P) - 1)).astype(np.int64) & 1)
    return bits ^ (1 << P), amp * sign


def _create(bits, amp, P):
    emp = ((bits >> P) & 1) == 0
    bits, amp = bits[emp], amp[emp]
    sign = 1 - 2 * (np.bitwise_count(bits & ((1 << P) - 1)).astype(np.int64) & 1)
    return bits | (1 << P), amp * sign


def brute_force_local_energy(h1e, chol, e0, psi_a, psi_b, phi_a, phi_b):
    """Returns (E, overlap) with overlap = <psi|phi> as a plain complex number."""
    N = h1e.shape[0]
    V = np.einsum("gpr,gqs->prqs", chol, chol)
    bits_phi, c_phi = _minor_expansion(phi_a, phi_b, N)
    bits_psi, c_psi = _minor_expansion(psi_a, psi_b, N)
    lookup = np.full(1 << (2 * N), -1, dtype=np.int64)
    lookup[bits_psi] = np.arange(len(bits_psi))
    bra = np.zeros(len(bits_psi), dtype=np.complex128)   # accumulates (H|phi>)_I in the psi ordering
    # overlap: <psi|phi> = sum_I conj(c_I(psi)) c_I(phi)   (Cauchy-Binet)
    pos = lookup[bits_phi]
    phi_vec = np.zeros(len(bits_psi), dtype=np.complex128)
    phi_vec[pos] = c_phi
    ovlp = np.sum(np.conj(c_psi) * phi_vec)

    def scatter(b, a):
        if len(b):
            np.add.at(bra, lookup[b], a)

    offs = (0, N)
    # one-body
    for so in offs:
        for q in range(N):
            b1, a1 = _annihilate(bits_phi, c_phi, so + q)
            for p in range(N):
                if h1e[p, q] == 0:
                    continue
                b2, a2 = _create(b1, a1, so + p)
                scatter(b2, h1e[p, q] * a2)
    # two-body: 1/2 sum (pr|qs) a+_{p,s1} a+_{q,s2} a_{s,s2} a_{r,s1}
    for s1 in offs:
        for r in range(N):
            b1, a1 = _annihilate(bits_phi, c_phi, s1 + r)
            for s2 in offs:
                for s in range(N):
                    b2, a2 = _annihilate(b1, a1, s2 + s)
                    if len(b2) == 0:
                        continue
                    for q in range(N):
                        b3, a3 = _create(b2, a2, s2 + q)
                        if len(b3) == 0:
                            continue
                        for p in range(N):
                            b4, a4 = _create(b3, a3, s1 + p)
                            scatter(b4, 0.5 * V[p, r, q, s] * a4)
    num = np.sum(np.conj(c_psi) * bra)
    return e0 + num / ovlp, ovlp


def hartree_fock_energy_mo(h1e, chol, e0, psi_a, psi_b):
    """Textbook closed-shell/open-shell HF energy of the determinant |psi> in its own orbital basis:

        E = E0 + sum_i h_ii + 1/2 sum_ij [ (ii|jj) - (ij|ji) ]      i, j over occupied SPIN orbitals,

    (Slater-Condon rule for a diagonal element, chemists' notation), with MO integrals
    h_ij = sum_pq conj(psi_pi) h_pq psi_qj and (ij|kl) = sum_g Lmo^g_ij Lmo^g_kl,
    Lmo^g_ij = sum_pq conj(psi_pi) L^g_pq psi_qj.  The exchange term only couples equal spins.
    """
    e = complex(e0)
    Lmo = []
    for psi in (psi_a, psi_b):
        hmo = psi.conj().T @ h1e @ psi
        e += np.trace(hmo)
        Lmo.append(np.einsum("pi,gpq,qj->gij", psi.conj(), chol, psi))
    tr = sum(np.einsum("gii->g", L) for L in Lmo)
    e += 0.5 * np.sum(tr * tr)                                   # 1/2 sum_ij (ii|jj), all spin pairs
    for L in Lmo:
        e -= 0.5 * np.einsum("gij,gji->", L, L)                  # 1/2 sum_ij (ij|ji), equal spins
    return e


def brute_force_spin_squared(psi_a, psi_b, phi_a, phi_b):
    """<psi|S^2|phi>/<psi|phi> with S^2 = S_- S_+ + S_z (S_z + 1), S_+ = sum_p a+_{p,up} a_{p,dn}, applied operator by
    operator to the determinant expansion of |phi> (no Green's function, no Wick's theorem).  alpha = up."""
    N = psi_a.shape[0]
    bits_phi, c_phi = _minor_expansion(phi_a, phi_b, N)
    bits_psi, c_psi = _minor_expansion(psi_a, psi_b, N)
    lookup = np.full(1 << (2 * N), -1, dtype=np.int64)
    lookup[bits_psi] = np.arange(len(bits_psi))
    phi_vec = np.zeros(len(bits_psi), dtype=np.complex128)
    phi_vec[lookup[bits_phi]] = c_phi
    ovlp = np.sum(np.conj(c_psi) * phi_vec)
    bra = np.zeros(len(bits_psi), dtype=np.complex128)
    for q in range(N):                      # S_+ = sum_q a+_{q,up} a_{q,dn}
        b1, a1 = _annihilate(bits_phi, c_phi, N + q)
        b2, a2 = _create(b1, a1, q)
        for p in range(N):                  # S_- = sum_p a+_{p,dn} a_{p,up}
            b3, a3 = _annihilate(b2, a2, p)
            b4, a4 = _create(b3, a3, N + p)
            if len(b4):
                np.add.at(bra, lookup[b4], a4)
    ms = 0.5 * (psi_a.shape[1] - psi_b.shape[1])
    return np.sum(np.conj(c_psi) * bra) / ovlp + ms * (ms + 1.0)


def brute_force_greens_function(psi_a, psi_b, phi_a, phi_b, spin):
    """G_pq = <psi|a+_{p,spin} a_{q,spin}|phi>/<psi|phi> (Eq. 20) by operator application on the
    determinant expansion; spin 0 = alpha, 1 = beta.  Fixes the index ORDER of the Green's function, which the energy
    (symmetric h and L) cannot see."""
    N = psi_a.shape[0]
    bits_phi, c_phi = _minor_expansion(phi_a, phi_b, N)
    bits_psi, c_psi = _minor_expansion(psi_a, psi_b, N)
    lookup = np.full(1 << (2 * N), -1, dtype=np.int64)
    lookup[bits_psi] = np.arange(len(bits_psi))
    phi_vec = np.zeros(len(bits_psi), dtype=np.complex128)
    phi_vec[lookup[bits_phi]] = c_phi
    ovlp = np.sum(np.conj(c_psi) * phi_vec)
    off = spin * N
    G = np.zeros((N, N), dtype=np.complex128)
    for q in range(N):
        b1, a1 = _annihilate(bits_phi, c_phi, off + q)
        for p in range(N):
            b2, a2 = _create(b1, a1, off + p)
            if len(b2):
                G[p, q] = np.sum(np.conj(c_psi[lookup[b2]]) * a2) / ovlp
    return G


# ---- dense many-body matrices in the (n_alpha, n_beta) determinant space (tiny systems only) -----------------------
def determinant_basis(N, na, nb):
    """Bitstrings of the basis determinants, in the order _minor_expansion produces them."""
    bits = []
    for Ia in combinations(range(N), na):
        ba = sum(1 << p for p in Ia)
        for Ib in combinations(range(N), nb):
            bits.append(ba | sum(1 << (N + p) for p in Ib))
    return np.array(bits, dtype=np.int64)


def determinant_vector(phi_a, phi_b, N):
    """Coefficients of |phi> = prod_j phi+_aj prod_k phi+_bk |0> in determinant_basis order (minors)."""
    return _minor_expansion(phi_a, phi_b, N)[1]


def _operator_matrix(apply, N, na, nb):
    basis = determinant_basis(N, na, nb)
    lookup = np.full(1 << (2 * N), -1, dtype=np.int64)
    lookup[basis] = np.arange(len(basis))
    M = np.zeros((len(basis), len(basis)), dtype=np.complex128)
    for col, b in enumerate(basis):
        for bits, amp in apply(np.array([b], dtype=np.int64), np.array([1.0 + 0j])):
            if len(bits):
                np.add.at(M[:, col], lookup[bits], amp)
    return M


def one_body_operator_matrix(A, N, na, nb):
    """Matrix of sum_{pq,spin} A_pq a+_{p,spin} a_{q,spin} (the same A for both spins) by operator application."""
    A = np.asarray(A)

    def apply(bits, amp):
        for so in (0, N):
            for q in range(N):
                b1, a1 = _annihilate(bits, amp, so + q)
                for p in range(N):
                    if A[p, q] != 0:
                        b2, a2 = _create(b1, a1, so + p)
                        yield b2, A[p, q] * a2
    return _operator_matrix(apply, N, na, nb)


def hamiltonian_matrix(h1e, chol, N, na, nb):
    """Matrix of H of PAPER.md:68 (Eq. 2) with (pr|qs) of Eq. 3, term by term, exactly as brute_force_local_energy
    applies it (normal-ordered two-body operator a+_p a+_q a_s a_r, no one-body shift)."""
    V = np.einsum("gpr,gqs->prqs", chol, chol)

    def apply(bits, amp):
        for so in (0, N):
            for q in range(N):
                b1, a1 = _annihilate(bits, amp, so + q)
                for p in range(N):
                    b2, a2 = _create(b1, a1, so + p)
                    yield b2, h1e[p, q] * a2
        for s1 in (0, N):
            for r in range(N):
                b1, a1 = _annihilate(bits, amp, s1 + r)
                for s2 in (0, N):
                    for s in range(N):
                        b2, a2 = _annihilate(b1, a1, s2 + s)
                        if len(b2) == 0:
                            continue
                        for q in range(N):
                            b3, a3 = _create(b2, a2, s2 + q)
                            if len(b3) == 0:
                                continue
                            for p in range(N):
                                b4, a4 = _create(b3, a3, s1 + p)
                                yield b4, 0.5 * V[p, r, q, s] * a4
    return _operator_matrix(apply, N, na, nb)
