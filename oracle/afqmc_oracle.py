"""CPU ORACLE for the ph-AFQMC local energy with a single-determinant trial.

TEST INFRASTRUCTURE ONLY.  Only ``tests/``, ``__graft_entry__.smoke()`` and the ``cpu_baseline`` /
``--impl reference`` legs of ``bench.py`` may import this module.  It shares no code, header, table
or helper with the CUDA path (``paper_2209_04015_b200/``) and neither imports the other; the only
common ground is the seeded input generator ``gen/``, which holds none of the method's arithmetic.

What it computes is the *plain definition* the paper's method re-associates exactly (half-rotation,
Eq. 21, and the "direct algorithm", are exact rewrites, not approximations), so none of
the GPU path's intermediates (half-rotated L, theta, T) appear here:

  overlap      <psi_T|phi> = prod_sigma det(psi_sigma^dagger phi_sigma)          PAPER.md:143 (Eq. 16)
  Green's fn   G^sigma_pq  = [phi (psi^dagger phi)^-1 psi^dagger]_qp   (N x N)   PAPER.md:174,187 (Eq. 20, 22)
  ERIs         V_prqs = (pr|qs) = sum_gamma L^gamma_pr L^gamma_qs               PAPER.md:72  (Eq. 3)
  local energy E = <psi_T|H|phi>/<psi_T|phi>                                     PAPER.md:224 (Eq. 26)
     with H of PAPER.md:68 (Eq. 2) and Wick's theorem for two non-orthogonal determinants,
     <a+_p,s a+_q,t a_s,t a_r,s> = G^s_pr G^t_qs - delta_st G^s_ps G^s_qr :
     E = E0 + sum_s sum_pq h_pq G^s_pq
            + 1/2 sum_prqs V_prqs [ Gtot_pr Gtot_qs - sum_s G^s_ps G^s_qr ],   Gtot = G^alpha + G^beta.

Precision: float64 / complex128 throughout (numpy).  Library primitives used as steps: ``numpy.matmul``
/ ``einsum`` / ``tensordot`` contractions.  The LU, determinant and inverse are written out below.

Three rungs, by memory only (same arithmetic, different bookkeeping):
  O1 ``local_energy_full_eri``      V stored [N][N][N][N]           tiny, small   (the literal definition)
  O2 ``local_energy_streamed_eri``  V generated one p-slab at a time medium, cu2o2 (V is 57 GB at N=290)
  O3 ``local_energy_cholesky``      Eq. 3 substituted, no V, full G, un-rotated L   large (V would be 500 GB)
O2 and O3 are pinned to O1 walker by walker in tests/test_oracle_pins.py; O1 is pinned by the closed-form
Hartree-Fock energy, phi -> phi C invariance, brute-force operator application over the full determinant
space, identity-Cholesky closed form, and symmetry checks.  Nothing here is "parity unpinned".

Readings of the paper where it is silent or garbled: E0 is an additive constant absent from
Eq. 2; h1e is used as given (Eq. 2 is already in a+a+aa order, no -1/2 sum (pr|rq) shift); the log-overlap
is reported as (sum_s log|det S_s|, arg prod_s det S_s in (-pi, pi]); pivot ties go to the lowest row.
"""
from __future__ import annotations

import math

import numpy as np


# ----------------------------------------------------------------------------------------------
# overlap matrix, LU with partial pivoting, determinant, inverse           (Eq. 16)
# ----------------------------------------------------------------------------------------------
def overlap_matrix(psi: np.ndarray, phi: np.ndarray) -> np.ndarray:
    """S = psi^dagger phi  (n x n).  PAPER.md:143, Eq. 16 (first form)."""
    return psi.conj().T @ phi


def lu_partial_pivot(S: np.ndarray):
    """Gaussian elimination with partial pivoting, P S = L U, written out row by row.

    Returns (LU, perm, nswaps): LU holds the unit-lower L below the diagonal and U on/above it,
    ``perm[k]`` is the original row now in position k.  Pivot = first row of maximal |a_ik|.
    """
    A = np.array(S, dtype=np.complex128, copy=True)
    n = A.shape[0]
    perm = list(range(n))
    nswaps = 0
    for k in range(n):
        piv = k
        best = abs(A[k, k])
        for i in range(k + 1, n):
            v = abs(A[i, k])
            if v > best:
                best, piv = v, i
        if piv != k:
            A[[k, piv], :] = A[[piv, k], :]
            perm[k], perm[piv] = perm[piv], perm[k]
            nswaps += 1
        if A[k, k] == 0:
            continue  # singular: det = 0; caller sees log|det| = -inf
        for i in range(k + 1, n):
            A[i, k] = A[i, k] / A[k, k]
            A[i, k + 1:] -= A[i, k] * A[k, k + 1:]
    return A, perm, nswaps


def logdet_and_inverse(S: np.ndarray):
    """(log|det S|, arg det S in (-pi,pi], S^-1) from the LU above.

    det S = (-1)^nswaps prod_k u_kk; the log is accumulated term by term because the overlaps of the
    synthetic walkers are ~e^-80..e^-160.  S^-1 by forward/back substitution on P.
    """
    n = S.shape[0]
    if n == 0:
        return 0.0, 0.0, np.zeros((0, 0), dtype=np.complex128)
    LU, perm, nswaps = lu_partial_pivot(S)
    logabs = 0.0
    phase = complex(-1.0 if (nswaps & 1) else 1.0)
    singular = False
    for k in range(n):
        u = LU[k, k]
        if u == 0:
            singular = True
            break
        logabs += math.log(abs(u))
        phase *= u / abs(u)
    if singular:
        return -math.inf, 0.0, np.full((n, n), np.nan + 1j * np.nan)
    arg = math.atan2(phase.imag, phase.real)
    # Solve L U X = P  (P = rows of the identity in pivot order)
    X = np.zeros((n, n), dtype=np.complex128)
    for k in range(n):
        X[k, perm[k]] = 1.0
    for k in range(n):                      # forward: unit lower triangular
        for i in range(k + 1, n):
            X[i, :] -= LU[i, k] * X[k, :]
    for k in range(n - 1, -1, -1):          # backward: upper triangular
        X[k, :] = X[k, :] / LU[k, k]
        for i in range(k):
            X[i, :] -= LU[i, k] * X[k, :]
    return logabs, arg, X


def greens_function(psi: np.ndarray, phi: np.ndarray):
    """Full N x N one-body Green's function of one spin sector and the log-overlap of that sector.

    G_pq = <psi|a+_p a_q|phi>/<psi|phi> = [phi (psi^dagger phi)^-1 psi^dagger]_qp   (note the
    transposed subscript ``qp`` in Eq. 22).  Returns (G, log|det S|, arg det S).
    """
    N, n = phi.shape
    if n == 0:
        return np.zeros((N, N), dtype=np.complex128), 0.0, 0.0
    S = overlap_matrix(psi, phi)
    logabs, arg, Sinv = logdet_and_inverse(S)
    G = (phi @ Sinv @ psi.conj().T).T
    return G, logabs, arg


def wrap_angle(a: float) -> float:
    """Wrap to (-pi, pi]."""
    a = math.fmod(a, 2.0 * math.pi)
    if a > math.pi:
        a -= 2.0 * math.pi
    elif a <= -math.pi:
        a += 2.0 * math.pi
    return a


def log_overlap(psi_a, psi_b, phi_a, phi_b):
    """(log|<psi_T|phi>|, arg<psi_T|phi>) with <psi_T|phi> = det S_alpha det S_beta  (Eq. 16, spins explicit)."""
    _, la, aa = greens_function(psi_a, phi_a)
    _, lb, ab = greens_function(psi_b, phi_b)
    return la + lb, wrap_angle(aa + ab)


# ----------------------------------------------------------------------------------------------
# ERIs                                                                          (Eq. 3)
# ----------------------------------------------------------------------------------------------
def eri_from_cholesky(chol: np.ndarray) -> np.ndarray:
    """V[p][r][q][s] = (pr|qs) = sum_gamma L^gamma_pr L^gamma_qs, stored in full."""
    ng, N, _ = chol.shape
    Lm = chol.reshape(ng, N * N)
    return (Lm.T @ Lm).reshape(N, N, N, N)


# ----------------------------------------------------------------------------------------------
# O1: the definition with V stored
# ----------------------------------------------------------------------------------------------
def energy_terms_from_G(h1e, V, Ga, Gb):
    """(E1, E_C, E_X) of Eq. 26 from full Green's functions and stored ERIs V[p][r][q][s]."""
    Gt = Ga + Gb
    e1 = np.sum(h1e * Ga) + np.sum(h1e * Gb)
    ec = 0.5 * np.einsum("prqs,pr,qs->", V, Gt, Gt, optimize=True)
    ex = 0.0
    for G in (Ga, Gb):
        ex += -0.5 * np.einsum("prqs,ps,qr->", V, G, G, optimize=True)
    return complex(e1), complex(ec), complex(ex)


def local_energy_full_eri(h1e, V, e0, psi_a, psi_b, phi_a, phi_b):
    """O1 for one walker.  Returns dict(E, E1, EC, EX, logabs, arg)."""
    Ga, la, aa = greens_function(psi_a, phi_a)
    Gb, lb, ab = greens_function(psi_b, phi_b)
    e1, ec, ex = energy_terms_from_G(h1e, V, Ga, Gb)
    return dict(E=e0 + e1 + ec + ex, E1=e1, EC=ec, EX=ex, logabs=la + lb, arg=wrap_angle(aa + ab))


def local_energy_explicit_loops(h1e, chol, e0, psi_a, psi_b, phi_a, phi_b):
    """O1 with every sum of Eq. 2/3/26 as an explicit Python loop (tiny systems only).

    Exists so that the index strings of the einsum version can be checked by eye against the paper.
    """
    ng, N, _ = chol.shape
    Ga, la, aa = greens_function(psi_a, phi_a)
    Gb, lb, ab = greens_function(psi_b, phi_b)
    V = np.zeros((N, N, N, N))
    for g in range(ng):
        for p in range(N):
            for r in range(N):
                for q in range(N):
                    for s in range(N):
                        V[p, r, q, s] += chol[g, p, r] * chol[g, q, s]
    e1 = 0j
    for p in range(N):
        for q in range(N):
            e1 += h1e[p, q] * (Ga[p, q] + Gb[p, q])
    ec = 0j
    ex = 0j
    for p in range(N):
        for r in range(N):
            for q in range(N):
                for s in range(N):
                    v = V[p, r, q, s]
                    ec += 0.5 * v * (Ga[p, r] + Gb[p, r]) * (Ga[q, s] + Gb[q, s])
                    ex -= 0.5 * v * (Ga[p, s] * Ga[q, r] + Gb[p, s] * Gb[q, r])
    return dict(E=e0 + e1 + ec + ex, E1=e1, EC=ec, EX=ex, logabs=la + lb, arg=wrap_angle(aa + ab))


# ----------------------------------------------------------------------------------------------
# O2: the same definition, V produced one p-slab at a time (never stored in full)
# ----------------------------------------------------------------------------------------------
def local_energy_streamed_eri(h1e, chol, e0, psi_a, psi_b, phis_a, phis_b):
    """O2 for a batch of walkers ``phis_* [nw][N][n]``.  Returns list of dicts as O1.

    For each p the slab V[p][r][q][s] = sum_g L^g_pr L^g_qs (N x N x N) is built from ``chol`` (Eq. 3),
    contracted with every walker's G exactly as in O1, and discarded.
    """
    ng, N, _ = chol.shape
    nw = phis_a.shape[0]
    Ga = np.empty((nw, N, N), dtype=np.complex128)
    Gb = np.empty((nw, N, N), dtype=np.complex128)
    logabs = np.empty(nw)
    arg = np.empty(nw)
    for w in range(nw):
        Ga[w], la, aa = greens_function(psi_a, phis_a[w])
        Gb[w], lb, ab = greens_function(psi_b, phis_b[w])
        logabs[w], arg[w] = la + lb, wrap_angle(aa + ab)
    Gt = Ga + Gb
    e1 = np.array([np.sum(h1e * Gt[w]) for w in range(nw)])
    ec = np.zeros(nw, dtype=np.complex128)
    ex = np.zeros(nw, dtype=np.complex128)
    Lm = chol.reshape(ng, N * N)
    for p in range(N):
        Vp = (chol[:, p, :].T @ Lm).reshape(N, N, N)          # Vp[r][q][s] = V[p][r][q][s]
        # Coulomb: 1/2 sum_r Gt[p][r] sum_qs Vp[r][q][s] Gt[q][s]
        J = np.einsum("rqs,wqs->wr", Vp, Gt, optimize=True)
        ec += 0.5 * np.einsum("wr,wr->w", Gt[:, p, :], J)
        # exchange: -1/2 sum_sigma sum_rqs Vp[r][q][s] G[p][s] G[q][r]
        for G in (Ga, Gb):
            W = np.einsum("rqs,ws->wrq", Vp, G[:, p, :], optimize=True)
            ex += -0.5 * np.einsum("wrq,wqr->w", W, G)
    return [dict(E=e0 + e1[w] + ec[w] + ex[w], E1=complex(e1[w]), EC=complex(ec[w]), EX=complex(ex[w]),
                 logabs=float(logabs[w]), arg=float(arg[w])) for w in range(nw)]


# ----------------------------------------------------------------------------------------------
# O3: Eq. 3 substituted into Eq. 26; full G, un-rotated L, no ERIs
# ----------------------------------------------------------------------------------------------
def local_energy_cholesky(h1e, chol, e0, psi_a, psi_b, phi_a, phi_b, gamma_block: int = 64):
    """O3 for one walker.

    E_C = 1/2 sum_g ( sum_pr L^g_pr Gtot_pr )^2
    E_X = -1/2 sum_g sum_sigma sum_prqs L^g_pr L^g_qs G_ps G_qr = -1/2 sum_g sum_sigma sum_rs A_rs A_sr,
          A = (L^g)^T G   (N x N per gamma).
    ``gamma_block`` only bounds the size of the temporary; every gamma is treated alike.
    """
    ng, N, _ = chol.shape
    Ga, la, aa = greens_function(psi_a, phi_a)
    Gb, lb, ab = greens_function(psi_b, phi_b)
    Gt = Ga + Gb
    e1 = complex(np.sum(h1e * Gt))
    ec = 0j
    ex = 0j
    for g0 in range(0, ng, gamma_block):
        Lb = chol[g0:g0 + gamma_block]                       # [g][p][r]
        tr = np.einsum("gpr,pr->g", Lb, Gt)
        ec += 0.5 * np.sum(tr * tr)
        LbT = Lb.transpose(0, 2, 1)
        for G in (Ga, Gb):
            if not G.any():
                continue
            A = np.matmul(LbT, G.real) + 1j * np.matmul(LbT, G.imag)   # A[g][r][s] = sum_p L_pr G_ps
            ex += -0.5 * np.sum(A * A.transpose(0, 2, 1))
    return dict(E=e0 + e1 + ec + ex, E1=e1, EC=complex(ec), EX=complex(ex), logabs=la + lb,
                arg=wrap_angle(aa + ab))


# ----------------------------------------------------------------------------------------------
# batch front end
# ----------------------------------------------------------------------------------------------
def local_energy_batch(inp, rung: str = "auto", walkers=None, V=None):
    """Energies and log-overlaps for walkers ``walkers`` (indices; default all) of a ``gen.Inputs``.

    Returns (E [k] complex128, logovlp [k] complex128 = log|ovlp| + i arg).  rung in {"O1","O2","O3","auto"};
    "auto" = O1 when the full ERI tensor is below 2 GB, else O3.
    """
    idx = list(range(inp.n_walkers)) if walkers is None else list(walkers)
    if rung == "auto":
        rung = "O1" if inp.N ** 4 * 8 <= 2 << 30 else "O3"
    E = np.empty(len(idx), dtype=np.complex128)
    lo = np.empty(len(idx), dtype=np.complex128)
    if rung == "O1":
        if V is None:
            V = eri_from_cholesky(inp.chol)
        res = [local_energy_full_eri(inp.h1e, V, inp.e0, inp.psi_a, inp.psi_b, inp.phi_a[w], inp.phi_b[w])
               for w in idx]
    elif rung == "O2":
        res = local_energy_streamed_eri(inp.h1e, inp.chol, inp.e0, inp.psi_a, inp.psi_b,
                                        inp.phi_a[idx], inp.phi_b[idx])
    elif rung == "O3":
        res = [local_energy_cholesky(inp.h1e, inp.chol, inp.e0, inp.psi_a, inp.psi_b, inp.phi_a[w], inp.phi_b[w])
               for w in idx]
    else:
        raise ValueError(rung)
    for k, r in enumerate(res):
        E[k] = r["E"]
        lo[k] = complex(r["logabs"], r["arg"])
    return E, lo


# ----------------------------------------------------------------------------------------------
# force bias: xbar^gamma = sum_pq G_pq L^gamma_pq        (Eq. 19)
# ----------------------------------------------------------------------------------------------
def force_bias(chol, psi_a, psi_b, phi_a, phi_b):
    """xbar[gamma] from the full Green's function (no half-rotation), Eq. 19 second line."""
    Ga, _, _ = greens_function(psi_a, phi_a)
    Gb, _, _ = greens_function(psi_b, phi_b)
    return np.einsum("gpq,pq->g", chol, Ga + Gb)


def spin_squared(psi_a, psi_b, phi_a, phi_b):
    """Mixed estimator <psi|S^2|phi>/<psi|phi> = N_dn + M_S (M_S + 1) - sum_pq G^dn_pq G^up_qp from the FULL Green's
    functions (Eq. 31; the transposed index order is Listing 6's ``einsum("zij,zji->z", Ga, Gb)``,
    PAPER.md:426, which is the correct Wick contraction of S_- S_+)."""
    Ga, _, _ = greens_function(psi_a, phi_a)
    Gb, _, _ = greens_function(psi_b, phi_b)
    n_up, n_dn = psi_a.shape[1], psi_b.shape[1]
    ms = 0.5 * (n_up - n_dn)
    return n_dn + ms * (ms + 1.0) - np.einsum("ij,ji->", Ga, Gb)


def phaseless_weight_update(weight, log_ovlp_old, log_ovlp_new, x, xbar):
    """Phaseless weight update of one walker, PAPER.md:100-123 (Eq. 7, 8, 10-12), step by step in the paper's order:
        O      = <Psi_T|B(x - xbar)|phi> / <Psi_T|phi>  = exp(log_ovlp_new - log_ovlp_old)               (Eq. 8)
        I      = O * exp(x . xbar - xbar . xbar / 2)                                                      (Eq. 7)
        theta  = arg O                                                                                    (Eq. 11)
        I_ph   = |I| * max(0, cos theta)                                                                  (Eq. 10)
        w_new  = I_ph * w                                                                                 (Eq. 12)
    log-overlaps are (log|ovlp|, arg ovlp) as returned by the local-energy call for the walker before and after the
    propagator was applied; x is the real auxiliary-field vector, xbar the complex force bias (Eq. 9).  The dot
    products are plain (unconjugated) sums over the auxiliary index."""
    x = np.asarray(x, dtype=np.float64)
    xbar = np.asarray(xbar, dtype=np.complex128)
    log_o = complex(log_ovlp_new) - complex(log_ovlp_old)
    expo = np.sum(x * xbar) - 0.5 * np.sum(xbar * xbar)
    big_i = np.exp(log_o + expo)
    theta = math.atan2(math.sin(log_o.imag), math.cos(log_o.imag))      # arg O in (-pi, pi]
    return abs(big_i) * max(0.0, math.cos(theta)) * weight
