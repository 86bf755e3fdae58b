"""The five synthetic configurations of BASELINE.json and their seeded generators.

Recipe (BASELINE.json ``configs``; restated in DESIGN.md §4):

* ``numpy.random.Generator(PCG64)``; one ``SeedSequence(seed).spawn(6)`` per config gives the
  streams (h1e, chol, trial-alpha, trial-beta, walkers-alpha, walkers-beta); seeds 1001..1005.
* h1e:  A ~ N(0,1)^{N x N} / sqrt(N);  h = (A + A^T)/2 + diag(d).
* chol: for gamma = 0..Ngamma-1:  B ~ N(0,1)^{N x N};  L^gamma = (B + B^T)/2 * exp(-gamma/tau).
* trial: Q factor of QR(N(0,1)^{N x N}) with columns re-phased so diag(R) > 0; psi = Q[:, :n]
  (complex128, zero imaginary part).  RHF-style: psi_beta = psi_alpha[:, :n_beta];
  UHF-style ("medium"): psi_beta from its own stream.
* walkers: phi_{sigma,w} = Q factor (reduced, diag(R) real positive) of psi_sigma + s (X + iY),
  X, Y ~ N(0,1)^{N x n}, independent per walker and per spin, drawn walker by walker so that the
  first k walkers do not depend on how many are requested.
* E0 = 0.5.

The paper measures on molecular integrals that are not available here; these
inputs take only their shapes ((52e,290o) from PAPER.md:13, 542) and a decaying Cholesky spectrum.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

CONFIGS = {
    "tiny": dict(N=10, n_alpha=3, n_beta=3, n_gamma=40, n_walkers=4, tau=10.0, hdiag=("arange",),
                 uhf=False, noise=0.1, seed=1001),
    "small": dict(N=100, n_alpha=20, n_beta=20, n_gamma=500, n_walkers=64, tau=100.0, hdiag=("arange",),
                  uhf=False, noise=0.2, seed=1002),
    "medium": dict(N=200, n_alpha=40, n_beta=40, n_gamma=1000, n_walkers=128, tau=200.0, hdiag=("arange",),
                   uhf=True, noise=0.2, seed=1003),
    "cu2o2": dict(N=290, n_alpha=26, n_beta=26, n_gamma=2000, n_walkers=256, tau=300.0,
                  hdiag=("linspace", 0.0, 50.0), uhf=False, noise=0.3, seed=1004),
    "large": dict(N=500, n_alpha=50, n_beta=50, n_gamma=3000, n_walkers=512, tau=500.0, hdiag=("arange",),
                  uhf=False, noise=0.3, seed=1005),
}
CONFIG_ORDER = ["tiny", "small", "medium", "cu2o2", "large"]
E0 = 0.5


@dataclass
class Inputs:
    name: str
    N: int
    n_alpha: int
    n_beta: int
    n_gamma: int
    e0: float
    h1e: np.ndarray        # [N][N] float64
    chol: np.ndarray       # [Ngamma][N][N] float64
    psi_a: np.ndarray      # [N][n_alpha] complex128
    psi_b: np.ndarray      # [N][n_beta] complex128
    phi_a: np.ndarray      # [Nw][N][n_alpha] complex128
    phi_b: np.ndarray      # [Nw][N][n_beta] complex128

    @property
    def n_walkers(self) -> int:
        return self.phi_a.shape[0]

    def trial_packed(self) -> np.ndarray:
        """ABI layout of the trial: alpha block [N][n_alpha] followed by beta block [N][n_beta]."""
        return np.concatenate([self.psi_a.ravel(), self.psi_b.ravel()])

    def walkers_packed(self, idx=None) -> np.ndarray:
        """ABI layout of the walkers: alpha block [Nw][N][n_alpha] then beta block [Nw][N][n_beta]."""
        pa = self.phi_a if idx is None else self.phi_a[idx]
        pb = self.phi_b if idx is None else self.phi_b[idx]
        return np.concatenate([np.ascontiguousarray(pa).ravel(), np.ascontiguousarray(pb).ravel()])


def _streams(seed: int):
    return [np.random.Generator(np.random.PCG64(s)) for s in np.random.SeedSequence(seed).spawn(6)]


def _qr_positive(a: np.ndarray) -> np.ndarray:
    """Reduced QR; columns re-phased so that diag(R) is real positive."""
    q, r = np.linalg.qr(a)
    d = np.diagonal(r)
    ph = np.where(np.abs(d) > 0, d / np.where(np.abs(d) > 0, np.abs(d), 1.0), 1.0)
    return q * ph[None, :]


def _hdiag(spec, N):
    if spec[0] == "arange":
        return np.arange(N, dtype=np.float64)
    if spec[0] == "linspace":
        return np.linspace(spec[1], spec[2], N)
    raise ValueError(spec)


def make_hamiltonian(cfg: dict, n_gamma: int | None = None):
    """h1e [N][N] and chol [Ngamma][N][N]; ``n_gamma`` < cfg value keeps the first vectors only."""
    N = cfg["N"]
    ng = cfg["n_gamma"] if n_gamma is None else n_gamma
    st = _streams(cfg["seed"])
    a = st[0].standard_normal((N, N)) / np.sqrt(N)
    h1e = 0.5 * (a + a.T) + np.diag(_hdiag(cfg["hdiag"], N))
    chol = np.empty((ng, N, N), dtype=np.float64)
    step = max(1, (1 << 24) // (N * N))
    for g0 in range(0, ng, step):
        g1 = min(ng, g0 + step)
        b = st[1].standard_normal((g1 - g0, N, N))
        dec = np.exp(-np.arange(g0, g1, dtype=np.float64) / cfg["tau"])
        chol[g0:g1] = 0.5 * (b + b.transpose(0, 2, 1)) * dec[:, None, None]
    return h1e, chol


def make_trial(cfg: dict):
    N, na, nb = cfg["N"], cfg["n_alpha"], cfg["n_beta"]
    st = _streams(cfg["seed"])
    qa = _qr_positive(st[2].standard_normal((N, N)))
    psi_a = qa[:, :na].astype(np.complex128)
    if cfg["uhf"]:
        qb = _qr_positive(st[3].standard_normal((N, N)))
        psi_b = qb[:, :nb].astype(np.complex128)
    else:
        psi_b = qa[:, :nb].astype(np.complex128)
    return np.ascontiguousarray(psi_a), np.ascontiguousarray(psi_b)


def make_walkers(cfg: dict, psi_a: np.ndarray, psi_b: np.ndarray, n_walkers: int | None = None):
    N = cfg["N"]
    nw = cfg["n_walkers"] if n_walkers is None else n_walkers
    st = _streams(cfg["seed"])
    out = []
    for rng, psi in ((st[4], psi_a), (st[5], psi_b)):
        n = psi.shape[1]
        phi = np.empty((nw, N, n), dtype=np.complex128)
        for w in range(nw):
            x = rng.standard_normal((N, n))
            y = rng.standard_normal((N, n))
            phi[w] = _qr_positive(psi + cfg["noise"] * (x + 1j * y)) if n > 0 else 0
        out.append(phi)
    return out[0], out[1]


def make_inputs(name: str, n_walkers: int | None = None, n_gamma: int | None = None) -> Inputs:
    cfg = CONFIGS[name]
    h1e, chol = make_hamiltonian(cfg, n_gamma)
    psi_a, psi_b = make_trial(cfg)
    phi_a, phi_b = make_walkers(cfg, psi_a, psi_b, n_walkers)
    return Inputs(name=name, N=cfg["N"], n_alpha=cfg["n_alpha"], n_beta=cfg["n_beta"],
                  n_gamma=chol.shape[0], e0=E0, h1e=h1e, chol=chol, psi_a=psi_a, psi_b=psi_b,
                  phi_a=phi_a, phi_b=phi_b)
