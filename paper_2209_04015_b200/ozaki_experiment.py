"""Ozaki-scheme experiment driver:  python -m paper_2209_04015_b200.ozaki_experiment [--large]

For the exchange contraction T = Ltilde theta^T (Eq. 29) it reports, per number of 7-bit digit planes,
  * the error of T and of the per-walker exchange energy x_w = sum_gamma sum_ij T_ij T_ji against an FP64 evaluation,
    and what that error is relative to the walker's total local energy (the library's own afqmc_local_energy),
  * the measured time of the tcgen05 kind::i8 kernel at the full Cu2O2-scale GEMM shape and its FP64-equivalent TFLOP/s,
and prints one JSON line.  An experiment harness, not the product path: Ltilde, theta and the FP64 reference products are
formed with torch (library GEMMs) because only the INT8 kernel is under test here."""
from __future__ import annotations

import argparse
import json
import os
import sys

import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def half_rotated(inp, spin, walkers, dev):
    """(Ltilde [Ng*n, N], theta columns [(plane, w, j), N]) of one spin for the listed walkers, float64 on `dev`."""
    psi = torch.from_numpy((inp.psi_a if spin == 0 else inp.psi_b).real.copy()).to(dev)          # real trial (all five configs)
    phi = torch.from_numpy((inp.phi_a if spin == 0 else inp.phi_b)[walkers]).to(dev)              # [nw, N, n] complex
    chol = torch.from_numpy(inp.chol).to(dev)
    n = psi.shape[1]
    Lt = torch.matmul(psi.T.unsqueeze(0), chol).reshape(-1, inp.N).contiguous()                     # [(g, i), p]
    S = torch.matmul(psi.T.to(torch.complex128).unsqueeze(0), phi)                                 # psi^T phi (psi real)
    theta = torch.matmul(phi, torch.linalg.inv(S)).transpose(1, 2).contiguous()                    # [nw, n, N]
    B = torch.cat([theta.real.reshape(-1, inp.N), theta.imag.reshape(-1, inp.N)], dim=0).contiguous()   # rows (plane, w, j)
    return Lt, B, n


def exchange_from_T(C, ng, n, nw):
    """x_w = sum_g sum_ij T_ij T_ji from C[(g, i), (plane, w, j)]  (Eq. 28)."""
    T = torch.complex(C[:, : nw * n], C[:, nw * n:]).reshape(ng, n, nw, n)                          # [g, i, w, j]
    return torch.einsum("giwj,gjwi->w", T, T)


def accuracy(name, walkers, slices_list, dev):
    from gen import make_inputs
    from paper_2209_04015_b200 import LocalEnergy
    from paper_2209_04015_b200.ozaki import ozaki_gemm
    inp = make_inputs(name, n_walkers=max(walkers) + 1)
    nw = len(walkers)
    le = LocalEnergy(torch.from_numpy(inp.h1e).to(dev), torch.from_numpy(inp.chol).to(dev),
                     torch.from_numpy(inp.trial_packed()).to(dev), inp.N, inp.n_alpha, inp.n_beta, inp.n_gamma, inp.e0, nw)
    E, _ = le.local_energy(torch.from_numpy(inp.walkers_packed(walkers)).to(dev), nw)
    E = E.clone()
    le.close()
    out = {"config": name, "N": inp.N, "n_gamma": inp.n_gamma, "walkers": list(walkers), "per_slices": {}}
    ref, oz = None, {s: 0 for s in slices_list}
    x_ref = torch.zeros(nw, dtype=torch.complex128, device=dev)
    x_oz = {s: torch.zeros(nw, dtype=torch.complex128, device=dev) for s in slices_list}
    t_err = {s: 0.0 for s in slices_list}
    for spin in (0, 1):
        Lt, B, n = half_rotated(inp, spin, walkers, dev)
        if n == 0:
            continue
        Cref = Lt @ B.T
        x_ref += exchange_from_T(Cref, inp.n_gamma, n, nw)
        tmax = Cref.abs().max().item()
        for s in slices_list:
            C = ozaki_gemm(Lt, B, s)["C"]
            x_oz[s] += exchange_from_T(C, inp.n_gamma, n, nw)
            t_err[s] = max(t_err[s], (C - Cref).abs().max().item() / tmax)
            del C
        del Cref, Lt, B
    for s in slices_list:
        dx = (x_oz[s] - x_ref).abs()
        out["per_slices"][s] = {"T_max_abs_err_over_max_T": t_err[s],
                                "exchange_rel_err_max": (dx / x_ref.abs()).max().item(),
                                "energy_rel_err_max": (0.5 * dx / E.abs()).max().item()}
    return out


def throughput(M, Ncol, K, slices_list, dev, repeats=3):
    from paper_2209_04015_b200.ozaki import ozaki_gemm
    g = torch.Generator(device=dev)
    g.manual_seed(7)
    A = torch.randn((M, K), dtype=torch.float64, device=dev, generator=g)
    B = torch.randn((Ncol, K), dtype=torch.float64, device=dev, generator=g)
    flops = 2.0 * M * Ncol * K
    res = {"M": M, "Ncol": Ncol, "K": K, "fp64_flops": flops, "per_slices": {}}
    for s in slices_list:
        ozaki_gemm(A, B, s, store=False)                      # warm-up
        r = ozaki_gemm(A, B, s, store=False, repeats=repeats)
        res["per_slices"][s] = {"ms_gemm": r["ms_gemm"], "ms_slice_both_operands": r["ms_slice"],
                                "int8_products": s * (s + 1) // 2,
                                "fp64_equiv_tflops": flops / (r["ms_gemm"] * 1e-3) * 1e-12,
                                "int8_tops": flops * (s * (s + 1) // 2) / (r["ms_gemm"] * 1e-3) * 1e-12}
    return res


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--large", action="store_true", help="also the accuracy leg on 'large' (minutes of host time to generate)")
    args = ap.parse_args()
    dev = torch.device("cuda", 0)
    slices = [3, 4, 5, 6, 7, 8]
    out = {"experiment": "ozaki_i8_exchange_contraction", "accuracy": [], "throughput": None}
    out["accuracy"].append(accuracy("small", list(range(16)), slices, dev))
    out["accuracy"].append(accuracy("cu2o2", [0, 1, 127, 128, 254, 255, 17, 200], slices, dev))
    if args.large:
        out["accuracy"].append(accuracy("large", [0, 255, 256, 511], slices, dev))
    # the exchange GEMM of one spin at the headline config: [Ngamma n x N] . [N x 2 Nw n]
    out["throughput"] = throughput(2000 * 26, 2 * 256 * 26, 290, slices, dev)
    print(json.dumps(out), flush=True)


if __name__ == "__main__":
    main()
