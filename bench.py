#!/usr/bin/env python
"""bench.py -- local-energy throughput of the B200-native AFQMC library (one JSON line on stdout).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config cu2o2] [--impl ours|reference]

A "step" is one pass of the whole hot path (K1 overlap/LU/inverse/theta -> K2 fused exchange, both spins ->
K3 assembly) over one batch of Nw synthetic walkers.  The default workload is the
configuration BASELINE.json's metric is quoted on: Cu2O2-scale, N=290, n_alpha=n_beta=26, Ngamma=2000, Nw=256.

  value      walkers/s, all ranks, inputs resident in HBM, CUDA events on the launch stream, max over ranks
  e2e        the same through afqmc_local_energy_host: pinned host walkers -> device, kernels, results -> host
  roofline   K2 (the dominant kernel): algorithmic flops 4 n^2 N per (walker, gamma, spin) / mean launch time,
             against the FP64 tensor (DMMA) peak measured live on this GPU with afqmc_fp64_peak
  cpu_baseline  the oracle (oracle/afqmc_oracle.py, rung O3) timed on this box's host cores on a bounded sample

N > 1: the path shards over walkers with no data-path collective -- the job has N * Nw walkers, rank r owns the r-th
block of Nw (weak scaling) and a replica of the half-rotated tensors; the only communication is the barrier, the
max-over-ranks of the timings and one gather of the per-walker energies for the result digest.  Launched under
torchrun by the driver; a plain `python bench.py --gpus N` re-launches itself that way.

--impl reference times the CPU oracle as it stands (rank 0 only) on a bounded sample per step.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "local-energy walkers/sec (complex128) at N=290,Ngamma=2000"
UNIT = "walkers/s"


def workload_desc(name, cfg, nw):
    return {"workload": f"{name}: N={cfg['N']} n_alpha={cfg['n_alpha']} n_beta={cfg['n_beta']} "
                        f"Ngamma={cfg['n_gamma']} Nw={nw} complex128, real RHF/UHF-style trial, seeded synthetic "
                        f"(gen/configs.py)",
            "config_name": name}


class ClockSampler(threading.Thread):
    """Samples SM clock / throttle reasons during the timed region (NVML, 20 ms period)."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.max_mhz = index, [], set(), None
        self._stop_evt = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception:
            self.ok = False

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        names = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap",
                 0x80: "hw_power_brake", 0x2: "applications_clocks", 0x100: "display_clocks"}
        while not self._stop_evt.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, nm in names.items():
                    if r & bit:
                        self.reasons.add(nm)
            except Exception:
                pass
            time.sleep(0.02)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=2)
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["unavailable"]}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


def oracle_threads():
    try:
        from threadpoolctl import threadpool_info
        n = [p.get("num_threads", 1) for p in threadpool_info() if p.get("user_api") == "blas"]
        return max(n) if n else os.cpu_count()
    except Exception:
        return os.cpu_count()


def time_oracle(inp, walkers, gamma_fraction=1):
    """Times the oracle (rung O3) as it stands on `walkers`; gamma_fraction = 1/k uses the first Ngamma/k vectors
    (cost is linear in Ngamma) and the caller scales.  Returns seconds."""
    from oracle import afqmc_oracle as orc
    chol = inp.chol if gamma_fraction == 1 else inp.chol[: inp.n_gamma // gamma_fraction]
    t0 = time.perf_counter()
    for w in walkers:
        orc.local_energy_cholesky(inp.h1e, chol, inp.e0, inp.psi_a, inp.psi_b, inp.phi_a[w], inp.phi_b[w])
    return time.perf_counter() - t0


def run_reference(args, cfg, rank, world):
    """--impl reference: the CPU oracle, rank 0 only."""
    if rank != 0:
        return
    from gen import make_inputs
    nw_total = cfg["n_walkers"]
    inp = make_inputs(args.config, n_walkers=min(nw_total, 4))
    # one walker per step on ALL Cholesky vectors (about 7 s per step at cu2o2 on 16 host threads); only `large`
    # (8 N^3 Ngamma = 3e12 flops per walker) is sampled on the first Ngamma / 8 vectors and scaled
    frac = 8 if 8.0 * cfg["N"] ** 3 * cfg["n_gamma"] > 1.0e12 else 1
    for _ in range(args.warmup):
        time_oracle(inp, [0], frac)
    t0 = time.perf_counter()
    for k in range(args.steps):
        time_oracle(inp, [k % inp.n_walkers], frac)
    dt = time.perf_counter() - t0
    walkers_equiv = args.steps / frac
    value = walkers_equiv / dt
    cores = oracle_threads()
    sample = (f"oracle rung O3 (full Green's function, un-rotated Cholesky vectors), 1 walker x "
              + (f"all {cfg['n_gamma']} Cholesky vectors per step" if frac == 1 else
                 f"first {cfg['n_gamma'] // frac}/{cfg['n_gamma']} Cholesky vectors per step; cost is linear in Ngamma, "
                 f"value scaled to the full Ngamma"))
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_desc(args.config, cfg, nw_total),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="cu2o2", choices=["tiny", "small", "medium", "cu2o2", "large"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-propagation", action="store_true", help="skip the propagation-step leg (SURVEY 8f-4)")
    ap.add_argument("--all-configs", action="store_true",
                    help="also time the other four configs (device-resident, fewer steps) and add them as "
                         "'other_configs' to the JSON line; generating 'large' takes a few minutes of host time")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    from gen import CONFIGS, make_inputs
    cfg = CONFIGS[args.config]
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))

    if args.impl == "reference":
        run_reference(args, cfg, rank, world)
        return

    if "WORLD_SIZE" not in os.environ and args.gpus > 1:
        # asked for N ranks from a plain `python bench.py --gpus N`: run the same command under torchrun
        from paper_2209_04015_b200.parallel import respawn_under_torchrun
        raise SystemExit(respawn_under_torchrun(os.path.abspath(__file__), args.gpus, sys.argv[1:]).returncode)
    if world != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}: launch one rank per GPU "
                         f"(torchrun --nproc-per-node {args.gpus}) or drop --gpus")

    import torch
    import torch.distributed as dist
    from paper_2209_04015_b200 import LocalEnergy, fp64_peak_tflops
    from paper_2209_04015_b200.parallel import (gather_walker_results, init_from_env, result_digest,
                                                weak_scaling_block)
    from paper_2209_04015_b200.parallel import max_over_ranks as _max_over_ranks

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (this library has no CPU path)")
    if torch.cuda.device_count() < world:
        raise SystemExit(f"bench.py: {world} ranks but only {torch.cuda.device_count()} GPUs are visible")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    init_from_env("nccl", dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def max_over_ranks(x):
        return _max_over_ranks(x, device=dev)

    # ---- inputs: same Hamiltonian/trial on every rank; the job's population is world * Nw walkers of the config's
    # generator (drawn walker by walker, so the first Nw are the one-rank job's) and rank r owns the r-th block.
    nw = cfg["n_walkers"]
    w_start, w_count = weak_scaling_block(nw, rank, world)
    assert w_count == nw
    inp = make_inputs(args.config, n_walkers=world * nw)
    my_walkers = list(range(w_start, w_start + w_count))
    h1e = torch.from_numpy(inp.h1e).to(dev)
    chol = torch.from_numpy(inp.chol).to(dev)
    trial = torch.from_numpy(inp.trial_packed()).to(dev)
    le = LocalEnergy(h1e, chol, trial, inp.N, inp.n_alpha, inp.n_beta, inp.n_gamma, inp.e0, nw)
    le.enable_force_bias(chol)          # operand of the dedicated force-bias GEMM (reported under "force_bias")
    PROP_DT, PROP_ORDER = 0.00005, 6    # customary Taylor order; 1/100 of the paper's Cu2O2 time step
    # because the synthetic Cholesky vectors are ~100x a molecule's: at 0.005 the overlap ratio overflows exp()
    if not args.no_propagation:
        le.enable_propagation(h1e, chol, PROP_DT)
    del chol
    torch.cuda.empty_cache()
    walkers_host = torch.from_numpy(inp.walkers_packed(my_walkers)).pin_memory()
    walkers = walkers_host.to(dev)
    outE = torch.empty(nw, dtype=torch.complex128, device=dev)
    outO = torch.empty(nw, dtype=torch.complex128, device=dev)
    outE_h = torch.empty(nw, dtype=torch.complex128).pin_memory()
    outO_h = torch.empty(nw, dtype=torch.complex128).pin_memory()
    info = le.info()
    walkers_bytes = int(walkers.numel() * 16)
    stream = torch.cuda.current_stream()

    # ---- FP64 peak, measured live (roofline denominator) ------------------------------------------------
    psamp = ClockSampler(local_rank)
    psamp.start()
    peak_dmma = fp64_peak_tflops("dmma", launches=20)
    peak_dfma = fp64_peak_tflops("dfma", launches=10)
    peak_record = {"how": "afqmc_fp64_peak: register-resident chains, 20 back-to-back launches of mode 0 (DMMA.8x8x4, "
                          "16 warps/SM x 8 accumulators) and 10 of mode 1 (DFMA), CUDA events around the sequence",
                   "dmma_launches": 20, "dfma_launches": 10, "clocks": psamp.stop()}

    # ---- device-resident timing ---------------------------------------------------------------------------
    for _ in range(args.warmup):
        le.local_energy(walkers, nw, outE, outO)
    barrier()
    launches0 = le.info()["kernel_launches"]
    le.set_profiling(True)
    sampler = ClockSampler(local_rank)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(stream)
    for _ in range(args.steps):
        le.local_energy(walkers, nw, outE, outO)
    e1.record(stream)
    barrier()
    clocks = sampler.stop()
    ms_total = max_over_ranks(e0.elapsed_time(e1))
    kms, kcalls = le.mean_kernel_ms()
    le.set_profiling(False)
    gpu_launches = le.info()["kernel_launches"] - launches0
    value = world * nw * args.steps / (ms_total * 1e-3)

    # ---- end to end through the host-buffer entry point -----------------------------------------------------
    for _ in range(2):
        le.local_energy_host(walkers_host, nw, outE_h, outO_h)
    barrier()
    e0.record(stream)
    for _ in range(args.steps):
        le.local_energy_host(walkers_host, nw, outE_h, outO_h)
    e1.record(stream)
    barrier()
    ms_e2e = max_over_ranks(e0.elapsed_time(e1))
    e2e_value = world * nw * args.steps / (ms_e2e * 1e-3)
    same = bool(torch.equal(outE_h.view(torch.float64), outE.cpu().view(torch.float64)))
    # per-walker energies of the whole job in walker order: equal digests between an N-rank and a 1-rank run (its
    # walkers are the first block) mean bit-identical results
    all_E = gather_walker_results(outE, world * nw)
    digest = {"first_block_sha256": result_digest(all_E[:nw]), "all_blocks_sha256": result_digest(all_E),
              "n_walkers_total": world * nw}

    # ---- the force bias without the energy: K1 + one DMMA GEMM per spin + combine ------------------
    fb_out = torch.empty((nw, inp.n_gamma), dtype=torch.complex128, device=dev)
    for _ in range(3):
        le.force_bias_only(walkers, nw, fb_out)
    barrier()
    e0.record(stream)
    for _ in range(args.steps):
        le.force_bias_only(walkers, nw, fb_out)
    e1.record(stream)
    barrier()
    ms_fb = max_over_ranks(e0.elapsed_time(e1)) / args.steps
    flops_fb = 4.0 * inp.N * inp.n_gamma * nw * (inp.n_alpha + inp.n_beta)

    # ---- one hybrid propagation step: K1, force bias, field GEMM, Taylor, K1, weights --
    prop = None
    if not args.no_propagation:
        from paper_2209_04015_b200 import sample_fields
        xf = sample_fields(1234, 0, nw, inp.n_gamma, first_walker=w_start, device=dev)     # Eq. 4's x, drawn before the timed region
        wts = torch.ones(nw, dtype=torch.float64, device=dev)
        wts_out, lo_out = torch.empty_like(wts), torch.empty(nw, dtype=torch.complex128, device=dev)
        wk = walkers.clone()
        le.set_profiling(True)
        for _ in range(3):
            wk.copy_(walkers)
            le.propagate(wk, nw, xf, wts, PROP_ORDER, wts_out, lo_out)
        barrier()
        phase = np.zeros(5)
        e0.record(stream)
        for _ in range(args.steps):
            wk.copy_(walkers)               # every step starts from the same determinants (62 MB device copy, timed)
            le.propagate(wk, nw, xf, wts, PROP_ORDER, wts_out, lo_out)
        e1.record(stream)
        barrier()
        phase = np.array(le.propagate_phase_ms())          # phases of the last step
        le.set_profiling(False)
        ms_prop = max_over_ranks(e0.elapsed_time(e1)) / args.steps
        ne = inp.n_alpha + inp.n_beta
        flops_field = 4.0 * nw * inp.n_gamma * inp.N * (inp.N + 1) / 2         # [N(N+1)/2 x Ng].[Ng x 2Nw] real GEMM (L symmetric)
        flops_taylor = (PROP_ORDER * 8.0 + 2 * 4.0) * inp.N ** 2 * ne * nw      # complex A T_k terms + two real E T products
        prop = {"value": world * nw / (ms_prop * 1e-3), "unit": UNIT, "ms_per_step": ms_prop, "dt": PROP_DT,
                "taylor_order": PROP_ORDER,
                "what": "afqmc_propagate: K1 + force-bias GEMM + field GEMM [N(N+1)/2 x Ng].[Ng x 2Nw] + (order + 2) batched "
                        "[N x N].[N x 2(na+nb)] products + K1 + phaseless weights; device-resident, x drawn beforehand",
                "phase_ms": {"k1_overlap": phase[0], "force_bias_gemm": phase[1], "fields_and_field_gemm": phase[2],
                             "one_body_and_taylor": phase[3], "k1_and_weights": phase[4]},
                "field_gemm": {"algorithmic_flops": flops_field, "tflops": flops_field / (phase[2] * 1e-3) * 1e-12},
                "taylor": {"algorithmic_flops": flops_taylor, "tflops": flops_taylor / (phase[3] * 1e-3) * 1e-12},
                "finite": bool(torch.isfinite(wts_out).all().item())}

    # ---- roofline of K2 -------------------------------------------------------------------------------------
    nspin_launches = int(inp.n_alpha > 0) + int(inp.n_beta > 0)
    flops_k2 = 4.0 * inp.N * inp.n_gamma * nw * (inp.n_alpha ** 2 + inp.n_beta ** 2)        # per step, both spins
    flops_per_launch = flops_k2 / nspin_launches
    k2_launch_ms = kms[1] / nspin_launches
    achieved = flops_per_launch / (k2_launch_ms * 1e-3) * 1e-12
    peak = max(peak_dmma, peak_dfma)
    if prop is not None:
        prop["field_gemm"]["frac_of_fp64_peak"] = prop["field_gemm"]["tflops"] / peak
        prop["taylor"]["frac_of_fp64_peak"] = prop["taylor"]["tflops"] / peak
    traffic = None
    tpath = os.path.join(ROOT, "profiles", "k2_dram_traffic.json")
    if os.path.exists(tpath):
        try:
            with open(tpath) as f:
                traffic = json.load(f).get(args.config, {}).get("dram_bytes_per_launch")
        except Exception:
            traffic = None
    bytes_l = info["ltilde_bytes"] + info["theta_bytes"]
    hbm_gbs, bf16_meas = None, None
    mp = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(mp):
        with open(mp) as f:
            mpj = json.load(f)
        hbm_gbs, bf16_meas = mpj.get("hbm_gbs"), mpj.get("bf16_tflops")
    hbm_gbs = hbm_gbs or 6650.0
    # the other way to an FP64 denominator: the driver-measured bf16 peak x the nominal FP64 : bf16 ratio of the
    # guides (45 : 2250 TFLOP/s dense).  It comes out BELOW the FP64 rate measured here, so the stricter one is used.
    bf16_scaled = (bf16_meas or 1590.0) * 45.0 / 2250.0
    t_roof_ms = max(flops_k2 / (peak * 1e12), bytes_l / (hbm_gbs * 1e9)) * 1e3
    roofline = {"bound": "tensor", "kernel": "k2_exchange (fused exchange + Coulomb traces), one launch per spin",
                "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak, "traffic": traffic,
                "traffic_source": "dram__bytes_read.sum + dram__bytes_write.sum of one ncu --set full capture of this "
                                  "kernel, stored in profiles/k2_dram_traffic.json; not re-measured in this run",
                "peak_measurement": peak_record,
                "peak_source": "FP64 DMMA.8x8x4 register-resident microbenchmark (afqmc_fp64_peak) measured live in "
                               "this run; MEASURED_PEAKS.json has no FP64 entry",
                "peak_dmma_tflops": peak_dmma, "peak_dfma_tflops": peak_dfma,
                "peak_bf16_measured_x_nominal_fp64_ratio": bf16_scaled, "frac_of_that": achieved / bf16_scaled,
                "algorithmic_flops_per_launch": flops_per_launch, "k2_ms_per_launch": k2_launch_ms,
                "kernel_ms_per_step": {"k1": kms[0], "k2": kms[1], "k3": kms[2]}, "profiled_calls": kcalls,
                "roofline_ms_per_step": t_roof_ms, "step_frac_of_roofline": t_roof_ms / (ms_total / args.steps),
                "hbm_bytes_algorithmic_per_step": bytes_l,
                # K1 (overlap / LU / inverse / theta): reads the walkers, writes the packed theta planes
                "k1": {"algorithmic_bytes": int(walkers_bytes + info["theta_bytes"]),
                       "achieved_gbs": (walkers_bytes + info["theta_bytes"]) / (kms[0] * 1e-3) * 1e-9,
                       "hbm_peak_gbs": hbm_gbs,
                       "note": "0.5 % of the step; its two products run on the tensor pipe, the inversion between them is "
                               "bound by dependent-issue latency (DESIGN.md section 6), not by HBM"}}

    # ---- CPU baseline: the oracle on a bounded sample (rank 0, N=1 only) ---------------------------------------
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        frac = 1
        per_walker_flops = 8.0 * inp.N ** 3 * inp.n_gamma
        if per_walker_flops > 1.0e12:        # keep the sample near 10-30 s
            frac = 8
        sample_w = [0]
        dt = time_oracle(inp, sample_w, frac)
        cpu = {"value": len(sample_w) / (dt * frac), "unit": UNIT, "cores": oracle_threads(), "kind": "oracle",
               "sample": f"oracle rung O3 on walker 0, {'all' if frac == 1 else f'first 1/{frac} of the'} "
                         f"{inp.n_gamma} Cholesky vectors ({dt:.1f} s{', scaled by ' + str(frac) if frac > 1 else ''})"}

    # ---- the other configs (north_star: report all five), device-resident timing only ------------------------
    others = None
    if args.all_configs and world == 1:
        le.close()
        del walkers, h1e, trial
        torch.cuda.empty_cache()
        others = {}
        for name in ("tiny", "small", "medium", "cu2o2", "large"):
            if name == args.config:
                continue
            oi = make_inputs(name)
            ole = LocalEnergy(torch.from_numpy(oi.h1e).to(dev), torch.from_numpy(oi.chol).to(dev),
                              torch.from_numpy(oi.trial_packed()).to(dev), oi.N, oi.n_alpha, oi.n_beta, oi.n_gamma,
                              oi.e0, oi.n_walkers)
            torch.cuda.empty_cache()
            ow = torch.from_numpy(oi.walkers_packed()).to(dev)
            oE = torch.empty(oi.n_walkers, dtype=torch.complex128, device=dev)
            oO = torch.empty_like(oE)
            nsteps = 3 if name == "large" else 20
            for _ in range(3):
                ole.local_energy(ow, oi.n_walkers, oE, oO)
            torch.cuda.synchronize()
            ole.set_profiling(True)
            e0.record(stream)
            for _ in range(nsteps):
                ole.local_energy(ow, oi.n_walkers, oE, oO)
            e1.record(stream)
            torch.cuda.synchronize()
            oms = e0.elapsed_time(e1) / nsteps
            okms, _ = ole.mean_kernel_ms()
            ofl = 4.0 * oi.N * oi.n_gamma * oi.n_walkers * (oi.n_alpha ** 2 + oi.n_beta ** 2)
            otf = ofl / (okms[1] * 1e-3) * 1e-12
            oinfo = ole.info()
            others[name] = {"walkers_per_s": oi.n_walkers / (oms * 1e-3), "ms_per_step": oms, "steps": nsteps,
                            "k2_tflops": otf, "k2_frac_of_peak": otf / peak,
                            "kernel_ms_per_step": {"k1": okms[0], "k2": okms[1], "k3": okms[2]},
                            "k2_tile": {k: oinfo[k] for k in ("tile_rows", "tile_cols", "stages", "ksteps_per_chunk")}}
            ole.close()
            del ow, oE, oO, oi
            torch.cuda.empty_cache()

    # ---- baseline B: the paper's own half-rotated CPU algorithm (Listing 4) restated in numpy, same host cores ----
    cpu_b = None
    if cpu is not None:
        from oracle.listing4_cpu import HalfRotated, local_energy_listing4
        t0 = time.perf_counter()
        hr = HalfRotated(inp.h1e, inp.chol, inp.psi_a, inp.psi_b)
        t_setup = time.perf_counter() - t0
        nb_w, t0 = 0, time.perf_counter()
        while nb_w < inp.n_walkers and (nb_w < 2 or time.perf_counter() - t0 < 5.0):
            local_energy_listing4(hr, inp.e0, inp.phi_a[nb_w], inp.phi_b[nb_w])
            nb_w += 1
        dt_b = time.perf_counter() - t0
        cpu_b = {"value": nb_w / dt_b, "unit": UNIT, "cores": oracle_threads(), "kind": "paper_listing4_numpy",
                 "sample": f"oracle/listing4_cpu.py on the first {nb_w} walkers ({dt_b:.1f} s; half-rotation setup "
                           f"{t_setup:.1f} s not included, as on the GPU)"}

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms_total / args.steps, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                "config": {**workload_desc(args.config, cfg, nw),
                           "parallelism": f"walker replicas x{world}, no data-path collective",
                           "l2": "no flush: per-step working set (packed Ltilde + theta + walkers = "
                                 f"{(bytes_l + walkers_bytes) / 1e6:.0f} MB) exceeds the 126 MB L2",
                           "k2_tile": {k: info[k] for k in ("tile_rows", "tile_cols", "gammas_per_tile",
                                                            "walkers_per_tile", "warps_m", "mt", "nt", "stages",
                                                            "k2_smem_bytes")}},
                "clocks": clocks,
                "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(walkers_host.numel() * 16),
                        "d2h_bytes_per_step": int(2 * nw * 16), "ms_per_step": ms_e2e / args.steps,
                        "matches_device_path_bitwise": same},
                "gpu_launches": int(gpu_launches),
                "result_digest": digest,
                "force_bias": {"value": world * nw / (ms_fb * 1e-3), "unit": UNIT, "ms_per_step": ms_fb,
                               "what": "afqmc_force_bias_only: K1 + [Ngamma x nN].[nN x 2Nw] DMMA GEMM per spin + "
                                       "combine; device-resident, same walkers",
                               "algorithmic_flops_per_step": flops_fb,
                               "tflops_incl_k1": flops_fb / (ms_fb * 1e-3) * 1e-12,
                               "speedup_vs_energy_step": (ms_total / args.steps) / ms_fb},
                "propagation": prop,
                "roofline": roofline,
                "cpu_baseline": cpu,
                "cpu_baseline_listing4": cpu_b}
        if others is not None:
            line["other_configs"] = others
        print(json.dumps(line), flush=True)
    le.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
