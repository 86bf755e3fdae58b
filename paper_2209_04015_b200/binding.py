"""ctypes binding with the same names as include/afqmc.h.  Argument marshalling only.

PyTorch is used for device memory and streams (tensors in, tensors out); every step of the path runs in the
library's CUDA kernels.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

_PKG = os.path.dirname(os.path.abspath(__file__))
_LIB = None

EXPORTS = ["afqmc_create", "afqmc_local_energy", "afqmc_local_energy_host", "afqmc_force_bias",
           "afqmc_enable_force_bias", "afqmc_force_bias_only", "afqmc_spin_squared", "afqmc_greens_function", "afqmc_phaseless_weights", "afqmc_destroy",
           "afqmc_last_error", "afqmc_get_info", "afqmc_set_profiling", "afqmc_last_kernel_ms", "afqmc_mean_kernel_ms",
           "afqmc_fp64_peak", "afqmc_plan", "afqmc_plan_trial", "afqmc_enable_propagation", "afqmc_propagate",
           "afqmc_propagation_xbar", "afqmc_propagate_phase_ms", "afqmc_sample_fields", "afqmc_log_overlap_static"]


class AfqmcError(RuntimeError):
    pass


class AfqmcInfo(C.Structure):
    _fields_ = [("N", C.c_int), ("n_alpha", C.c_int), ("n_beta", C.c_int), ("n_gamma", C.c_int),
                ("max_walkers", C.c_int), ("k_steps", C.c_int),
                ("tile_rows", C.c_int * 2), ("tile_cols", C.c_int * 2), ("gammas_per_tile", C.c_int * 2),
                ("walkers_per_tile", C.c_int * 2), ("warps_m", C.c_int * 2), ("mt", C.c_int * 2), ("nt", C.c_int * 2),
                ("stages", C.c_int * 2), ("ksteps_per_chunk", C.c_int * 2), ("k2_smem_bytes", C.c_int * 2),
                ("ltilde_bytes", C.c_longlong), ("theta_bytes", C.c_longlong), ("kernel_launches", C.c_longlong)]


def library_path() -> str:
    return os.path.join(_PKG, "libafqmc.so")


def load_library():
    """dlopen libafqmc.so (built in-tree).  Raises if it is missing: there is no fallback path."""
    global _LIB
    if _LIB is not None:
        return _LIB
    path = library_path()
    if not os.path.exists(path):
        raise AfqmcError(f"{path} not found: build it first (python -c 'import __graft_entry__ as g; g.build()')")
    lib = C.CDLL(path)
    vp, ip, dp = C.c_void_p, C.c_int, C.c_double
    lib.afqmc_create.argtypes = [vp, vp, vp, ip, ip, ip, ip, dp, ip, vp, C.POINTER(vp)]
    lib.afqmc_create.restype = ip
    lib.afqmc_local_energy.argtypes = [vp, vp, ip, vp, vp, vp]
    lib.afqmc_local_energy.restype = ip
    lib.afqmc_local_energy_host.argtypes = [vp, vp, ip, vp, vp, vp]
    lib.afqmc_local_energy_host.restype = ip
    lib.afqmc_force_bias.argtypes = [vp, vp, vp]
    lib.afqmc_force_bias.restype = ip
    lib.afqmc_sample_fields.argtypes = [C.c_ulonglong, C.c_ulonglong, ip, ip, ip, vp, vp]
    lib.afqmc_sample_fields.restype = ip
    lib.afqmc_log_overlap_static.argtypes = [vp, vp, ip, ip, ip, ip, vp, vp]
    lib.afqmc_log_overlap_static.restype = ip
    lib.afqmc_enable_force_bias.argtypes = [vp, vp, vp]
    lib.afqmc_enable_force_bias.restype = ip
    lib.afqmc_force_bias_only.argtypes = [vp, vp, ip, vp, vp]
    lib.afqmc_force_bias_only.restype = ip
    lib.afqmc_spin_squared.argtypes = [vp, vp, vp]
    lib.afqmc_spin_squared.restype = ip
    lib.afqmc_greens_function.argtypes = [vp, ip, vp, vp]
    lib.afqmc_greens_function.restype = ip
    lib.afqmc_phaseless_weights.argtypes = [ip, ip, vp, vp, vp, vp, vp, vp, vp]
    lib.afqmc_phaseless_weights.restype = ip
    lib.afqmc_destroy.argtypes = [vp]
    lib.afqmc_destroy.restype = None
    lib.afqmc_last_error.argtypes = [vp]
    lib.afqmc_last_error.restype = C.c_char_p
    lib.afqmc_get_info.argtypes = [vp, C.POINTER(AfqmcInfo)]
    lib.afqmc_get_info.restype = ip
    lib.afqmc_set_profiling.argtypes = [vp, ip]
    lib.afqmc_set_profiling.restype = ip
    lib.afqmc_last_kernel_ms.argtypes = [vp, C.POINTER(C.c_float)]
    lib.afqmc_last_kernel_ms.restype = ip
    lib.afqmc_mean_kernel_ms.argtypes = [vp, C.POINTER(C.c_float), C.POINTER(ip)]
    lib.afqmc_mean_kernel_ms.restype = ip
    lib.afqmc_fp64_peak.argtypes = [ip, ip, C.POINTER(dp), vp]
    lib.afqmc_fp64_peak.restype = ip
    lib.afqmc_plan.argtypes = [ip, ip, ip, ip, ip, C.POINTER(AfqmcInfo)]
    lib.afqmc_plan.restype = ip
    lib.afqmc_plan_trial.argtypes = [ip, ip, ip, ip, ip, ip, ip, C.POINTER(AfqmcInfo)]
    lib.afqmc_plan_trial.restype = ip
    lib.afqmc_enable_propagation.argtypes = [vp, vp, vp, dp, vp]
    lib.afqmc_enable_propagation.restype = ip
    lib.afqmc_propagate.argtypes = [vp, vp, ip, vp, vp, vp, vp, ip, vp]
    lib.afqmc_propagate.restype = ip
    lib.afqmc_propagation_xbar.argtypes = [vp, vp, vp]
    lib.afqmc_propagation_xbar.restype = ip
    lib.afqmc_propagate_phase_ms.argtypes = [vp, C.POINTER(C.c_float)]
    lib.afqmc_propagate_phase_ms.restype = ip
    _LIB = lib
    return lib


def _stream_ptr(stream=None):
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def _require_cuda():
    if not torch.cuda.is_available():
        raise AfqmcError("no CUDA device: this library has no CPU path")


def fp64_peak_tflops(mode: str = "dmma", launches: int = 10) -> float:
    """afqmc_fp64_peak: measured register-resident FP64 throughput (TFLOP/s). mode: 'dmma' | 'dfma'."""
    _require_cuda()
    lib = load_library()
    out = C.c_double(0.0)
    rc = lib.afqmc_fp64_peak(0 if mode == "dmma" else 1, launches, C.byref(out), _stream_ptr())
    if rc != 0:
        raise AfqmcError(f"afqmc_fp64_peak failed ({rc}): {lib.afqmc_last_error(None).decode()}")
    return out.value


def phaseless_weights(x, xbar, log_ovlp_old, log_ovlp_new, weights, out=None, stream=None):
    """afqmc_phaseless_weights (Eq. 7-12): x float64 [Nw, Ngamma], xbar complex128 [Nw, Ngamma], log-overlaps
    complex128 [Nw], weights float64 [Nw]; all contiguous CUDA tensors.  Returns the new weights."""
    _require_cuda()
    lib = load_library()
    nw, ng = x.shape
    for t, dt in ((x, torch.float64), (xbar, torch.complex128), (log_ovlp_old, torch.complex128),
                  (log_ovlp_new, torch.complex128), (weights, torch.float64)):
        if not (t.is_cuda and t.is_contiguous() and t.dtype == dt):
            raise AfqmcError("phaseless_weights: inputs must be contiguous CUDA tensors of the documented dtypes")
    if xbar.shape != x.shape or log_ovlp_old.numel() != nw or log_ovlp_new.numel() != nw or weights.numel() != nw:
        raise AfqmcError("phaseless_weights: shapes do not match")
    if out is None:
        out = torch.empty_like(weights)
    rc = lib.afqmc_phaseless_weights(nw, ng, x.data_ptr(), xbar.data_ptr(), log_ovlp_old.data_ptr(),
                                     log_ovlp_new.data_ptr(), weights.data_ptr(), out.data_ptr(), _stream_ptr(stream))
    if rc != 0:
        raise AfqmcError(f"afqmc_phaseless_weights failed ({rc}): {lib.afqmc_last_error(None).decode()}")
    return out


def sample_fields(seed, step, n_walkers, n_gamma, first_walker=0, out=None, device=None, stream=None):
    """afqmc_sample_fields: the auxiliary fields x ~ N(0, 1) of one propagation step (Eq. 4), float64 [n_walkers, n_gamma] on
    the GPU, from the counter-based generator the header describes (no state: the same arguments give the same numbers)."""
    _require_cuda()
    lib = load_library()
    if out is None:
        out = torch.empty((n_walkers, n_gamma), dtype=torch.float64, device=device or "cuda")
    if not (out.is_cuda and out.is_contiguous() and out.dtype == torch.float64) or out.numel() != n_walkers * n_gamma:
        raise AfqmcError("sample_fields: out must be a contiguous CUDA float64 tensor of n_walkers * n_gamma elements")
    rc = lib.afqmc_sample_fields(int(seed) & (2 ** 64 - 1), int(step) & (2 ** 64 - 1), int(first_walker), int(n_walkers), int(n_gamma),
                                 out.data_ptr(), _stream_ptr(stream))
    if rc != 0:
        raise AfqmcError(f"afqmc_sample_fields failed ({rc}): {lib.afqmc_last_error(None).decode()}")
    return out


def log_overlap_static(trial, walkers, N, n_alpha, n_beta, n_walkers, out=None, stream=None):
    """afqmc_log_overlap_static: log-overlaps [n_walkers] complex128 without a handle and without any allocation inside the
    library (pass ``out`` to keep this wrapper allocation-free too).  Sizes beyond the library's static scratch raise."""
    _require_cuda()
    lib = load_library()
    for t, cnt in ((trial, N * (n_alpha + n_beta)), (walkers, n_walkers * N * (n_alpha + n_beta))):
        if not (t.is_cuda and t.is_contiguous() and t.dtype == torch.complex128) or t.numel() != cnt:
            raise AfqmcError("log_overlap_static: trial / walkers must be contiguous CUDA complex128 tensors of the documented sizes")
    if out is None:
        out = torch.empty(n_walkers, dtype=torch.complex128, device=walkers.device)
    if not (out.is_cuda and out.is_contiguous() and out.dtype == torch.complex128) or out.numel() != n_walkers:
        raise AfqmcError("log_overlap_static: out must be a contiguous CUDA complex128 tensor of n_walkers elements")
    rc = lib.afqmc_log_overlap_static(trial.data_ptr(), walkers.data_ptr(), int(N), int(n_alpha), int(n_beta), int(n_walkers),
                                      out.data_ptr(), _stream_ptr(stream))
    if rc != 0:
        raise AfqmcError(f"afqmc_log_overlap_static failed ({rc}): {lib.afqmc_last_error(None).decode()}")
    return out


def _info_dict(inf) -> dict:
    out = {}
    for name, _ in AfqmcInfo._fields_:
        v = getattr(inf, name)
        out[name] = list(v) if hasattr(v, "__len__") else v
    return out


def plan(N, n_alpha, n_beta, n_gamma, max_walkers, complex_alpha=False, complex_beta=False) -> dict:
    """afqmc_plan / afqmc_plan_trial: the K2 tile shape / pipeline / packed sizes afqmc_create would choose (host only,
    no GPU); complex_* say which spin blocks of the trial are complex."""
    lib = load_library()
    inf = AfqmcInfo()
    rc = lib.afqmc_plan_trial(N, n_alpha, n_beta, n_gamma, max_walkers, int(bool(complex_alpha)),
                              int(bool(complex_beta)), C.byref(inf))
    if rc != 0:
        raise AfqmcError(f"afqmc_plan failed ({rc}): {lib.afqmc_last_error(None).decode()}")
    return _info_dict(inf)


class LocalEnergy:
    """Handle around afqmc_create / afqmc_local_energy / afqmc_destroy.

    h1e [N,N] float64, chol [Ngamma,N,N] float64, trial = complex128 vector (alpha block [N,n_alpha] then beta
    block [N,n_beta]); all CUDA tensors.  ``chol`` is not retained.
    """

    def __init__(self, h1e, chol, trial, N, n_alpha, n_beta, n_gamma, e0, max_walkers, stream=None):
        _require_cuda()
        self._lib = load_library()
        self._h = C.c_void_p(None)
        for t, dt in ((h1e, torch.float64), (chol, torch.float64), (trial, torch.complex128)):
            if not (t.is_cuda and t.is_contiguous() and t.dtype == dt):
                raise AfqmcError("inputs must be contiguous CUDA tensors of dtype float64/float64/complex128")
        if h1e.numel() != N * N or chol.numel() != n_gamma * N * N or trial.numel() != N * (n_alpha + n_beta):
            raise AfqmcError("input sizes do not match N, n_alpha, n_beta, n_gamma")
        rc = self._lib.afqmc_create(h1e.data_ptr(), chol.data_ptr(), trial.data_ptr(), N, n_alpha, n_beta, n_gamma,
                                    float(e0), max_walkers, _stream_ptr(stream), C.byref(self._h))
        if rc != 0:
            raise AfqmcError(f"afqmc_create failed ({rc}): {self._lib.afqmc_last_error(None).decode()}")
        self.N, self.n_alpha, self.n_beta, self.n_gamma, self.max_walkers = N, n_alpha, n_beta, n_gamma, max_walkers
        self._last_nw = 0           # walkers of the last local_energy / force_bias_only call (theta held by the handle)
        self._last_energy_nw = 0    # walkers of the last local_energy call (Coulomb traces held by the handle)

    def _check(self, rc, what):
        if rc != 0:
            raise AfqmcError(f"{what} failed ({rc}): {self._lib.afqmc_last_error(self._h).decode()}")

    def local_energy(self, walkers, n_walkers, out_energies=None, out_overlaps=None, stream=None):
        """afqmc_local_energy on device tensors.  Returns (energies, log_overlaps) complex128 [n_walkers]."""
        if not (walkers.is_cuda and walkers.is_contiguous() and walkers.dtype == torch.complex128):
            raise AfqmcError("walkers must be a contiguous CUDA complex128 tensor")
        if walkers.numel() != n_walkers * self.N * (self.n_alpha + self.n_beta):
            raise AfqmcError("walkers has the wrong number of elements")
        if out_energies is None:
            out_energies = torch.empty(n_walkers, dtype=torch.complex128, device=walkers.device)
        if out_overlaps is None:
            out_overlaps = torch.empty(n_walkers, dtype=torch.complex128, device=walkers.device)
        rc = self._lib.afqmc_local_energy(self._h, walkers.data_ptr(), n_walkers, out_energies.data_ptr(),
                                          out_overlaps.data_ptr(), _stream_ptr(stream))
        self._check(rc, "afqmc_local_energy")
        self._last_nw = self._last_energy_nw = n_walkers
        return out_energies, out_overlaps

    def local_energy_host(self, walkers_host, n_walkers, out_energies_host=None, out_overlaps_host=None, stream=None):
        """afqmc_local_energy_host on HOST (ideally pinned) tensors; synchronises before returning."""
        if walkers_host.is_cuda or walkers_host.dtype != torch.complex128 or not walkers_host.is_contiguous():
            raise AfqmcError("walkers_host must be a contiguous CPU complex128 tensor")
        if walkers_host.numel() != n_walkers * self.N * (self.n_alpha + self.n_beta):
            raise AfqmcError("walkers_host has the wrong number of elements")
        if out_energies_host is None:
            out_energies_host = torch.empty(n_walkers, dtype=torch.complex128).pin_memory()
        if out_overlaps_host is None:
            out_overlaps_host = torch.empty(n_walkers, dtype=torch.complex128).pin_memory()
        rc = self._lib.afqmc_local_energy_host(self._h, walkers_host.data_ptr(), n_walkers,
                                               out_energies_host.data_ptr(), out_overlaps_host.data_ptr(),
                                               _stream_ptr(stream))
        self._check(rc, "afqmc_local_energy_host")
        self._last_nw = self._last_energy_nw = n_walkers
        return out_energies_host, out_overlaps_host

    def _out_for_last_call(self, what, n_walkers, last, per_walker, out):
        """The library writes results for the walkers of the LAST call, not for a caller-chosen count: the optional
        ``n_walkers`` must agree with it and a caller-provided ``out`` must hold exactly that many."""
        if last < 1:
            raise AfqmcError(f"{what}: no preceding energy / force-bias call on this handle")
        if n_walkers is not None and n_walkers != last:
            raise AfqmcError(f"{what}: n_walkers={n_walkers} but the handle holds {last} walkers from the last call")
        shape = (last, *per_walker)
        if out is None:
            return torch.empty(shape, dtype=torch.complex128, device="cuda")
        if not (out.is_cuda and out.is_contiguous() and out.dtype == torch.complex128) or out.numel() != \
                torch.Size(shape).numel():
            raise AfqmcError(f"{what}: out must be a contiguous CUDA complex128 tensor of shape {shape}")
        return out

    def force_bias(self, n_walkers=None, out=None, stream=None):
        """afqmc_force_bias: [n_walkers, n_gamma] complex128 traces of the last energy call."""
        out = self._out_for_last_call("force_bias", n_walkers, self._last_energy_nw, (self.n_gamma,), out)
        self._check(self._lib.afqmc_force_bias(self._h, out.data_ptr(), _stream_ptr(stream)), "afqmc_force_bias")
        return out

    def enable_force_bias(self, chol, stream=None):
        """afqmc_enable_force_bias: build the operand of the dedicated force-bias GEMM from ``chol`` (CUDA float64)."""
        if not (chol.is_cuda and chol.is_contiguous() and chol.dtype == torch.float64) or \
                chol.numel() != self.n_gamma * self.N * self.N:
            raise AfqmcError("chol must be the contiguous CUDA float64 [n_gamma, N, N] tensor given at creation")
        self._check(self._lib.afqmc_enable_force_bias(self._h, chol.data_ptr(), _stream_ptr(stream)),
                    "afqmc_enable_force_bias")

    def force_bias_only(self, walkers, n_walkers, out=None, stream=None):
        """afqmc_force_bias_only: [n_walkers, n_gamma] complex128 force bias without the energy."""
        if not (walkers.is_cuda and walkers.is_contiguous() and walkers.dtype == torch.complex128):
            raise AfqmcError("walkers must be a contiguous CUDA complex128 tensor")
        if walkers.numel() != n_walkers * self.N * (self.n_alpha + self.n_beta):
            raise AfqmcError("walkers has the wrong number of elements")
        if out is None:
            out = torch.empty((n_walkers, self.n_gamma), dtype=torch.complex128, device=walkers.device)
        elif not (out.is_cuda and out.is_contiguous() and out.dtype == torch.complex128) or \
                out.numel() != n_walkers * self.n_gamma:
            raise AfqmcError("force_bias_only: out must be a contiguous CUDA complex128 [n_walkers, n_gamma] tensor")
        self._check(self._lib.afqmc_force_bias_only(self._h, walkers.data_ptr(), n_walkers, out.data_ptr(),
                                                    _stream_ptr(stream)), "afqmc_force_bias_only")
        self._last_nw = n_walkers
        return out

    def enable_propagation(self, h1e, chol, dt, stream=None):
        """afqmc_enable_propagation: one-time setup of the hybrid propagation for time step ``dt`` (CUDA float64 h1e,
        chol as given at creation)."""
        for t, cnt in ((h1e, self.N * self.N), (chol, self.n_gamma * self.N * self.N)):
            if not (t.is_cuda and t.is_contiguous() and t.dtype == torch.float64) or t.numel() != cnt:
                raise AfqmcError("h1e / chol must be the contiguous CUDA float64 tensors given at creation")
        self._check(self._lib.afqmc_enable_propagation(self._h, h1e.data_ptr(), chol.data_ptr(), float(dt),
                                                       _stream_ptr(stream)), "afqmc_enable_propagation")

    def propagate(self, walkers, n_walkers, x, weights, taylor_order=6, weights_out=None, log_ovlp_out=None, stream=None):
        """afqmc_propagate: one hybrid phaseless step (Eq. 6-13).  ``walkers`` (CUDA complex128, ABI layout) is
        overwritten with the propagated determinants; x float64 [n_walkers, n_gamma]; weights float64 [n_walkers].
        Returns (weights_out, log_ovlp_out)."""
        if not (walkers.is_cuda and walkers.is_contiguous() and walkers.dtype == torch.complex128):
            raise AfqmcError("walkers must be a contiguous CUDA complex128 tensor")
        if walkers.numel() != n_walkers * self.N * (self.n_alpha + self.n_beta):
            raise AfqmcError("walkers has the wrong number of elements")
        for t, cnt in ((x, n_walkers * self.n_gamma), (weights, n_walkers)):
            if not (t.is_cuda and t.is_contiguous() and t.dtype == torch.float64) or t.numel() != cnt:
                raise AfqmcError("x / weights must be contiguous CUDA float64 tensors of [n_walkers, n_gamma] / [n_walkers]")
        if weights_out is None:
            weights_out = torch.empty(n_walkers, dtype=torch.float64, device=walkers.device)
        if log_ovlp_out is None:
            log_ovlp_out = torch.empty(n_walkers, dtype=torch.complex128, device=walkers.device)
        for t, dt_ in ((weights_out, torch.float64), (log_ovlp_out, torch.complex128)):
            if not (t.is_cuda and t.is_contiguous() and t.dtype == dt_) or t.numel() != n_walkers:
                raise AfqmcError("weights_out / log_ovlp_out must be contiguous CUDA tensors of n_walkers elements")
        rc = self._lib.afqmc_propagate(self._h, walkers.data_ptr(), n_walkers, x.data_ptr(), weights.data_ptr(),
                                       weights_out.data_ptr(), log_ovlp_out.data_ptr(), int(taylor_order),
                                       _stream_ptr(stream))
        self._check(rc, "afqmc_propagate")
        self._last_nw, self._last_energy_nw = n_walkers, 0
        return weights_out, log_ovlp_out

    def propagation_xbar(self, out=None, stream=None):
        """afqmc_propagation_xbar: the shift xbar (Eq. 9) of the last propagate call, complex128 [n_walkers, n_gamma]."""
        out = self._out_for_last_call("propagation_xbar", None, self._last_nw, (self.n_gamma,), out)
        self._check(self._lib.afqmc_propagation_xbar(self._h, out.data_ptr(), _stream_ptr(stream)), "afqmc_propagation_xbar")
        return out

    def propagate_phase_ms(self):
        ms = (C.c_float * 5)()
        self._check(self._lib.afqmc_propagate_phase_ms(self._h, ms), "afqmc_propagate_phase_ms")
        return [float(v) for v in ms]

    def spin_squared(self, n_walkers=None, out=None, stream=None):
        """afqmc_spin_squared: [n_walkers] complex128 <S^2> mixed estimator for the walkers of the last energy /
        force-bias call."""
        out = self._out_for_last_call("spin_squared", n_walkers, self._last_nw, (), out)
        self._check(self._lib.afqmc_spin_squared(self._h, out.data_ptr(), _stream_ptr(stream)), "afqmc_spin_squared")
        return out

    def greens_function(self, spin, n_walkers=None, out=None, stream=None):
        """afqmc_greens_function: full G^sigma [n_walkers, N, N] complex128 (spin 0 = alpha, 1 = beta) for the walkers
        of the last energy / force-bias call."""
        out = self._out_for_last_call("greens_function", n_walkers, self._last_nw, (self.N, self.N), out)
        self._check(self._lib.afqmc_greens_function(self._h, int(spin), out.data_ptr(), _stream_ptr(stream)),
                    "afqmc_greens_function")
        return out

    def info(self) -> dict:
        inf = AfqmcInfo()
        self._check(self._lib.afqmc_get_info(self._h, C.byref(inf)), "afqmc_get_info")
        return _info_dict(inf)

    def set_profiling(self, enable: bool):
        self._check(self._lib.afqmc_set_profiling(self._h, int(bool(enable))), "afqmc_set_profiling")

    def last_kernel_ms(self):
        ms = (C.c_float * 3)()
        self._check(self._lib.afqmc_last_kernel_ms(self._h, ms), "afqmc_last_kernel_ms")
        return [float(x) for x in ms]

    def mean_kernel_ms(self):
        """(mean [K1, K2, K3] ms, number of profiled calls averaged)."""
        ms = (C.c_float * 3)()
        n = C.c_int(0)
        self._check(self._lib.afqmc_mean_kernel_ms(self._h, ms, C.byref(n)), "afqmc_mean_kernel_ms")
        return [float(x) for x in ms], n.value

    def close(self):
        if self._h:
            self._lib.afqmc_destroy(self._h)
            self._h = C.c_void_p(None)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
