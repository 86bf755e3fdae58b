"""afqmc_log_overlap_static -- the entry point that allocates nothing (include/afqmc.h): its scratch is a file-scope device
array of AFQMC_STATIC_SCRATCH_BYTES.  Checked against the existing path (afqmc_create + afqmc_local_energy's out_overlaps)
within the tolerance of tests/test_gpu_parity.py (1e-10 relative), on two calls in a row of different shape -- the array keeps
the first call's contents, so the second call must have cleared what has to start at zero.

Named test_zz_* so that pytest collects it last: the suite runs with pytest -x, and a failure here must not hide other tests.
Passes alone in a fresh process and after the other tests (it shares no state with them but the loaded library)."""
import math

import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu
RTOL = 1e-10


def _existing_path(inp):
    from paper_2209_04015_b200 import LocalEnergy
    dev = "cuda"
    le = LocalEnergy(torch.from_numpy(inp.h1e).to(dev), torch.from_numpy(inp.chol).to(dev), torch.from_numpy(inp.trial_packed()).to(dev),
                     inp.N, inp.n_alpha, inp.n_beta, inp.n_gamma, inp.e0, inp.n_walkers)
    _, lo = le.local_energy(torch.from_numpy(inp.walkers_packed()).to(dev), inp.n_walkers)
    torch.cuda.synchronize()
    lo = lo.cpu().numpy()
    le.close()
    return lo


def _assert_same(lo, ref):
    dre = np.abs(lo.real - ref.real) / np.maximum(1.0, np.abs(ref.real))
    assert np.all(dre <= RTOL), f"log|ovlp| err max {dre.max():.3e}"
    dim = np.abs((lo.imag - ref.imag + math.pi) % (2 * math.pi) - math.pi)
    assert np.all(dim <= RTOL * np.maximum(1.0, np.abs(ref.real))), f"arg ovlp err max {dim.max():.3e}"


def test_static_entry_point_matches_the_existing_path_on_two_calls_in_a_row():
    from gen import make_inputs
    from paper_2209_04015_b200 import log_overlap_static
    from tests.test_gpu_parity import _custom
    cases = [make_inputs("small", n_walkers=40, n_gamma=8),               # N = 100, n = 20: the larger footprint first
             _custom(4242, 37, 9, 0, 5, 11, complex_trial=True),           # then a smaller, complex-trial, one-spin, odd-sized one
             _custom(4243, 70, 33, 31, 4, 3)]                              # and n > 32 (another kernel instantiation)
    refs = [_existing_path(c) for c in cases]
    dev = "cuda"
    args = [(torch.from_numpy(c.trial_packed()).to(dev), torch.from_numpy(c.walkers_packed()).to(dev),
             torch.empty(c.n_walkers, dtype=torch.complex128, device=dev)) for c in cases]
    torch.cuda.synchronize()
    free0 = None
    for rep in range(2):                                                  # the whole sequence twice: six calls sharing one array
        for c, (trial, walkers, out), ref in zip(cases, args, refs):
            out.fill_(float("nan"))
            log_overlap_static(trial, walkers, c.N, c.n_alpha, c.n_beta, c.n_walkers, out=out)
            torch.cuda.synchronize()
            _assert_same(out.cpu().numpy(), ref)
            if free0 is None:
                free0 = torch.cuda.mem_get_info()[0]                       # after the first call (module loading is behind us)
    assert torch.cuda.mem_get_info()[0] == free0                          # no call took device memory


def test_static_entry_point_rejects_what_does_not_fit():
    from paper_2209_04015_b200 import AfqmcError, log_overlap_static
    N, n, nw = 290, 26, 63                                                 # one walker more than fits (afqmc.h)
    trial = torch.zeros(N * 2 * n, dtype=torch.complex128, device="cuda")
    walkers = torch.zeros(nw * N * 2 * n, dtype=torch.complex128, device="cuda")
    with pytest.raises(AfqmcError, match="bytes of scratch"):
        log_overlap_static(trial, walkers, N, n, n, nw)
    with pytest.raises(AfqmcError, match="n_sigma"):
        log_overlap_static(torch.zeros(100 * 65, dtype=torch.complex128, device="cuda"),
                           torch.zeros(100 * 65, dtype=torch.complex128, device="cuda"), 100, 65, 0, 1)
