"""GPU checks of the Ozaki-scheme experiment (include/afqmc_ozaki.h): the INT8 tcgen05 GEMM must be
EXACT where the digits represent the inputs exactly, and its error must fall by 2^-7 per extra digit plane otherwise."""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu


def _gemm(A, B, slices):
    from paper_2209_04015_b200.ozaki import ozaki_gemm
    out = ozaki_gemm(torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda(), slices)
    torch.cuda.synchronize()
    return out["C"].cpu().numpy(), out


@pytest.mark.parametrize("M,Ncol,K", [(128, 64, 32), (200, 100, 70), (390, 333, 290)])
def test_small_integer_inputs_are_reproduced_exactly(M, Ncol, K):
    """Integers of magnitude <= 60 fit ONE 7-bit digit after the power-of-two scaling, so with two planes every kept
    product is exact: the result must equal the integer matrix product bit for bit (tests the UMMA descriptors, the
    core-matrix packing, the weight-class accumulation in TMEM and ragged edge tiles)."""
    rng = np.random.default_rng(M + K)
    A = rng.integers(-60, 61, (M, K)).astype(np.float64) * 0.25
    B = rng.integers(-60, 61, (Ncol, K)).astype(np.float64) * 8.0
    C, _ = _gemm(A, B, 2)
    assert np.array_equal(C, A @ B.T)


def test_error_falls_by_seven_bits_per_digit_plane_and_reaches_double_precision():
    rng = np.random.default_rng(5)
    M, Ncol, K = 300, 260, 290
    A = rng.standard_normal((M, K)) * np.exp(rng.uniform(-3, 3, (M, 1)))      # rows of very different scale
    B = rng.standard_normal((Ncol, K)) * np.exp(rng.uniform(-3, 3, (Ncol, 1)))
    ref = (A.astype(np.longdouble) @ B.T.astype(np.longdouble)).astype(np.float64)
    scale = np.max(np.abs(A), axis=1)[:, None] * np.max(np.abs(B), axis=1)[None, :] * K
    errs = []
    for s in range(1, 9):
        C, _ = _gemm(A, B, s)
        errs.append(np.max(np.abs(C - ref) / scale))
    for s in range(1, 7):
        assert errs[s] < errs[s - 1] / 30, errs           # ~2^-7 = 1/128 per plane, with slack
    assert errs[7] < 1e-15, errs


def test_argument_errors():
    from paper_2209_04015_b200 import AfqmcError
    from paper_2209_04015_b200.ozaki import ozaki_gemm
    A = torch.zeros((8, 8), dtype=torch.float64, device="cuda")
    with pytest.raises(AfqmcError, match="slices"):
        ozaki_gemm(A, A, 9)
    with pytest.raises(AfqmcError, match="share K"):
        ozaki_gemm(A, torch.zeros((8, 9), dtype=torch.float64, device="cuda"), 2)
