"""GPU parity of afqmc_sample_fields (the auxiliary fields of Eq. 4) against oracle/rng_oracle.py: the generator is
counter-based, so both sides must produce the same numbers from (seed, step, walker, gamma) alone.  The integer stream
is bit-exact by construction; what is compared here are the normals, which go through log / sqrt / sincos on both sides:
a few ulp of |x| <= 8.7, i.e. 1e-14 absolute."""
import numpy as np
import pytest
import torch

from oracle import rng_oracle as rng

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("seed,step,nw,ng,first", [
    (0, 0, 1, 1, 0),                                   # a single field (half a pair)
    (0x0123456789ABCDEF, 3, 7, 9, 0),                  # odd Ngamma, 64-bit seed
    (2 ** 64 - 1, 2 ** 40 + 5, 5, 64, 1000),           # step beyond 32 bits, walker offset
    (1234, 17, 256, 2000, 0),                          # the bench's shape (Cu2O2 scale)
])
def test_fields_equal_the_oracle(seed, step, nw, ng, first):
    from paper_2209_04015_b200 import sample_fields
    x = sample_fields(seed, step, nw, ng, first_walker=first).cpu().numpy()
    ref = rng.sample_fields(seed, step, nw, ng, first_walker=first)
    assert x.shape == ref.shape
    assert np.max(np.abs(x - ref)) <= 1e-14
    assert np.mean(x == ref) > 0.5                     # most values agree to the last bit


def test_fields_do_not_depend_on_the_batch_and_are_reproducible():
    from paper_2209_04015_b200 import sample_fields
    a = sample_fields(99, 4, 40, 33)
    b = sample_fields(99, 4, 10, 33, first_walker=25)
    c = sample_fields(99, 4, 40, 33)
    assert torch.equal(a[25:35], b) and torch.equal(a, c)
    assert not torch.equal(a, sample_fields(99, 5, 40, 33)) and not torch.equal(a, sample_fields(98, 4, 40, 33))


def test_propagate_with_library_drawn_fields_matches_oracle_with_oracle_drawn_fields():
    """The whole step with x from afqmc_sample_fields against the oracle's step with x from its own generator."""
    from oracle import propagation_oracle as prop
    from paper_2209_04015_b200 import sample_fields
    from tests.test_gpu_parity import _le
    from gen import make_inputs
    inp = make_inputs("tiny")
    nw, dt = inp.n_walkers, 0.002
    le = _le(inp)
    le.enable_propagation(torch.from_numpy(inp.h1e).cuda(), torch.from_numpy(inp.chol).cuda(), dt)
    x = sample_fields(7, 0, nw, inp.n_gamma)
    wk = torch.from_numpy(inp.walkers_packed()).cuda()
    w_new, _ = le.propagate(wk, nw, x, torch.ones(nw, dtype=torch.float64, device="cuda"), taylor_order=40)
    torch.cuda.synchronize()
    xo = rng.sample_fields(7, 0, nw, inp.n_gamma)
    out = wk.cpu().numpy()[: nw * inp.N * inp.n_alpha].reshape(nw, inp.N, inp.n_alpha)
    for w in range(nw):
        ref = prop.propagate_walker(inp.h1e, inp.chol, inp.psi_a, inp.psi_b, inp.phi_a[w], inp.phi_b[w], 1.0, xo[w], dt)
        assert np.max(np.abs(out[w] - ref["phi_a"])) <= 1e-10 * np.max(np.abs(ref["phi_a"]))
        assert abs(w_new[w].item() - ref["weight"]) <= 1e-9 * max(abs(ref["weight"]), 1e-300)
    le.close()
