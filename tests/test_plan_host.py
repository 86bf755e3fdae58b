"""Host logic of the library that runs without a GPU: afqmc_plan (the K2 tile-shape planner) and argument checks."""
import pytest

from gen import CONFIGS
from paper_2209_04015_b200 import AfqmcError, plan

SMEM_MAX = 232448     # 227 KB opt-in dynamic shared memory per CTA on sm_100


@pytest.mark.parametrize("name", list(CONFIGS))
def test_plan_is_consistent_for_the_five_configs(name):
    c = CONFIGS[name]
    p = plan(c["N"], c["n_alpha"], c["n_beta"], c["n_gamma"], c["n_walkers"])
    assert p["k_steps"] == (c["N"] + 3) // 4
    for s, n in enumerate((c["n_alpha"], c["n_beta"])):
        rows, cols = p["tile_rows"][s], p["tile_cols"][s]
        gT, wT = p["gammas_per_tile"][s], p["walkers_per_tile"][s]
        assert rows % 8 == 0 and cols % 8 == 0
        assert gT * n <= rows < gT * n + 8              # whole gamma blocks, padded only in the last strip
        assert 2 * wT * n <= cols < 2 * wT * n + 8      # both planes of wT walkers, padded only in the last block
        assert rows // 8 <= p["mt"][s] * p["warps_m"][s] and cols // 8 == p["nt"][s]
        assert p["mt"][s] * p["nt"][s] <= 26            # accumulator tiles per warp (register budget)
        assert p["stages"][s] >= 2 and p["ksteps_per_chunk"][s] >= 1
        assert 0 < p["k2_smem_bytes"][s] <= SMEM_MAX
    assert p["ltilde_bytes"] >= 8 * c["n_gamma"] * c["N"] * (c["n_alpha"] + c["n_beta"])
    assert p["theta_bytes"] >= 16 * c["n_walkers"] * c["N"] * (c["n_alpha"] + c["n_beta"])


def test_headline_tile_wastes_little():
    c = CONFIGS["cu2o2"]
    p = plan(c["N"], c["n_alpha"], c["n_beta"], c["n_gamma"], c["n_walkers"])
    useful = (p["gammas_per_tile"][0] * 26) * (2 * p["walkers_per_tile"][0] * 26)
    assert useful / (p["tile_rows"][0] * p["tile_cols"][0]) > 0.95


@pytest.mark.parametrize("args", [(0, 1, 1, 1, 1), (10, 11, 1, 1, 1), (10, -1, 1, 1, 1), (10, 0, 0, 5, 1), (10, 3, 3, 0, 1), (10, 3, 3, 5, 0)])
def test_plan_rejects_bad_sizes(args):
    with pytest.raises(AfqmcError, match="out of range"):
        plan(*args)


def test_plan_reports_unsupported_occupation():
    with pytest.raises(AfqmcError, match="not supported"):
        plan(200, 65, 3, 10, 4)


@pytest.mark.parametrize("n", [1, 2, 3, 7, 8, 9, 31, 33, 64])
def test_plan_handles_any_occupation(n):
    p = plan(max(n, 70), n, max(n - 1, 0), 50, 9)
    assert p["k2_smem_bytes"][0] <= SMEM_MAX and p["tile_rows"][0] >= n


def test_every_compiled_k2_instantiation_has_a_witness_shape():
    """k2_pick (csrc/afqmc.cu) instantiates k2_exchange<MT, NT> for NT = 1..NTmax(MT); tests/k2_instances.py must name,
    for each of them, a problem the planner maps to it (the GPU suite launches every row against the oracle)."""
    import os
    import re
    from tests.k2_instances import WITNESS
    src = open(os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "paper_2209_04015_b200", "csrc",
                            "afqmc.cu")).read()
    compiled = set()
    for mt, ntmax in re.findall(r"case (\d): return k2_pick_nt<\d, (\d+)>\(nt\);", src):
        compiled |= {(int(mt), nt) for nt in range(1, int(ntmax) + 1)}
    assert len(compiled) == 43 and compiled == set(WITNESS)
    for (mt, nt), (n, cx, N, ng, nw) in WITNESS.items():
        p = plan(N, n, 0, ng, nw, complex_alpha=bool(cx))
        assert (p["mt"][0], p["nt"][0], p["warps_m"][0]) == (mt, nt, 12), ((mt, nt), p)


def test_complex_trial_occupation_limit_is_reported():
    """A complex trial block stacks Re / Im rows (2 n rows per gamma block): it fits a K2 tile up to n = 52."""
    plan(60, 52, 3, 10, 4, complex_alpha=True)
    with pytest.raises(AfqmcError, match="no K2 tile shape"):
        plan(60, 53, 3, 10, 4, complex_alpha=True)
