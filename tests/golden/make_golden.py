"""Writes tests/golden/oracle_energies.json: oracle energies/log-overlaps for sampled walkers of the five
configs, so that the full-size GPU parity tests need not re-run the expensive rungs each time.

Calls ONLY ``gen/`` (inputs) and ``oracle/`` (values).  Nothing here touches the CUDA path.

    python tests/golden/make_golden.py            # all configs  (~2 h on 8 cores, needs ~20 GB RAM)
    python tests/golden/make_golden.py tiny small # a subset (merged into the existing file)

Rungs (oracle/afqmc_oracle.py): O1 = stored ERIs (the literal definition), O2 = the same definition with the
ERIs generated slab by slab, O3 = Eq. 3 substituted (full G, un-rotated L).  Where two rungs are stored for the
same walker the script asserts that they agree to 1e-11 relative before writing.
"""
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from gen import make_inputs  # noqa: E402
from oracle import afqmc_oracle as orc  # noqa: E402

OUT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_energies.json")

PLAN = {
    # name: (definition rung, its walkers, O3 walkers)
    "tiny": ("O1", "all", "all"),
    "small": ("O1", "all", "all"),
    "medium": ("O2", [0, 1, 2, 63, 64, 126, 127], list(range(0, 128, 8)) + [1, 2, 63, 126, 127]),
    # the headline config: every walker on the Cholesky-direct rung (about 1.7 h on 8 cores), six on the streamed definition
    "cu2o2": ("O2", [0, 1, 127, 128, 254, 255], "all"),
    # large runs K2 with one walker per column tile (wT = 1) and is the only config on the <2,13> kernel with a 6 x 2
    # ring: first / last walkers, both sides of the 148-CTA round boundaries of the tile schedule (147|148, 295|296,
    # 443|444), both sides of the power-of-two marks and a few in between.
    "large": (None, [], [0, 1, 2, 63, 64, 127, 128, 147, 148, 191, 192, 255, 256, 295, 296, 319, 320, 383, 384, 443, 444,
                         447, 448, 477, 500, 509, 510, 511, 37, 101, 222, 350, 413, 470]),
}


def pack(E, lo):
    return dict(E_re=[float(x.real) for x in E], E_im=[float(x.imag) for x in E],
                logabs=[float(x.real) for x in lo], arg=[float(x.imag) for x in lo])


def main(names):
    data = {}
    if os.path.exists(OUT):
        with open(OUT) as f:
            data = json.load(f)
    for name in names:
        t0 = time.time()
        inp = make_inputs(name)
        rung, wdef, wo3 = PLAN[name]
        wdef = list(range(inp.n_walkers)) if wdef == "all" else wdef
        wo3 = list(range(inp.n_walkers)) if wo3 == "all" else sorted(set(wo3))
        entry = dict(config=name, N=inp.N, n_alpha=inp.n_alpha, n_beta=inp.n_beta, n_gamma=inp.n_gamma,
                     n_walkers=inp.n_walkers)
        E3, lo3 = [], []
        for c0 in range(0, len(wo3), 32):                # in chunks, the file is rewritten after each (a long run can be resumed by hand)
            Ec, loc = orc.local_energy_batch(inp, rung="O3", walkers=wo3[c0:c0 + 32])
            E3 += list(Ec); lo3 += list(loc)
            entry["O3"] = dict(walkers=wo3[:len(E3)], **pack(E3, lo3))
            if name in data and "definition" in data[name] and "definition" not in entry:
                entry["definition"] = data[name]["definition"]
            data[name] = entry
            with open(OUT, "w") as f:
                json.dump(data, f, indent=1)
            print(name, "O3", len(E3), "of", len(wo3), time.time() - t0, flush=True)
        print(name, "O3 done", time.time() - t0, flush=True)
        if rung is not None:
            Ed, lod = orc.local_energy_batch(inp, rung=rung, walkers=wdef)
            entry["definition"] = dict(rung=rung, walkers=wdef, **pack(Ed, lod))
            for k, w in enumerate(wdef):
                if w in wo3:
                    j = wo3.index(w)
                    assert abs(Ed[k] - E3[j]) <= 1e-11 * abs(Ed[k]), (name, w, Ed[k], E3[j])
                    assert lod[k] == lo3[j]
            print(name, rung, "done", time.time() - t0, flush=True)
        data[name] = entry
        with open(OUT, "w") as f:
            json.dump(data, f, indent=1)
    print("wrote", OUT)


if __name__ == "__main__":
    main(sys.argv[1:] or list(PLAN))
