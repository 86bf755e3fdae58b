"""One rank of the N > 1 host protocol bench.py uses, on CPU: rank and world from the torchrun environment, `gloo`
process group, this rank's block of the weak-scaling population, evaluation of ITS walkers (the CPU oracle stands in for
the GPU call, which needs a device), gather in global walker order, digest and max-over-ranks timing.  Rank 0 prints
one JSON line.  Started by tests/test_multirank_host.py through parallel.respawn_under_torchrun."""
import json
import os
import sys

import numpy as np
import torch

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))

from gen import make_inputs  # noqa: E402
from oracle import afqmc_oracle as orc  # noqa: E402
from paper_2209_04015_b200.parallel import (gather_walker_results, init_from_env, max_over_ranks, result_digest,  # noqa: E402
                                            weak_scaling_block)


def main():
    nw = int(sys.argv[1])
    rank, world, _ = init_from_env("gloo")
    start, count = weak_scaling_block(nw, rank, world)
    inp = make_inputs("tiny", n_walkers=world * nw)
    E, _ = orc.local_energy_batch(inp, rung="O3", walkers=list(range(start, start + count)))
    all_E = gather_walker_results(torch.from_numpy(np.asarray(E, dtype=np.complex128)), world * nw)
    tmax = max_over_ranks(10.0 + rank)
    if rank == 0:
        print(json.dumps({"world": world, "first_block_sha256": result_digest(all_E[:nw]),
                          "all_blocks_sha256": result_digest(all_E), "tmax": tmax}), flush=True)
    if world > 1:
        torch.distributed.barrier()
        torch.distributed.destroy_process_group()


if __name__ == "__main__":
    main()
