"""World-size-2 `gloo` test (CPU) of the N > 1 host logic: walker sharding, gathering of per-walker results in the
global order, max-over-ranks of a timing.  Each rank evaluates ITS walkers (here with the CPU oracle standing in for
the GPU call, which needs a device) and the gathered vector must equal the single-process result."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2209_04015_b200.parallel import gather_walker_results, max_over_ranks, walker_shard


def test_walker_shard_partitions_exactly():
    for nw in (0, 1, 4, 7, 256, 513):
        for world in (1, 2, 3, 8):
            blocks = [walker_shard(nw, r, world) for r in range(world)]
            assert sum(c for _, c in blocks) == nw
            pos = 0
            for s, c in blocks:
                assert s == pos and c >= 0
                pos += c
            counts = [c for _, c in blocks]
            assert max(counts) - min(counts) <= 1
    with pytest.raises(ValueError):
        walker_shard(4, 2, 2)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, nw, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from gen import make_inputs
        from oracle import afqmc_oracle as orc
        inp = make_inputs("tiny", n_walkers=nw)
        start, count = walker_shard(nw, rank, world)
        idx = list(range(start, start + count))
        if count:
            E, lo = orc.local_energy_batch(inp, rung="O3", walkers=idx)
        else:
            E, lo = np.zeros(0, complex), np.zeros(0, complex)
        Eg = gather_walker_results(torch.from_numpy(np.asarray(E, dtype=np.complex128)), nw)
        log = gather_walker_results(torch.from_numpy(np.asarray(lo, dtype=np.complex128)), nw)
        tmax = max_over_ranks(10.0 + rank)
        if rank == 0:
            q.put((Eg.numpy(), log.numpy(), tmax))
        dist.barrier()
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("nw", [4, 3])
def test_two_ranks_gather_equals_single_process(nw):
    from gen import make_inputs
    from oracle import afqmc_oracle as orc
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, nw, q)) for r in range(world)]
    for p in procs:
        p.start()
    Eg, log, tmax = q.get(timeout=240)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    inp = make_inputs("tiny", n_walkers=nw)
    E, lo = orc.local_energy_batch(inp, rung="O3")
    assert np.array_equal(Eg, np.asarray(E)) and np.array_equal(log, np.asarray(lo))
    assert tmax == 11.0


def test_respawn_under_torchrun_runs_the_weak_scaling_protocol():
    """`python bench.py --gpus N` without torchrun re-launches itself with parallel.respawn_under_torchrun; here the
    same helper starts tests/multirank_worker.py as 2 gloo ranks.  The first block's digest must equal the one-rank
    run's (bit-identical energies), and the whole job's digest the single-process evaluation of all walkers."""
    import json
    import subprocess
    import sys
    from paper_2209_04015_b200.parallel import respawn_under_torchrun, result_digest, torchrun_command, weak_scaling_block
    from gen import make_inputs
    from oracle import afqmc_oracle as orc
    worker = os.path.join(os.path.dirname(os.path.abspath(__file__)), "multirank_worker.py")
    cmd = torchrun_command(worker, 2, ["3"], port=1234)
    assert cmd[1:3] == ["-m", "torch.distributed.run"] and "--nproc-per-node=2" in cmd and "127.0.0.1" in cmd
    assert weak_scaling_block(3, 1, 2) == (3, 3)
    two = respawn_under_torchrun(worker, 2, ["3"], stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True, timeout=600)
    assert two.returncode == 0, two.stderr[-2000:]
    r2 = json.loads([ln for ln in two.stdout.splitlines() if ln.startswith("{")][-1])
    one = subprocess.run([sys.executable, worker, "3"], stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True, timeout=600,
                         env={k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK")})
    assert one.returncode == 0, one.stderr[-2000:]
    r1 = json.loads([ln for ln in one.stdout.splitlines() if ln.startswith("{")][-1])
    assert r2["world"] == 2 and r1["world"] == 1 and r2["tmax"] == 11.0
    assert r2["first_block_sha256"] == r1["first_block_sha256"] == r1["all_blocks_sha256"]
    E, _ = orc.local_energy_batch(make_inputs("tiny", n_walkers=6), rung="O3")
    assert r2["all_blocks_sha256"] == result_digest(torch.from_numpy(np.asarray(E, dtype=np.complex128)))
