"""A C99 program as a client of the C ABI (tests/c_caller/afqmc_c_caller.c): the header must compile as plain C and link
against libafqmc.so without any C++ or Python in between (CPU test), and its results must equal the Python binding's bit
for bit and the oracle's to 1e-10 (GPU test)."""
import os
import struct
import subprocess

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = os.path.join(ROOT, "tests", "c_caller", "afqmc_c_caller.c")
CUDA = os.environ.get("CUDA_HOME", "/usr/local/cuda")


def _build(tmp_path):
    from paper_2209_04015_b200.build import build_library
    lib = build_library()
    exe = str(tmp_path / "afqmc_c_caller")
    cmd = ["gcc", "-std=c99", "-O1", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), "-I", os.path.join(CUDA, "include"), SRC,
           "-o", exe, lib, "-L", os.path.join(CUDA, "lib64"), "-lcudart", f"-Wl,-rpath,{os.path.dirname(lib)}",
           f"-Wl,-rpath,{os.path.join(CUDA, 'lib64')}"]
    res = subprocess.run(cmd, capture_output=True, text=True)
    assert res.returncode == 0, res.stderr
    return exe


def test_header_is_plain_c_and_the_library_links_from_c(tmp_path):
    exe = _build(tmp_path)
    res = subprocess.run([exe], capture_output=True, text=True)          # no arguments: usage message, no CUDA call
    assert res.returncode == 1 and "usage" in res.stderr


@pytest.mark.gpu
def test_c_program_reproduces_the_binding_and_the_oracle(tmp_path):
    import torch
    from gen import make_inputs
    from oracle import afqmc_oracle as orc
    from paper_2209_04015_b200 import LocalEnergy
    exe = _build(tmp_path)
    inp = make_inputs("small", n_walkers=21, n_gamma=37)
    fin, fout = str(tmp_path / "in.bin"), str(tmp_path / "out.bin")
    with open(fin, "wb") as f:
        f.write(struct.pack("<5id", inp.N, inp.n_alpha, inp.n_beta, inp.n_gamma, inp.n_walkers, inp.e0))
        for a in (inp.h1e, inp.chol, inp.trial_packed(), inp.walkers_packed()):
            f.write(np.ascontiguousarray(a).tobytes())
    res = subprocess.run([exe, fin, fout], capture_output=True, text=True, timeout=600)
    assert res.returncode == 0, res.stdout + res.stderr
    nw = inp.n_walkers
    out = np.fromfile(fout, dtype=np.complex128).reshape(4, nw)
    assert np.array_equal(out[0].view(np.float64), out[2].view(np.float64))      # host entry = device entry, bit for bit
    assert np.array_equal(out[1].view(np.float64), out[3].view(np.float64))
    dev = "cuda"
    le = LocalEnergy(torch.from_numpy(inp.h1e).to(dev), torch.from_numpy(inp.chol).to(dev), torch.from_numpy(inp.trial_packed()).to(dev),
                     inp.N, inp.n_alpha, inp.n_beta, inp.n_gamma, inp.e0, nw)
    E, lo = le.local_energy(torch.from_numpy(inp.walkers_packed()).to(dev), nw)
    torch.cuda.synchronize()
    assert np.array_equal(E.cpu().numpy().view(np.float64), out[2].view(np.float64))   # same library, same bits
    le.close()
    Eo, loo = orc.local_energy_batch(inp, rung="O3")
    assert np.all(np.abs(out[0] - Eo) <= 1e-10 * np.abs(Eo))
    assert np.all(np.abs(out[1].real - np.asarray(loo).real) <= 1e-10 * np.maximum(1.0, np.abs(np.asarray(loo).real)))
