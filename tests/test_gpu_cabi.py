"""The boundary is a C ABI with plain pointers: tests/cabi_client.c, a C program with no Python and no torch in
it, is compiled against include/nyxrt.h, linked with libnyxrt.so and the CUDA runtime, and run on config 1; what it
prints must equal the Python binding's result bit for bit where integers are concerned and to the summation order
otherwise, and the oracle's by the parity rule."""
import os
import shutil
import subprocess

import numpy as np
import pytest

from paper_2512_12466_b200 import synth
from parity import run_gpu, run_oracle

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_plain_c_client(O, tmp_path):
    import __graft_entry__
    __graft_entry__.build()
    cuda = os.environ.get("CUDA_HOME", "/usr/local/cuda")
    if not shutil.which("gcc") or not os.path.exists(os.path.join(cuda, "include", "cuda_runtime.h")):
        pytest.skip("no C toolchain / CUDA headers on this box")
    exe = str(tmp_path / "cabi_client")
    libdir = os.path.join(ROOT, "paper_2512_12466_b200")
    subprocess.check_call(["gcc", "-std=c99", "-O1", "-Wall", "-I", os.path.join(ROOT, "include"), "-I",
                           os.path.join(cuda, "include"), os.path.join(ROOT, "tests", "cabi_client.c"), "-o", exe,
                           "-L", libdir, "-lnyxrt", "-L", os.path.join(cuda, "lib64"), "-lcudart",
                           "-Wl,-rpath," + libdir, "-Wl,-rpath," + os.path.join(cuda, "lib64")])
    r = subprocess.run([exe], capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, (r.returncode, r.stderr)
    v = r.stdout.split()
    ints = [int(x) for x in v[:7]]
    absorbed, emitted, gsum, gnb = [float(x) for x in v[7:]]
    cfg = synth.make(1)
    gam, heat, st, cat = run_gpu(cfg)
    go, ho, so, co = run_oracle(O, cfg)
    assert ints == [st.segments] + list(st.spawned[:5]) + [sum(st.killed_tau)]
    assert ints == [so.segments] + list(so.spawned[:5]) + [sum(so.killed_tau)]
    assert emitted == 5e48 and abs(absorbed - so.photons_absorbed) <= 1e-12 * so.photons_absorbed
    assert abs(gsum - go.sum()) <= 1e-9 * go.sum() and abs(gnb - go[16, 16, 17]) <= 1e-9 * go[16, 16, 17]
    assert abs(gsum - gam.sum()) <= 1e-12 * gam.sum()
