"""Register FFT building blocks (fe_fft2.cuh) on the host against the O(N^2) DFT definition.

The butterflies, recursions and pruning rules the CUDA passes are built from are `__host__ __device__`
templates; this test compiles them for the host with nvcc (no GPU needed) and checks every instantiated
length / direction / pruning mode against the definition of the discrete Fourier transform.  A wrong twiddle
constant, sign or pruning rule fails here before any kernel runs.
"""
import os
import shutil
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")


@pytest.mark.skipif(not (os.path.exists(NVCC) or shutil.which("nvcc")), reason="nvcc not available")
def test_register_fft_blocks_match_dft_definition(tmp_path):
    nvcc = NVCC if os.path.exists(NVCC) else shutil.which("nvcc")
    exe = str(tmp_path / "host_fft_blocks")
    src = os.path.join(ROOT, "tests", "host_fft_blocks.cu")
    inc = [os.path.join(ROOT, "paper_2605_28800_b200", "csrc"), os.path.join(ROOT, "include")]
    cmd = [nvcc, "-std=c++17", "-O1", "-w", "-o", exe, src] + ["-I" + i for i in inc]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr
    out = subprocess.run([exe], capture_output=True, text=True, timeout=60)
    assert out.returncode == 0, out.stderr
    lines = [l.split() for l in out.stdout.strip().splitlines()]
    assert len(lines) >= 26
    for name, n, err in lines:
        tol = 2e-6 if name.startswith("f32") else 2e-14       # a few ulp times log2(N) stages
        assert float(err) < tol, (name, n, err)
