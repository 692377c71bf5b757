"""Hardware-layout contract of the tcgen05 forward planned in DESIGN.md 5.8 (round 2).

Two tiny standalone CUDA programs (tests/umma_probe/*.cu, compiled here with nvcc for sm_100a) check, with
exact small-integer fp16 data, that `tcgen05.mma` reads the shared-memory tiles this library already
produces exactly as DESIGN.md 5.8 states:

* umma_mn_major_probe: S^T = V^T K over a [16 rows x 128 channels] K and V tile loaded by the same 2-D TMA
  boxes as the forward kernels (64 channels x rows, 128-byte swizzle), both operands MN-major
  (leading byte offset = distance between the two 64-channel boxes, stride byte offset = 1024);
* umma_k_major_probe: O = A B^T with A = a [128 x 128] TMA tile used in place (K-major, one k-step of 16
  channels = +32 bytes inside the swizzled row, the second 64 channels in the next box) and B = a
  [144 x 128] operand written by the threads with the 128-byte swizzle applied by hand.

They share no code with the product kernels or the oracle; the expected values are brute-force host loops.
"""
import os
import shutil
import subprocess

import pytest

HERE = os.path.dirname(os.path.abspath(__file__))
PROBES = {
    "umma_mn_major_probe": "lbo 2048 sbo 1024: max err vs V^T K: 0 ;",
    "umma_k_major_probe": "K-major M=128 N=144 K=128: max err 0",
}


@pytest.mark.gpu
@pytest.mark.parametrize("name", sorted(PROBES))
def test_umma_layout_probe(name, tmp_path):
    nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(nvcc):
        pytest.skip("nvcc not available on this box")
    exe = str(tmp_path / name)
    src = os.path.join(HERE, "umma_probe", name + ".cu")
    subprocess.check_call([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O2", "-std=c++17", src, "-o", exe])
    out = subprocess.run([exe], capture_output=True, text=True, timeout=120)
    assert out.returncode == 0, out.stdout + out.stderr
    assert "kernel: no error" in out.stdout, out.stdout
    assert PROBES[name] in out.stdout, out.stdout
