"""Host-side emulation of the CUDA FFT engine (csrc/fft.cuh): butterflies, Stockham indexing, pass schedule and
shared-memory padding, checked against a direct O(N^2) DFT in fp64 written inside tests/fft_engine_host.cu.
Needs nvcc (host compile only), no GPU and no oracle."""
import os
import shutil
import subprocess

import pytest

HERE = os.path.dirname(os.path.abspath(__file__))


@pytest.mark.skipif(shutil.which("nvcc") is None, reason="nvcc not on PATH")
def test_fft_engine_host_emulation(tmp_path):
    exe = str(tmp_path / "fft_engine_host")
    subprocess.check_call(["nvcc", "-std=c++17", "-O2", "-Wno-deprecated-gpu-targets", "-x", "cu", "-o", exe,
                           os.path.join(HERE, "fft_engine_host.cu")])
    out = subprocess.run([exe], capture_output=True, text=True)
    assert out.returncode == 0, out.stdout + out.stderr
    assert "worst=" in out.stdout
