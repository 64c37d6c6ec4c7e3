"""CPU check of the shared-memory FFT core of the fused theta chains (csrc/fft_smem.cuh): its stage
functions are __host__ __device__, so tests/fft_smem_host_check.cu runs the "threads" sequentially on
the host and compares every supported length with a direct long-double DFT (a definition, not another
FFT): forward chain at digit-reversed positions, inverse chain as its exact inverse."""
import os
import shutil
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_fft_smem_against_direct_dft(tmp_path):
    nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(nvcc):
        pytest.skip("nvcc not available")
    exe = str(tmp_path / "fft_check")
    src = os.path.join(ROOT, "tests", "fft_smem_host_check.cu")
    subprocess.check_call([nvcc, "-std=c++17", "-O1", "-Wno-deprecated-gpu-targets", "-o", exe, src])
    out = subprocess.run([exe], capture_output=True, text=True)
    assert out.returncode == 0, out.stdout + out.stderr
    assert "OK" in out.stdout


def test_fft_reg_against_direct_dft(tmp_path):
    """The register-tiled 4096-point transform of the fused phi kernels (csrc/fft_reg.cuh), phase by phase on the host."""
    nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(nvcc):
        pytest.skip("nvcc not available")
    exe = str(tmp_path / "fft_reg_check")
    src = os.path.join(ROOT, "tests", "fft_reg_host_check.cu")
    subprocess.check_call([nvcc, "-std=c++17", "-O1", "-Wno-deprecated-gpu-targets", "-o", exe, src])
    out = subprocess.run([exe], capture_output=True, text=True)
    assert out.returncode == 0, out.stdout + out.stderr
    assert "OK" in out.stdout
