"""CPU-only: the register-resident DFT codelets of the PME transforms (csrc/fftx.cuh) and the index algebra of the two-step
kernels built on them (x / y axes; the real z axis as a half-length transform with an even/odd split), compiled as HOST
code and compared with naive fp64 DFTs (tests/host/fft_codelets_check.cu) -- for every size the library instantiates."""
import os
import re
import subprocess

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")


def test_codelets_and_two_step_algebra_on_the_host(tmp_path):
    exe = str(tmp_path / "fft_check")
    src = os.path.join(ROOT, "tests", "host", "fft_codelets_check.cu")
    r = subprocess.run([NVCC, "-O1", "-std=c++17", "-Wno-deprecated-gpu-targets", "-o", exe, src], capture_output=True, text=True)
    assert r.returncode == 0, r.stderr[-2000:]
    out = subprocess.run([exe], capture_output=True, text=True, check=True).stdout
    rows = dict(line.split() for line in out.strip().splitlines())
    sizes = [int(m) for m in re.findall(r"X\((\d+),", open(os.path.join(ROOT, "paper_2503_21176_b200", "csrc", "fftx.cuh")).read())]
    assert len(sizes) == 14
    for n in (2, 3, 4, 5, 6, 8, 9, 10, 12, 16):
        assert float(rows[f"dft{n}"]) < 1e-6, (n, rows[f"dft{n}"])
    for k in sizes:
        # inputs of magnitude 0.5, sums of up to 256 terms in fp32: errors of a few 1e-6 absolute
        assert float(rows[f"twostep{k}"]) < 1e-5, (k, rows[f"twostep{k}"])
        assert float(rows[f"real{k}"]) < 2e-5, (k, rows[f"real{k}"])
