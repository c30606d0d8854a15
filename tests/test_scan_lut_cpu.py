"""k_scan's permutation tables against the plain definition of run naming, on the host (-m "not gpu"): the table
generator is constexpr C++ shared with the kernel (paper_1105_5804_b200/csrc/scan_kernel.cuh), the checker
tests/host/scan_lut_check.cu emulates PRMT and enumerates every pattern."""
import os
import subprocess
import tempfile

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_scan_tables_match_the_definition_of_run_naming():
    src = os.path.join(ROOT, "tests", "host", "scan_lut_check.cu")
    with tempfile.TemporaryDirectory() as d:
        exe = os.path.join(d, "scan_lut_check")
        cmd = ["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-std=c++17", "-O1", "-o", exe, src]
        r = subprocess.run(cmd, capture_output=True, text=True)
        assert r.returncode == 0, r.stderr
        r = subprocess.run([exe], capture_output=True, text=True)
        assert r.returncode == 0 and "scan tables ok: 4096 cases" in r.stdout, r.stdout + r.stderr
