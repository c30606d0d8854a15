"""k_scan's row logic against the plain definition of connectivity, on the host (-m "not gpu"): the naming tables
(constexpr C++) and the per-lane row functions are shared with the kernel (paper_1105_5804_b200/csrc/scan_kernel.cuh);
the checker tests/host/scan_row_check.cu emulates PRMT and the two shuffles and runs whole rows of lanes."""
import os
import subprocess
import tempfile

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_scan_rows_match_the_definition_of_connectivity():
    src = os.path.join(ROOT, "tests", "host", "scan_row_check.cu")
    with tempfile.TemporaryDirectory() as d:
        exe = os.path.join(d, "scan_row_check")
        cmd = ["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-std=c++17", "-O1", "-o", exe, src]
        r = subprocess.run(cmd, capture_output=True, text=True)
        assert r.returncode == 0, r.stderr
        r = subprocess.run([exe], capture_output=True, text=True)
        assert r.returncode == 0 and "scan rows ok: 72000 rows" in r.stdout, r.stdout + r.stderr
