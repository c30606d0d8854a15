"""CPU-side checks of the C-ABI library: it loads, exports every symbol the header declares, validates arguments and
computes the same thresholds as the oracle.  No kernel is launched here (-m "not gpu")."""
import ctypes as C
import math
import os
import re

import pytest

import oracle
from paper_1105_5804_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()                      # nvcc cross-compiles sm_100a without a GPU
    return binding.lib()


def header_functions():
    text = open(os.path.join(ROOT, "include", "swb200.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    names = re.findall(r"\b(?:int|size_t|const char\*)\s+(\w+)\s*\(", text)
    return sorted(set(names))


def test_library_exports_every_declared_symbol(lib):
    declared = header_functions()
    assert len(declared) >= 19 and "sw_sweep" in declared and "wolff_step" in declared
    assert sorted(binding.SYMBOLS) == declared
    for name in declared:
        assert hasattr(lib, name), name


def test_library_is_sm100a_cuda_code():
    import subprocess
    out = subprocess.run(["cuobjdump", "-lelf", binding.LIB_PATH], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_create_validates_arguments(lib):
    h = C.c_void_p()
    bc = oracle.beta_c(2)
    for L, q, beta in [(2, 2, bc), (6, 2, bc), (65536, 2, bc), (64, 1, bc), (64, 9, bc), (64, 2, -0.1),
                       (64, 2, float("nan")), (64, 2, float("inf"))]:
        assert lib.sw_create(C.byref(h), L, q, beta, 1) == binding.SW_EINVAL, (L, q, beta)
        assert not h.value
    assert lib.sw_create(None, 64, 2, bc, 1) == binding.SW_EINVAL
    assert lib.sw_create(C.byref(h), 64, 2, bc, 1) == binding.SW_OK
    # unbound handle: every device entry point refuses without touching CUDA
    assert lib.sw_sweep(h, 1, None) == binding.SW_ESTATE
    assert lib.sw_init_spins(h, 1, None) == binding.SW_ESTATE
    assert lib.sw_label(h, None, None, None) == binding.SW_ESTATE
    assert lib.sw_activate(h, None) == binding.SW_ESTATE
    assert lib.wolff_step(h, 1, None, None) == binding.SW_ESTATE
    obs = binding.sw_obs()
    assert lib.sw_observables(h, C.byref(obs), None) == binding.SW_ESTATE
    assert lib.sw_sweep(h, -1, None) == binding.SW_EINVAL
    assert lib.sw_fewcluster_step(h, 1, 4, 1, None, None) == binding.SW_ESTATE
    assert lib.sw_fewcluster_step(h, 1, 70000, 1, None, None) == binding.SW_EINVAL
    # misaligned / NULL buffers, short workspace
    wb = lib.sw_workspace_bytes(64, 2)
    assert lib.sw_bind(h, None, 16, None, 32, wb, None) == binding.SW_EINVAL
    assert lib.sw_bind(h, 16 + 1, 32, None, 48, wb, None) == binding.SW_EINVAL
    assert lib.sw_bind(h, 16, 32, None, 48, wb - 1, None) == binding.SW_EINVAL
    # counter / threshold accessors
    t = C.c_uint64()
    assert lib.sw_get_counter(h, C.byref(t)) == 0 and t.value == 0
    assert lib.sw_set_counter(h, (7 << 32) | 5) == 0
    assert lib.sw_get_counter(h, C.byref(t)) == 0 and t.value == (7 << 32) | 5
    T = C.c_uint32()
    assert lib.sw_set_threshold(h, 123) == 0 and lib.sw_get_threshold(h, C.byref(T)) == 0 and T.value == 123
    assert lib.sw_destroy(h) == 0
    assert lib.sw_destroy(None) == binding.SW_EINVAL
    hp = C.c_void_p()
    assert lib.sw_create(C.byref(hp), 64, 3, 1.0, 1) == 0
    assert lib.wolff_step(hp, 1, None, None) == binding.SW_EINVAL      # Wolff is defined for q=2 only
    lib.sw_destroy(hp)


def test_thresholds_equal_the_oracles(lib):
    cases = [(2, oracle.beta_c(2)), (2, 0.40), (2, 0.50), (2, 0.0), (2, 0.3), (3, oracle.beta_c(3)),
             (4, math.log(3.0)), (4, 0.7), (8, oracle.beta_c(8)), (2, 50.0)]
    for q, beta in cases:
        h = C.c_void_p()
        assert lib.sw_create(C.byref(h), 16, q, beta, 0) == 0
        T = C.c_uint32()
        assert lib.sw_get_threshold(h, C.byref(T)) == 0
        assert T.value == oracle.threshold(q, beta), (q, beta)
        lib.sw_destroy(h)


def test_workspace_bytes_and_strerror(lib):
    assert lib.sw_workspace_bytes(6, 2) == 0 and lib.sw_workspace_bytes(64, 9) == 0
    for L in (4, 64, 100, 1024, 16384):
        wb = lib.sw_workspace_bytes(L, 2)
        ntx, nty = -(-L // 128), -(-L // 32)
        # cluster sizes + the two int32 edge arrays (the draw cache is not part of the default build: nothing reserved for it)
        need = 4 * L * L + 2 * 4 * (ntx + nty) * L
        assert need <= wb < need + 65536 + 4096 * 16 + 16384    # + the (sat, minus) ring of sw_series_read, accumulators
    assert lib.sw_workspace_bytes(32768, 2) > 0 and lib.sw_workspace_bytes(32768, 3) == 0   # q > 2: L <= 16384
    assert lib.sw_strerror(0) == b"ok"
    for code in (-1, -2, -3, -4, -5, -99):
        assert len(lib.sw_strerror(code)) > 0


def test_struct_layouts_match_header():
    assert C.sizeof(binding.sw_obs) == 8 * (3 + 8 + 5)
    assert C.sizeof(binding.sw_cstats) == 8 * (3 + 32)
