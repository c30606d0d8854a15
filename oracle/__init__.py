"""oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

ctypes front end of ``oracle/sw_oracle.c``: the plain serial CPU statement of the
Swendsen-Wang / Wolff update (M. Weigel, arXiv:1105.5804; PAPER.md P:51-55 steps
1-3, P:111 breadth-first search, P:330 Wolff).  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl
reference`` legs may import this package.  It shares no code with
``paper_1105_5804_b200`` and never imports it.

This file holds no arithmetic of the method: it only marshals numpy arrays into
the C functions.  The one exception is :func:`beta_c`, a literature constant.
"""
from __future__ import annotations

import ctypes as C
import math
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sw_oracle.c")


def _machine_tag() -> str:
    """The library is built -O3 -march=native (SURVEY.md 8(d) "CPU baseline beside it"), so it is tied to the CPU it was
    built on: one file per CPU model, rebuilt where it is missing (the GPU box has gcc; the in-tree .so travels with the
    repository snapshot but may come from another CPU)."""
    import hashlib
    try:
        with open("/proc/cpuinfo") as f:
            txt = "".join(l for l in f if l.startswith(("model name", "flags")))[:20000]
    except OSError:
        txt = "unknown"
    return hashlib.sha256(txt.encode()).hexdigest()[:10]


_FLAGS = ["-O3", "-march=native"]
_LIB = os.path.join(_HERE, "libsw_oracle.%s.so" % _machine_tag())


def build_flags() -> str:
    return "gcc " + " ".join(_FLAGS)


def build(force: bool = False) -> str:
    """Compile sw_oracle.c with gcc -O3 -march=native for this machine (integer code: the flags change no result)."""
    if force or (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(["gcc"] + _FLAGS + ["-std=c11", "-fPIC", "-shared", "-Wall", "-Wextra",
                                                  "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


class Obs(C.Structure):
    _fields_ = [("sat_bonds", C.c_int64), ("energy", C.c_int64), ("magnetisation", C.c_int64),
                ("state_count", C.c_int64 * 8)]


class CStats(C.Structure):
    _fields_ = [("n_clusters", C.c_int64), ("max_cluster", C.c_int64),
                ("sum_sq_cluster", C.c_uint64), ("hist32", C.c_int64 * 32)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        p8, pu8, p32, p64, pu32 = (C.POINTER(C.c_int8), C.POINTER(C.c_uint8), C.POINTER(C.c_int32),
                                   C.POINTER(C.c_int64), C.POINTER(C.c_uint32))
        L.orc_philox4x32_10.argtypes = [pu32, pu32, pu32]
        L.orc_philox4x32_10.restype = None
        L.orc_threshold.argtypes = [C.c_int, C.c_double]
        L.orc_threshold.restype = C.c_uint32
        L.orc_threshold_from_p.argtypes = [C.c_double]
        L.orc_threshold_from_p.restype = C.c_uint32
        L.orc_init_spins.argtypes = [C.c_int32, C.c_int32, C.c_uint64, C.c_int32, p8]
        L.orc_init_spins.restype = C.c_int
        L.orc_bonds.argtypes = [C.c_int32, C.c_uint32, C.c_uint64, C.c_uint64, p8, pu8]
        L.orc_bonds.restype = C.c_int64
        L.orc_pack_bonds.argtypes = [C.c_int64, pu8, pu8]
        L.orc_pack_bonds.restype = None
        L.orc_unpack_bonds.argtypes = [C.c_int64, pu8, pu8]
        L.orc_unpack_bonds.restype = None
        L.orc_label.argtypes = [C.c_int32, pu8, p32]
        L.orc_label.restype = C.c_int64
        L.orc_flip.argtypes = [C.c_int32, C.c_int32, C.c_uint64, C.c_uint64, p32, p8]
        L.orc_flip.restype = None
        L.orc_observables.argtypes = [C.c_int32, C.c_int32, p8, C.POINTER(Obs)]
        L.orc_observables.restype = None
        L.orc_cluster_stats.argtypes = [C.c_int64, p32, C.POINTER(CStats)]
        L.orc_cluster_stats.restype = C.c_int
        L.orc_sweep.argtypes = [C.c_int32, C.c_int32, C.c_uint32, C.c_uint64, C.c_uint64, p8, p32, pu8, p64]
        L.orc_sweep.restype = C.c_int64
        L.orc_run_chain.argtypes = [C.c_int32, C.c_int32, C.c_uint32, C.c_uint64, C.c_uint64, C.c_int64, p8, p64]
        L.orc_run_chain.restype = C.c_int
        L.orc_wolff_step.argtypes = [C.c_int32, C.c_int32, C.c_uint32, C.c_uint64, C.c_uint64, p8, p64, p64]
        L.orc_wolff_step.restype = C.c_int64
        L.orc_wolff_chain.argtypes = [C.c_int32, C.c_uint32, C.c_uint64, C.c_uint64, C.c_int64, p8, p64]
        L.orc_wolff_chain.restype = C.c_int
        L.orc_fewcluster_step.argtypes = [C.c_int32, C.c_int32, C.c_uint32, C.c_uint64, C.c_uint64, C.c_int32, C.c_uint32, p8,
                                          C.POINTER(C.c_int32), p64]
        L.orc_fewcluster_step.restype = C.c_int64
        L.orc_fewcluster_chain.argtypes = [C.c_int32, C.c_uint32, C.c_uint64, C.c_uint64, C.c_int64, C.c_int32, C.c_uint32, p8, p64]
        L.orc_fewcluster_chain.restype = C.c_int
        L.orc_fnv1a64.argtypes = [pu8, C.c_int64]
        L.orc_fnv1a64.restype = C.c_uint64
        # simple cubic lattice
        L.orc3_init_spins.argtypes = [C.c_int32, C.c_int32, C.c_uint64, C.c_int32, p8]
        L.orc3_init_spins.restype = C.c_int
        L.orc3_bonds.argtypes = [C.c_int32, C.c_uint32, C.c_uint64, C.c_uint64, p8, pu8]
        L.orc3_bonds.restype = C.c_int64
        L.orc3_label.argtypes = [C.c_int32, pu8, p32]
        L.orc3_label.restype = C.c_int64
        L.orc3_flip.argtypes = [C.c_int64, C.c_int32, C.c_uint64, C.c_uint64, p32, p8]
        L.orc3_flip.restype = None
        L.orc3_observables.argtypes = [C.c_int32, C.c_int32, p8, C.POINTER(Obs)]
        L.orc3_observables.restype = None
        L.orc3_sweep.argtypes = [C.c_int32, C.c_int32, C.c_uint32, C.c_uint64, C.c_uint64, p8, p32, pu8, p64]
        L.orc3_sweep.restype = C.c_int64
        L.orc3_run_chain.argtypes = [C.c_int32, C.c_int32, C.c_uint32, C.c_uint64, C.c_uint64, C.c_int64, p8, p64]
        L.orc3_run_chain.restype = C.c_int
        _lib = L
    return _lib


def _p(a, ct):
    return a.ctypes.data_as(C.POINTER(ct))


def beta_c(q: int) -> float:
    """Critical coupling in the library's convention (SURVEY 8(b)/8(c) issue 4; P:166 gives
    ln(1+sqrt 2) for the delta-Hamiltonian of q=2): q=2 Ising +-1 -> ln(1+sqrt 2)/2, else ln(1+sqrt q)."""
    return 0.5 * math.log(1.0 + math.sqrt(2.0)) if q == 2 else math.log(1.0 + math.sqrt(q))


def philox(ctr, key):
    c = np.asarray(ctr, dtype=np.uint32).copy()
    k = np.asarray(key, dtype=np.uint32).copy()
    out = np.zeros(4, dtype=np.uint32)
    lib().orc_philox4x32_10(_p(c, C.c_uint32), _p(k, C.c_uint32), _p(out, C.c_uint32))
    return out


def threshold(q: int, beta: float) -> int:
    return int(lib().orc_threshold(q, beta))


def threshold_from_p(p: float) -> int:
    return int(lib().orc_threshold_from_p(p))


def init_spins(L: int, q: int, seed: int, mode: int) -> np.ndarray:
    s = np.empty(L * L, dtype=np.int8)
    rc = lib().orc_init_spins(L, q, seed, mode, _p(s, C.c_int8))
    if rc != 0:
        raise ValueError("orc_init_spins: bad arguments")
    return s


def bonds(L: int, T: int, seed: int, t: int, spins: np.ndarray):
    """-> (codes uint8[N] with bit0 = east, bit1 = north, number of active bonds)"""
    assert spins.dtype == np.int8 and spins.size == L * L and spins.flags.c_contiguous
    codes = np.empty(L * L, dtype=np.uint8)
    n = lib().orc_bonds(L, T, seed, t, _p(spins, C.c_int8), _p(codes, C.c_uint8))
    return codes, int(n)


def pack_bonds(codes: np.ndarray) -> np.ndarray:
    codes = np.ascontiguousarray(codes, dtype=np.uint8)
    packed = np.zeros((codes.size + 3) // 4, dtype=np.uint8)
    lib().orc_pack_bonds(codes.size, _p(codes, C.c_uint8), _p(packed, C.c_uint8))
    return packed


def unpack_bonds(packed: np.ndarray, N: int) -> np.ndarray:
    packed = np.ascontiguousarray(packed, dtype=np.uint8)
    codes = np.empty(N, dtype=np.uint8)
    lib().orc_unpack_bonds(N, _p(packed, C.c_uint8), _p(codes, C.c_uint8))
    return codes


def label(L: int, codes: np.ndarray):
    """-> (labels int32[N], number of clusters)"""
    codes = np.ascontiguousarray(codes, dtype=np.uint8)
    assert codes.size == L * L
    labels = np.empty(L * L, dtype=np.int32)
    nc = lib().orc_label(L, _p(codes, C.c_uint8), _p(labels, C.c_int32))
    if nc < 0:
        raise MemoryError
    return labels, int(nc)


def flip(L: int, q: int, seed: int, t: int, labels: np.ndarray) -> np.ndarray:
    labels = np.ascontiguousarray(labels, dtype=np.int32)
    spins = np.empty(L * L, dtype=np.int8)
    lib().orc_flip(L, q, seed, t, _p(labels, C.c_int32), _p(spins, C.c_int8))
    return spins


def observables(L: int, q: int, spins: np.ndarray) -> dict:
    assert spins.dtype == np.int8 and spins.size == L * L and spins.flags.c_contiguous
    o = Obs()
    lib().orc_observables(L, q, _p(spins, C.c_int8), C.byref(o))
    return {"sat_bonds": o.sat_bonds, "energy": o.energy, "magnetisation": o.magnetisation,
            "state_count": list(o.state_count)}


def cluster_stats(labels: np.ndarray) -> dict:
    labels = np.ascontiguousarray(labels, dtype=np.int32)
    c = CStats()
    if lib().orc_cluster_stats(labels.size, _p(labels, C.c_int32), C.byref(c)) != 0:
        raise MemoryError
    return {"n_clusters": c.n_clusters, "max_cluster": c.max_cluster,
            "sum_sq_cluster": c.sum_sq_cluster, "hist32": list(c.hist32)}


def sweep(L: int, q: int, T: int, seed: int, t: int, spins: np.ndarray):
    """One SW sweep in place on `spins`. -> (labels, codes, n_clusters, n_active_bonds)"""
    assert spins.dtype == np.int8 and spins.size == L * L and spins.flags.c_contiguous
    labels = np.empty(L * L, dtype=np.int32)
    codes = np.empty(L * L, dtype=np.uint8)
    nb = C.c_int64(0)
    nc = lib().orc_sweep(L, q, T, seed, t, _p(spins, C.c_int8), _p(labels, C.c_int32),
                         _p(codes, C.c_uint8), C.byref(nb))
    if nc < 0:
        raise MemoryError
    return labels, codes, int(nc), int(nb.value)


def run_chain(L: int, q: int, T: int, seed: int, t0: int, n: int, spins: np.ndarray) -> np.ndarray:
    """n sweeps in place; -> int64[n,4] = (E, M, n_clusters, sum size^2) after every sweep."""
    assert spins.dtype == np.int8 and spins.size == L * L and spins.flags.c_contiguous
    series = np.zeros((n, 4), dtype=np.int64)
    if lib().orc_run_chain(L, q, T, seed, t0, n, _p(spins, C.c_int8), _p(series, C.c_int64)) != 0:
        raise MemoryError
    return series


def wolff_step(L: int, T: int, seed: int, t: int, spins: np.ndarray):
    """One Wolff step in place (q=2). -> (|C|, seed site, min site index of C)"""
    assert spins.dtype == np.int8 and spins.size == L * L and spins.flags.c_contiguous
    s0, r0 = C.c_int64(0), C.c_int64(0)
    sz = lib().orc_wolff_step(L, 2, T, seed, t, _p(spins, C.c_int8), C.byref(s0), C.byref(r0))
    if sz < 0:
        raise MemoryError
    return int(sz), int(s0.value), int(r0.value)


def wolff_chain(L: int, T: int, seed: int, t0: int, n: int, spins: np.ndarray) -> np.ndarray:
    """n Wolff steps in place; -> int64[n,3] = (E, M, |C|) after every step."""
    assert spins.dtype == np.int8 and spins.size == L * L and spins.flags.c_contiguous
    series = np.zeros((n, 3), dtype=np.int64)
    if lib().orc_wolff_chain(L, T, seed, t0, n, _p(spins, C.c_int8), _p(series, C.c_int64)) != 0:
        raise MemoryError
    return series


def fewcluster_step(L: int, T: int, seed: int, t: int, n_seeds: int, T_flip: int, spins: np.ndarray):
    """One few-cluster step in place (q=2, reading 21). -> (flipped sites, flipped clusters, labels)"""
    assert spins.dtype == np.int8 and spins.size == L * L and spins.flags.c_contiguous
    labels = np.empty(L * L, dtype=np.int32)
    nfc = C.c_int64(0)
    f = lib().orc_fewcluster_step(L, 2, T, seed, t, n_seeds, T_flip, _p(spins, C.c_int8), _p(labels, C.c_int32), C.byref(nfc))
    if f < 0:
        raise MemoryError
    return int(f), int(nfc.value), labels


def fewcluster_chain(L: int, T: int, seed: int, t0: int, n: int, n_seeds: int, T_flip: int, spins: np.ndarray) -> np.ndarray:
    """n few-cluster steps in place; -> int64[n,3] = (E, M, flipped sites) after every step."""
    assert spins.dtype == np.int8 and spins.size == L * L and spins.flags.c_contiguous
    series = np.zeros((n, 3), dtype=np.int64)
    if lib().orc_fewcluster_chain(L, T, seed, t0, n, n_seeds, T_flip, _p(spins, C.c_int8), _p(series, C.c_int64)) != 0:
        raise MemoryError
    return series


def fnv1a64(buf: np.ndarray) -> int:
    b = np.ascontiguousarray(buf).view(np.uint8).reshape(-1)
    return int(lib().orc_fnv1a64(_p(b, C.c_uint8), b.size))


# ---- simple cubic lattice: site i = z L^2 + y L + x, bond codes bit 0 east, 1 north, 2 up ----------
def init_spins3(L: int, q: int, seed: int, mode: int) -> np.ndarray:
    s = np.empty(L ** 3, dtype=np.int8)
    if lib().orc3_init_spins(L, q, seed, mode, _p(s, C.c_int8)) != 0:
        raise ValueError("orc3_init_spins: bad arguments")
    return s


def bonds3(L: int, T: int, seed: int, t: int, spins: np.ndarray):
    assert spins.dtype == np.int8 and spins.size == L ** 3 and spins.flags.c_contiguous
    codes = np.empty(L ** 3, dtype=np.uint8)
    n = lib().orc3_bonds(L, T, seed, t, _p(spins, C.c_int8), _p(codes, C.c_uint8))
    return codes, int(n)


def label3(L: int, codes: np.ndarray):
    codes = np.ascontiguousarray(codes, dtype=np.uint8)
    assert codes.size == L ** 3
    labels = np.empty(L ** 3, dtype=np.int32)
    nc = lib().orc3_label(L, _p(codes, C.c_uint8), _p(labels, C.c_int32))
    if nc < 0:
        raise MemoryError
    return labels, int(nc)


def flip3(q: int, seed: int, t: int, labels: np.ndarray) -> np.ndarray:
    labels = np.ascontiguousarray(labels, dtype=np.int32)
    spins = np.empty(labels.size, dtype=np.int8)
    lib().orc3_flip(labels.size, q, seed, t, _p(labels, C.c_int32), _p(spins, C.c_int8))
    return spins


def observables3(L: int, q: int, spins: np.ndarray) -> dict:
    assert spins.dtype == np.int8 and spins.size == L ** 3 and spins.flags.c_contiguous
    o = Obs()
    lib().orc3_observables(L, q, _p(spins, C.c_int8), C.byref(o))
    return {"sat_bonds": o.sat_bonds, "energy": o.energy, "magnetisation": o.magnetisation,
            "state_count": list(o.state_count)}


def sweep3(L: int, q: int, T: int, seed: int, t: int, spins: np.ndarray):
    """One SW sweep of the L^3 lattice in place. -> (labels, codes, n_clusters, n_active_bonds)"""
    assert spins.dtype == np.int8 and spins.size == L ** 3 and spins.flags.c_contiguous
    labels = np.empty(L ** 3, dtype=np.int32)
    codes = np.empty(L ** 3, dtype=np.uint8)
    nb = C.c_int64(0)
    nc = lib().orc3_sweep(L, q, T, seed, t, _p(spins, C.c_int8), _p(labels, C.c_int32), _p(codes, C.c_uint8), C.byref(nb))
    if nc < 0:
        raise MemoryError
    return labels, codes, int(nc), int(nb.value)


def run_chain3(L: int, q: int, T: int, seed: int, t0: int, n: int, spins: np.ndarray) -> np.ndarray:
    assert spins.dtype == np.int8 and spins.size == L ** 3 and spins.flags.c_contiguous
    series = np.zeros((n, 4), dtype=np.int64)
    if lib().orc3_run_chain(L, q, T, seed, t0, n, _p(spins, C.c_int8), _p(series, C.c_int64)) != 0:
        raise MemoryError
    return series
