"""Thin ctypes binding of libswb200.so (include/swb200.h): same names, argument marshalling only.

torch is used for device memory and streams only.  If the shared library is missing or cannot be loaded this
module raises -- there is no CPU fallback and nothing here imports ``oracle``.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libswb200.so")

SW_OK, SW_EINVAL, SW_ESTATE, SW_ECUDA, SW_ENOMEM, SW_ELIMIT = 0, -1, -2, -3, -4, -5
STATIC_MAX_SITES = 1 << 20                                # SW_STATIC_MAX_SITES of include/swb200.h
OBS_SPINS, OBS_CLUSTERS = 1, 2                            # SW_OBS_* of include/swb200.h
NPHASE = 3                                                # SW_NPHASE of include/swb200.h

# every symbol include/swb200.h declares (tests check that the library exports all of them)
SYMBOLS = [
    "sw_create", "sw_destroy", "sw_workspace_bytes", "sw_bind", "sw_set_threshold", "sw_get_threshold",
    "sw_set_counter", "sw_get_counter", "sw_init_spins", "sw_sweep", "sw_activate", "sw_label",
    "sw_cluster_stats", "wolff_step", "sw_observables", "sw_observables_ex", "sw_series_read", "sw_wolff_frontier", "sw_sweep_host", "sw_sweep_host_ex", "sw_launch_count", "sw_strerror",
    "sw_last_cuda_error", "sw_profile_enable", "sw_profile_read", "sw_create3d", "sw_workspace_bytes3d", "sw_label_paper",
    "sw_set_band", "sw_band_layout", "sw_sweep_band_begin", "sw_sweep_band_end", "sw_band_counters",
    "sw_cluster_stats_static", "sw_fewcluster_step",
]


class sw_obs(C.Structure):
    _fields_ = [("sat_bonds", C.c_int64), ("energy", C.c_int64), ("magnetisation", C.c_int64),
                ("state_count", C.c_int64 * 8), ("n_clusters", C.c_int64), ("n_active_bonds", C.c_int64),
                ("max_cluster", C.c_int64), ("sum_sq_cluster", C.c_uint64), ("counter", C.c_uint64)]

    def as_dict(self):
        return {"sat_bonds": self.sat_bonds, "energy": self.energy, "magnetisation": self.magnetisation,
                "state_count": list(self.state_count), "n_clusters": self.n_clusters,
                "n_active_bonds": self.n_active_bonds, "max_cluster": self.max_cluster,
                "sum_sq_cluster": self.sum_sq_cluster, "counter": self.counter}


class sw_cstats(C.Structure):
    _fields_ = [("n_clusters", C.c_int64), ("max_cluster", C.c_int64), ("sum_sq_cluster", C.c_uint64),
                ("hist32", C.c_int64 * 32)]

    def as_dict(self):
        return {"n_clusters": self.n_clusters, "max_cluster": self.max_cluster,
                "sum_sq_cluster": self.sum_sq_cluster, "hist32": list(self.hist32)}


class sw_paper_stats(C.Structure):
    _fields_ = [("selflabel_passes_max", C.c_int32), ("relax_iterations", C.c_int32), ("sewing_levels", C.c_int32),
                ("reserved", C.c_int32), ("ms_local", C.c_double), ("ms_consolidate", C.c_double), ("ms_flatten", C.c_double),
                ("ms_wrap", C.c_double)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_ if k != "reserved"}


_lib = None


def lib():
    """Load libswb200.so (building it first if the sources are newer and nvcc is present)."""
    global _lib
    if _lib is not None:
        return _lib
    from . import build as _build
    if not os.path.exists(LIB_PATH) or (_build.needs_build() and _build.have_nvcc()):
        _build.build()                                    # raises if nvcc is missing; a no-op when up to date
    L = C.CDLL(LIB_PATH)
    vp, i32, i64, u32, u64 = C.c_void_p, C.c_int32, C.c_int64, C.c_uint32, C.c_uint64
    L.sw_create.argtypes = [C.POINTER(vp), i32, i32, C.c_double, u64]
    L.sw_destroy.argtypes = [vp]
    L.sw_workspace_bytes.argtypes = [i32, i32]
    L.sw_workspace_bytes.restype = C.c_size_t
    L.sw_create3d.argtypes = [C.POINTER(vp), i32, i32, C.c_double, u64]
    L.sw_workspace_bytes3d.argtypes = [i32, i32]
    L.sw_workspace_bytes3d.restype = C.c_size_t
    L.sw_bind.argtypes = [vp, vp, vp, vp, vp, C.c_size_t, vp]
    L.sw_set_threshold.argtypes = [vp, u32]
    L.sw_get_threshold.argtypes = [vp, C.POINTER(u32)]
    L.sw_set_counter.argtypes = [vp, u64]
    L.sw_get_counter.argtypes = [vp, C.POINTER(u64)]
    L.sw_init_spins.argtypes = [vp, C.c_int, vp]
    L.sw_sweep.argtypes = [vp, i64, vp]
    L.sw_activate.argtypes = [vp, vp]
    L.sw_label.argtypes = [vp, vp, vp, vp]
    L.sw_cluster_stats.argtypes = [vp, vp, C.POINTER(sw_cstats), vp]
    L.sw_cluster_stats_static.argtypes = [i32, vp, vp, vp]
    L.sw_label_paper.argtypes = [vp, C.c_int, C.c_int, vp, vp, C.POINTER(sw_paper_stats), vp]
    L.sw_set_band.argtypes = [vp, C.c_int, C.c_int]
    L.sw_band_layout.argtypes = [vp, C.c_int, C.POINTER(i32), C.POINTER(i32), C.POINTER(i32), C.POINTER(C.c_size_t),
                                 C.POINTER(C.c_size_t)]
    L.sw_sweep_band_begin.argtypes = [vp, vp]
    L.sw_sweep_band_end.argtypes = [vp, vp]
    L.sw_band_counters.argtypes = [vp, C.POINTER(i64), vp]
    L.wolff_step.argtypes = [vp, i64, C.POINTER(i64), vp]
    L.sw_fewcluster_step.argtypes = [vp, i64, i32, u32, C.POINTER(i64), vp]
    L.sw_observables.argtypes = [vp, C.POINTER(sw_obs), vp]
    L.sw_observables_ex.argtypes = [vp, C.POINTER(sw_obs), C.c_int, vp]
    L.sw_wolff_frontier.argtypes = [vp, C.c_int]
    L.sw_series_read.argtypes = [vp, u64, i64, C.POINTER(i64), C.POINTER(i64), vp]
    L.sw_sweep_host.argtypes = [vp, vp, i64, vp, vp, C.POINTER(sw_obs), vp]
    L.sw_sweep_host_ex.argtypes = [vp, vp, i64, vp, vp, C.POINTER(sw_obs), C.c_int, vp]
    L.sw_launch_count.argtypes = [vp, C.POINTER(u64)]
    L.sw_profile_enable.argtypes = [vp, C.c_int]
    L.sw_profile_read.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(u64)]
    L.sw_strerror.argtypes = [C.c_int]
    L.sw_strerror.restype = C.c_char_p
    L.sw_last_cuda_error.argtypes = [vp]
    L.sw_last_cuda_error.restype = C.c_char_p
    for name in SYMBOLS:
        if name not in ("sw_workspace_bytes", "sw_workspace_bytes3d", "sw_strerror", "sw_last_cuda_error"):
            getattr(L, name).restype = C.c_int
    _lib = L
    return L


class SwError(RuntimeError):
    def __init__(self, code, detail=""):
        self.code = code
        msg = lib().sw_strerror(code).decode()
        super().__init__("swb200: %s (%d)%s" % (msg, code, (": " + detail) if detail else ""))


def cluster_stats_static(L: int, labels, out=None) -> "object":
    """sw_cluster_stats_static: cluster statistics of an L x L label tensor with no workspace and no handle, for callers that
    cannot allocate device memory (the scratch is an array built into the library; L * L <= STATIC_MAX_SITES).

    labels: int32 CUDA tensor of L * L canonical labels.  out: a CUDA tensor of >= 35 int64 on the same GPU that receives the
    sw_cstats (n_clusters, max_cluster, sum_sq_cluster, hist32[32]); if None one is created here (which allocates -- pass your
    own to stay allocation-free).  Asynchronous on torch's current stream of that GPU; returns `out`.  Calls that overlap on
    one GPU race on the shared array."""
    import torch
    if out is None:
        out = torch.empty(C.sizeof(sw_cstats) // 8, dtype=torch.int64, device=labels.device)
    stream = C.c_void_p(torch.cuda.current_stream(labels.device).cuda_stream)
    rc = lib().sw_cluster_stats_static(L, labels.data_ptr(), out.data_ptr(), stream)
    if rc != SW_OK:
        raise SwError(rc)
    return out


def cstats_from_tensor(out) -> dict:
    """The sw_cstats a cluster_stats_static call left in `out`, as the dict Lattice.cluster_stats returns (synchronising copy)."""
    v = out.cpu().tolist()
    return {"n_clusters": v[0], "max_cluster": v[1], "sum_sq_cluster": v[2] & 0xFFFFFFFFFFFFFFFF, "hist32": v[3:35]}


class Lattice:
    """One bound sw_handle plus the torch tensors it is bound to (device memory only; no arithmetic here)."""

    def __init__(self, L: int, q: int, beta: float, seed: int, device="cuda:0", with_bonds: bool = False, dim: int = 2):
        """dim = 2: L x L square lattice (sw_create); dim = 3: L x L x L simple cubic lattice (sw_create3d)."""
        import torch
        self._torch = torch
        self._h = C.c_void_p()
        self._lib = lib()
        if dim not in (2, 3):
            raise ValueError("dim must be 2 or 3")
        rc = (self._lib.sw_create3d if dim == 3 else self._lib.sw_create)(C.byref(self._h), L, q, beta, seed)
        if rc != SW_OK:
            raise SwError(rc)
        self.L, self.q, self.N, self.dim = L, q, L ** dim, dim
        self.device = torch.device(device)
        if self.device.type != "cuda":
            raise RuntimeError("swb200 needs a CUDA device; there is no CPU path")
        self.spins = torch.empty(self.N, dtype=torch.int8, device=self.device)
        self.labels = torch.empty(self.N, dtype=torch.int32, device=self.device)
        # bonds: packed, 4 sites per byte (square lattice); one byte per site (cubic lattice)
        self.bonds = torch.empty(self.N // 4 if dim == 2 else self.N, dtype=torch.uint8, device=self.device) if with_bonds else None
        wb = (self._lib.sw_workspace_bytes3d if dim == 3 else self._lib.sw_workspace_bytes)(L, q)
        self.work = torch.empty(wb, dtype=torch.uint8, device=self.device)
        self._check(self._lib.sw_bind(self._h, self.spins.data_ptr(), self.labels.data_ptr(),
                                      self.bonds.data_ptr() if with_bonds else None, self.work.data_ptr(), wb,
                                      self._stream()))

    # -- helpers ------------------------------------------------------------------------------------------
    def _stream(self):
        return C.c_void_p(self._torch.cuda.current_stream(self.device).cuda_stream)

    def _check(self, rc):
        if rc != SW_OK:
            raise SwError(rc, self._lib.sw_last_cuda_error(self._h).decode() if rc == SW_ECUDA else "")

    def close(self):
        if self._h:
            self._torch.cuda.synchronize(self.device)
            self._lib.sw_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- the C-ABI, one method per entry point ---------------------------------------------------------------
    def set_threshold(self, T: int):
        self._check(self._lib.sw_set_threshold(self._h, T))

    def get_threshold(self) -> int:
        v = C.c_uint32()
        self._check(self._lib.sw_get_threshold(self._h, C.byref(v)))
        return v.value

    def set_counter(self, t: int):
        self._check(self._lib.sw_set_counter(self._h, t))

    def get_counter(self) -> int:
        v = C.c_uint64()
        self._check(self._lib.sw_get_counter(self._h, C.byref(v)))
        return v.value

    def init_spins(self, mode: int):
        self._check(self._lib.sw_init_spins(self._h, mode, self._stream()))

    def sweep(self, n: int = 1):
        self._check(self._lib.sw_sweep(self._h, n, self._stream()))

    def activate(self):
        self._check(self._lib.sw_activate(self._h, self._stream()))

    def label(self, bonds=None, labels_out=None):
        self._check(self._lib.sw_label(self._h, bonds.data_ptr() if bonds is not None else None,
                                       labels_out.data_ptr() if labels_out is not None else None, self._stream()))

    def label_paper(self, method: int, B: int, bonds=None, labels_out=None) -> dict:
        """The paper's own pipeline (ablation baseline): method 0 = label relaxation, 1 = hierarchical sewing."""
        st = sw_paper_stats()
        self._check(self._lib.sw_label_paper(self._h, method, B, bonds.data_ptr() if bonds is not None else None,
                                             labels_out.data_ptr() if labels_out is not None else None, C.byref(st),
                                             self._stream()))
        return st.as_dict()

    # -- multi-GPU row bands (include/swb200.h "MULTI-GPU ROW BANDS"; the exchange itself is in bands.py) ----------------------
    def set_band(self, rank: int, nranks: int):
        self._check(self._lib.sw_set_band(self._h, rank, nranks))

    def band_layout(self, band: int) -> dict:
        y0, n, yh = C.c_int32(), C.c_int32(), C.c_int32()
        oa, ob = C.c_size_t(), C.c_size_t()
        self._check(self._lib.sw_band_layout(self._h, band, C.byref(y0), C.byref(n), C.byref(yh), C.byref(oa), C.byref(ob)))
        return {"y_first": y0.value, "n_rows": n.value, "y_halo": yh.value, "off_rootN": oa.value, "off_rootS": ob.value}

    def sweep_band_begin(self):
        self._check(self._lib.sw_sweep_band_begin(self._h, self._stream()))

    def sweep_band_end(self):
        self._check(self._lib.sw_sweep_band_end(self._h, self._stream()))

    def band_counters(self) -> dict:
        out = (C.c_int64 * 4)()
        self._check(self._lib.sw_band_counters(self._h, out, self._stream()))
        return {"n_active_bonds": out[0], "n_clusters": out[1], "sat_before": out[2], "minus_before": out[3]}

    def cluster_stats(self, labels=None) -> dict:
        out = sw_cstats()
        self._check(self._lib.sw_cluster_stats(self._h, labels.data_ptr() if labels is not None else None,
                                               C.byref(out), self._stream()))
        return out.as_dict()

    def wolff_step(self, n: int = 1, want_sizes: bool = True):
        if want_sizes:
            sizes = (C.c_int64 * n)()
            self._check(self._lib.wolff_step(self._h, n, sizes, self._stream()))
            return list(sizes)
        self._check(self._lib.wolff_step(self._h, n, None, self._stream()))
        return None

    def fewcluster_step(self, n: int, n_seeds: int, T_flip: int, want_counts: bool = True):
        """n few-cluster steps (sw_fewcluster_step) -> list of flipped sites per step, or None"""
        if want_counts:
            out = (C.c_int64 * n)()
            self._check(self._lib.sw_fewcluster_step(self._h, n, n_seeds, T_flip, out, self._stream()))
            return list(out)
        self._check(self._lib.sw_fewcluster_step(self._h, n, n_seeds, T_flip, None, self._stream()))
        return None

    def wolff_frontier(self, max_levels: int):
        self._check(self._lib.sw_wolff_frontier(self._h, max_levels))

    def observables(self, spins: bool = True, clusters: bool = True) -> dict:
        out = sw_obs()
        if spins and clusters:
            self._check(self._lib.sw_observables(self._h, C.byref(out), self._stream()))
        else:
            flags = (OBS_SPINS if spins else 0) | (OBS_CLUSTERS if clusters else 0)
            self._check(self._lib.sw_observables_ex(self._h, C.byref(out), flags, self._stream()))
        return out.as_dict()

    def series(self, t_first: int, n: int, magnetisation: bool = True):
        """-> (energies, magnetisations or None) of the configurations at counters t_first .. t_first + n - 1"""
        E = (C.c_int64 * n)()
        M = (C.c_int64 * n)() if magnetisation else None
        self._check(self._lib.sw_series_read(self._h, t_first, n, E, M, self._stream()))
        return list(E), (list(M) if magnetisation else None)

    def sweep_host(self, h_spins_in, n: int, h_spins_out=None, h_labels_out=None, want_obs: bool = True,
                   obs_flags: int = OBS_SPINS | OBS_CLUSTERS):
        """Host-buffer end-to-end call: torch CPU tensors (ideally pinned) in and out."""
        out = sw_obs()
        self._check(self._lib.sw_sweep_host_ex(
            self._h, h_spins_in.data_ptr() if h_spins_in is not None else None, n,
            h_spins_out.data_ptr() if h_spins_out is not None else None,
            h_labels_out.data_ptr() if h_labels_out is not None else None,
            C.byref(out) if want_obs else None, obs_flags, self._stream()))
        return out.as_dict() if want_obs else None

    def profile_enable(self, on: bool):
        self._check(self._lib.sw_profile_enable(self._h, 1 if on else 0))

    def profile_read(self):
        """-> (ms per phase summed over the timed sweeps [k_scan, k_seam, k_final], number of sweeps)"""
        ms = (C.c_double * NPHASE)(*([0.0] * NPHASE))
        n = C.c_uint64(0)
        self._check(self._lib.sw_profile_read(self._h, ms, C.byref(n)))
        return list(ms), n.value

    def launch_count(self) -> int:
        v = C.c_uint64()
        self._check(self._lib.sw_launch_count(self._h, C.byref(v)))
        return v.value

    # -- convenience (copies only) -------------------------------------------------------------------------
    def set_spins(self, host_array):
        t = self._torch.from_numpy(host_array).view(self._torch.int8)
        self.spins.copy_(t.to(self.device))

    def spins_host(self):
        return self.spins.cpu().numpy()

    def labels_host(self):
        return self.labels.cpu().numpy()
