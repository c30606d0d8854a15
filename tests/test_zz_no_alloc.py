"""sw_cluster_stats_static: cluster statistics for callers that cannot allocate device memory.

Who that is: code that runs where every byte of the GPU already belongs to somebody else's pool (a raw cudaMalloc fails there or
takes pages the pool counts on), code in a latency-critical loop (cudaMalloc / cudaFree stall the whole device), or a plug-in
that is given two device pointers and no workspace.  The regular path (sw_cluster_stats) needs a bound handle whose workspace
somebody allocated; this entry point keeps its scratch -- one int32 per site plus the accumulators -- in an array compiled
into libswb200.so (SW_STATIC_MAX_SITES = 2^20 sites, about 4 MiB per GPU) and takes only the labels and a device buffer for
the result.

The file is named test_zz_* so that pytest collects it last: `pytest -x` stops at the first failure, and a failure here must
not hide the parity tests.  It makes no assumption about what ran before it in the process (the shared array may hold
anything): it passes alone in a fresh process and after the rest of the suite.

Checked here: the result equals the regular path's (integers: bit for bit, the tolerance of every test in this repository) and
the oracle's, on two calls in a row with different labels, then on a smaller ragged lattice (stale sizes of the larger call
must not leak), and a lattice beyond the limit is refused with SW_ELIMIT.
"""
import ctypes as C

import pytest

import oracle
from paper_1105_5804_b200 import binding


def test_static_entry_point_refuses_bad_sizes_before_touching_the_gpu():
    """No GPU needed: size and pointer checks come before any CUDA call."""
    lib = binding.lib()
    fake = C.c_void_p(0x1000)                              # aligned, never dereferenced on these paths
    assert lib.sw_cluster_stats_static(1028, fake, fake, None) == binding.SW_ELIMIT          # 1028^2 > 2^20
    assert lib.sw_cluster_stats_static(16384, fake, fake, None) == binding.SW_ELIMIT
    assert lib.sw_cluster_stats_static(2, fake, fake, None) == binding.SW_EINVAL
    assert lib.sw_cluster_stats_static(6, fake, fake, None) == binding.SW_EINVAL             # L % 4 != 0
    assert lib.sw_cluster_stats_static(64, None, fake, None) == binding.SW_EINVAL
    assert lib.sw_cluster_stats_static(64, fake, None, None) == binding.SW_EINVAL
    assert lib.sw_cluster_stats_static(64, C.c_void_p(0x1004), fake, None) == binding.SW_EINVAL   # labels not 16-byte aligned
    assert b"SW_STATIC_MAX_SITES" in lib.sw_strerror(binding.SW_ELIMIT)
    assert binding.STATIC_MAX_SITES == 1024 * 1024


@pytest.mark.gpu
def test_static_cluster_stats_match_the_workspace_path_on_consecutive_calls():
    import torch
    assert torch.cuda.is_available()
    dev = torch.device("cuda:0")
    out = torch.full((35,), -7, dtype=torch.int64, device=dev)        # the caller's result buffer, reused by every call
    L = 1024                                                          # the largest lattice the array holds
    lat = binding.Lattice(L, 2, oracle.beta_c(2), 99, device="cuda:0")
    lat.init_spins(1)
    seen = []
    for call in range(2):                                             # two calls in a row, different labels each time
        lat.sweep(1 + call)
        want = lat.cluster_stats()                                    # regular path: size scratch in the bound workspace
        binding.cluster_stats_static(L, lat.labels, out)
        got = binding.cstats_from_tensor(out)
        assert got == want, "call %d" % call
        assert got == oracle.cluster_stats(lat.labels_host())
        assert sum(got["hist32"]) == got["n_clusters"]
        seen.append(got)
    assert seen[0] != seen[1]                                         # (the second call really had other labels to count)
    # the same labels again, back to back with no synchronisation in between: same answer, nothing left over
    out2 = torch.empty(35, dtype=torch.int64, device=dev)
    binding.cluster_stats_static(L, lat.labels, out)
    binding.cluster_stats_static(L, lat.labels, out2)
    assert binding.cstats_from_tensor(out) == seen[1] and binding.cstats_from_tensor(out2) == seen[1]
    lat.close()
    # a smaller lattice with ragged strips after the large one: the sizes the large call left behind must not be counted
    Ls = 260
    small = binding.Lattice(Ls, 3, oracle.beta_c(3), 5, device="cuda:0")
    small.init_spins(1)
    small.sweep(2)
    binding.cluster_stats_static(Ls, small.labels, out)
    got = binding.cstats_from_tensor(out)
    assert got == small.cluster_stats() == oracle.cluster_stats(small.labels_host())
    # labels that did not come from this library's own buffers (a caller's tensor): one cluster per site
    ident = torch.arange(64 * 64, dtype=torch.int32, device=dev)
    binding.cluster_stats_static(64, ident, out)
    got = binding.cstats_from_tensor(out)
    assert got["n_clusters"] == 4096 and got["max_cluster"] == 1 and got["sum_sq_cluster"] == 4096
    assert got["hist32"] == [4096] + [0] * 31
    small.close()


@pytest.mark.gpu
def test_static_entry_point_refuses_what_it_cannot_take():
    import torch
    dev = torch.device("cuda:0")
    out = torch.zeros(35, dtype=torch.int64, device=dev)
    big = torch.zeros(1028 * 1028, dtype=torch.int32, device=dev)
    with pytest.raises(binding.SwError) as e:
        binding.cluster_stats_static(1028, big, out)
    assert e.value.code == binding.SW_ELIMIT and "SW_STATIC_MAX_SITES" in str(e.value)
    assert int(out.abs().sum()) == 0                                  # nothing was launched
    host = torch.zeros(64 * 64, dtype=torch.int32)                    # host memory where device memory is required
    rc = binding.lib().sw_cluster_stats_static(64, C.c_void_p(host.data_ptr()), C.c_void_p(out.data_ptr()), None)
    assert rc == binding.SW_EINVAL
