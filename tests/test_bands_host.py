"""The N>1 path of the multi-GPU row bands on CPU (-m "not gpu"): the exchange of paper_1105_5804_b200/bands.py (halo row, the two
root rows of every band, the counter sum) over a world_size-2 gloo group, with a stand-in for the lattice that holds CPU tensors
and launches nothing -- what is tested is which rows travel where, in which order relative to the two C-ABI calls."""
import json
import os
import socket
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


class FakeLat:
    """Rows of band b carry the value 10 * (t + 1) + b in the 'true' configuration after t sweeps; foreign rows hold -1."""

    def __init__(self, L, G):
        import torch
        self._torch, self.L, self.G, self.t = torch, L, G, 0
        self.device = torch.device("cpu")
        self.rows = L // G
        self.spins = torch.full((L * L,), -1, dtype=torch.int8)
        self.work = torch.zeros(G * 2 * 4 * L, dtype=torch.uint8)
        self.log = []

    def set_band(self, rank, nranks):
        assert nranks == self.G
        self.rank = rank
        self._fill_band()

    def _fill_band(self):
        lo = self.rank * self.rows * self.L
        self.spins[lo: lo + self.rows * self.L] = 10 * (self.t + 1) + self.rank

    def band_layout(self, b):
        L = self.L
        return {"y_first": b * self.rows, "n_rows": self.rows, "y_halo": ((b + 1) * self.rows) % L,
                "off_rootN": (2 * b) * 4 * L, "off_rootS": (2 * b + 1) * 4 * L}

    def _rows(self, b):
        from paper_1105_5804_b200 import bands
        return bands.row_views(self, self.band_layout(b))

    def sweep_band_begin(self):
        L, r = self.L, self.rank
        yh = self.band_layout(r)["y_halo"]
        halo = self.spins[yh * L: (yh + 1) * L]
        assert bool((halo == 10 * (self.t + 1) + (r + 1) % self.G).all()), "halo row is not the first row of the band above"
        a, b = self._rows(r)
        a.copy_(self._torch.arange(L, dtype=self._torch.int32) + 1000 * (r + 1) + self.t)
        b.copy_(self._torch.arange(L, dtype=self._torch.int32) + 2000 * (r + 1) + self.t)
        self.log.append("begin")

    def sweep_band_end(self):
        L = self.L
        for bnd in range(self.G):
            a, b = self._rows(bnd)
            assert int(a[0]) == 1000 * (bnd + 1) + self.t and int(a[L - 1]) == 1000 * (bnd + 1) + self.t + L - 1
            assert int(b[0]) == 2000 * (bnd + 1) + self.t and int(b[L - 1]) == 2000 * (bnd + 1) + self.t + L - 1
        self.t += 1
        self._fill_band()
        self.log.append("end")

    def band_counters(self):
        return {"n_active_bonds": 100 + self.rank, "n_clusters": 7, "sat_before": 1000 * (self.rank + 1), "minus_before": self.rank}

    def close(self):
        pass


def _worker(rank, world, port, out):
    import torch
    import torch.distributed as dist
    from paper_1105_5804_b200 import bands
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    L = 64
    rows = bands.gather_rows(dist, torch.full((5,), rank, dtype=torch.int32))
    ok_gather = [int(t[0]) for t in rows] == list(range(world))
    band = bands.DistBand(L, 2, 0.4, 1, dist, "cpu", lat=FakeLat(L, world))
    band.sweep(3)                                        # the stand-in asserts what it sees at begin / end
    c = band.counters()
    with open(out % rank, "w") as f:
        json.dump({"gather": ok_gather, "log": band.lat.log, "counters": c, "t": band.lat.t}, f)
    dist.destroy_process_group()


def test_band_exchange_gloo_world2(tmp_path):
    pytest.importorskip("torch")
    import torch.multiprocessing as mp
    out = str(tmp_path / "r%d.json")
    mp.spawn(_worker, args=(2, _free_port(), out), nprocs=2, join=True)
    for r in range(2):
        got = json.load(open(out % r))
        assert got["gather"] and got["t"] == 3 and got["log"] == ["begin", "end"] * 3
        assert got["counters"] == {"minus_before": 1, "n_active_bonds": 201, "n_clusters": 14, "sat_before": 3000}
