"""Multi-GPU Swendsen-Wang by row bands (include/swb200.h "MULTI-GPU ROW BANDS"; csrc/band_kernels.cuh): the exchange around
the C-ABI calls.  Nothing here computes anything of the method: it copies one row of spins and two rows of int32 roots per
rank and sweep, and sums counters.

Two drivers over the same steps:
  * :class:`BandGroup`  -- G bands in ONE process (one or several devices), rows copied tensor to tensor.  Used by the
    `-m gpu` tests to run the G-rank algorithm on a single GPU, band after band (no kernel waits for another rank's kernel).
  * :class:`DistBand`   -- one band per process under ``torch.distributed`` (NCCL on GPUs): the halo row and the two root rows
    travel by ``all_gather``.  :func:`gather_rows` is the only collective and works on CPU tensors with gloo too (tested so).
"""
from __future__ import annotations

from . import binding


def row_views(lat, layout_of_band: dict):
    """(rootN row, rootS row) of one band as int32 views of `lat`'s workspace tensor."""
    L = lat.L
    w = lat.work
    a = w[layout_of_band["off_rootN"]: layout_of_band["off_rootN"] + 4 * L].view(lat._torch.int32)
    b = w[layout_of_band["off_rootS"]: layout_of_band["off_rootS"] + 4 * L].view(lat._torch.int32)
    return a, b


def spin_row(lat, y: int):
    return lat.spins[y * lat.L: (y + 1) * lat.L]


def gather_rows(dist, mine):
    """all_gather of one tensor per rank -> list of tensors in rank order (any backend, any device)."""
    import torch
    out = [torch.empty_like(mine) for _ in range(dist.get_world_size())]
    dist.all_gather(out, mine.contiguous())
    return out


class BandGroup:
    """G bands of one L x L lattice in one process.  devices: one per band, or one for all."""

    def __init__(self, L: int, q: int, beta: float, seed: int, nbands: int, devices="cuda:0"):
        if isinstance(devices, str):
            devices = [devices] * nbands
        self.G, self.L, self.N = nbands, L, L * L
        self.lats = [binding.Lattice(L, q, beta, seed, device=d) for d in devices]
        for r, lat in enumerate(self.lats):
            lat.set_band(r, nbands)
        self.layout = [self.lats[0].band_layout(b) for b in range(nbands)]

    def init_spins(self, mode: int):
        for lat in self.lats:
            lat.init_spins(mode)                          # every rank initialises the whole lattice (one cheap kernel)

    def sweep(self, n: int = 1):
        G = self.G
        for _ in range(n):
            for r, lat in enumerate(self.lats):           # 1. north halo row from the band above (periodic)
                yh = self.layout[r]["y_halo"]
                spin_row(lat, yh).copy_(spin_row(self.lats[(r + 1) % G], yh))
            for lat in self.lats:                         # 2. band-local part
                lat.sweep_band_begin()
            for r, lat in enumerate(self.lats):           # 3. "all-gather" of the two root rows of every band
                for b in range(G):
                    if b != r:
                        src = row_views(self.lats[b], self.layout[b])
                        dst = row_views(lat, self.layout[b])
                        dst[0].copy_(src[0]); dst[1].copy_(src[1])
            for lat in self.lats:                         # 4. cross-band seams, flatten + flip
                lat.sweep_band_end()

    def counters(self) -> dict:
        tot = {}
        for lat in self.lats:
            for k, v in lat.band_counters().items():
                tot[k] = tot.get(k, 0) + v
        return tot

    def spins_host(self):
        """the bands' rows stitched together"""
        import numpy as np
        out = np.empty(self.N, dtype=np.int8)
        for r, lat in enumerate(self.lats):
            lo = self.layout[r]["y_first"] * self.L
            hi = lo + self.layout[r]["n_rows"] * self.L
            out[lo:hi] = lat.spins[lo:hi].cpu().numpy()
        return out

    def labels_host(self):
        import numpy as np
        out = np.empty(self.N, dtype=np.int32)
        for r, lat in enumerate(self.lats):
            lo = self.layout[r]["y_first"] * self.L
            hi = lo + self.layout[r]["n_rows"] * self.L
            out[lo:hi] = lat.labels[lo:hi].cpu().numpy()
        return out

    def close(self):
        for lat in self.lats:
            lat.close()


class DistBand:
    """One band per process; `dist` is an initialised torch.distributed (NCCL: one GPU per rank)."""

    def __init__(self, L: int, q: int, beta: float, seed: int, dist, device, lat=None):
        """lat: an object with the band methods of binding.Lattice (the gloo test of the exchange passes a stand-in that holds
        CPU tensors and launches nothing); default: a binding.Lattice on `device`."""
        self.dist, self.rank, self.G = dist, dist.get_rank(), dist.get_world_size()
        self.L, self.N = L, L * L
        self.lat = lat if lat is not None else binding.Lattice(L, q, beta, seed, device=device)
        self.lat.set_band(self.rank, self.G)
        self.layout = [self.lat.band_layout(b) for b in range(self.G)]

    def init_spins(self, mode: int):
        self.lat.init_spins(mode)

    def sweep(self, n: int = 1):
        import torch
        lat, G, r = self.lat, self.G, self.rank
        for _ in range(n):
            # 1. every rank publishes the first row of its band; I need the one of the band above
            first = gather_rows(self.dist, spin_row(lat, self.layout[r]["y_first"]))
            spin_row(lat, self.layout[r]["y_halo"]).copy_(first[(r + 1) % G])
            lat.sweep_band_begin()
            # 3. the two root rows of every band
            mine = torch.stack(row_views(lat, self.layout[r]))
            rows = gather_rows(self.dist, mine)
            for b in range(G):
                if b != r:
                    dst = row_views(lat, self.layout[b])
                    dst[0].copy_(rows[b][0]); dst[1].copy_(rows[b][1])
            lat.sweep_band_end()

    def counters(self) -> dict:
        import torch
        c = self.lat.band_counters()
        keys = sorted(c)
        t = torch.tensor([c[k] for k in keys], dtype=torch.int64, device=self.lat.device)
        self.dist.all_reduce(t)
        return dict(zip(keys, t.tolist()))

    def close(self):
        self.lat.close()
