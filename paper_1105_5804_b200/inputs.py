"""Seeded synthetic input generators shared by tests, bench.py and smoke().

This module holds NONE of the method's arithmetic (no Philox, no bond rule, no labelling): it only draws
plain numpy random arrays of the shapes the boundary accepts, so that the CUDA path and the oracle can be fed
identical bytes.  It imports neither the CUDA binding nor ``oracle``.

Recipes: the paper's workloads are themselves synthetic -- equilibrium Potts
configurations and percolation bond sets on periodic L x L lattices (Table I) -- so
nothing stands in for a dataset.
"""
from __future__ import annotations

import numpy as np


def random_bond_codes(L: int, p_east: float, p_north: float, seed: int) -> np.ndarray:
    """uint8[N] codes, bit0 = east bond open, bit1 = north bond open, i.i.d. (bond percolation, BJ config 4)."""
    rng = np.random.default_rng(seed)
    e = rng.random(L * L) < p_east
    n = rng.random(L * L) < p_north
    return (e.astype(np.uint8) | (n.astype(np.uint8) << 1)).astype(np.uint8)


def pack_codes(codes: np.ndarray) -> np.ndarray:
    """Boundary layout (include/swb200.h): byte b holds sites 4b..4b+3, site j in bits 2(j&3), 2(j&3)+1."""
    c = np.ascontiguousarray(codes, dtype=np.uint8).reshape(-1, 4) & 3
    return (c[:, 0] | (c[:, 1] << 2) | (c[:, 2] << 4) | (c[:, 3] << 6)).astype(np.uint8)


def unpack_codes(packed: np.ndarray) -> np.ndarray:
    p = np.ascontiguousarray(packed, dtype=np.uint8)
    out = np.empty((p.size, 4), dtype=np.uint8)
    for j in range(4):
        out[:, j] = (p >> (2 * j)) & 3
    return out.reshape(-1)


def random_spins(L: int, q: int, seed: int) -> np.ndarray:
    """int8[N]: q=2 -> +-1, else 0..q-1, i.i.d. uniform from numpy (NOT the library's Philox init)."""
    rng = np.random.default_rng(seed)
    k = rng.integers(0, q, size=L * L)
    return (1 - 2 * k).astype(np.int8) if q == 2 else k.astype(np.int8)


def striped_spins(L: int, q: int, width: int) -> np.ndarray:
    """Vertical stripes of `width` columns cycling through the q states (structured edge case)."""
    x = np.arange(L * L) % L
    k = (x // width) % q
    return (1 - 2 * k).astype(np.int8) if q == 2 else k.astype(np.int8)


def snake_codes(L: int) -> np.ndarray:
    """A single cluster that is a boustrophedon path through the whole lattice: the longest possible chain,
    the degenerate worst case for pointer chasing.  Row y is fully east-connected; rows y and y+1 are joined
    at alternating ends; no wrap bonds."""
    codes = np.zeros((L, L), dtype=np.uint8)
    codes[:, : L - 1] |= 1
    for y in range(L - 1):
        codes[y, L - 1 if y % 2 == 0 else 0] |= 2
    return codes.reshape(-1)


def spiral_codes(L: int) -> np.ndarray:
    """Comb: one full row (y=0) plus every column as a tooth -> one cluster with long vertical runs."""
    codes = np.zeros((L, L), dtype=np.uint8)
    codes[0, : L - 1] |= 1
    codes[: L - 1, :] |= 2
    return codes.reshape(-1)


def blob_image(L: int, levels: int, seed: int, smooth: int = 3) -> np.ndarray:
    """uint8[L, L] synthetic grey-level image: seeded uniform noise, box-smoothed `smooth` times (3 x 3, no wrap), quantised to
    `levels` grey levels of equal population -- blobs of all sizes with ragged outlines, the structure of a segmentation input
    ("image segmentation").  Stands in for no dataset."""
    rng = np.random.default_rng(seed)
    a = rng.random((L, L))
    for _ in range(smooth):
        b = np.pad(a, 1, mode="edge")
        a = sum(b[1 + dy:1 + dy + L, 1 + dx:1 + dx + L] for dy in (-1, 0, 1) for dx in (-1, 0, 1)) / 9.0
    ranks = a.reshape(-1).argsort(kind="stable").argsort(kind="stable")
    return (ranks * levels // (L * L)).astype(np.uint8).reshape(L, L)


def image_bond_codes(img: np.ndarray) -> np.ndarray:
    """uint8[N] bond codes (the boundary's format: bit0 east, bit1 north) of the pixel-adjacency graph of an L x L image with
    4-connectivity: a bond joins two neighbouring pixels of equal value.  Row 0 of the array is lattice row y = 0.  An image
    has no periodic boundary: the east bonds of the last column and the north bonds of the last row stay open.  This is input
    preparation for sw_label (a graph handed to the labeller), not part of the method."""
    L = img.shape[0]
    assert img.shape == (L, L)
    codes = np.zeros((L, L), dtype=np.uint8)
    codes[:, : L - 1] |= (img[:, : L - 1] == img[:, 1:]).astype(np.uint8)
    codes[: L - 1, :] |= ((img[: L - 1, :] == img[1:, :]).astype(np.uint8) << 1)
    return codes.reshape(-1)
