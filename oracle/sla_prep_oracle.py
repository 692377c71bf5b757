"""CPU oracle for the upstream sequence preparation: voxel coordinates -> window key ->
window-sorted order -> gathered rows.

TEST INFRASTRUCTURE ONLY: importable from tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs.  The product package never imports this module, and this module shares no code
with the CUDA path.

What the paper fixes (section 3.2): "we arrange the voxels of the entire scene into a single
flattened matrix ... These voxels are ordered based on their window coordinates, ensuring that voxels from
the same window form a sub-matrix in contiguous memory."  Windows are S_h x S_w cells of the bird's-eye-view
grid ("(S_w, S_h) ... (12, 12) and (20, 20)").  Everything here is integer work with a plain
definition, written out as that definition (reading A16 for what the paper leaves open):

  * coords[i] = (b, z, y, x), int32: sample index in the batch, then the voxel's cell, slowest axis first.
    z takes no part: windows tile the ground plane only.
  * window coordinate of a voxel = (b, y // S_h, x // S_w); its key is the row-major index of that triple in
    the [batch, ceil(grid_h / S_h), ceil(grid_w / S_w)] array of windows, W of them.  A voxel outside the
    grid (b, y or x out of range) gets the key W: it sorts behind every window and belongs to none.
  * the window-sorted order is the STABLE sort by key: voxels of one window keep their input order.  The
    paper does not order voxels inside a window (the op is invariant to it, reading A8); stability makes
    the permutation unique, hence testable bit for bit, and the op's rounding reproducible.
  * perm[j] = input position of the voxel that lands at sorted position j; gather: dst[j] = src[perm[j]];
    scatter (the way back for the op's output): dst[perm[j]] = src[j].

Pins (tests/test_prep_oracle_pins.py): a hand-worked example under tests/golden/, brute force with Python's
sorted() on (key, position) pairs, the permutation/sortedness/stability invariants, scatter(gather(x)) = x.
"""
from __future__ import annotations

import numpy as np


def n_windows(batch: int, grid_h: int, grid_w: int, S_h: int, S_w: int) -> int:
    """W = batch * ceil(grid_h / S_h) * ceil(grid_w / S_w)."""
    return batch * (-(-grid_h // S_h)) * (-(-grid_w // S_w))


def window_keys(coords, batch: int, grid_h: int, grid_w: int, S_h: int, S_w: int):
    """key[i] of every voxel, int32 [N]; W for a voxel outside the grid (reading A16)."""
    coords = np.asarray(coords, dtype=np.int64).reshape(-1, 4)
    nwy = -(-grid_h // S_h)
    nwx = -(-grid_w // S_w)
    W = batch * nwy * nwx
    key = np.empty(coords.shape[0], dtype=np.int32)
    for i in range(coords.shape[0]):
        b, _z, y, x = (int(c) for c in coords[i])
        if 0 <= b < batch and 0 <= y < grid_h and 0 <= x < grid_w:
            key[i] = (b * nwy + y // S_h) * nwx + x // S_w
        else:
            key[i] = W
    return key


def sort_by_window(key):
    """Stable sort by key: returns (perm int32 [N], key_sorted int32 [N]) with key_sorted = key[perm]."""
    key = np.asarray(key, dtype=np.int32)
    perm = np.argsort(key, kind="stable").astype(np.int32)
    return perm, key[perm]


def gather_rows(src, perm):
    """dst[j] = src[perm[j]]: the flattened window-sorted matrix of PAPER.md:77."""
    src = np.asarray(src)
    dst = np.empty_like(src)
    for j in range(len(perm)):
        dst[j] = src[perm[j]]
    return dst


def scatter_rows(src, perm):
    """dst[perm[j]] = src[j]: window-sorted rows back to the input order."""
    src = np.asarray(src)
    dst = np.empty_like(src)
    for j in range(len(perm)):
        dst[perm[j]] = src[j]
    return dst


def window_offsets(key_sorted, W: int):
    """offsets[w] = #{ j : key_sorted[j] < w }, w = 0..W ("offsets generation").

    offsets[W] is the number of voxels inside the grid; rows behind it carry the key W.
    """
    key_sorted = np.asarray(key_sorted, dtype=np.int64)
    off = np.zeros(W + 1, dtype=np.int32)
    for w in range(W + 1):
        off[w] = int(np.sum(key_sorted < w))
    return off
