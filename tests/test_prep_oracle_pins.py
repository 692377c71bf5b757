"""Pins for oracle/sla_prep_oracle.py: the hand-worked example, brute force with Python's
sorted() on tiny inputs, and the invariants that make the window-sorted order unique."""
import os

import numpy as np
import pytest

from oracle import sla_prep_oracle as P
from oracle import sla_oracle as O

GOLD = os.path.join(os.path.dirname(__file__), "golden", "prep_golden_12vox.txt")


def _golden():
    out = {}
    with open(GOLD) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            name, *vals = line.split()
            out[name] = np.array([int(v) for v in vals], dtype=np.int64)
    return out


def test_golden_example():
    g = _golden()
    batch, gh, gw, sh, sw = (int(v) for v in g["params"])
    coords = g["coords"].reshape(-1, 4)
    W = P.n_windows(batch, gh, gw, sh, sw)
    assert W == 18
    key = P.window_keys(coords, batch, gh, gw, sh, sw)
    assert key.tolist() == g["key"].tolist()
    perm, ks = P.sort_by_window(key)
    assert perm.tolist() == g["perm"].tolist()
    assert ks.tolist() == g["key_sorted"].tolist()
    assert P.window_offsets(ks, W).tolist() == g["offsets"].tolist()


def _random_scene(rng, n, batch, gh, gw, p_out=0.1):
    coords = np.stack([rng.integers(0, batch, n), rng.integers(0, 40, n), rng.integers(0, gh, n),
                       rng.integers(0, gw, n)], axis=1).astype(np.int32)
    bad = rng.random(n) < p_out                       # some voxels off the grid, on every axis and both sides
    which = rng.integers(0, 6, n)
    coords[bad & (which == 0), 0] = batch
    coords[bad & (which == 1), 0] = -1
    coords[bad & (which == 2), 2] = gh
    coords[bad & (which == 3), 2] = -3
    coords[bad & (which == 4), 3] = gw + 5
    coords[bad & (which == 5), 3] = -1
    return coords


@pytest.mark.parametrize("seed", range(6))
def test_brute_force_small(seed):
    rng = np.random.default_rng(seed)
    batch, gh, gw = int(rng.integers(1, 4)), int(rng.integers(1, 30)), int(rng.integers(1, 30))
    sh, sw = int(rng.integers(1, 9)), int(rng.integers(1, 9))
    n = int(rng.integers(0, 200))
    coords = _random_scene(rng, n, batch, gh, gw)
    W = P.n_windows(batch, gh, gw, sh, sw)
    key = P.window_keys(coords, batch, gh, gw, sh, sw)
    # the key, from the definition of a row-major index, via numpy's own index arithmetic
    nwy, nwx = -(-gh // sh), -(-gw // sw)
    for i in range(n):
        b, _, y, x = coords[i]
        inside = 0 <= b < batch and 0 <= y < gh and 0 <= x < gw
        want = np.ravel_multi_index((b, y // sh, x // sw), (batch, nwy, nwx)) if inside else W
        assert key[i] == want
    perm, ks = P.sort_by_window(key)
    brute = sorted(range(n), key=lambda i: (int(key[i]), i))      # stable order, by brute force
    assert perm.tolist() == brute
    assert ks.tolist() == [int(key[i]) for i in brute]
    off = P.window_offsets(ks, W)
    assert off.tolist() == [sum(1 for kk in key if kk < w) for w in range(W + 1)]
    # the same offsets through the SLA oracle's own routine on the in-grid prefix
    n_in = int(off[W])
    assert O.offsets_from_window_ids(ks[:n_in], W).tolist() == off.tolist()


def test_invariants_and_round_trip():
    rng = np.random.default_rng(11)
    coords = _random_scene(rng, 5000, 2, 468, 468, p_out=0.02)
    W = P.n_windows(2, 468, 468, 12, 12)
    assert W == 2 * 39 * 39
    key = P.window_keys(coords, 2, 468, 468, 12, 12)
    perm, ks = P.sort_by_window(key)
    assert sorted(perm.tolist()) == list(range(5000))             # a permutation
    assert np.all(np.diff(ks) >= 0)                                # sorted
    same = np.diff(ks) == 0
    assert np.all(np.diff(perm)[same] > 0)                         # stable: ties keep the input order
    x = rng.standard_normal((5000, 3)).astype(np.float32)
    g = P.gather_rows(x, perm)
    assert np.array_equal(g, x[perm])
    assert np.array_equal(P.scatter_rows(g, perm), x)              # scatter undoes gather
    # every window is a contiguous block whose voxels share one window coordinate
    off = P.window_offsets(ks, W)
    for w in rng.integers(0, W, 50):
        rows = perm[off[w]:off[w + 1]]
        for r in rows:
            b, _, y, xx = coords[r]
            assert (b * 39 + y // 12) * 39 + xx // 12 == w


def test_degenerate():
    key = P.window_keys(np.zeros((0, 4), np.int32), 1, 4, 4, 2, 2)
    perm, ks = P.sort_by_window(key)
    assert key.size == 0 and perm.size == 0 and ks.size == 0
    assert P.window_offsets(ks, 4).tolist() == [0] * 5
    # a window larger than the grid: one window per sample
    c = np.array([[0, 0, 3, 3], [1, 0, 0, 0], [0, 0, 0, 0]], np.int32)
    assert P.n_windows(2, 4, 4, 9, 9) == 2
    assert P.window_keys(c, 2, 4, 4, 9, 9).tolist() == [0, 1, 0]
    assert P.sort_by_window([0, 1, 0])[0].tolist() == [0, 2, 1]
