"""Seeded random sweeps: many small scenes of random structure through every tensor-core path against the oracles
(forward, backward, both feature maps, both head sizes, both 16-bit dtypes), and random shapes through the sequence
preparation.  Same tolerances as the targeted parity tests."""
import numpy as np
import pytest

import paper_2401_00912_b200 as pkg
from paper_2401_00912_b200 import workloads as wl
from oracle import sla_oracle
from oracle import sla_prep_oracle as P
import test_gpu_parity as T

pytestmark = pytest.mark.gpu


def _random_lengths(rng):
    kind = rng.integers(0, 4)
    if kind == 0:      # mostly tiny windows with empties
        ln = rng.integers(0, 5, rng.integers(1, 400))
    elif kind == 1:    # mid-sized windows around the tile and packing limits
        ln = rng.choice([1, 2, 15, 16, 17, 31, 32, 33, 63, 64, 65, 143, 144, 200], rng.integers(1, 40))
    elif kind == 2:    # a few long windows around the fuse limit and beyond, with tiny ones in between
        ln = rng.choice([1, 3, 255, 256, 257, 300, 511, 700, 1500], rng.integers(1, 10))
    else:              # geometric mix
        ln = np.minimum(rng.geometric(0.03, rng.integers(1, 120)), 900)
    ln = np.asarray(ln, dtype=np.int64)
    if ln.sum() == 0:
        ln[0] = 1
    return ln


@pytest.mark.parametrize("seed", range(24))
def test_random_scenes_forward_backward(seed):
    torch = T._torch()
    rng = np.random.default_rng(1000 + seed)
    dtype = ("f16", "bf16")[seed % 2]
    H, d = [(8, 16), (8, 32), (4, 16), (2, 32), (12, 16), (16, 32)][seed % 6]
    relu = (seed // 6) % 2 == 1
    scale = (1.0, 3.0)[(seed // 12) % 2]
    sc = wl.make_scene(_random_lengths(rng), H, d, dtype, seed=5000 + seed, scale=scale, name=f"rand{seed}")
    if relu:
        T._relu_case(sc)
        return
    out, ref = T.run_forward(sc)
    T.check(f"{sc.name}.out", out, ref, dtype, sc.lengths)
    grads, gref = T.run_backward(sc)
    T.check_grads(grads, gref, sc)


@pytest.mark.parametrize("seed", range(12))
def test_random_sequence_preparation(seed):
    torch = T._torch()
    rng = np.random.default_rng(2000 + seed)
    batch, gh, gw = int(rng.integers(1, 5)), int(rng.integers(1, 300)), int(rng.integers(1, 300))
    sh, sw = int(rng.integers(1, 25)), int(rng.integers(1, 25))
    n = int(rng.integers(0, 30000))
    coords = np.stack([rng.integers(-1, batch + 1, n), rng.integers(0, 40, n), rng.integers(-3, gh + 3, n),
                       rng.integers(-3, gw + 3, n)], axis=1).astype(np.int32)
    W = P.n_windows(batch, gh, gw, sh, sw)
    key = P.window_keys(coords, batch, gh, gw, sh, sw)
    perm_w, ks_w = P.sort_by_window(key)
    cd = torch.from_numpy(coords).cuda().reshape(n, 4)
    perm, ks, off = pkg.sla_sequence_from_coords(cd, batch, gh, gw, sh, sw)
    torch.cuda.synchronize()
    assert np.array_equal(perm.cpu().numpy(), perm_w) and np.array_equal(ks.cpu().numpy(), ks_w)
    n_in = int((key < W).sum())
    off_w = sla_oracle.offsets_from_window_ids(ks_w[:n_in], W)
    assert np.array_equal(off.cpu().numpy(), off_w)
