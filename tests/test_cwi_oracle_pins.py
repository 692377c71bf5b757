"""Pins for oracle/sla_cwi_oracle.py: the hand-worked example, scipy.ndimage.correlate on the dense
zero-filled volume, delta kernels, an isolated voxel, a shifted delta, linearity."""
import os

import numpy as np
import scipy.ndimage as ndi

from oracle import sla_cwi_oracle as O

GOLD = os.path.join(os.path.dirname(__file__), "golden", "cwi_golden_5vox.txt")


def _golden():
    out = {}
    with open(GOLD) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            name, *vals = line.split()
            out[name] = np.array([float(v) for v in vals])
    return out


def test_golden_example():
    g = _golden()
    S_h, S_w = (int(v) for v in g["params"])
    w3 = np.arange(1, 28, dtype=np.float64).reshape(1, 27)
    out = O.cwi_forward(g["x"].reshape(5, 4), g["coords"].reshape(5, 4).astype(np.int64), S_h, S_w,
                        g["w_h"].reshape(1, 3), g["w_w"].reshape(1, 3), w3)
    assert np.array_equal(out, g["out"].reshape(5, 4))


def _scene(rng, n, batch, gz, gh, gw, C):
    cells = rng.choice(batch * gz * gh * gw, size=n, replace=False)
    b, r = np.divmod(cells, gz * gh * gw)
    z, r = np.divmod(r, gh * gw)
    y, xx = np.divmod(r, gw)
    return np.stack([b, z, y, xx], axis=1).astype(np.int64), rng.standard_normal((n, C))


def test_against_scipy_correlate_on_the_dense_volume():
    rng = np.random.default_rng(0)
    batch, gz, gh, gw, c, S_h, S_w = 2, 4, 11, 9, 3, 4, 6
    coords, x = _scene(rng, 150, batch, gz, gh, gw, 4 * c)
    w_h, w_w, w_3 = rng.standard_normal((c, S_h + 1)), rng.standard_normal((c, S_w + 1)), rng.standard_normal((c, 27))
    got = O.cwi_forward(x, coords, S_h, S_w, w_h, w_w, w_3)
    dense = np.zeros((batch, gz, gh, gw, 4 * c))
    dense[coords[:, 0], coords[:, 1], coords[:, 2], coords[:, 3]] = x
    want = np.zeros_like(dense)
    for b in range(batch):
        for ch in range(c):
            want[b, ..., ch] = ndi.correlate1d(dense[b, ..., ch], w_h[ch], axis=1, mode="constant", cval=0.0)
            want[b, ..., c + ch] = ndi.correlate1d(dense[b, ..., c + ch], w_w[ch], axis=2, mode="constant", cval=0.0)
            want[b, ..., 2 * c + ch] = ndi.correlate(dense[b, ..., 2 * c + ch], w_3[ch].reshape(3, 3, 3),
                                                     mode="constant", cval=0.0)
            want[b, ..., 3 * c + ch] = dense[b, ..., 3 * c + ch]
    assert np.allclose(got, want[coords[:, 0], coords[:, 1], coords[:, 2], coords[:, 3]], rtol=1e-12, atol=1e-12)


def test_delta_isolated_shift_and_linearity():
    rng = np.random.default_rng(1)
    c, S_h, S_w = 2, 2, 4
    coords, x = _scene(rng, 60, 1, 3, 8, 8, 4 * c)
    delta_h = np.zeros((c, S_h + 1)); delta_h[:, S_h // 2] = 1
    delta_w = np.zeros((c, S_w + 1)); delta_w[:, S_w // 2] = 1
    delta_3 = np.zeros((c, 27)); delta_3[:, 13] = 1
    assert np.array_equal(O.cwi_forward(x, coords, S_h, S_w, delta_h, delta_w, delta_3), x)       # centre taps: identity
    # an isolated voxel sees only its own centre taps
    w_h, w_w, w_3 = rng.standard_normal((c, S_h + 1)), rng.standard_normal((c, S_w + 1)), rng.standard_normal((c, 27))
    one = O.cwi_forward(x[:1], np.array([[0, 5, 5, 5]]), S_h, S_w, w_h, w_w, w_3)
    want = np.concatenate([w_h[:, S_h // 2] * x[0, :c], w_w[:, S_w // 2] * x[0, c:2 * c], w_3[:, 13] * x[0, 2 * c:3 * c],
                           x[0, 3 * c:]])
    assert np.allclose(one[0], want, rtol=1e-15)
    # a delta at offset +1 along x copies the right-hand neighbour's feature (correlation, not a flipped convolution)
    sh = np.zeros((c, S_w + 1)); sh[:, S_w // 2 + 1] = 1
    two = O.cwi_forward(x[:2], np.array([[0, 0, 3, 3], [0, 0, 3, 4]]), S_h, S_w, delta_h, sh, delta_3)
    assert np.array_equal(two[0, c:2 * c], x[1, c:2 * c]) and np.all(two[1, c:2 * c] == 0)
    # and along y for the first branch
    shy = np.zeros((c, S_h + 1)); shy[:, S_h // 2 - 1] = 1
    two = O.cwi_forward(x[:2], np.array([[0, 0, 3, 3], [0, 0, 2, 3]]), S_h, S_w, shy, delta_w, delta_3)
    assert np.array_equal(two[0, :c], x[1, :c]) and np.all(two[1, :c] == 0)
    x2 = rng.standard_normal(x.shape)
    a, b = 1.5, -0.25
    lhs = O.cwi_forward(a * x + b * x2, coords, S_h, S_w, w_h, w_w, w_3)
    rhs = a * O.cwi_forward(x, coords, S_h, S_w, w_h, w_w, w_3) + b * O.cwi_forward(x2, coords, S_h, S_w, w_h, w_w, w_3)
    assert np.allclose(lhs, rhs, rtol=1e-12, atol=1e-12)
