"""Pins for oracle/sla_proj_oracle.py: the hand-worked example, a pure-Python triple loop, selector and
identity weights, linearity, zero input."""
import os

import numpy as np

from oracle import sla_proj_oracle as P

GOLD = os.path.join(os.path.dirname(__file__), "golden", "proj_golden_c2.txt")


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
    q, k, v = P.project_qkv(g["x"].reshape(3, 2), g["w"].reshape(6, 2), g["bias"])
    assert np.array_equal(q, g["q"].reshape(3, 2))
    assert np.array_equal(k, g["k"].reshape(3, 2))
    assert np.array_equal(v, g["v"].reshape(3, 2))


def test_triple_loop_brute_force():
    rng = np.random.default_rng(0)
    N, C = 7, 5
    x = rng.standard_normal((N, C))
    w = rng.standard_normal((3 * C, C))
    b = rng.standard_normal(3 * C)
    want = [[0.0] * (3 * C) for _ in range(N)]
    for i in range(N):
        for j in range(3 * C):
            acc = float(b[j])
            for c in range(C):
                acc += float(x[i, c]) * float(w[j, c])
            want[i][j] = acc
    want = np.array(want)
    q, k, v = P.project_qkv(x, w, b)
    assert np.allclose(np.concatenate([q, k, v], axis=1), want, rtol=1e-13, atol=1e-13)


def test_selector_identity_and_zero():
    rng = np.random.default_rng(1)
    N, C = 9, 6
    x = rng.standard_normal((N, C))
    # output feature j copies input column sel[j]: a transposed operand or a wrong block order cannot pass
    sel = rng.integers(0, C, 3 * C)
    w = np.zeros((3 * C, C))
    w[np.arange(3 * C), sel] = 1.0
    q, k, v = P.project_qkv(x, w)
    y = np.concatenate([q, k, v], axis=1)
    for j in range(3 * C):
        assert np.array_equal(y[:, j], x[:, sel[j]])
    eye3 = np.concatenate([np.eye(C), 2 * np.eye(C), -np.eye(C)], axis=0)
    q, k, v = P.project_qkv(x, eye3)
    assert np.array_equal(q, x) and np.array_equal(k, 2 * x) and np.array_equal(v, -x)
    b = rng.standard_normal(3 * C)
    q, k, v = P.project_qkv(np.zeros((N, C)), rng.standard_normal((3 * C, C)), b)
    assert np.array_equal(np.concatenate([q, k, v], axis=1), np.tile(b, (N, 1)))


def test_linearity_and_bound():
    rng = np.random.default_rng(2)
    N, C = 11, 8
    x1, x2 = rng.standard_normal((N, C)), rng.standard_normal((N, C))
    w = rng.standard_normal((3 * C, C))
    a, b = 0.75, -2.5
    y12 = np.concatenate(P.project_qkv(a * x1 + b * x2, w), axis=1)
    y1 = np.concatenate(P.project_qkv(x1, w), axis=1)
    y2 = np.concatenate(P.project_qkv(x2, w), axis=1)
    assert np.allclose(y12, a * y1 + b * y2, rtol=1e-12, atol=1e-12)
    # the accumulation bound covers an fp32 evaluation of the same product (inputs exactly representable in fp32)
    xf, wf = x1.astype(np.float32), w.astype(np.float32)
    acc, mag = P.accumulation_bound(xf, wf)
    y32 = (xf @ wf.T).astype(np.float64)
    yex = xf.astype(np.float64) @ wf.T.astype(np.float64)
    assert np.all(np.abs(y32 - yex) <= acc) and np.all(mag >= np.abs(yex) * (1 - 1e-12))
