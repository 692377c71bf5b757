"""CPU oracle for the shared Q/K/V projection around the SLA op.

TEST INFRASTRUCTURE ONLY: importable from tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs.  The product package never imports this module, and it shares no code with the CUDA path.

What the paper fixes: "Self-attention first linearly projects the input to queries, keys, and values using weight
matrices W_Q, W_K and W_V, such that Q = x W_Q, K = x W_K, V = x W_V" and "we use a shared projection layer
to map all the voxels in the scene to query, key, and value representations, denoted Q, K, V".  The
definition is a matrix product, written out as one (numpy matmul in fp64 is the library primitive of this step).
What the paper leaves open is fixed by DESIGN.md reading A17:
  * x is [N, C] with C = H * d_h; "shared" = one layer for every voxel of the scene, one [3C, C] weight: row j holds the
    weights of output feature j (the layout of a linear layer's weight), rows 0..C-1 give Q, C..2C-1 give K, 2C..3C-1
    give V; so W_Q of the paper is w[0:C].T and Q = x @ w[0:C].T.  Head h of Q is its columns h*d_h .. (h+1)*d_h-1.
  * an optional bias [3C] is added (the paper's formula has none: pass None).
  * the module = projection, then SLA on (Q, K, V) rounded to the I/O dtype (they are tensors of that dtype in memory).

Pins (tests/test_proj_oracle_pins.py): a hand-worked example under tests/golden/, a pure-Python triple loop on tiny
inputs, selector weights (output column j copies input column i: catches a transposed operand), identity, linearity,
zero input -> bias.
"""
from __future__ import annotations

import numpy as np


def project_qkv(x, w, bias=None):
    """(Q, K, V), each fp64 [N, C]: y = x @ w.T (+ bias), split into three blocks of C output features."""
    x = np.asarray(x, dtype=np.float64)
    w = np.asarray(w, dtype=np.float64)
    C = x.shape[1]
    assert w.shape == (3 * C, C), "w must be [3C, C]: one row per output feature"
    y = np.matmul(x, w.T)
    if bias is not None:
        y = y + np.asarray(bias, dtype=np.float64).reshape(1, 3 * C)
    return y[:, :C].copy(), y[:, C:2 * C].copy(), y[:, 2 * C:].copy()


def accumulation_bound(x, w, bias=None):
    """(bound, mag): mag = sum_k |x_k w_k| (+ |bias|), and bound = (K + 1) * 2^-24 * mag, which covers the error of
    accumulating the K products (and the bias) in fp32 in any order (Higham, Accuracy and Stability, 3.5, to first
    order in 2^-24).  The parity test adds the final rounding to the storage format on top of it."""
    x = np.abs(np.asarray(x, dtype=np.float64))
    w = np.abs(np.asarray(w, dtype=np.float64))
    K = x.shape[1]
    mag = np.matmul(x, w.T)
    if bias is not None:
        mag = mag + np.abs(np.asarray(bias, dtype=np.float64)).reshape(1, -1)
    return (K + 1) * 2.0 ** -24 * mag, mag
