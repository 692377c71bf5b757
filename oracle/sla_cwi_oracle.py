"""CPU oracle for the Cross-Window Interaction module: depth-wise sparse convolutions.

TEST INFRASTRUCTURE ONLY: importable from tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs.  The product package never imports this module, and it shares no code with the CUDA path.

What the paper fixes (Eq. 4-7): the input features of 4c channels are split along the channel
dimension into four branches, X' = Concat(X_k, X_w, X_h, X^{3c:4c}) with
    X_k = DWConv_{(S_h+1) x 1 x 1}(X^{:c}),   X_w = DWConv_{1 x (S_w+1) x 1}(X^{c:2c}),   X_h = DWConv_{3x3x3}(X^{2c:3c}),
and the last branch an identity mapping; (S_w, S_h) is the window size, DWConv a depth-wise (per-channel) convolution.
The definition is a plain sum over taps, written out as that sum.  What the paper leaves open is fixed by DESIGN.md
reading A18:
  * voxels are sparse: coords[i] = (b, z, y, x) int32, all distinct; the output lives on the same voxels as the input
    (a submanifold convolution: OpenPCDet-style sparse backbones keep the active set), and a tap that lands on a cell
    with no voxel, or outside the grid, or in another sample, contributes nothing;
  * the (S_h+1)-tap kernel runs along y, the (S_w+1)-tap kernel along x (S_h, S_w even, so the kernels are odd and
    centred: offsets -S/2 .. +S/2), the 3x3x3 kernel over (z, y, x) with offsets -1..1, tap index (dz+1)*9+(dy+1)*3+(dx+1);
  * cross-correlation as in every deep-learning "convolution": out[i] = sum_t w[t] * X[voxel at coords[i] + offset(t)];
  * weights are per channel: w_h [c, S_h+1], w_w [c, S_w+1], w_3 [c, 27]; no bias.

Pins (tests/test_cwi_oracle_pins.py): a hand-worked example under tests/golden/, scipy.ndimage.correlate on the dense
zero-filled volume (inactive cells are zeros there, which is the same rule), delta kernels -> identity, an isolated
voxel -> centre weight times input, a shifted delta -> the neighbour's feature, linearity.
"""
from __future__ import annotations

import numpy as np


def cwi_forward(x, coords, S_h: int, S_w: int, w_h, w_w, w_3):
    """x [N, 4c] -> out fp64 [N, 4c] (Eq. 4-7).  coords int [N, 4] rows (b, z, y, x), all distinct."""
    x = np.asarray(x, dtype=np.float64)
    coords = np.asarray(coords, dtype=np.int64).reshape(-1, 4)
    N, C = x.shape
    assert C % 4 == 0 and S_h % 2 == 0 and S_w % 2 == 0
    c = C // 4
    w_h = np.asarray(w_h, dtype=np.float64).reshape(c, S_h + 1)
    w_w = np.asarray(w_w, dtype=np.float64).reshape(c, S_w + 1)
    w_3 = np.asarray(w_3, dtype=np.float64).reshape(c, 27)
    where = {tuple(int(v) for v in coords[i]): i for i in range(N)}
    assert len(where) == N, "coords must be distinct"
    out = np.zeros((N, C))
    for i in range(N):
        b, z, y, xx = (int(v) for v in coords[i])
        for t in range(S_h + 1):                                   # Eq. 5: (S_h+1)-tap kernel along y, channels [0, c)
            j = where.get((b, z, y + t - S_h // 2, xx))
            if j is not None:
                out[i, 0:c] += w_h[:, t] * x[j, 0:c]
        for t in range(S_w + 1):                                   # Eq. 6: (S_w+1)-tap kernel along x, channels [c, 2c)
            j = where.get((b, z, y, xx + t - S_w // 2))
            if j is not None:
                out[i, c:2 * c] += w_w[:, t] * x[j, c:2 * c]
        for dz in (-1, 0, 1):                                      # Eq. 7: 3x3x3, channels [2c, 3c)
            for dy in (-1, 0, 1):
                for dx in (-1, 0, 1):
                    j = where.get((b, z + dz, y + dy, xx + dx))
                    if j is not None:
                        out[i, 2 * c:3 * c] += w_3[:, (dz + 1) * 9 + (dy + 1) * 3 + (dx + 1)] * x[j, 2 * c:3 * c]
        out[i, 3 * c:] = x[i, 3 * c:]                              # Eq. 4: identity branch
    return out


def magnitude(x, coords, S_h: int, S_w: int, w_h, w_w, w_3):
    """sum over taps of |w| |x| per output element (the same sums on absolute values): scale of the fp32 accumulation
    error the parity test allows."""
    return cwi_forward(np.abs(np.asarray(x, dtype=np.float64)), coords, S_h, S_w, np.abs(w_h), np.abs(w_w), np.abs(w_3))
