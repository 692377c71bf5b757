"""Pins for the CPU oracle (oracle/sla_oracle.cpp) against things OTHER than itself:
P1 brute-force quadratic form, P2 closed forms, P3 invariants (Eq. 2),
P4 zero-padded masked group attention (Fig. 1a), P5 golden example
(tests/golden/sla_golden_d2.txt), P6 gradient identities, P7 finite differences + torch autograd
on the quadratic definition.  CPU only; no CUDA path is touched here.
"""
import os

import numpy as np
import pytest
import torch

from oracle import sla_oracle as orc
from paper_2401_00912_b200 import workloads as wl

GOLD = os.path.join(os.path.dirname(__file__), "golden", "sla_golden_d2.txt")


def np_phi(x):
    # independent restatement of reading A1 via numpy primitives (elu(x)+1)
    return np.where(x > 0, x + 1.0, np.exp(np.minimum(x, 0.0)))


def offsets_of(lengths):
    return np.concatenate([[0], np.cumsum(lengths)]).astype(np.int32)


def rand_qkv(rng, N, H, d, scale=1.0):
    return tuple(scale * rng.standard_normal((N, H, d)) for _ in range(3))


def quadratic_window(q, k, v):
    """(phi(Q) phi(K)^T) V / rowsum for ONE window; q,k,v [m,H,d] -> [m,H,d] (numpy matmul)."""
    a, b = np_phi(q), np_phi(k)
    A = np.einsum("ihp,jhp->hij", a, b)               # [H,m,m] attention map phi(Q)phi(K)^T
    num = np.einsum("hij,jhr->ihr", A, v)
    den = A.sum(axis=2).T[:, :, None]                 # [m,H,1]
    return num / den


def load_golden():
    out, name, rows = {}, None, 0
    with open(GOLD) as f:
        lines = [ln.strip() for ln in f if ln.strip() and not ln.startswith("#")]
    i = 0
    while i < len(lines):
        name, r, c = lines[i].split()
        r, c = int(r), int(c)
        out[name] = np.array([[float(x) for x in lines[i + 1 + t].split()] for t in range(r)])
        assert out[name].shape == (r, c)
        i += 1 + r
    return out


# ---------------------------------------------------------------- P5 golden
def test_p5_golden_forward_and_state():
    g = load_golden()
    q, k, v = (g[n].reshape(3, 1, 2) for n in ("q", "k", "v"))
    off = np.array([0, 3], dtype=np.int32)
    o, S, z = orc.forward(q, k, v, off, return_state=True)
    np.testing.assert_allclose(S[0, 0], g["S"], rtol=0, atol=2e-12)
    np.testing.assert_allclose(z[0, 0], g["z"][0], rtol=0, atol=2e-12)
    np.testing.assert_allclose(o[:, 0, :], g["o"], rtol=0, atol=2e-12)


def test_p5_golden_hand_checkable_subcase():
    g = load_golden()
    q, k, v = (g[n][:2].reshape(2, 1, 2) for n in ("q", "k", "v"))
    o, S, z = orc.forward(q, k, v, np.array([0, 2], dtype=np.int32), return_state=True)
    np.testing.assert_allclose(S[0, 0], [[1, 2], [1, 1]], atol=1e-15)
    np.testing.assert_allclose(z[0, 0], [3, 2], atol=1e-15)
    np.testing.assert_allclose(o[:, 0, :], g["sub_o"], atol=1e-15)


def test_p5_golden_backward():
    g = load_golden()
    q, k, v, do = (g[n].reshape(3, 1, 2) for n in ("q", "k", "v", "dO"))
    dq, dk, dv = orc.backward(q, k, v, do, np.array([0, 3], dtype=np.int32))
    np.testing.assert_allclose(dq[:, 0, :], g["dq"], rtol=0, atol=2e-11)
    np.testing.assert_allclose(dk[:, 0, :], g["dk"], rtol=0, atol=2e-11)
    np.testing.assert_allclose(dv[:, 0, :], g["dv"], rtol=0, atol=2e-11)


# ---------------------------------------------------------------- P1 quadratic brute force
@pytest.mark.parametrize("H,d", [(1, 1), (2, 4), (4, 16), (3, 32)])
def test_p1_linear_equals_quadratic(H, d):
    rng = np.random.default_rng(1234 + 10 * H + d)
    lengths = np.array([1, 2, 3, 7, 0, 16, 17, 33, 64, 0, 5])
    off = offsets_of(lengths)
    q, k, v = rand_qkv(rng, int(lengths.sum()), H, d, scale=1.5)
    o = orc.forward(q, k, v, off)
    for w in range(len(lengths)):
        s, e = off[w], off[w + 1]
        if e > s:
            ref = quadratic_window(q[s:e], k[s:e], v[s:e])
            np.testing.assert_allclose(o[s:e], ref, rtol=1e-12, atol=1e-13)
    assert not np.isnan(o).any()


def test_p1_python_loop_definition_tiny():
    """Pure-Python triple loop of Eq. 3 on a tiny case (catches transposed S / wrong index)."""
    rng = np.random.default_rng(7)
    m, d = 5, 3
    q, k, v = rand_qkv(rng, m, 1, d)
    o = orc.forward(q, k, v, np.array([0, m], dtype=np.int32))
    import math
    ph = lambda x: x + 1.0 if x > 0 else math.exp(x)
    for i in range(m):
        wts = [sum(ph(q[i, 0, p]) * ph(k[j, 0, p]) for p in range(d)) for j in range(m)]
        for r in range(d):
            ref = sum(wts[j] * v[j, 0, r] for j in range(m)) / sum(wts)
            assert abs(o[i, 0, r] - ref) < 1e-13


# ---------------------------------------------------------------- P2 closed forms
def test_p2_length_one_windows_return_v():
    rng = np.random.default_rng(2)
    N, H, d = 37, 4, 16
    q, k, v = rand_qkv(rng, N, H, d, scale=3.0)
    o = orc.forward(q, k, v, np.arange(N + 1, dtype=np.int32))
    np.testing.assert_allclose(o, v, rtol=1e-14, atol=1e-14)


def test_p2_equal_keys_give_window_mean_of_v():
    rng = np.random.default_rng(3)
    lengths = np.array([4, 9, 1, 30])
    off = offsets_of(lengths)
    N, H, d = int(lengths.sum()), 2, 8
    q, k, v = rand_qkv(rng, N, H, d)
    for w in range(len(lengths)):
        k[off[w]:off[w + 1]] = k[off[w]]
    o = orc.forward(q, k, v, off)
    for w in range(len(lengths)):
        mean = v[off[w]:off[w + 1]].mean(axis=0, keepdims=True)
        np.testing.assert_allclose(o[off[w]:off[w + 1]], np.broadcast_to(mean, o[off[w]:off[w + 1]].shape),
                                   rtol=1e-12, atol=1e-13)


def test_p2_equal_values_returned_unchanged():
    rng = np.random.default_rng(4)
    lengths = np.array([6, 13])
    off = offsets_of(lengths)
    q, k, v = rand_qkv(rng, 19, 3, 4)
    for w in range(2):
        v[off[w]:off[w + 1]] = v[off[w]]
    o = orc.forward(q, k, v, off)
    np.testing.assert_allclose(o, v, rtol=1e-12, atol=1e-13)


def test_p2_dh1_output_independent_of_q():
    rng = np.random.default_rng(5)
    q, k, v = rand_qkv(rng, 11, 2, 1)
    off = np.array([0, 4, 11], dtype=np.int32)
    o1 = orc.forward(q, k, v, off)
    o2 = orc.forward(rng.standard_normal(q.shape), k, v, off)
    np.testing.assert_allclose(o1, o2, rtol=1e-12, atol=1e-13)
    b = np_phi(k)
    for s, e in [(0, 4), (4, 11)]:
        ref = (b[s:e] * v[s:e]).sum(0) / b[s:e].sum(0)
        np.testing.assert_allclose(o1[s:e], np.broadcast_to(ref, o1[s:e].shape), rtol=1e-12)


# ---------------------------------------------------------------- P3 invariants
def test_p3_convex_combination_bounds():
    s = wl.make_config(0)
    q, k, v = s.tensor("q"), s.tensor("k"), s.tensor("v")
    off = s.offsets
    o = orc.forward(q, k, v, off)
    for w in range(s.W):
        a, b = off[w], off[w + 1]
        vw = v[a:b].astype(np.float64)
        lo, hi = vw.min(axis=0), vw.max(axis=0)
        assert np.all(o[a:b] >= lo - 1e-12) and np.all(o[a:b] <= hi + 1e-12)


def test_p3_permutation_within_window():
    rng = np.random.default_rng(6)
    lengths = np.array([5, 12, 1, 20])
    off = offsets_of(lengths)
    N, H, d = int(lengths.sum()), 2, 8
    q, k, v = rand_qkv(rng, N, H, d)
    perm = np.arange(N)
    for w in range(len(lengths)):
        perm[off[w]:off[w + 1]] = off[w] + rng.permutation(lengths[w])
    o, S, z = orc.forward(q, k, v, off, return_state=True)
    o2, S2, z2 = orc.forward(q[perm], k[perm], v[perm], off, return_state=True)
    np.testing.assert_allclose(S2, S, rtol=1e-13, atol=1e-13)
    np.testing.assert_allclose(z2, z, rtol=1e-13, atol=1e-13)
    np.testing.assert_allclose(o2, o[perm], rtol=1e-12, atol=1e-13)


def test_p3_window_and_head_independence_and_concat():
    rng = np.random.default_rng(8)
    lengths = np.array([3, 0, 8, 21, 2])
    off = offsets_of(lengths)
    N, H, d = int(lengths.sum()), 3, 4
    q, k, v = rand_qkv(rng, N, H, d)
    o = orc.forward(q, k, v, off)
    # Eq. 2: concatenation of per-window LA
    for w in range(len(lengths)):
        s, e = off[w], off[w + 1]
        if e > s:
            ow = orc.forward(q[s:e], k[s:e], v[s:e], np.array([0, e - s], dtype=np.int32))
            np.testing.assert_array_equal(ow, o[s:e])
    # perturbing window 3 changes only its rows; perturbing head 1 changes only head 1
    k2 = k.copy(); k2[off[3]:off[4]] += 1.0
    o2 = orc.forward(q, k2, v, off)
    changed = np.abs(o2 - o).max(axis=(1, 2)) > 0
    assert changed[off[3]:off[4]].all() and not changed[:off[3]].any() and not changed[off[4]:].any()
    v3 = v.copy(); v3[:, 1, :] *= 2.0
    o3 = orc.forward(q, k, v3, off)
    np.testing.assert_array_equal(o3[:, [0, 2]], o[:, [0, 2]])
    np.testing.assert_allclose(o3[:, 1], 2.0 * o[:, 1], rtol=1e-13)


def test_p3_multithreaded_variant_identical():
    s = wl.make_config(0)
    q, k, v = s.tensor("q"), s.tensor("k"), s.tensor("v")
    o1 = orc.forward(q, k, v, s.offsets, nthreads=1)
    o4 = orc.forward(q, k, v, s.offsets, nthreads=4)
    np.testing.assert_array_equal(o1, o4)


# ---------------------------------------------------------------- P4 padded masked group attention
def test_p4_padded_masked_group_attention():
    rng = np.random.default_rng(9)
    lengths = np.array([1, 4, 9, 2, 16, 30, 7])
    off = offsets_of(lengths)
    N, H, d = int(lengths.sum()), 2, 8
    q, k, v = rand_qkv(rng, N, H, d)
    o = orc.forward(q, k, v, off)
    W, L = len(lengths), int(lengths.max())
    Qp = np.zeros((W, L, H, d)); Kp = np.zeros((W, L, H, d)); Vp = np.zeros((W, L, H, d))
    mask = np.zeros((W, L), dtype=bool)
    for w in range(W):
        m = lengths[w]
        Qp[w, :m], Kp[w, :m], Vp[w, :m] = q[off[w]:off[w + 1]], k[off[w]:off[w + 1]], v[off[w]:off[w + 1]]
        mask[w, :m] = True
    A = np.einsum("wihp,wjhp->whij", np_phi(Qp), np_phi(Kp))      # phi(0)=1 != 0: key mask is essential
    A = A * mask[:, None, None, :]
    Op = np.einsum("whij,wjhr->wihr", A, Vp) / A.sum(-1).transpose(0, 2, 1)[..., None]
    for w in range(W):
        np.testing.assert_allclose(Op[w, :lengths[w]], o[off[w]:off[w + 1]], rtol=1e-12, atol=1e-13)
    # without the mask the padded result differs (shows the mask matters under elu+1)
    A_nomask = np.einsum("wihp,wjhp->whij", np_phi(Qp), np_phi(Kp))
    O_nomask = np.einsum("whij,wjhr->wihr", A_nomask, Vp) / A_nomask.sum(-1).transpose(0, 2, 1)[..., None]
    assert np.abs(O_nomask[0, :1] - o[0:1]).max() > 1e-3


# ---------------------------------------------------------------- gradients: P6 identities
def _grad_case(seed=11, H=2, d=8, lengths=(1, 6, 19, 0, 3), scale=1.0):
    rng = np.random.default_rng(seed)
    lengths = np.array(lengths)
    off = offsets_of(lengths)
    N = int(lengths.sum())
    q, k, v = rand_qkv(rng, N, H, d, scale)
    g = rng.standard_normal((N, H, d))
    return q, k, v, g, off, lengths


def test_p6_gradient_identities():
    q, k, v, g, off, lengths = _grad_case()
    dq, dk, dv = orc.backward(q, k, v, g, off)
    phi_q, phi_k = np_phi(q), np_phi(k)
    dphi_q = np.where(q > 0, 1.0, np.exp(np.minimum(q, 0)))
    dphi_k = np.where(k > 0, 1.0, np.exp(np.minimum(k, 0)))
    da, db = dq / dphi_q, dk / dphi_k
    # o is degree-0 homogeneous in a_i  =>  a_i . da_i = 0
    assert np.abs((phi_q * da).sum(-1)).max() < 1e-12
    for w in range(len(lengths)):
        s, e = off[w], off[w + 1]
        if e == s:
            continue
        # o invariant to a common scaling of all b_j in the window => sum_j b_j . db_j = 0
        assert np.abs((phi_k[s:e] * db[s:e]).sum(axis=(0, 2))).max() < 1e-11
        # rows of the attention map sum to 1 => sum_j dv_j = sum_i g_i
        np.testing.assert_allclose(dv[s:e].sum(0), g[s:e].sum(0), rtol=1e-11, atol=1e-12)
        if e - s == 1:
            assert np.abs(dq[s:e]).max() < 1e-13 and np.abs(dk[s:e]).max() < 1e-13
            np.testing.assert_allclose(dv[s:e], g[s:e], rtol=1e-13)


# ---------------------------------------------------------------- gradients: P7 FD + autograd
def test_p7_torch_autograd_on_quadratic_form():
    q, k, v, g, off, lengths = _grad_case(seed=12, H=3, d=4, lengths=(2, 9, 1, 14))
    dq, dk, dv = orc.backward(q, k, v, g, off)
    tq, tk, tv = (torch.tensor(x, dtype=torch.float64, requires_grad=True) for x in (q, k, v))
    tg = torch.tensor(g)
    loss = 0.0
    for w in range(len(lengths)):
        s, e = int(off[w]), int(off[w + 1])
        a = torch.nn.functional.elu(tq[s:e]) + 1
        b = torch.nn.functional.elu(tk[s:e]) + 1
        A = torch.einsum("ihp,jhp->hij", a, b)
        o = torch.einsum("hij,jhr->ihr", A, tv[s:e]) / A.sum(-1).transpose(0, 1)[..., None]
        loss = loss + (o * tg[s:e]).sum()
    loss.backward()
    np.testing.assert_allclose(dq, tq.grad.numpy(), rtol=1e-10, atol=1e-12)
    np.testing.assert_allclose(dk, tk.grad.numpy(), rtol=1e-10, atol=1e-12)
    np.testing.assert_allclose(dv, tv.grad.numpy(), rtol=1e-10, atol=1e-12)


def test_p7_finite_differences_500_voxel_slice():
    """Central differences of L = sum(dO*O) on a 500-voxel slice of the config-4 layout
    (BASELINE.json configs[4]): a random scalar subset + 8 directional derivatives."""
    s4 = wl.make_config(4)
    off_full = s4.offsets
    wend = int(np.searchsorted(off_full, 500, side="right")) - 1
    off = off_full[: wend + 1].copy()
    n = int(off[-1])
    assert 300 <= n <= 500
    rng = np.random.default_rng(13)
    H, d = 8, 16
    q, k, v = rand_qkv(rng, n, H, d)
    g = rng.standard_normal((n, H, d))
    dq, dk, dv = orc.backward(q, k, v, g, off)
    L = lambda q_, k_, v_: float((orc.forward(q_, k_, v_, off) * g).sum())
    h = 1e-5
    grads = {"q": dq, "k": dk, "v": dv}
    base = {"q": q, "k": k, "v": v}
    for _ in range(8):   # directional derivatives over the whole slice
        dirs = {n_: rng.standard_normal(x.shape) for n_, x in base.items()}
        plus = L(*(base[n_] + h * dirs[n_] for n_ in "qkv"))
        minus = L(*(base[n_] - h * dirs[n_] for n_ in "qkv"))
        fd = (plus - minus) / (2 * h)
        an = sum(float((grads[n_] * dirs[n_]).sum()) for n_ in "qkv")
        assert abs(fd - an) <= 1e-6 * max(1.0, abs(an)), (fd, an)
    # per-scalar on a random subset: only the touched window needs recomputation
    wid = np.repeat(np.arange(len(off) - 1), np.diff(off))
    worst = 0.0
    for _ in range(150):
        name = "qkv"[rng.integers(3)]
        i, hh, c = rng.integers(n), rng.integers(H), rng.integers(d)
        w = wid[i]
        s, e = int(off[w]), int(off[w + 1])
        sub = {n_: base[n_][s:e].copy() for n_ in "qkv"}
        o2 = np.array([0, e - s], dtype=np.int32)
        f = lambda t: float((orc.forward(t["q"], t["k"], t["v"], o2) * g[s:e]).sum())
        sub[name][i - s, hh, c] += h
        fp = f(sub)
        sub[name][i - s, hh, c] -= 2 * h
        fm = f(sub)
        fd = (fp - fm) / (2 * h)
        an = grads[name][i, hh, c]
        worst = max(worst, abs(fd - an) / max(1e-3, abs(an)))
    assert worst < 1e-5, worst


# ---------------------------------------------------------------- offsets prep
def test_offsets_against_searchsorted_and_bruteforce():
    rng = np.random.default_rng(14)
    for W, N in [(1, 0), (1, 5), (7, 0), (10, 33), (64, 2000), (500, 300)]:
        ids = np.sort(rng.integers(0, W, size=N)).astype(np.int32)
        off = orc.offsets_from_window_ids(ids, W)
        ref = np.searchsorted(ids, np.arange(W + 1), side="left").astype(np.int32)
        np.testing.assert_array_equal(off, ref)
        if N <= 40:
            brute = np.array([int((ids < w).sum()) for w in range(W + 1)], dtype=np.int32)
            np.testing.assert_array_equal(off, brute)
        assert off[0] == 0 and off[-1] == N
    s = wl.make_config(3)
    np.testing.assert_array_equal(orc.offsets_from_window_ids(s.window_ids, s.W), s.offsets)


# ---------------------------------------------------------------- ReLU feature map with eps (reading A15)
GOLD_RELU = os.path.join(os.path.dirname(__file__), "golden", "sla_golden_relu_d2.txt")


def quadratic_window_relu(q, k, v, eps):
    """(relu(Q) relu(K)^T) V / (rowsum + eps) for ONE window (numpy restatement, PAPER.md:73 with reading A15)."""
    a, b = np.maximum(q, 0.0), np.maximum(k, 0.0)
    A = np.einsum("ihp,jhp->hij", a, b)
    return np.einsum("hij,jhr->ihr", A, v) / (A.sum(axis=2).T[:, :, None] + eps)


def test_relu_golden_hand_example():
    global GOLD
    saved, GOLD = GOLD, GOLD_RELU
    try:
        g = load_golden()
    finally:
        GOLD = saved
    q, k, v = (g[n][:, None, :] for n in ("q", "k", "v"))
    eps = float(g["eps"][0, 0])
    out, S, z = orc.forward(q, k, v, offsets_of([3]), return_state=True, phi="relu", eps=eps)
    np.testing.assert_allclose(S[0, 0], g["S"], rtol=0, atol=1e-15)
    np.testing.assert_allclose(z[0, 0], g["z"][0], rtol=0, atol=1e-15)
    np.testing.assert_allclose(out[:, 0, :], g["o"], rtol=1e-15, atol=1e-16)
    # the first two rows at eps = 0: (1,5)/6 and (0,1)
    out0 = orc.forward(q[:2], k[:2], v[:2], offsets_of([2]), phi="relu", eps=0.0)
    np.testing.assert_allclose(out0[:, 0, :], [[1 / 6, 5 / 6], [0.0, 1.0]], rtol=1e-15)


@pytest.mark.parametrize("H,d", [(1, 1), (2, 4), (3, 16), (2, 32)])
def test_relu_linear_equals_quadratic_with_eps(H, d):
    rng = np.random.default_rng(100 + d)
    lengths = [1, 2, 3, 7, 16, 33, 64]
    q, k, v = rand_qkv(rng, sum(lengths), H, d)
    off = offsets_of(lengths)
    for eps in (1e-6, 0.25):
        out = orc.forward(q, k, v, off, phi="relu", eps=eps)
        for w in range(len(lengths)):
            s, e = off[w], off[w + 1]
            np.testing.assert_allclose(out[s:e], quadratic_window_relu(q[s:e], k[s:e], v[s:e], eps), rtol=1e-12, atol=1e-14)


def test_relu_homogeneity_and_eps_closed_form():
    """relu(c x) = c relu(x) for c > 0: at eps = 0 the output is invariant to a positive scaling of q and of all k
    of a window (SURVEY f1's pin); and o(eps) = o(0) den / (den + eps) wherever den > 0."""
    rng = np.random.default_rng(7)
    lengths = [5, 40, 9]
    q, k, v = rand_qkv(rng, sum(lengths), 2, 8)
    off = offsets_of(lengths)
    o0, S, z = orc.forward(q, k, v, off, return_state=True, phi="relu", eps=0.0)
    assert np.isfinite(o0).all()                    # d = 8, windows >= 5 rows: den > 0 on this draw
    np.testing.assert_allclose(orc.forward(3.7 * q, k, v, off, phi="relu", eps=0.0), o0, rtol=1e-12, atol=1e-14)
    np.testing.assert_allclose(orc.forward(q, 0.2 * k, v, off, phi="relu", eps=0.0), o0, rtol=1e-12, atol=1e-14)
    eps = 0.3
    oe = orc.forward(q, k, v, off, phi="relu", eps=eps)
    for w in range(len(lengths)):
        s, e = off[w], off[w + 1]
        den = np.einsum("ihp,hp->ih", np.maximum(q[s:e], 0.0), z[w])[:, :, None]
        np.testing.assert_allclose(oe[s:e], o0[s:e] * den / (den + eps), rtol=1e-12, atol=1e-14)


def test_relu_length_one_windows():
    """m = 1: o = v (a.b)/(a.b + eps); exactly 0 when a.b = 0 (probability (3/4)^d per head)."""
    rng = np.random.default_rng(8)
    q, k, v = rand_qkv(rng, 400, 3, 4)
    off = offsets_of([1] * 400)
    eps = 1e-3
    out = orc.forward(q, k, v, off, phi="relu", eps=eps)
    ab = (np.maximum(q, 0.0) * np.maximum(k, 0.0)).sum(-1, keepdims=True)
    np.testing.assert_allclose(out, v * ab / (ab + eps), rtol=1e-13, atol=0)
    assert (ab == 0).any() and np.all(out[np.broadcast_to(ab == 0, out.shape)] == 0.0)


def test_relu_backward_autograd_and_finite_differences():
    rng = np.random.default_rng(21)
    lengths = (2, 9, 1, 14)
    N, H, d = sum(lengths), 3, 4
    q, k, v = rand_qkv(rng, N, H, d)
    # keep every input away from the kink of relu so that derivatives (and central differences) are well defined
    q = np.where(np.abs(q) < 0.05, 0.05 * np.sign(q) + (q == 0) * 0.05, q)
    k = np.where(np.abs(k) < 0.05, 0.05 * np.sign(k) + (k == 0) * 0.05, k)
    g = rng.standard_normal((N, H, d))
    off = offsets_of(lengths)
    eps = 1e-2
    dq, dk, dv = orc.backward(q, k, v, g, off, phi="relu", eps=eps)
    tq, tk, tv = (torch.tensor(x, dtype=torch.float64, requires_grad=True) for x in (q, k, v))
    tg = torch.tensor(g)
    loss = 0.0
    for w in range(len(lengths)):
        s, e = int(off[w]), int(off[w + 1])
        A = torch.einsum("ihp,jhp->hij", torch.relu(tq[s:e]), torch.relu(tk[s:e]))
        o = torch.einsum("hij,jhr->ihr", A, tv[s:e]) / (A.sum(-1).transpose(0, 1)[..., None] + eps)
        loss = loss + (o * tg[s:e]).sum()
    loss.backward()
    np.testing.assert_allclose(dq, tq.grad.numpy(), rtol=1e-10, atol=1e-12)
    np.testing.assert_allclose(dk, tk.grad.numpy(), rtol=1e-10, atol=1e-12)
    np.testing.assert_allclose(dv, tv.grad.numpy(), rtol=1e-10, atol=1e-12)
    # central differences of L = sum(g * forward) on a few scalars of each tensor
    def L(qq, kk, vv):
        return float((g * orc.forward(qq, kk, vv, off, phi="relu", eps=eps)).sum())
    h = 1e-6
    for name, x, grad in (("q", q, dq), ("k", k, dk), ("v", v, dv)):
        for _ in range(12):
            idx = tuple(rng.integers(0, n) for n in x.shape)
            xp, xm = x.copy(), x.copy()
            xp[idx] += h
            xm[idx] -= h
            args_p = {"q": (xp, k, v), "k": (q, xp, v), "v": (q, k, xp)}[name]
            args_m = {"q": (xm, k, v), "k": (q, xm, v), "v": (q, k, xm)}[name]
            fd = (L(*args_p) - L(*args_m)) / (2 * h)
            assert abs(fd - grad[idx]) <= 1e-6 * max(1.0, abs(grad[idx])), (name, idx, fd, grad[idx])
