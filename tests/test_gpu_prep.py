"""GPU parity for the sequence preparation (include/sla.h "Sequence preparation"): window keys,
the stable sort by key, gather/scatter of rows and the offsets, bit for bit against oracle/sla_prep_oracle.py on
the same seeded inputs; then the whole path coordinates -> sorted sequence -> SLA -> input order against the
oracles chained the same way."""
import numpy as np
import pytest

import paper_2401_00912_b200 as pkg
from paper_2401_00912_b200 import workloads as wl
from oracle import sla_oracle
from oracle import sla_prep_oracle as P

pytestmark = pytest.mark.gpu


def _torch():
    import torch
    return torch


def _dev(a):
    return _torch().from_numpy(np.ascontiguousarray(a)).cuda()


GRIDS = [  # batch, grid_h, grid_w, S_h, S_w
    (1, 468, 468, 12, 12),      # Waymo-like
    (2, 360, 360, 20, 20),      # nuScenes-like
    (3, 50, 70, 7, 12),         # windows that do not divide the grid
    (1, 5, 5, 9, 9),            # one window
]


@pytest.mark.parametrize("grid", GRIDS)
@pytest.mark.parametrize("n", [0, 1, 33, 513, 20011])
def test_window_keys(grid, n):
    torch = _torch()
    batch, gh, gw, sh, sw = grid
    rng = np.random.default_rng(n + gh)
    coords = np.stack([rng.integers(-1, batch + 1, n), rng.integers(0, 40, n), rng.integers(-2, gh + 2, n),
                       rng.integers(-2, gw + 2, n)], axis=1).astype(np.int32)
    want = P.window_keys(coords, batch, gh, gw, sh, sw)
    got = pkg.sla_window_keys(_dev(coords).reshape(n, 4), batch, gh, gw, sh, sw)
    torch.cuda.synchronize()
    assert pkg.sla_window_count(batch, gh, gw, sh, sw) == P.n_windows(batch, gh, gw, sh, sw)
    assert np.array_equal(got.cpu().numpy(), want)


def _keys(kind, n, W, rng):
    if kind == "uniform":
        return rng.integers(0, W + 1, n).astype(np.int32)
    if kind == "equal":
        return np.full(n, W // 2, np.int32)
    if kind == "descending":
        return (W - (np.arange(n) * (W + 1) // max(n, 1))).astype(np.int32)
    if kind == "few":                                   # long runs of a handful of keys
        return np.clip(rng.choice(np.array([0, 1, W // 3, W - 1, W], dtype=np.int64), n), 0, W).astype(np.int32)
    raise ValueError(kind)


@pytest.mark.parametrize("W", [0, 1, 255, 256, 3042, 65535, 65536, (1 << 24) + 5, (1 << 31) - 2])   # 1..4 passes
@pytest.mark.parametrize("n", [1, 31, 32, 512, 513, 2049, 70001])
def test_sort_by_window(W, n):
    torch = _torch()
    rng = np.random.default_rng(W % 1000 + n)
    for kind in ("uniform", "equal", "descending", "few"):
        key = _keys(kind, n, W, rng)
        perm_w, ks_w = P.sort_by_window(key)
        perm, ks = pkg.sla_sort_by_window(_dev(key), W)
        torch.cuda.synchronize()
        assert np.array_equal(ks.cpu().numpy(), ks_w), (kind, "key_sorted")
        assert np.array_equal(perm.cpu().numpy(), perm_w), (kind, "perm")


@pytest.mark.parametrize("n", [131072, 131073, 200001, 262144, 262145, 300001, 524289])
def test_sort_by_window_kernel_variants(n):
    """Sizes on both sides of the library's switches (short/long warp tiles, scan inside the scatter kernel or
    as a kernel of its own), two and three passes."""
    torch = _torch()
    for W in (3042, 70000):
        rng = np.random.default_rng(n + W)
        key = _keys("uniform", n, W, rng)
        perm_w, ks_w = P.sort_by_window(key)
        perm, ks = pkg.sla_sort_by_window(_dev(key), W)
        torch.cuda.synchronize()
        assert np.array_equal(ks.cpu().numpy(), ks_w)
        assert np.array_equal(perm.cpu().numpy(), perm_w)


def test_sort_empty_and_errors():
    torch = _torch()
    perm, ks = pkg.sla_sort_by_window(torch.empty(0, dtype=torch.int32, device="cuda"), 10)
    assert perm.numel() == 0 and ks.numel() == 0
    key = torch.zeros(100, dtype=torch.int32, device="cuda")
    with pytest.raises(pkg.SlaError):
        pkg.sla_sort_by_window(key, 10, workspace=torch.empty(16, dtype=torch.uint8, device="cuda"))
    with pytest.raises(pkg.SlaError):
        pkg.sla_sort_by_window(key, -1)
    with pytest.raises(pkg.SlaError):
        pkg.sla_window_keys(torch.zeros(4, 4, dtype=torch.int32, device="cuda"), 1, 10, 10, 0, 3)
    with pytest.raises(pkg.SlaError):
        pkg.sla_window_count(1 << 15, 1 << 15, 1 << 15, 1, 1)


def test_sort_one_million_properties():
    """Full-size property check (the oracle's argsort is a library sort, so it serves here too)."""
    torch = _torch()
    rng = np.random.default_rng(5)
    n, W = 1 << 20, 2 * 39 * 39
    key = rng.integers(0, W + 1, n).astype(np.int32)
    perm, ks = pkg.sla_sort_by_window(_dev(key), W)
    torch.cuda.synchronize()
    perm, ks = perm.cpu().numpy(), ks.cpu().numpy()
    assert np.array_equal(np.sort(perm), np.arange(n))
    assert np.array_equal(ks, key[perm]) and np.all(np.diff(ks) >= 0)
    assert np.all(np.diff(perm)[np.diff(ks) == 0] > 0)            # stable
    assert np.array_equal(perm, P.sort_by_window(key)[0])


@pytest.mark.parametrize("case", ["f16_rows256", "f32_rows12", "unaligned_base", "bf16_d32", "int8_rows4"])
def test_gather_scatter(case):
    torch = _torch()
    rng = np.random.default_rng(3)
    n = 7001
    perm = rng.permutation(n).astype(np.int32)
    if case == "f16_rows256":
        x = torch.from_numpy(rng.standard_normal((n, 8, 16)).astype(np.float16)).cuda()
    elif case == "f32_rows12":
        x = torch.from_numpy(rng.standard_normal((n, 3)).astype(np.float32)).cuda()
    elif case == "unaligned_base":                       # 16-byte rows at a base that is only 4-byte aligned
        buf = torch.from_numpy(rng.standard_normal(n * 4 + 1).astype(np.float32)).cuda()
        x = buf[1:].view(n, 4)
        assert x.data_ptr() % 16 == 4
    elif case == "bf16_d32":
        x = torch.from_numpy(rng.standard_normal((n, 4, 32)).astype(np.float32)).cuda().to(torch.bfloat16)
    else:
        x = torch.from_numpy(rng.integers(-128, 127, (n, 4)).astype(np.int8)).cuda()
    xn = x.view(torch.uint8).cpu().numpy().reshape(n, -1)
    g = pkg.sla_gather_rows(x, _dev(perm))
    s = pkg.sla_scatter_rows(g, _dev(perm))
    torch.cuda.synchronize()
    assert np.array_equal(g.view(torch.uint8).cpu().numpy().reshape(n, -1), P.gather_rows(xn, perm))
    assert np.array_equal(s.view(torch.uint8).cpu().numpy().reshape(n, -1), xn)
    assert np.array_equal(pkg.sla_scatter_rows(x, _dev(perm)).view(torch.uint8).cpu().numpy().reshape(n, -1),
                          P.scatter_rows(xn, perm))


def test_gather_skips_bad_perm_entries():
    torch = _torch()
    n = 100
    x = torch.arange(n * 4, dtype=torch.int32, device="cuda").view(n, 4)
    perm = torch.arange(n, dtype=torch.int32, device="cuda")
    perm[7], perm[50] = -1, n
    out = torch.full_like(x, -5)
    pkg.sla_gather_rows(x, perm, out=out)
    torch.cuda.synchronize()
    want = x.clone()
    want[7], want[50] = -5, -5
    assert torch.equal(out, want)
    with pytest.raises(pkg.SlaError):
        pkg.sla_gather_rows(torch.zeros(n, 3, dtype=torch.int8, device="cuda"), perm)   # 3-byte rows


@pytest.mark.parametrize("batch,n,n_outside", [(1, 60000, 0), (2, 30011, 13), (1, 700, 5)])
def test_sequence_from_coords(batch, n, n_outside):
    torch = _torch()
    coords = wl.coords_waymo_like(77 + n, N=n, batch=batch, n_outside=n_outside)
    W = P.n_windows(batch, 468, 468, 12, 12)
    key = P.window_keys(coords, batch, 468, 468, 12, 12)
    perm_w, ks_w = P.sort_by_window(key)
    off_w = P.window_offsets(ks_w, W)
    assert off_w[W] == n - n_outside
    perm, ks, off = pkg.sla_sequence_from_coords(_dev(coords), batch, 468, 468, 12, 12)
    torch.cuda.synchronize()
    assert np.array_equal(perm.cpu().numpy(), perm_w)
    assert np.array_equal(ks.cpu().numpy(), ks_w)
    assert np.array_equal(off.cpu().numpy(), off_w)


def test_coords_to_attention_and_back():
    """Voxels in voxeliser order -> window-sorted sequence -> SLA -> back to voxeliser order, every step in the
    library, against the two oracles chained the same way."""
    torch = _torch()
    n, n_outside, H, d = 20000, 9, 8, 16
    coords = wl.coords_waymo_like(901, N=n, batch=1, n_outside=n_outside)
    rng = np.random.default_rng(902)
    q, k, v = (wl.round_to_dtype(rng.standard_normal((n, H, d)).astype(np.float32), "f16") for _ in range(3))
    W = P.n_windows(1, 468, 468, 12, 12)
    # oracle chain
    perm_w, ks_w = P.sort_by_window(P.window_keys(coords, 1, 468, 468, 12, 12))
    off_w = P.window_offsets(ks_w, W)
    n_in = int(off_w[W])
    qs, ks_, vs = (P.gather_rows(t, perm_w)[:n_in] for t in (q, k, v))
    o_sorted = sla_oracle.forward(qs, ks_, vs, off_w, nthreads=8)
    want = np.zeros((n, H, d))
    want[perm_w[:n_in]] = o_sorted
    # library chain
    perm, _, off = pkg.sla_sequence_from_coords(_dev(coords), 1, 468, 468, 12, 12)
    assert int(off[W]) == n_in
    qd, kd, vd = (pkg.sla_gather_rows(_dev(t).to(torch.float16), perm) for t in (q, k, v))
    o = torch.zeros(n, H, d, dtype=torch.float16, device="cuda")
    pkg.sla_forward(qd[:n_in], kd[:n_in], vd[:n_in], off, out=o[:n_in])
    back = torch.zeros_like(o)
    # rows behind n_in belong to no window: zero them so that the scatter writes the zeros the oracle chain holds
    o[n_in:] = 0
    pkg.sla_scatter_rows(o, perm, out=back)
    torch.cuda.synchronize()
    got = back.double().cpu().numpy()
    err = np.abs(got - want) / (1e-3 + 2e-2 * np.abs(want))
    assert err.max() <= 1.0, err.max()
