"""GPU parity for the Cross-Window Interaction module (include/sla.h): the depth-wise sparse convolutions
against oracle/sla_cwi_oracle.py on the same seeded inputs.

Tolerance (reading A18): every output is a sum of at most T = S_h + S_w + 29 products accumulated in fp32 and
rounded once to the I/O dtype: |got - ref| <= acc + u (|ref| + acc) + 2^-24 with acc = (T + 1) 2^-24 sum_t |w_t x_t|
(oracle.magnitude) and u = 2^-24 / 2^-11 / 2^-8 for fp32 / fp16 / bf16.  The identity branch must come out bit for bit."""
import numpy as np
import pytest

import paper_2401_00912_b200 as pkg
from paper_2401_00912_b200 import workloads as wl
from oracle import sla_cwi_oracle as O

pytestmark = pytest.mark.gpu

UNIT = {"f32": 2.0 ** -24, "f16": 2.0 ** -11, "bf16": 2.0 ** -8}


def _torch():
    import torch
    return torch


def _tdt(dtype):
    torch = _torch()
    return {"f32": torch.float32, "f16": torch.float16, "bf16": torch.bfloat16}[dtype]


def _weights(rng, c, S_h, S_w):
    return tuple((rng.standard_normal((c, t)) / np.sqrt(t)).astype(np.float32) for t in (S_h + 1, S_w + 1, 27))


def _run(x, coords, grid, S_h, S_w, ws, dtype):
    torch = _torch()
    xd = torch.from_numpy(x).cuda().to(_tdt(dtype))
    out = pkg.sla_cwi_forward(xd, torch.from_numpy(coords.astype(np.int32)).cuda(), grid, S_h, S_w,
                              *(torch.from_numpy(w).cuda() for w in ws))
    torch.cuda.synchronize()
    return out


def _check(out, x, coords, S_h, S_w, ws, dtype):
    ref = O.cwi_forward(x, coords, S_h, S_w, *ws)
    mag = O.magnitude(x, coords, S_h, S_w, *ws)
    acc = (S_h + S_w + 30) * 2.0 ** -24 * mag
    allowed = acc + UNIT[dtype] * (np.abs(ref) + acc) + 2.0 ** -24
    g = out.double().cpu().numpy()
    assert np.isfinite(g).all()
    ratio = np.abs(g - ref) / allowed
    worst = np.unravel_index(np.argmax(ratio), ratio.shape)
    assert ratio.max() <= 1.0, f"worst err/bound {ratio.max():.3f} at {worst}: got {g[worst]} want {ref[worst]}"
    c = x.shape[1] // 4
    assert np.array_equal(g[:, 3 * c:], x[:, 3 * c:].astype(np.float64))          # identity branch: exact


def _dense_scene(rng, n, batch, gz, gh, gw):
    cells = rng.choice(batch * gz * gh * gw, size=n, replace=False)
    b, r = np.divmod(cells, gz * gh * gw)
    z, r = np.divmod(r, gh * gw)
    y, xx = np.divmod(r, gw)
    return np.stack([b, z, y, xx], axis=1).astype(np.int32)


@pytest.mark.parametrize("dtype", ["f32", "f16", "bf16"])
@pytest.mark.parametrize("C,S_h,S_w", [(128, 12, 12), (256, 20, 20), (64, 2, 4), (8, 12, 12), (512, 0, 0),
                                       (128, 16, 16), (128, 4, 6), (256, 32, 0), (64, 0, 0), (128, 18, 16), (128, 30, 2)])
def test_cwi_dense_neighbourhoods(dtype, C, S_h, S_w):
    """A small, densely occupied grid: most taps hit a voxel, windows reach over the borders and into other samples."""
    rng = np.random.Generator(np.random.PCG64(C + S_h))
    grid = (2, 3, 17, 19)
    coords = _dense_scene(rng, 1200, *grid)
    x = wl.round_to_dtype(rng.standard_normal((1200, C)).astype(np.float32), dtype)
    ws = _weights(rng, C // 4, S_h, S_w)
    _check(_run(x, coords, grid, S_h, S_w, ws, dtype), x, coords, S_h, S_w, ws, dtype)


@pytest.mark.parametrize("gz", [32, 33, 40])
def test_cwi_tall_grids_and_dirty_workspace(gz):
    """grid_z = 32 is the largest grid that takes the occupancy words (bit 31 in use); above, the index grid is cleared
    on every call.  The workspace starts full of values that look like voxel indices: none of them may be read as one."""
    torch = _torch()
    rng = np.random.Generator(np.random.PCG64(gz))
    grid = (2, gz, 9, 11)
    n = 900
    coords = _dense_scene(rng, n, *grid)
    coords[:8, 1] = gz - 1                                                # the top cell is occupied
    coords = np.unique(coords, axis=0).astype(np.int32)
    n = coords.shape[0]
    x = wl.round_to_dtype(rng.standard_normal((n, 128)).astype(np.float32), "f16")
    ws = _weights(rng, 32, 4, 4)
    nbytes = int(pkg.load_library().sla_cwi_workspace_bytes(*grid))
    buf = torch.randint(0, n, (nbytes // 4,), dtype=torch.int32, device="cuda").view(torch.uint8)
    out = pkg.sla_cwi_forward(torch.from_numpy(x).cuda().half(), torch.from_numpy(coords).cuda(), grid, 4, 4,
                              *(torch.from_numpy(w).cuda() for w in ws), workspace=buf)
    torch.cuda.synchronize()
    _check(out, x, coords, 4, 4, ws, "f16")


@pytest.mark.parametrize("n", [1, 31, 257])
def test_cwi_small_and_isolated(n):
    rng = np.random.Generator(np.random.PCG64(n))
    grid = (1, 8, 64, 64)
    coords = _dense_scene(rng, n, *grid)
    x = wl.round_to_dtype(rng.standard_normal((n, 128)).astype(np.float32), "f16")
    ws = _weights(rng, 32, 12, 12)
    _check(_run(x, coords, grid, 12, 12, ws, "f16"), x, coords, 12, 12, ws, "f16")


def test_cwi_waymo_like_scene_two_calls():
    """The bench's scene shape (468 x 468 ground grid, 32 cells in z, 12 x 12 windows), 20 000 voxels so that the
    oracle's loops finish in seconds; two calls in a row on different scenes share the index grid workspace."""
    torch = _torch()
    grid = (1, 32, 468, 468)
    ws_buf = torch.empty(int(pkg.load_library().sla_cwi_workspace_bytes(*grid)), dtype=torch.uint8, device="cuda")
    rng = np.random.Generator(np.random.PCG64(5))
    ws = _weights(rng, 32, 12, 12)
    for seed in (11, 12):
        coords = wl.coords_waymo_like(seed, N=20000, batch=1, nz=4)       # 4 occupied z cells: real 3-D neighbourhoods
        x = wl.round_to_dtype(rng.standard_normal((20000, 128)).astype(np.float32), "f16")
        out = pkg.sla_cwi_forward(torch.from_numpy(x).cuda().half(), torch.from_numpy(coords).cuda(), grid, 12, 12,
                                  *(torch.from_numpy(w).cuda() for w in ws), workspace=ws_buf)
        torch.cuda.synchronize()
        _check(out, x, coords, 12, 12, ws, "f16")


def test_cwi_writes_nothing_beyond_n_and_ignores_voxels_off_the_grid():
    torch = _torch()
    rng = np.random.Generator(np.random.PCG64(77))
    grid = (1, 2, 16, 16)
    coords = _dense_scene(rng, 200, *grid)
    x = wl.round_to_dtype(rng.standard_normal((200, 64)).astype(np.float32), "f16")
    ws = _weights(rng, 16, 4, 4)
    buf = torch.full((264, 64), 5.0, dtype=torch.float16, device="cuda")
    pkg.sla_cwi_forward(torch.from_numpy(x).cuda().half(), torch.from_numpy(coords).cuda(), grid, 4, 4,
                        *(torch.from_numpy(w).cuda() for w in ws), out=buf[:200])
    torch.cuda.synchronize()
    assert bool((buf[200:] == 5.0).all())
    _check(buf[:200], x, coords, 4, 4, ws, "f16")
    # a voxel off the grid: nobody sees it, its own convolution branches are zero, its identity branch is copied
    co2 = coords.copy()
    co2[7] = (0, 0, 16, 3)
    out = pkg.sla_cwi_forward(torch.from_numpy(x).cuda().half(), torch.from_numpy(co2).cuda(), grid, 4, 4,
                              *(torch.from_numpy(w).cuda() for w in ws))
    torch.cuda.synchronize()
    keep = np.ones(200, bool)
    keep[7] = False
    ref = O.cwi_forward(x[keep], co2[keep], 4, 4, *ws)
    got = out.double().cpu().numpy()
    assert np.allclose(got[keep], ref, rtol=2e-3, atol=2e-3)
    assert np.all(got[7, :48] == 0) and np.array_equal(got[7, 48:], x[7, 48:].astype(np.float64))


def test_cwi_full_size_properties():
    """The bench's size (60 000 voxels, 468 x 468 x 32 grid), where the oracle's Python loops would take minutes:
    properties that hold at any size.  (a) Relabelling the voxels permutes the output rows and changes nothing else
    (fixed tap order: bit for bit).  (b) Shifting the whole scene inside the grid changes nothing.  (c) Sampled
    voxels against the oracle evaluated on their neighbourhoods only."""
    torch = _torch()
    grid = (1, 32, 468, 468)
    rng = np.random.Generator(np.random.PCG64(2024))
    coords = wl.coords_waymo_like(2024, N=60000, batch=1, nz=6)
    coords[:, 2] = np.clip(coords[:, 2], 8, 459)             # room for the shift of (b)
    coords[:, 3] = np.clip(coords[:, 3], 8, 459)
    coords = np.unique(coords, axis=0).astype(np.int32)
    n = coords.shape[0]
    x = wl.round_to_dtype(rng.standard_normal((n, 128)).astype(np.float32), "f16")
    ws = _weights(rng, 32, 12, 12)
    wd = [torch.from_numpy(w).cuda() for w in ws]
    xd, cd = torch.from_numpy(x).cuda().half(), torch.from_numpy(coords).cuda()
    out = pkg.sla_cwi_forward(xd, cd, grid, 12, 12, *wd)
    perm = torch.from_numpy(rng.permutation(n)).cuda()
    out_p = pkg.sla_cwi_forward(xd[perm].contiguous(), cd[perm].contiguous(), grid, 12, 12, *wd)
    shift = torch.tensor([0, 1, 7, -5], dtype=torch.int32, device="cuda")
    out_s = pkg.sla_cwi_forward(xd, (cd + shift).contiguous(), grid, 12, 12, *wd)
    torch.cuda.synchronize()
    assert torch.equal(out_p, out[perm])
    assert torch.equal(out_s, out)
    sample = rng.choice(n, 300, replace=False)
    near = np.zeros(n, bool)
    for i in sample:                                          # every voxel any tap of a sampled voxel can reach
        d = np.abs(coords - coords[i])
        near |= (d[:, 0] == 0) & (d[:, 1] <= 1) & (d[:, 2] <= 6) & (d[:, 3] <= 6)
    idx = np.flatnonzero(near)
    ref = O.cwi_forward(x[idx], coords[idx], 12, 12, *ws)
    mag = O.magnitude(x[idx], coords[idx], 12, 12, *ws)
    pos = {int(v): j for j, v in enumerate(idx)}
    rows = np.array([pos[int(i)] for i in sample])
    acc = 54 * 2.0 ** -24 * mag[rows]
    got = out[torch.from_numpy(sample).cuda()].double().cpu().numpy()
    assert np.all(np.abs(got - ref[rows]) <= acc + UNIT["f16"] * (np.abs(ref[rows]) + acc) + 2.0 ** -24)


def test_cwi_errors():
    torch = _torch()
    x = torch.zeros(10, 128, dtype=torch.float16, device="cuda")
    co = torch.zeros(10, 4, dtype=torch.int32, device="cuda")
    w = [torch.zeros(32, t, dtype=torch.float32, device="cuda") for t in (13, 13, 27)]
    with pytest.raises(pkg.SlaError, match="INVALID_ARG"):
        pkg.sla_cwi_forward(x, co, (1, 4, 8, 8), 11, 12, torch.zeros(32, 12, dtype=torch.float32, device="cuda"), w[1], w[2])
    with pytest.raises(pkg.SlaError, match="WORKSPACE"):
        pkg.sla_cwi_forward(x, co, (1, 4, 8, 8), 12, 12, *w, workspace=torch.empty(16, dtype=torch.uint8, device="cuda"))
    with pytest.raises(pkg.SlaError):
        pkg.sla_cwi_forward(x, co, (1, 4, 8, 8), 12, 12, w[0], w[1], torch.zeros(32, 9, dtype=torch.float32, device="cuda"))
    with pytest.raises(pkg.SlaError, match="INVALID_ARG"):
        pkg.sla_cwi_forward(x, co, (1 << 12, 1 << 10, 1 << 10, 1 << 10), 12, 12, *w)
    e = torch.empty(0, 128, dtype=torch.float16, device="cuda")
    assert pkg.sla_cwi_forward(e, torch.empty(0, 4, dtype=torch.int32, device="cuda"), (1, 4, 8, 8), 12, 12, *w).numel() == 0
