"""GPU parity: the CUDA path (through the C ABI) against the fp64 CPU oracle, element by element on
the same seeded inputs.  Tolerances (BASELINE.json north_star; reading A11):
  |gpu - ref| <= atol + rtol*|ref|,  fp32: rtol 1e-5, atol 1e-6;  fp16/bf16: rtol 2e-2, atol 1e-3.
Gradients additionally: relative L2 error <= 1e-2 (fp16/bf16), 1e-5 (fp32), taken over the rows
of windows with >= 2 voxels and, separately, over the rows of windows longer than 256 voxels (whose small
gradients would pass the atol of the elementwise check trivially).  Rows of length-1 windows (dq = dk = 0
exactly, so a relative norm is ill-posed there) keep the elementwise check only."""
import numpy as np
import pytest

import paper_2401_00912_b200 as pkg
from paper_2401_00912_b200 import workloads as wl
from oracle import sla_oracle

pytestmark = pytest.mark.gpu

TOL = {"f32": (1e-5, 1e-6), "f16": (2e-2, 1e-3), "bf16": (2e-2, 1e-3)}
REL_L2 = {"f32": 1e-5, "f16": 1e-2, "bf16": 1e-2}


def _torch():
    import torch
    return torch


def to_dev(a, dtype):
    torch = _torch()
    tdt = {"f32": torch.float32, "f16": torch.float16, "bf16": torch.bfloat16}[dtype]
    return torch.from_numpy(a).cuda().to(tdt)   # values are already exactly representable


def check(name, got_t, want, dtype, lengths=None):
    rtol, atol = TOL[dtype]
    got = got_t.double().cpu().numpy()
    assert np.isfinite(got).all(), f"{name}: non-finite output"
    err = np.abs(got - want) / (atol + rtol * np.abs(want))
    worst = np.unravel_index(np.argmax(err), err.shape)
    msg = f"{name}: worst err/tol {err.max():.3f} at {worst} got {got[worst]} want {want[worst]}"
    if lengths is not None:
        off = np.concatenate([[0], np.cumsum(lengths)])
        w = int(np.searchsorted(off, worst[0], side="right") - 1)
        msg += f" (window {w}, length {int(lengths[w])})"
    assert err.max() <= 1.0, msg
    return float(err.max())


def run_forward(sc, workspace=None):
    torch = _torch()
    q, k, v = sc.tensor("q"), sc.tensor("k"), sc.tensor("v")
    off = torch.from_numpy(sc.offsets).cuda()
    out = pkg.sla_forward(to_dev(q, sc.dtype), to_dev(k, sc.dtype), to_dev(v, sc.dtype), off)
    torch.cuda.synchronize()
    ref = sla_oracle.forward(q, k, v, sc.offsets, nthreads=8)
    return out, ref


def run_backward(sc):
    torch = _torch()
    q, k, v, g = sc.tensor("q"), sc.tensor("k"), sc.tensor("v"), sc.tensor("do")
    off = torch.from_numpy(sc.offsets).cuda()
    grads = pkg.sla_backward(to_dev(q, sc.dtype), to_dev(k, sc.dtype), to_dev(v, sc.dtype), off,
                             to_dev(g, sc.dtype))
    torch.cuda.synchronize()
    ref = sla_oracle.backward(q, k, v, g, sc.offsets, nthreads=8)
    return grads, ref


def check_grads(grads, ref, sc):
    lengths = np.asarray(sc.lengths)
    row_len = np.repeat(lengths, lengths)                 # window length of every row
    groups = [("windows>=2", row_len >= 2), ("windows>256", row_len > 256)]
    for name, got, want in zip(("dq", "dk", "dv"), grads, ref):
        check(f"{sc.name}.{name}", got, want, sc.dtype, sc.lengths)
        gotd = got.double().cpu().numpy()
        for gname, rows in groups:
            if not rows.any():
                continue
            den = np.linalg.norm(want[rows])
            if den == 0.0:
                continue
            rel = np.linalg.norm(gotd[rows] - want[rows]) / den
            assert rel <= REL_L2[sc.dtype], f"{sc.name}.{name} [{gname}]: relative L2 error {rel:.3e} > {REL_L2[sc.dtype]:.0e}"


# ---- prep kernel: bit-exact ----------------------------------------------------------------------
@pytest.mark.parametrize("case", ["config0", "config1", "config3", "gaps", "single", "empty_tail", "n0"])
def test_offsets_bit_exact(case):
    torch = _torch()
    if case.startswith("config"):
        sc = wl.make_config(int(case[-1]))
        lengths = sc.lengths
    elif case == "gaps":
        lengths = np.array([0, 0, 3, 0, 1, 0, 0, 0, 700, 0, 2, 0, 0])
    elif case == "single":
        lengths = np.array([1000])
    elif case == "empty_tail":
        lengths = np.array([5, 0, 0, 0])
    else:
        lengths = np.array([0, 0, 0])
    W = len(lengths)
    ids = np.repeat(np.arange(W, dtype=np.int32), lengths)
    want = sla_oracle.offsets_from_window_ids(ids, W)
    got = pkg.sla_offsets_from_window_ids(torch.from_numpy(ids).cuda(), W)
    torch.cuda.synchronize()
    assert np.array_equal(got.cpu().numpy(), want)
    assert np.array_equal(want, np.concatenate([[0], np.cumsum(lengths)]).astype(np.int32))


# ---- the five BASELINE.json configs, full size, every element --------------------------------------
@pytest.mark.parametrize("c", [0, 1, 2, 3])
def test_forward_configs(c):
    sc = wl.make_config(c)
    out, ref = run_forward(sc)
    check(f"{sc.name}.out", out, ref, sc.dtype, sc.lengths)


def test_forward_backward_config4():
    sc = wl.make_config(4)
    out, ref = run_forward(sc)
    check(f"{sc.name}.out", out, ref, sc.dtype, sc.lengths)
    grads, gref = run_backward(sc)
    check_grads(grads, gref, sc)


@pytest.mark.parametrize("c", [0, 2, 3])
def test_backward_other_configs(c):
    sc = wl.make_config(c)
    grads, gref = run_backward(sc)
    check_grads(grads, gref, sc)


# ---- edge cases (SURVEY.md §8c list) ---------------------------------------------------------------
EDGE_LAYOUTS = {
    "one_window": [777],
    "all_len1": [1] * 333,
    "empty_start_end_consecutive": [0, 0, 5, 0, 0, 0, 9, 40, 0],
    "around_rowbatch_4_8": [3, 4, 5, 7, 8, 9, 15, 16, 17, 31, 32, 33],
    "around_tile_64": [63, 64, 65, 1, 127, 128, 129],
    "around_fuse_256": [255, 256, 257, 2, 258, 1, 511, 513],
    "huge_and_tiny": [1, 2, 3000, 1, 1, 2, 4097, 3],
    "ragged_not_mult16": [13, 29, 101, 7],
}


@pytest.mark.parametrize("layout", sorted(EDGE_LAYOUTS))
@pytest.mark.parametrize("dtype,H,d", [("f32", 4, 32), ("f32", 2, 16), ("f16", 8, 16), ("f16", 8, 32),
                                       ("bf16", 8, 32), ("bf16", 4, 16), ("f16", 1, 16), ("f32", 1, 32),
                                       ("f16", 3, 16), ("bf16", 16, 32), ("f16", 2, 32), ("bf16", 6, 32)])
def test_edge_layouts_forward_backward(layout, dtype, H, d):
    sc = wl.make_scene(EDGE_LAYOUTS[layout], H, d, dtype, seed=77 + len(layout), name=layout)
    out, ref = run_forward(sc)
    check(f"{layout}.out", out, ref, dtype, sc.lengths)
    grads, gref = run_backward(sc)
    check_grads(grads, gref, sc)


@pytest.mark.parametrize("d", [16, 32])
@pytest.mark.parametrize("dtype", ["f32", "f16", "bf16"])
def test_large_magnitude_inputs(dtype, d):
    """q,k entries of +-20: phi spans e^-20 .. 21; the normaliser must stay finite and accurate."""
    sc = wl.make_scene([1, 2, 9, 40, 300], 4, d, dtype, seed=5)
    rng = np.random.Generator(np.random.PCG64(99))
    q, k, v = sc.tensor("q"), sc.tensor("k"), sc.tensor("v")
    sel = rng.random(q.shape) < 0.2
    q = wl.round_to_dtype(np.where(sel, np.sign(q) * 20.0, q).astype(np.float32), dtype)
    sel = rng.random(k.shape) < 0.2
    k = wl.round_to_dtype(np.where(sel, np.sign(k) * 20.0, k).astype(np.float32), dtype)
    torch = _torch()
    off = torch.from_numpy(sc.offsets).cuda()
    out = pkg.sla_forward(to_dev(q, dtype), to_dev(k, dtype), to_dev(v, dtype), off)
    ref = sla_oracle.forward(q, k, v, sc.offsets)
    check("large_magnitude.out", out, ref, dtype, sc.lengths)
    # backward on the same inputs: phi' spans e^-20 .. 1, den spans orders of magnitude
    g = sc.tensor("do")
    grads = pkg.sla_backward(to_dev(q, dtype), to_dev(k, dtype), to_dev(v, dtype), off, to_dev(g, dtype))
    torch.cuda.synchronize()
    gref = sla_oracle.backward(q, k, v, g, sc.offsets)
    for name, got, want in zip(("dq", "dk", "dv"), grads, gref):
        check(f"large_magnitude.{name}", got, want, dtype, sc.lengths)


@pytest.mark.parametrize("entry", ["tc", "tcgen05"])
@pytest.mark.parametrize("dtype", ["f16", "bf16"])
@pytest.mark.parametrize("shift,lengths", [(-8.0, [3, 12, 17, 40, 144, 200, 700]), (-11.0, [3, 12, 17, 40, 144, 200, 700]),
                                           (-12.0, [17, 40, 144, 200, 700])])
def test_forward_windows_whose_keys_are_all_far_below_zero(shift, lengths, dtype, entry):
    """Every key of a window around -8 ... -12: phi(k) ~ 3e-4 ... 6e-6, so z / m lies far below the fp16 normal range
    (6.1e-5).  The kernels scale the state by the exponent of its own largest z before the fp16 rounding (Eq. 3 is a
    ratio: any common factor of S and z cancels), so windows that go through a state stay accurate.  Windows of <= 16
    rows (packed quadratic tiles) use phi(k) itself as an fp16 operand and keep their accuracy down to k ~ -11; below
    -12 the fp16 subnormal spacing of phi(k) itself (6e-8) is what limits every path."""
    if entry == "tcgen05" and dtype != "f16":
        pytest.skip("the tcgen05 entry takes fp16")
    sc = wl.make_scene(lengths, 8, 16, dtype, seed=21)
    q, v = sc.tensor("q"), sc.tensor("v")
    k = wl.round_to_dtype((0.5 * sc.tensor("k") + shift).astype(np.float32), dtype)
    torch = _torch()
    off = torch.from_numpy(sc.offsets).cuda()
    out = pkg.sla_forward(to_dev(q, dtype), to_dev(k, dtype), to_dev(v, dtype), off, tcgen05=(entry == "tcgen05"))
    torch.cuda.synchronize()
    ref = sla_oracle.forward(q, k, v, sc.offsets)
    check(f"keys_at_{shift}.out", out, ref, dtype, sc.lengths)


@pytest.mark.parametrize("d", [16, 32])
@pytest.mark.parametrize("dtype", ["f16", "bf16"])
@pytest.mark.parametrize("shift,lengths", [(-8.0, [3, 12, 17, 40, 144, 200, 700]), (-11.0, [3, 12, 17, 40, 144, 200, 700]),
                                           (-12.0, [40, 144, 200, 700])])
def test_backward_windows_whose_keys_are_all_far_below_zero(shift, lengths, dtype, d):
    """The same regime for the gradients: den = phi(q) . z is ~ m * 1e-4, so g / den and dS are large while phi'(k) is
    tiny; the tensor-core backward scales S, z, dS and dz by the exponent of the window's largest z."""
    sc = wl.make_scene(lengths, 8 if d == 16 else 4, d, dtype, seed=22)
    q, v, g = sc.tensor("q"), sc.tensor("v"), sc.tensor("do")
    k = wl.round_to_dtype((0.5 * sc.tensor("k") + shift).astype(np.float32), dtype)
    torch = _torch()
    off = torch.from_numpy(sc.offsets).cuda()
    grads = pkg.sla_backward(to_dev(q, dtype), to_dev(k, dtype), to_dev(v, dtype), off, to_dev(g, dtype))
    torch.cuda.synchronize()
    gref = sla_oracle.backward(q, k, v, g, sc.offsets)
    for name, got, want in zip(("dq", "dk", "dv"), grads, gref):
        check(f"keys_at_{shift}.{name}", got, want, dtype, sc.lengths)


# ---- the tcgen05 forward (sla_forward_tcgen05): same oracle, same tolerance --------------------------
TCGEN05_LAYOUTS = dict(EDGE_LAYOUTS, mixed_pack_wrap=[2, 6, 3, 15, 8, 53, 88, 53, 76, 107, 121, 144, 144] * 40,
                       dense_144=[144] * 400, tiny_3=[3] * 3000)


@pytest.mark.parametrize("c", [1, 3, 4])
def test_forward_tcgen05_configs(c):
    torch = _torch()
    sc = wl.make_config(c)
    q, k, v = sc.tensor("q"), sc.tensor("k"), sc.tensor("v")
    off = torch.from_numpy(sc.offsets).cuda()
    out = pkg.sla_forward(to_dev(q, sc.dtype), to_dev(k, sc.dtype), to_dev(v, sc.dtype), off, tcgen05=True)
    torch.cuda.synchronize()
    check(f"{sc.name}.tcgen05", out, sla_oracle.forward(q, k, v, sc.offsets, nthreads=8), sc.dtype, sc.lengths)


@pytest.mark.parametrize("layout", sorted(TCGEN05_LAYOUTS))
@pytest.mark.parametrize("H", [8, 16])
def test_forward_tcgen05_edge_layouts(layout, H):
    torch = _torch()
    sc = wl.make_scene(TCGEN05_LAYOUTS[layout], H, 16, "f16", seed=177 + len(layout), name=layout)
    q, k, v = sc.tensor("q"), sc.tensor("k"), sc.tensor("v")
    off = torch.from_numpy(sc.offsets).cuda()
    out = pkg.sla_forward(to_dev(q, "f16"), to_dev(k, "f16"), to_dev(v, "f16"), off, tcgen05=True)
    torch.cuda.synchronize()
    check(f"{layout}.tcgen05", out, sla_oracle.forward(q, k, v, sc.offsets, nthreads=8), "f16", sc.lengths)


def test_forward_tcgen05_unsupported_shapes():
    torch = _torch()
    off = torch.tensor([0, 4], dtype=torch.int32, device="cuda")
    for shape, dt in (((4, 4, 16), torch.float16), ((4, 8, 32), torch.float16), ((4, 8, 16), torch.bfloat16)):
        q = torch.zeros(*shape, dtype=dt, device="cuda")
        with pytest.raises(pkg.SlaError, match="UNSUPPORTED"):
            pkg.sla_forward(q, q, q, off, tcgen05=True)


# ---- ReLU feature map with eps (sla_forward_phi / sla_backward_phi) ------------------
RELU_EPS = 1e-6


UNIT = {"f32": 2.0 ** -24, "f16": 2.0 ** -11, "bf16": 2.0 ** -8}


def _relu_grad_amplification(q, k, v, g, offsets, eps):
    """Forward-error scale of the ReLU map's gradients.  With max(x,0) the denominator a.z + eps can be arbitrarily
    small, and dq = (dnum S^T + dden z) phi'(q) is then a difference of two large terms (for a length-1 window they
    cancel to O(eps)): any arithmetic with unit roundoff u has an error of order u times the sum of the ABSOLUTE
    values of the terms.  This returns that sum per element for dq, dk, dv (numpy, from the definition)."""
    a, b = np.maximum(q, 0.0), np.maximum(k, 0.0)
    amp_q, amp_k, amp_v = np.zeros_like(q), np.zeros_like(q), np.zeros_like(q)
    for w in range(len(offsets) - 1):
        s, e = int(offsets[w]), int(offsets[w + 1])
        if e == s:
            continue
        S = np.einsum("jhp,jhr->hpr", b[s:e], np.abs(v[s:e]))        # |S| (b >= 0)
        z = b[s:e].sum(0)                                             # [H,d]
        Sv = np.einsum("jhp,jhr->hpr", b[s:e], v[s:e])
        den = np.einsum("ihp,hp->ih", a[s:e], z) + eps                # [m,H]
        o = np.einsum("ihp,hpr->ihr", a[s:e], Sv) / den[..., None]
        dnum = np.abs(g[s:e]) / den[..., None]                        # |dnum|
        dden = np.abs((g[s:e] * o).sum(-1)) / den                     # |dden|
        amp_q[s:e] = np.einsum("ihr,hpr->ihp", dnum, S) + dden[..., None] * z[None]
        dS = np.einsum("ihp,ihr->hpr", a[s:e], dnum)                  # |dS|
        dz = np.einsum("ih,ihp->hp", dden, a[s:e])                    # |dz|
        amp_k[s:e] = np.einsum("jhr,hpr->jhp", np.abs(v[s:e]), dS) + dz[None]
        amp_v[s:e] = np.einsum("jhp,hpr->jhr", b[s:e], dS)
    return amp_q, amp_k, amp_v


def _relu_case(sc, backward=True):
    torch = _torch()
    q, k, v, g = sc.tensor("q"), sc.tensor("k"), sc.tensor("v"), sc.tensor("do")
    off = torch.from_numpy(sc.offsets).cuda()
    tq, tk, tv, tg = (to_dev(a, sc.dtype) for a in (q, k, v, g))
    out = pkg.sla_forward(tq, tk, tv, off, phi="relu", eps=RELU_EPS)
    torch.cuda.synchronize()
    ref = sla_oracle.forward(q, k, v, sc.offsets, nthreads=8, phi="relu", eps=RELU_EPS)
    check(f"{sc.name}.relu.out", out, ref, sc.dtype, sc.lengths)
    if backward:
        grads = pkg.sla_backward(tq, tk, tv, off, tg, phi="relu", eps=RELU_EPS)
        torch.cuda.synchronize()
        gref = sla_oracle.backward(q, k, v, g, sc.offsets, nthreads=8, phi="relu", eps=RELU_EPS)
        amps = _relu_grad_amplification(*(x.astype(np.float64) for x in (q, k, v, g)), sc.offsets, RELU_EPS)
        rtol, atol = TOL[sc.dtype]
        for name, got, want, amp in zip(("dq", "dk", "dv"), grads, gref, amps):
            gotd = got.double().cpu().numpy()
            assert np.isfinite(gotd).all(), f"{sc.name}.relu.{name}: non-finite"
            # the north-star tolerance plus the conditioning of the element itself (see _relu_grad_amplification)
            err = np.abs(gotd - want) / (atol + rtol * np.abs(want) + 16 * UNIT[sc.dtype] * amp)
            worst = np.unravel_index(np.argmax(err), err.shape)
            assert err.max() <= 1.0, f"{sc.name}.relu.{name}: worst err/tol {err.max():.3f} at {worst} got {gotd[worst]} want {want[worst]} amp {amp[worst]}"


@pytest.mark.parametrize("c", [0, 1, 3])
def test_relu_forward_configs(c):
    _relu_case(wl.make_config(c), backward=False)


@pytest.mark.parametrize("c", [4, 2, 3])
def test_relu_backward_configs(c):
    """The ReLU map's backward at full size: config 4 (d_h = 16) and config 2 (d_h = 32) on the tensor-core kernels,
    config 3 (tiny windows packed into quadratic tiles + four windows of 27 500 rows through the split passes)."""
    _relu_case(wl.make_config(c))


@pytest.mark.parametrize("layout", sorted(EDGE_LAYOUTS))
@pytest.mark.parametrize("dtype,H,d", [("f32", 4, 32), ("f16", 8, 16), ("bf16", 8, 32), ("f16", 3, 16)])
def test_relu_edge_layouts_forward_backward(layout, dtype, H, d):
    _relu_case(wl.make_scene(EDGE_LAYOUTS[layout], H, d, dtype, seed=277 + len(layout), name=layout))


def test_relu_zero_denominator_rows_and_errors():
    """A query whose every channel is negative has phi(q) = 0: the output row is 0/(0+eps) = 0, finite."""
    torch = _torch()
    sc = wl.make_scene([1, 5, 40], 8, 16, "f16", seed=9)
    q, k, v = sc.tensor("q").copy(), sc.tensor("k"), sc.tensor("v")
    q[3] = -np.abs(q[3]) - 0.5
    q[20] = -np.abs(q[20]) - 0.5
    off = torch.from_numpy(sc.offsets).cuda()
    out = pkg.sla_forward(to_dev(q, "f16"), to_dev(k, "f16"), to_dev(v, "f16"), off, phi="relu", eps=RELU_EPS)
    assert torch.all(out[3] == 0) and torch.all(out[20] == 0) and torch.isfinite(out).all()
    check("relu.zero_den", out, sla_oracle.forward(q, k, v, sc.offsets, phi="relu", eps=RELU_EPS), "f16", sc.lengths)
    t = to_dev(q, "f16")
    with pytest.raises(pkg.SlaError, match="INVALID_ARG"):
        pkg.sla_forward(t, t, t, off, phi="relu", eps=-1.0)


def test_n0_w0_and_errors():
    torch = _torch()
    q = torch.empty(0, 8, 16, dtype=torch.float16, device="cuda")
    off = torch.zeros(1, dtype=torch.int32, device="cuda")
    assert pkg.sla_forward(q, q, q, off).shape == (0, 8, 16)
    off3 = torch.zeros(4, dtype=torch.int32, device="cuda")
    assert pkg.sla_forward(q, q, q, off3).shape == (0, 8, 16)
    q2 = torch.zeros(4, 8, 16, dtype=torch.float16, device="cuda")
    off2 = torch.tensor([0, 4], dtype=torch.int32, device="cuda")
    small = torch.empty(16, dtype=torch.uint8, device="cuda")
    with pytest.raises(pkg.SlaError, match="WORKSPACE"):
        pkg.sla_forward(q2, q2, q2, off2, workspace=small)
    q3 = torch.zeros(4, 8, 24, dtype=torch.float16, device="cuda")
    with pytest.raises(pkg.SlaError, match="UNSUPPORTED"):
        pkg.sla_forward(q3, q3, q3, off2)


def test_closed_forms_on_gpu():
    """Pins that need no oracle: length-1 windows return v (Eq. 3 with m=1); equal values returned."""
    torch = _torch()
    sc = wl.make_scene([1] * 50 + [7, 90], 8, 16, "f16", seed=3)
    q, k, v = (to_dev(sc.tensor(n), "f16") for n in ("q", "k", "v"))
    off = torch.from_numpy(sc.offsets).cuda()
    out = pkg.sla_forward(q, k, v, off)
    assert torch.allclose(out[:50].float(), v[:50].float(), rtol=2e-3, atol=1e-3)
    v2 = v.clone()
    v2[50:57] = v[50]
    out2 = pkg.sla_forward(q, k, v2, off)
    assert torch.allclose(out2[50:57].float(), v2[50:57].float(), rtol=2e-3, atol=1e-3)


def test_host_entry_matches_device_entry():
    torch = _torch()
    sc = wl.make_config(0)
    q, k, v = (torch.from_numpy(sc.tensor(n)).pin_memory() for n in ("q", "k", "v"))
    ids = torch.from_numpy(sc.window_ids).pin_memory()
    out_h = pkg.sla_forward_host(q, k, v, ids, sc.W)
    off = torch.from_numpy(sc.offsets).cuda()
    out_d = pkg.sla_forward(q.cuda(), k.cuda(), v.cuda(), off)
    assert torch.equal(out_h, out_d.cpu())


def test_host_entry_repeated_calls_reuse_the_pool():
    """sla_forward_host takes its staging block from a library-owned memory pool that keeps the block between calls:
    calls of different sizes, interleaved and repeated, must each match the oracle and the device entry (a stale or
    too-small reused block would show here).  Scenes of >= 16 384 rows are cut at window boundaries into chunks that
    travel and compute in a pipeline; a window's tile-mates then differ from the one-call layout, so the comparison with
    the device entry allows the last bits of the fp16 result (the oracle check is the parity statement)."""
    torch = _torch()
    scenes = [wl.make_config(0), wl.make_config(1), wl.make_config(0), wl.make_config(1)]
    for sc in scenes:
        tdt = torch.float16 if sc.dtype == "f16" else torch.float32
        q, k, v = (torch.from_numpy(sc.tensor(n)).to(tdt).pin_memory() for n in ("q", "k", "v"))
        ids = torch.from_numpy(sc.window_ids).pin_memory()
        out_h = pkg.sla_forward_host(q, k, v, ids, sc.W)
        off = torch.from_numpy(sc.offsets).cuda()
        out_d = pkg.sla_forward(q.cuda(), k.cuda(), v.cuda(), off)
        if sc.N < 16384:
            assert torch.equal(out_h, out_d.cpu()), sc.name
        else:
            assert torch.allclose(out_h.float(), out_d.cpu().float(), rtol=4e-3, atol=2e-4), sc.name
        ref = sla_oracle.forward(sc.tensor("q"), sc.tensor("k"), sc.tensor("v"), sc.offsets, nthreads=8)
        check(f"{sc.name}.host_entry", out_h, ref, sc.dtype, sc.lengths)


def test_host_entry_chunk_boundaries_and_bad_ids():
    """Chunk cuts fall on window boundaries even when a long window straddles the nominal cut, and ids that are not
    sorted window indices are refused at the cuts."""
    torch = _torch()
    sc = wl.make_scene([9000, 3, 1, 12000, 40, 7000, 1, 1, 2, 5000], 8, 16, "f16", seed=31)
    q, k, v = (torch.from_numpy(sc.tensor(n)).to(torch.float16).pin_memory() for n in ("q", "k", "v"))
    ids = torch.from_numpy(sc.window_ids).pin_memory()
    out_h = pkg.sla_forward_host(q, k, v, ids, sc.W)
    check("host_entry.straddle", out_h, sla_oracle.forward(sc.tensor("q"), sc.tensor("k"), sc.tensor("v"), sc.offsets, nthreads=8),
          "f16", sc.lengths)
    bad = ids.clone()
    bad[:] = sc.W + 5
    with pytest.raises(pkg.SlaError, match="INVALID_ARG"):
        pkg.sla_forward_host(q, k, v, bad.pin_memory(), sc.W)


@pytest.mark.parametrize("c", [1, 4])
def test_forward_bounded_entry_matches_general_and_oracle(c):
    """sla_forward_bounded (one launch, no workspace; windows <= 144 rows by construction of the
    12x12-window configs) must give exactly what sla_forward gives, and match the oracle."""
    torch = _torch()
    sc = wl.make_config(c)
    assert int(sc.lengths.max()) <= 144
    q, k, v = sc.tensor("q"), sc.tensor("k"), sc.tensor("v")
    off = torch.from_numpy(sc.offsets).cuda()
    tq, tk, tv = (to_dev(a, sc.dtype) for a in (q, k, v))
    out_b = pkg.sla_forward(tq, tk, tv, off, max_window_len=144)
    out_g = pkg.sla_forward(tq, tk, tv, off)
    torch.cuda.synchronize()
    assert torch.equal(out_b, out_g)
    ref = sla_oracle.forward(q, k, v, sc.offsets, nthreads=8)
    check(f"{sc.name}.bounded", out_b, ref, sc.dtype, sc.lengths)


def test_forward_bounded_generic_path_and_errors():
    torch = _torch()
    sc = wl.make_scene([5, 1, 144, 33, 2, 100, 16, 17], 4, 32, "f32", seed=12)
    q, k, v = sc.tensor("q"), sc.tensor("k"), sc.tensor("v")
    off = torch.from_numpy(sc.offsets).cuda()
    out = pkg.sla_forward(*(to_dev(a, "f32") for a in (q, k, v)), off, max_window_len=144)
    check("bounded_f32.out", out, sla_oracle.forward(q, k, v, sc.offsets), "f32", sc.lengths)
    with pytest.raises(pkg.SlaError, match="UNSUPPORTED"):
        pkg.sla_forward(*(to_dev(a, "f32") for a in (q, k, v)), off, max_window_len=1000)


@pytest.mark.parametrize("c", [1, 4])
def test_backward_bounded_entry_matches_general_and_oracle(c):
    """sla_backward_bounded (one launch, no workspace) must give exactly what sla_backward gives, and pass the
    gradient criterion against the oracle."""
    torch = _torch()
    sc = wl.make_config(c)
    assert int(sc.lengths.max()) <= 144
    q, k, v, g = (sc.tensor(n) for n in ("q", "k", "v", "do"))
    off = torch.from_numpy(sc.offsets).cuda()
    tq, tk, tv, tg = (to_dev(a, sc.dtype) for a in (q, k, v, g))
    gb = pkg.sla_backward(tq, tk, tv, off, tg, max_window_len=144)
    gg = pkg.sla_backward(tq, tk, tv, off, tg)
    torch.cuda.synchronize()
    for a, b in zip(gb, gg):
        assert torch.equal(a, b)
    check_grads(gb, sla_oracle.backward(q, k, v, g, sc.offsets, nthreads=8), sc)


@pytest.mark.parametrize("dtype,d", [("f32", 32), ("bf16", 32), ("f32", 16)])     # bf16, d_h = 32: sla_bwd_tc32.cu
def test_backward_bounded_generic_path_and_errors(dtype, d):
    torch = _torch()
    sc = wl.make_scene([5, 1, 144, 33, 2, 100, 16, 17, 256], 4, d, dtype, seed=13)
    q, k, v, g = (sc.tensor(n) for n in ("q", "k", "v", "do"))
    off = torch.from_numpy(sc.offsets).cuda()
    dev = [to_dev(a, dtype) for a in (q, k, v)]
    grads = pkg.sla_backward(*dev, off, to_dev(g, dtype), max_window_len=256)
    torch.cuda.synchronize()
    check_grads(grads, sla_oracle.backward(q, k, v, g, sc.offsets), sc)
    with pytest.raises(pkg.SlaError, match="UNSUPPORTED"):
        pkg.sla_backward(*dev, off, to_dev(g, dtype), max_window_len=257)
    with pytest.raises(pkg.SlaError):
        pkg.sla_backward(*dev, off, to_dev(g, dtype), max_window_len=16, phi="relu", eps=1e-6)


@pytest.mark.parametrize("dtype,H,d", [("f16", 8, 16), ("bf16", 8, 32), ("f16", 2, 32)])
def test_backward_writes_nothing_beyond_n(dtype, H, d):
    """Guard rows behind dq, dk, dv keep their sentinel (ragged last tiles, split windows, partial slabs)."""
    torch = _torch()
    sc = wl.make_scene([13, 300, 1, 29, 257, 7], H, d, dtype, seed=91)
    q, k, v, g = (to_dev(sc.tensor(n), dtype) for n in ("q", "k", "v", "do"))
    off = torch.from_numpy(sc.offsets).cuda()
    pad = 64
    bufs = [torch.full((sc.N + pad, H, d), 3.0, dtype=q.dtype, device="cuda") for _ in range(3)]
    pkg.sla_backward(q, k, v, off, g, dq=bufs[0][:sc.N], dk=bufs[1][:sc.N], dv=bufs[2][:sc.N])
    torch.cuda.synchronize()
    for b in bufs:
        assert bool((b[sc.N:] == 3.0).all())
    ref = sla_oracle.backward(sc.tensor("q"), sc.tensor("k"), sc.tensor("v"), sc.tensor("do"), sc.offsets)
    check_grads([b[:sc.N] for b in bufs], ref, sc)


def _span_table_restated(off, N, span, nspans):
    """The work list of include/sla.h (sla_build_span_table), restated on the host: per span the window of its first
    row and the rows it streams under the middle-row ownership rule (windows of more than 256 rows are cut at the span)."""
    off = np.asarray(off, dtype=np.int64)
    t = np.zeros((nspans, 4), dtype=np.int32)
    win_of = lambda r: int(np.searchsorted(off, r, side="right") - 1)       # skips zero-length windows
    for i in range(nspans):
        r0, r1 = i * span, min((i + 1) * span, N)
        w0, wl = win_of(r0), win_of(r1 - 1)
        s, e = int(off[w0]), int(off[w0 + 1])
        begin = (s if s + (e - s) // 2 >= r0 else e) if e - s <= 256 else r0
        s, e = int(off[wl]), int(off[wl + 1])
        end = (e if s + (e - s) // 2 < r1 else s) if e - s <= 256 else r1
        t[i] = (w0, begin, end, 0)
    return t


@pytest.mark.parametrize("case", ["config1", "config3", "config2", "gaps_and_long", "one_window", "len1"])
def test_span_table_bit_exact(case):
    """SURVEY 8(a) a1 (work list): integer work, bit for bit against the host restatement above."""
    torch = _torch()
    if case.startswith("config"):
        sc = wl.make_config(int(case[-1]))
    elif case == "gaps_and_long":
        sc = wl.make_scene([0, 0, 5, 300, 0, 1, 256, 257, 0, 17, 1000, 2, 0], 8, 16, "f16", seed=71)
    elif case == "one_window":
        sc = wl.make_scene([777], 8, 16, "f16", seed=72)
    else:
        sc = wl.make_scene([1] * 5000, 8, 16, "f16", seed=73)
    off = torch.from_numpy(sc.offsets).cuda()
    raw = pkg.sla_build_span_table(off, sc.N, sc.H, sc.d_h)
    torch.cuda.synchronize()
    tab = raw.cpu().numpy().view(np.int32).reshape(-1, 4)
    magic, span, nspans, n = (int(x) for x in tab[0])
    assert n == sc.N and span % 16 == 0 and nspans == (sc.N + span - 1) // span
    assert tab.shape[0] >= nspans + 1
    want = _span_table_restated(sc.offsets, sc.N, span, nspans)
    got = tab[1:nspans + 1]
    bad = np.nonzero((got != want).any(axis=1))[0]
    assert bad.size == 0, f"span {bad[0]}: got {got[bad[0]]} want {want[bad[0]]} (span {span} rows)"


@pytest.mark.parametrize("case", ["config1", "config4", "tiny", "mixed_d32", "bf16_partial_slab", "small_n"])
def test_forward_planned_matches_bounded_bit_for_bit(case):
    """sla_forward_planned: the span table (built once per scene) replaces the in-kernel window search and must not
    change a bit of the result; a table of another scene's size is detected on the device and ignored."""
    torch = _torch()
    if case == "config1":
        sc = wl.make_config(1)
    elif case == "config4":
        sc = wl.make_config(4)
    elif case == "tiny":
        sc = wl.make_scene([1, 0, 2, 1, 3, 0, 0, 1, 5, 2] * 300, 8, 16, "f16", seed=61)
    elif case == "mixed_d32":
        sc = wl.make_scene([256, 1, 17, 0, 144, 33, 2, 255, 64, 63, 65] * 20, 8, 32, "f16", seed=62)
    elif case == "bf16_partial_slab":
        sc = wl.make_scene([100, 7, 256, 1, 1, 31], 12, 16, "bf16", seed=63)
    else:
        sc = wl.make_scene([5, 3], 8, 16, "f16", seed=64)
    q, k, v = (to_dev(sc.tensor(n), sc.dtype) for n in ("q", "k", "v"))
    off = torch.from_numpy(sc.offsets).cuda()
    table = pkg.sla_build_span_table(off, sc.N, sc.H, sc.d_h)
    out_p = pkg.sla_forward_planned(q, k, v, off, table, 256)
    out_b = pkg.sla_forward(q, k, v, off, max_window_len=256)
    torch.cuda.synchronize()
    assert torch.equal(out_p, out_b)
    ref = sla_oracle.forward(sc.tensor("q"), sc.tensor("k"), sc.tensor("v"), sc.offsets, nthreads=8)
    check(f"{sc.name}.planned", out_p, ref, sc.dtype, sc.lengths)
    # a table of another problem size: ignored, same result
    other = wl.make_scene([50, 60, 70], sc.H, sc.d_h, sc.dtype, seed=65)
    t2 = pkg.sla_build_span_table(torch.from_numpy(other.offsets).cuda(), other.N, other.H, other.d_h)
    big = torch.zeros(max(table.numel(), t2.numel()), dtype=torch.uint8, device="cuda")
    big[:t2.numel()] = t2
    out_w = pkg.sla_forward_planned(q, k, v, off, big, 256)
    torch.cuda.synchronize()
    assert torch.equal(out_w, out_b)
    with pytest.raises(pkg.SlaError, match="WORKSPACE"):
        pkg.sla_forward_planned(q, k, v, off, torch.zeros(16, dtype=torch.uint8, device="cuda")[:0].contiguous() if False else torch.zeros(0, dtype=torch.uint8, device="cuda"), 256)


def test_forward_under_cuda_graph_replay():
    """The C-ABI calls are capturable: a graph of prep + forward replays to the same result."""
    torch = _torch()
    sc = wl.make_config(1)
    q, k, v = (to_dev(sc.tensor(n), sc.dtype) for n in ("q", "k", "v"))
    ids = torch.from_numpy(sc.window_ids).cuda()
    off = torch.empty(sc.W + 1, dtype=torch.int32, device="cuda")
    out = torch.empty_like(q)
    ws = torch.empty(pkg.workspace_bytes(sc.N, sc.W, sc.H, sc.d_h, pkg.SLA_F16), dtype=torch.uint8, device="cuda")
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        pkg.sla_offsets_from_window_ids(ids, sc.W, out=off, stream=s)
        pkg.sla_forward(q, k, v, off, out=out, workspace=ws, stream=s)
        torch.cuda.synchronize()
        want = out.clone()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s):
            pkg.sla_offsets_from_window_ids(ids, sc.W, out=off, stream=s)
            pkg.sla_forward(q, k, v, off, out=out, workspace=ws, stream=s)
        out.zero_()
        g.replay()
        torch.cuda.synchronize()
    assert torch.equal(out, want)


def test_second_device_after_first():
    """Per-device state (shared-memory opt-ins, SM count, the static workspace's address, tensor maps): the same calls
    on cuda:1 after cuda:0 must give the same results.  Skipped on a one-GPU box."""
    torch = _torch()
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs")
    sc = wl.make_scene([300, 5, 1, 1000, 17, 64], 8, 16, "f16", seed=55)
    ref = sla_oracle.forward(sc.tensor("q"), sc.tensor("k"), sc.tensor("v"), sc.offsets)
    outs = []
    for dev in ("cuda:0", "cuda:1", "cuda:0"):
        with torch.cuda.device(dev):
            q, k, v = (to_dev(sc.tensor(n), "f16").to(dev) for n in ("q", "k", "v"))
            off = torch.from_numpy(sc.offsets).to(dev)
            o1 = pkg.sla_forward(q, k, v, off)
            o2 = pkg.sla_forward_static(q, k, v, off)
            g = pkg.sla_backward(q, k, v, off, to_dev(sc.tensor("do"), "f16").to(dev))
            torch.cuda.synchronize()
            check(f"{dev}.out", o1, ref, "f16", sc.lengths)
            check(f"{dev}.static", o2, ref, "f16", sc.lengths)
            outs.append((o1.cpu(), g[0].cpu()))
    assert torch.equal(outs[0][0][:5], outs[2][0][:5])
