"""GPU parity for the shared Q/K/V projection and the module (include/sla.h): the tcgen05 GEMM against
oracle/sla_proj_oracle.py on the same seeded inputs.

Tolerance (reading A17): fp32 accumulation of K = C products in any order, one rounding to the I/O dtype:
  |got - ref| <= acc + u (|ref| + acc) + 2^-24,   acc = (C + 1) 2^-24 sum_k |x_k w_k|  (oracle.accumulation_bound),
u = 2^-11 (fp16) / 2^-8 (bf16); 2^-24 covers fp16 subnormal spacing.  Selector weights must come out bit for bit."""
import numpy as np
import pytest

import paper_2401_00912_b200 as pkg
from paper_2401_00912_b200 import workloads as wl
from oracle import sla_oracle
from oracle import sla_proj_oracle as P

pytestmark = pytest.mark.gpu

UNIT = {"f32": 2.0 ** -24, "f16": 2.0 ** -11, "bf16": 2.0 ** -8}
TOL = {"f16": (2e-2, 1e-3), "bf16": (2e-2, 1e-3)}      # the SLA tolerance, for the module test


def _torch():
    import torch
    return torch


def _tdt(dtype):
    torch = _torch()
    return {"f32": torch.float32, "f16": torch.float16, "bf16": torch.bfloat16}[dtype]


def _inputs(N, C, dtype, seed, bias):
    rng = np.random.Generator(np.random.PCG64(seed))
    x = wl.round_to_dtype(rng.standard_normal((N, C)).astype(np.float32), dtype)
    w = wl.round_to_dtype((rng.standard_normal((3 * C, C)) / np.sqrt(C)).astype(np.float32), dtype)
    b = rng.standard_normal(3 * C).astype(np.float32) if bias else None
    return x, w, b


def _dev(a, dtype=None):
    torch = _torch()
    t = torch.from_numpy(np.ascontiguousarray(a)).cuda()
    return t.to(_tdt(dtype)) if dtype else t


def _check_proj(got, x, w, b, dtype):
    ref = np.concatenate(P.project_qkv(x, w, b), axis=1)
    acc, _ = P.accumulation_bound(x, w, b)
    allowed = acc + UNIT[dtype] * (np.abs(ref) + acc) + 2.0 ** -24
    g = np.concatenate([t.double().cpu().numpy() for t in got], axis=1)
    assert np.isfinite(g).all()
    ratio = np.abs(g - ref) / allowed
    worst = np.unravel_index(np.argmax(ratio), ratio.shape)
    assert ratio.max() <= 1.0, f"worst err/bound {ratio.max():.3f} at {worst}: got {g[worst]} want {ref[worst]}"
    return float(ratio.max())


@pytest.mark.parametrize("bias", [False, True])
@pytest.mark.parametrize("dtype", ["f16", "bf16"])
@pytest.mark.parametrize("C", [128, 256])
@pytest.mark.parametrize("N", [1, 127, 128, 129, 1000, 20011])
def test_projection_against_oracle(N, C, dtype, bias):
    torch = _torch()
    x, w, b = _inputs(N, C, dtype, 1000 + N + C, bias)
    got = pkg.sla_qkv_projection(_dev(x, dtype), _dev(w, dtype), _dev(b) if bias else None)
    torch.cuda.synchronize()
    _check_proj(got, x, w, b, dtype)


@pytest.mark.parametrize("C,dtype", [(128, "f16"), (256, "bf16")])
def test_projection_selector_weights_bit_exact(C, dtype):
    """Output feature j copies input column sel[j]: every product is exact, so the result is x's columns bit for bit;
    a transposed operand, a wrong k-step offset or a wrong q/k/v block cannot pass."""
    torch = _torch()
    rng = np.random.Generator(np.random.PCG64(7))
    N = 777
    x = wl.round_to_dtype(rng.standard_normal((N, C)).astype(np.float32), dtype)
    sel = rng.integers(0, C, 3 * C)
    w = np.zeros((3 * C, C), np.float32)
    w[np.arange(3 * C), sel] = 1.0
    q, k, v = pkg.sla_qkv_projection(_dev(x, dtype), _dev(w, dtype))
    torch.cuda.synchronize()
    y = np.concatenate([t.float().cpu().numpy() for t in (q, k, v)], axis=1)
    assert np.array_equal(y, x[:, sel])


def test_projection_full_size_configs():
    """The bench's sizes: config 1 (N = 60 000, C = 128, fp16) and config 2 (N = 200 000, C = 256, bf16), every element."""
    torch = _torch()
    for N, C, dtype in ((60000, 128, "f16"), (200000, 256, "bf16")):
        x, w, b = _inputs(N, C, dtype, 5 + C, True)
        xd, wd, bd = _dev(x, dtype), _dev(w, dtype), _dev(b)
        got = pkg.sla_qkv_projection(xd, wd, bd)
        again = pkg.sla_qkv_projection(xd, wd, bd)
        torch.cuda.synchronize()
        _check_proj(got, x, w, b, dtype)
        for a, c in zip(got, again):
            assert torch.equal(a, c)                      # deterministic: no atomics, fixed accumulation order


@pytest.mark.parametrize("N", [1, 129, 300])
def test_projection_writes_nothing_beyond_n(N):
    """The last tile is clipped by the TMA unit: rows N.. of larger output buffers keep their sentinel."""
    torch = _torch()
    x, w, _ = _inputs(N, 128, "f16", 40 + N, False)
    pad = 200
    bufs = [torch.full((N + pad, 128), 7.0, dtype=torch.float16, device="cuda") for _ in range(3)]
    pkg.sla_qkv_projection(_dev(x, "f16"), _dev(w, "f16"), q=bufs[0][:N], k=bufs[1][:N], v=bufs[2][:N])
    torch.cuda.synchronize()
    for b in bufs:
        assert bool((b[N:] == 7.0).all())
    _check_proj([b[:N] for b in bufs], x, w, None, "f16")


@pytest.mark.parametrize("N,C,dtype,bias", [(1000, 128, "f16", True), (333, 256, "bf16", False), (60000, 128, "f16", False)])
def test_linear_against_oracle(N, C, dtype, bias):
    """sla_linear (one [C, C] layer, e.g. the output projection) = the first block of the projection oracle."""
    torch = _torch()
    rng = np.random.Generator(np.random.PCG64(N + C))
    x = wl.round_to_dtype(rng.standard_normal((N, C)).astype(np.float32), dtype)
    w = wl.round_to_dtype((rng.standard_normal((C, C)) / np.sqrt(C)).astype(np.float32), dtype)
    b = rng.standard_normal(C).astype(np.float32) if bias else None
    got = pkg.sla_linear(_dev(x, dtype), _dev(w, dtype), _dev(b) if bias else None)
    torch.cuda.synchronize()
    w3 = np.concatenate([w, np.zeros((2 * C, C), np.float32)], axis=0)
    b3 = np.concatenate([b, np.zeros(2 * C, np.float32)]) if bias else None
    ref = P.project_qkv(x, w3, b3)[0]
    acc = P.accumulation_bound(x, w3, b3)[0][:, :C]
    allowed = acc + UNIT[dtype] * (np.abs(ref) + acc) + 2.0 ** -24
    g = got.double().cpu().numpy()
    assert np.isfinite(g).all() and (np.abs(g - ref) / allowed).max() <= 1.0


@pytest.mark.parametrize("N,C,dtype,bias", [(2000, 128, "f32", True), (777, 64, "f16", False), (130, 48, "bf16", True),
                                            (65, 20, "f32", False), (1, 512, "f16", True)])
def test_projection_generic_path(N, C, dtype, bias):
    """fp32 I/O (config 0's dtype) and the C the tensor-core kernel does not take: the plain tiled kernel."""
    torch = _torch()
    x, w, b = _inputs(N, C, dtype, 2000 + N + C, bias)
    got = pkg.sla_qkv_projection(_dev(x, dtype), _dev(w, dtype), _dev(b) if bias else None)
    torch.cuda.synchronize()
    _check_proj(got, x, w, b, dtype)
    y = pkg.sla_linear(_dev(x, dtype), _dev(w[:C], dtype), _dev(b[:C]) if bias else None)
    torch.cuda.synchronize()
    assert torch.equal(y, got[0])                         # the same sums in the same order


def test_module_forward_fp32_config0():
    """The module on the fp32 configuration (generic projection + generic SLA kernels), SLA tolerance of fp32."""
    torch = _torch()
    sc = wl.make_config(0)
    C = sc.H * sc.d_h
    x, w, _ = _inputs(sc.N, C, "f32", 311, False)
    out, q, k, v = pkg.sla_module_forward(_dev(x), _dev(w), torch.from_numpy(sc.offsets).cuda(), sc.H)
    torch.cuda.synchronize()
    _check_proj([t.reshape(sc.N, C) for t in (q, k, v)], x, w, None, "f32")
    # the oracle chain on the GPU's q, k, v would break the rule that no oracle input comes from the CUDA path; fp32
    # roundings of q, k, v (2^-24) are far below the SLA tolerance, so the chained oracles are compared directly
    qr, kr, vr = (t.astype(np.float32).reshape(sc.N, sc.H, sc.d_h) for t in P.project_qkv(x, w))
    ref = sla_oracle.forward(qr, kr, vr, sc.offsets)
    g = out.double().cpu().numpy()
    assert np.isfinite(g).all() and (np.abs(g - ref) / (1e-5 + 1e-4 * np.abs(ref))).max() <= 1.0


def test_projection_errors_and_empty():
    torch = _torch()
    with pytest.raises(pkg.SlaError):
        pkg.sla_qkv_projection(torch.zeros(10, 128, dtype=torch.float16, device="cuda"),
                               torch.zeros(128, 384, dtype=torch.float16, device="cuda"))
    e = torch.empty(0, 128, dtype=torch.float16, device="cuda")
    q, k, v = pkg.sla_qkv_projection(e, torch.zeros(384, 128, dtype=torch.float16, device="cuda"))
    assert q.numel() == 0


@pytest.mark.parametrize("c", [1, 2])
def test_module_forward_against_oracle_chain(c):
    """x -> projection -> SLA, in one C call.  (a) q, k, v within the projection bound; (b) `out` bit for bit what
    sla_forward gives on the separately projected q, k, v (same kernels, the chain adds no arithmetic); (c) `out` against
    the two oracles chained: Q, K, V of the projection oracle rounded to the I/O dtype, then the SLA oracle.  In (c) the
    GPU's q, k, v may differ from the oracle's by one rounding of the I/O dtype wherever the fp32 sum lands within the
    accumulation error of a rounding boundary, so the absolute floor of the SLA tolerance becomes one unit roundoff of
    the I/O dtype at the outputs' scale (bf16: 2^-8; fp16's 2^-11 is already below the SLA atol of 1e-3)."""
    torch = _torch()
    sc = wl.make_config(c)
    C = sc.H * sc.d_h
    x, w, _ = _inputs(sc.N, C, sc.dtype, 300 + c, False)
    xd, wd, off = _dev(x, sc.dtype), _dev(w, sc.dtype), torch.from_numpy(sc.offsets).cuda()
    out, q, k, v = pkg.sla_module_forward(xd, wd, off, sc.H)
    q2, k2, v2 = pkg.sla_qkv_projection(xd, wd)
    out2 = pkg.sla_forward(*(t.view(sc.N, sc.H, sc.d_h) for t in (q2, k2, v2)), off)
    torch.cuda.synchronize()
    _check_proj([t.reshape(sc.N, C) for t in (q, k, v)], x, w, None, sc.dtype)
    assert torch.equal(q.reshape(sc.N, C), q2) and torch.equal(k.reshape(sc.N, C), k2) and torch.equal(v.reshape(sc.N, C), v2)
    if int(sc.lengths.max()) <= 256:
        assert torch.equal(out, out2)        # split windows accumulate with atomics: order-dependent in the last bit
    qr, kr, vr = (wl.round_to_dtype(t.astype(np.float32), sc.dtype).reshape(sc.N, sc.H, sc.d_h)
                  for t in P.project_qkv(x, w))
    ref = sla_oracle.forward(qr, kr, vr, sc.offsets, nthreads=8)
    rtol, atol = TOL[sc.dtype]
    atol = max(atol, UNIT[sc.dtype])
    g = out.double().cpu().numpy()
    err = np.abs(g - ref) / (atol + rtol * np.abs(ref))
    assert np.isfinite(g).all() and err.max() <= 1.0, err.max()
    err2 = np.abs(out2.double().cpu().numpy() - ref) / (atol + rtol * np.abs(ref))
    assert err2.max() <= 1.0, err2.max()
