"""sla_forward_static (include/sla.h): the forward with its workspace in the library's static device array, for callers
that cannot allocate.  Collected last on purpose (the file name sorts behind the other test files).

Checked against the existing path (sla_forward with a caller-owned workspace) on the same inputs, within the tolerance
the parity tests use, on two calls in a row: the second call runs on a different scene, so contents the first call
left in the shared array would show.  The scenes hold windows longer than 256 rows, the only ones that use scratch."""
import numpy as np
import pytest

import paper_2401_00912_b200 as pkg
from paper_2401_00912_b200 import workloads as wl

pytestmark = pytest.mark.gpu

TOL = {"f32": (1e-5, 1e-6), "f16": (2e-2, 1e-3), "bf16": (2e-2, 1e-3)}     # as tests/test_gpu_parity.py
STATIC_BYTES = 4 << 20                                                     # SLA_STATIC_WORKSPACE_BYTES


def _torch():
    import torch
    return torch


def _dev(sc):
    torch = _torch()
    tdt = {"f32": torch.float32, "f16": torch.float16, "bf16": torch.bfloat16}[sc.dtype]
    q, k, v = (torch.from_numpy(sc.tensor(n)).cuda().to(tdt) for n in ("q", "k", "v"))
    return q, k, v, torch.from_numpy(sc.offsets).cuda()


def _close(name, got, want, dtype):
    rtol, atol = TOL[dtype]
    g, w = got.double().cpu().numpy(), want.double().cpu().numpy()
    assert np.isfinite(g).all(), f"{name}: non-finite output"
    err = np.abs(g - w) / (atol + rtol * np.abs(w))
    assert err.max() <= 1.0, f"{name}: worst err/tol {err.max():.3f}"


SCENES = {
    # two scenes per case, different lengths and seeds; each has split windows (> 256 rows) and short ones
    "f16_d16": [([300, 5, 1, 1000, 17, 64, 2, 700, 33], 8, 16, "f16", 31),
                ([40, 2000, 3, 257, 16, 900, 1, 1, 120], 8, 16, "f16", 32)],
    "bf16_d32": [([513, 9, 1, 300, 77], 8, 32, "bf16", 33), ([2, 1200, 31, 260], 8, 32, "bf16", 34)],
    "f32_generic": [([300, 5, 1, 600, 17], 4, 32, "f32", 35), ([1, 800, 3, 258], 4, 32, "f32", 36)],
}


@pytest.mark.parametrize("case", sorted(SCENES))
def test_static_matches_existing_path_two_calls_in_a_row(case):
    torch = _torch()
    scenes = [wl.make_scene(ln, H, d, dt, seed=seed) for ln, H, d, dt, seed in SCENES[case]]
    dev = [_dev(sc) for sc in scenes]
    want = [pkg.sla_forward(q, k, v, off) for q, k, v, off in dev]       # existing path, its own workspace
    outs = [torch.empty_like(t[0]) for t in dev]
    torch.cuda.synchronize()
    for (q, k, v, off), out in zip(dev, outs):                           # back to back on one stream, no sync between
        pkg.sla_forward_static(q, k, v, off, out=out)
    torch.cuda.synchronize()
    for sc, got, ref in zip(scenes, outs, want):
        _close(f"{case}.{sc.name}", got, ref, sc.dtype)
    # and once more in the other order: the array now holds the second scene's states
    for (q, k, v, off), out in reversed(list(zip(dev, outs))):
        out.zero_()
        pkg.sla_forward_static(q, k, v, off, out=out)
    torch.cuda.synchronize()
    for sc, got, ref in zip(scenes, outs, want):
        _close(f"{case}.{sc.name}.again", got, ref, sc.dtype)


def test_static_on_the_metric_config():
    """BASELINE.json config 1 (N = 60 000, no split window) and config 4 (N = 120 000, near the limit)."""
    torch = _torch()
    for c in (1, 4):
        sc = wl.make_config(c)
        q, k, v, off = _dev(sc)
        assert pkg.workspace_bytes(sc.N, sc.W, sc.H, sc.d_h, pkg.SLA_F16) <= STATIC_BYTES
        want = pkg.sla_forward(q, k, v, off)
        got = pkg.sla_forward_static(q, k, v, off)
        again = pkg.sla_forward_static(q, k, v, off)
        torch.cuda.synchronize()
        _close(f"config{c}", got, want, sc.dtype)
        _close(f"config{c}.again", again, want, sc.dtype)


def test_static_rejects_what_does_not_fit_and_launches_nothing():
    torch = _torch()
    N, H, d = 140000, 8, 16                                               # needs 4.7 MB of scratch
    assert pkg.workspace_bytes(N, 1, H, d, pkg.SLA_F16) > STATIC_BYTES
    q = torch.zeros(N, H, d, dtype=torch.float16, device="cuda")
    off = torch.tensor([0, N], dtype=torch.int32, device="cuda")
    out = torch.full_like(q, 7.0)
    with pytest.raises(pkg.SlaError, match="SLA_ERR_TOO_LARGE"):
        pkg.sla_forward_static(q, q, q, off, out=out)
    torch.cuda.synchronize()
    assert bool((out == 7.0).all())
    # the largest N that fits at this shape is accepted
    slot = H * (d + 1) * d * 4
    n_fit = N
    while pkg.workspace_bytes(n_fit, 1, H, d, pkg.SLA_F16) > STATIC_BYTES:
        n_fit -= 257
    assert pkg.workspace_bytes(n_fit, 1, H, d, pkg.SLA_F16) > STATIC_BYTES - slot - 1
    sc = wl.make_scene([n_fit - 300, 300], H, d, "f16", seed=37)
    qd, kd, vd, offd = _dev(sc)
    _close("largest", pkg.sla_forward_static(qd, kd, vd, offd), pkg.sla_forward(qd, kd, vd, offd), "f16")
    # empty problem: nothing to do
    e = torch.empty(0, H, d, dtype=torch.float16, device="cuda")
    assert pkg.sla_forward_static(e, e, e, torch.zeros(1, dtype=torch.int32, device="cuda")).numel() == 0
