"""CPU-side checks of the boundary: the C-ABI library builds for sm_100a, loads, and exports every
symbol include/sla.h declares; argument validation that needs no GPU.  No compute calls."""
import os
import re

import pytest

import paper_2401_00912_b200 as pkg
from paper_2401_00912_b200 import build as sla_build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    sla_build.build()
    return pkg.load_library()


def test_header_symbols_match_binding_and_library(lib):
    hdr = open(os.path.join(ROOT, "include", "sla.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(sla_[a-z_0-9]+)\s*\(", hdr))
    assert declared == set(pkg.SYMBOLS)
    for s in declared:
        assert getattr(lib, s) is not None


def test_status_strings_and_version(lib):
    assert lib.sla_status_string(0) == b"SLA_OK"
    assert lib.sla_status_string(3) == b"SLA_ERR_WORKSPACE"
    assert b"sm_100a" in lib.sla_version()


def test_workspace_bytes(lib):
    # one fp32 [H,d+1,d] slot per possible split window (> 256 rows): N//257 + 1 slots
    one = 16 + (60000 // 257 + 1) * 8 * 17 * 16 * 4        # 16-byte header + slots
    assert lib.sla_workspace_bytes(60000, 1340, 8, 16, pkg.SLA_F16, 0) == one
    assert lib.sla_workspace_bytes(60000, 1340, 8, 16, pkg.SLA_F16, 1) == 2 * one
    assert lib.sla_workspace_bytes(100, 4, 8, 24, pkg.SLA_F16, 0) == 0      # unsupported d_h
    assert lib.sla_workspace_bytes(-1, 4, 8, 16, pkg.SLA_F16, 0) == 0


def test_argument_validation_without_gpu(lib):
    # all of these return before any CUDA call
    assert lib.sla_forward(None, None, None, None, 10, 2, 8, 16, pkg.SLA_F16, None, None, 0, None) == 1
    assert lib.sla_forward(None, None, None, None, 0, 0, 8, 16, pkg.SLA_F16, None, None, 0, None) == 0
    assert lib.sla_forward(None, None, None, None, 10, 2, 8, 20, pkg.SLA_F16, None, None, 0, None) == 2
    assert lib.sla_forward(None, None, None, None, 10, 2, 8, 16, 7, None, None, 0, None) == 2
    assert lib.sla_forward(None, None, None, None, 2**31, 2, 8, 16, 1, None, None, 0, None) == 1
    assert lib.sla_forward(16, 16, 16, 16, 10, 2, 8, 16, pkg.SLA_F16, 16, None, 0, None) == 3
    assert lib.sla_forward(8, 16, 16, 16, 10, 2, 8, 16, pkg.SLA_F16, 16, 16, 1 << 20, None) == 2
    assert lib.sla_backward(None, None, None, None, 10, 2, 8, 16, 1, None, None, None, None, None, 0, None) == 1
    assert lib.sla_offsets_from_window_ids(None, 10, 2, None, None) == 1


def test_binding_refuses_cpu_tensors():
    import torch
    q = torch.zeros(4, 1, 16)
    off = torch.tensor([0, 4], dtype=torch.int32)
    with pytest.raises(pkg.SlaError):
        pkg.sla_forward(q, q, q, off)


def test_product_never_imports_oracle():
    """The product path must not route through the oracle (no import, load or link of oracle/)."""
    for dirpath, _, files in os.walk(os.path.join(ROOT, "paper_2401_00912_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle", src, flags=re.M), f
                assert "sla_oracle" not in src and "libsla_oracle" not in src, f
