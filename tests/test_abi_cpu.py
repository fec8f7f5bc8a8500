"""CPU-side checks of the boundary: libtwk.so loads without a GPU and exports every symbol include/twk.h declares;
host-only entry points behave; compute entry points refuse to run without CUDA (no CPU fallback)."""
import os
import re

import pytest

import paper_2501_03322_b200 as P

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "twk.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(twk_[a-z0-9_]+)\s*\(", src)))


def test_header_symbols_exported():
    decl = declared_symbols()
    assert "twk_magnify" in decl and "twk_images_fixed" in decl and len(decl) >= 10
    L = P.lib()
    missing = [s for s in decl if not hasattr(L, s)]
    assert not missing, missing
    assert sorted(P.exported_symbols()) == decl


def test_workspace_bytes_is_host_arithmetic():
    a = P.twk_workspace_bytes(1000)
    b = P.twk_workspace_bytes(4096000)
    assert 0 < a < b < 1 << 34
    # the hand-over arena (14,720 B per slot, default min(max_sources, 2^19) slots) is the bulk of a large context; with it
    # come the 1024 carry-over slots between the refinement stages (512 samples x (26 + 3) doubles + ids + header)
    lean = P.twk_workspace_bytes(4096000, handoff_slots=0)
    carry_slot = (512 * 29 + 512 // 4 + 8) * 8
    assert lean < 1 << 31 and b - lean == (1 << 19) * 14720 + 1024 * carry_slot
    assert P.twk_workspace_bytes(1000, handoff_slots=-2) == 0        # invalid
    assert P.twk_workspace_bytes(1000, max_samples=512) < a          # no stage-3 arena
    assert P.twk_workspace_bytes(1000, max_samples=5000) == 0        # invalid options
    assert "sm_100a" in P.twk_version() and "src:" in P.twk_version()


def test_strerror():
    L = P.lib()
    assert L.twk_strerror(0) == b"ok"
    assert b"invalid" in L.twk_strerror(-1)


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(P.TwkError):
        P.Context(16)


def test_product_does_not_import_oracle():
    """The product path must not reach into oracle/ (and the oracle not into the product)."""
    pkg = os.path.join(ROOT, "paper_2501_03322_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                for needle in ("import oracle", "from oracle", "libtwk_oracle", "twk_oracle", "oracle/api", "oracle."):
                    assert needle not in txt, (f, needle)
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2501_03322_b200" not in txt and "csrc" not in txt
