"""CPU-side checks: the C-ABI library loads and exports every symbol include/scatman.h declares; with
no CUDA device the product path fails loudly (no fallback)."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2202_03411_b200 import build, binding
    build.build()
    return binding.load_library()


def test_exports_match_header(lib):
    from paper_2202_03411_b200 import binding
    hdr = open(os.path.join(ROOT, "include", "scatman.h")).read()
    declared = set(re.findall(r"\b(scatman_[a-z_]+)\s*\(", hdr))
    assert declared == set(binding.EXPORTS), declared ^ set(binding.EXPORTS)
    for name in declared:
        assert getattr(lib, name) is not None


def test_version_and_status_strings(lib):
    assert lib.scatman_version() >= 100
    assert lib.scatman_status_string(0) == b"ok"
    assert b"workspace" in lib.scatman_status_string(3)
    assert lib.scatman_destroy(None) == 0


def test_struct_layout_matches_header():
    from paper_2202_03411_b200 import binding as B
    assert C.sizeof(B.Grid) == 40 and C.sizeof(B.Detector) == 32 and C.sizeof(B.Options) == 16
    assert C.sizeof(B.Shape) == 136 and B.Shape.quat.offset == 16 and B.Shape.h_coef.offset == 80 and B.Shape.vdx.offset == 128


def test_no_device_fails_loudly(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    ctx = C.c_void_p()
    rc = lib.scatman_create(C.byref(ctx), 0)
    assert rc == 2 and not ctx.value          # SCATMAN_UNSUPPORTED_DEVICE, no context, no fallback
    from paper_2202_03411_b200 import binding as B
    with pytest.raises(B.ScatmanError):
        B.Scatman(0)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2202_03411_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"(import\s+oracle|from\s+oracle|oracle/|libmsft_oracle|msft_oracle)", src), \
                    f"{f} reaches into the oracle"
