"""CPU-side checks of the boundary: libpdp.so builds, loads and exports every symbol declared in
include/pdp.h; error paths that need no GPU behave as documented."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1903_06838_b200 import build, binding
    build.build()
    return binding.load_library()


def test_exports_match_header(lib):
    from paper_1903_06838_b200 import binding
    hdr = open(os.path.join(ROOT, "include", "pdp.h")).read()
    declared = set(re.findall(r"\b(pdp_[a-z_]+)\s*\(", hdr))
    assert declared == set(binding.EXPORTS), declared ^ set(binding.EXPORTS)
    for name in declared:
        assert hasattr(lib, name), name


def test_version_and_strerror(lib):
    assert lib.pdp_version() == 100
    assert lib.pdp_strerror(0) == b"ok"
    assert b"aligned" in lib.pdp_strerror(-5)
    assert lib.pdp_destroy(None) == 0


def test_create_argument_errors(lib):
    from paper_1903_06838_b200 import binding
    h = ctypes.c_void_p()
    prm = binding.pdp_params(50.0, 20.0, 100.0, 0, 0)
    assert lib.pdp_create(None, None, None, ctypes.byref(prm), ctypes.byref(h)) == -1
    buf = (ctypes.c_float * 16)(*([1.0] * 16))
    bad = binding.pdp_geometry(1, 2, 8, 3, 4)          # seg_cols does not divide cols
    assert lib.pdp_create(ctypes.byref(bad), buf, buf, ctypes.byref(prm), ctypes.byref(h)) == -2
    geo = binding.pdp_geometry(1, 2, 8, 4, 4)
    badp = binding.pdp_params(50.0, 20.0, 0.0, 0, 0)   # photon_adu must be > 0
    assert lib.pdp_create(ctypes.byref(geo), buf, buf, ctypes.byref(badp), ctypes.byref(h)) == -3
    assert h.value is None


def test_no_gpu_fails_loudly(lib):
    """Without an sm_100 device there is no fallback: pdp_create must fail."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_1903_06838_b200 import binding
    with pytest.raises(binding.PdpError):
        binding.Context(panels=1, rows=2, cols=8, seg_cols=4, max_frames_per_batch=1,
                        pedestal=[0.0] * 16, gain=[1.0] * 16, seed_adu=50, cm_adu=20, photon_adu=100)


def test_product_does_not_import_oracle():
    for dirpath, _, files in os.walk(os.path.join(ROOT, "paper_1903_06838_b200")):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, fn)).read()
                assert "oracle" not in src.replace("oracle/ ", "").replace("oracle/)", "") or fn in ("synth.py",) or \
                    "import oracle" not in src and "from oracle" not in src and "pdp_oracle" not in src, fn
