"""CPU-only checks of the C-ABI boundary: the library loads without a GPU, exports every
symbol include/sn.h declares, and its host-side argument validation returns the documented
error codes before touching the device (no compute calls are made here)."""
import ctypes
import os
import re

import numpy as np
import pytest

from paper_1909_08354_b200 import build, sn

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return sn.lib()


def test_exports_match_header(lib):
    hdr = open(os.path.join(ROOT, "include", "sn.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(sn_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(sn.EXPORTS)
    for name in declared:
        assert hasattr(lib, name), name


def test_workspace_bytes(lib):
    assert sn.workspace_bytes((64, 64)) > 64 * 64 * 8
    w = sn.workspace_bytes((512, 512, 512))
    cells = 512 ** 3
    # default: psi (8 B) + half spectrum (~4 B) + FFT tables -- the stepper alone
    assert cells * 12 < w < cells * 12.1
    assert w % 256 == 0
    # + staging scratch (4 B) + external potential (4 B) + beta, gamma tables of eq. (12) (8 B)
    assert cells * 28 < sn.workspace_bytes((512, 512, 512), features=sn.FEAT_ALL) < cells * 28.2
    assert sn.workspace_bytes((512, 512, 512), features=sn.FEAT_VEXT) - w == cells * 4
    assert sn.workspace_bytes((64, 64), features=8) == 0          # unknown feature bit
    # ensembles whose line counts overflow a 32-bit int are rejected, not wrapped
    assert sn.workspace_bytes((4096, 4096), batch=1 << 20) == 0
    assert sn.workspace_bytes((64, 64), batch=1 << 20) > 0
    for bad in [(64,), (64, 64, 64, 64), (48, 64), (16, 64), (8192, 64), (64, 100), (0, 64), (160, 64), (6144, 64), (288, 64)]:
        assert sn.workspace_bytes(bad) == 0


def _create(lib, dims=(64, 64), L=(10.0, 10.0), A=-0.5, B=1.0, C=0.0, D=1.0, g=(0.1,), dtau=1e-3,
            ws=0x1000, ws_bytes=None, out=True):
    h = ctypes.c_void_p()
    nd = len(dims)
    c_dims = (ctypes.c_int64 * nd)(*dims)
    c_L = (ctypes.c_double * nd)(*L)
    c_g = (ctypes.c_double * max(1, len(g)))(*(g or (0.0,)))
    nbytes = sn.workspace_bytes(dims) if ws_bytes is None else ws_bytes
    rc = lib.sn_create(ctypes.byref(h) if out else None, nd, c_dims, c_L, A, B, C, D, c_g, len(g), dtau,
                       ctypes.c_void_p(ws), nbytes, None)
    return rc, h


def test_create_validation_codes(lib):
    # every case fails in host-side validation, before any CUDA call (fake workspace pointer)
    assert _create(lib, out=False)[0] == -1                       # SN_ERR_NULL
    assert _create(lib, ws=0)[0] == -1
    assert _create(lib, dims=(64, 48))[0] == -2                   # SN_ERR_DIMS
    assert _create(lib, dims=(64,), L=(10.0,))[0] == -2
    assert _create(lib, A=float("nan"))[0] == -3                  # SN_ERR_PARAM
    assert _create(lib, L=(10.0, -1.0))[0] == -3
    assert _create(lib, g=(0.1,) * 5)[0] == -3
    assert _create(lib, dtau=float("inf"))[0] == -3
    assert _create(lib, ws_bytes=1024)[0] == -5                   # SN_ERR_WORKSPACE
    assert _create(lib, ws=0x1010)[0] == -5                       # not 256-byte aligned
    # reading Q5: C > 0 equal to k^2 of a grid mode -> singular; L = 2 pi makes k integer
    L = (2 * np.pi, 2 * np.pi)
    assert _create(lib, L=L, C=25.0)[0] == -4                     # 3^2 + 4^2
    assert _create(lib, L=L, C=2.0)[0] == -4                      # 1^2 + 1^2
    rc, h = _create(lib, out=True, ws=0)
    assert rc == -1 and not h.value                               # *out untouched on error


def test_null_context_calls(lib):
    assert lib.sn_step(None, 1) == -1
    assert lib.sn_set_state(None, None, 0) == -1
    assert lib.sn_get_state(None, None, 0) == -1
    assert lib.sn_diagnostics(None, None) == -1
    assert lib.sn_set_dtau(None, 0.1) == -1
    assert lib.sn_destroy(None) == -1
    assert lib.sn_debug_fft(None, 1) == -1
    assert lib.sn_launch_count(None) == 0
    assert lib.sn_step_order4(None, 1) == -1
    assert lib.sn_set_local_terms(None, 0.0, 0.0, 1.0, 1e-6) == -1
    assert lib.sn_set_external_potential(None, None, 0) == -1
    assert lib.sn_set_source_tables(None, None, None, 0) == -1
    assert lib.sn_set_bohm(None, 0.0, 1e-6) == -1
    assert lib.sn_profile(None, 1) == -1
    assert lib.sn_debug_potential(None, None, 0) == -1
    assert lib.sn_set_option(None, 1, 0) == -1
    assert lib.sn_create_opt(None, 2, None, None, 0.0, 0.0, 0.0, 0.0, None, 0, 0.0, None, 0, None, None) == -1
    assert lib.sn_strerror(-9).decode().startswith("the call needs")
    assert lib.sn_strerror(-4).decode().startswith("C > 0")
    assert lib.sn_strerror(0).decode() == "ok"


def test_library_reads_no_environment_variables():
    """every switch is an argument (sn_options, sn_set_option), none an environment variable."""
    for f in os.listdir(os.path.join(ROOT, "paper_1909_08354_b200", "csrc")):
        assert "getenv" not in open(os.path.join(ROOT, "paper_1909_08354_b200", "csrc", f)).read(), f


def test_no_cpu_fallback():
    """The product path must fail loudly without a GPU (this container has none)."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError):
        sn.Simulation((64, 64), 10.0, -0.5, 1.0, 0.0, 1.0, (), 1e-3)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1909_08354_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in text.replace("oracle/", "").replace("the oracle", "").replace(
                    "float64 oracle", ""), f
