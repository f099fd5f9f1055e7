"""CPU-only checks of the boundary: libgint.so builds (nvcc cross-compiles sm_100a without a GPU), loads, exports every
function include/gint.h declares, and fails loudly -- never falls back -- when no CUDA device is present."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "gint.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(gint_[a-z0-9_]+)\s*\(", src)) - {"gint_ctx"})


def test_header_declares_the_north_star_calls():
    names = _declared()
    for must in ("gint_init", "gint_vlocal", "gint_rho", "gint_free", "gint_get_pairs", "gint_last_error"):
        assert must in names


def test_library_exports_every_declared_symbol():
    from paper_2409_09399_b200 import gint as G
    lib = G.lib()
    for name in _declared():
        assert hasattr(lib, name), f"libgint.so does not export {name}"
    assert sorted(G.EXPORTS) == _declared()


def test_no_cpu_fallback_and_argument_errors():
    import torch
    from paper_2409_09399_b200 import gint as G
    from paper_2409_09399_b200 import workloads as W
    lib = G.lib()
    ctx = C.c_void_p()
    # NULL arrays are rejected before anything else
    rc = lib.gint_init(C.byref(ctx), 1, None, None, None, C.c_double(0.01), None, None, None, 0, None, None, None, None, 0, C.c_ulonglong(0))
    assert rc == -1 and b"NULL" in lib.gint_last_error()
    assert lib.gint_free(None) == -5
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present: the no-device error path cannot be exercised")
    w = W.make_workload(0)
    with pytest.raises(G.GintError, match="no CPU fallback|CUDA"):
        G.Gint.from_workload(w)


def test_oracle_is_not_imported_by_the_product():
    for root, _, files in os.walk(os.path.join(ROOT, "paper_2409_09399_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".h")):
                txt = open(os.path.join(root, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", txt, flags=re.M), f
                assert "liboracle" not in txt and "gint_oracle" not in txt, f


def test_batch_flag_packing():
    from paper_2409_09399_b200.gint import batch_flag
    assert batch_flag(8, 4, 2) == 8 | (4 << 8) | (2 << 16)
    assert np.int64(batch_flag(1, 1, 1)) == 0x010101
    # the fields of the flags word do not overlap (include/gint.h): batch edges 0..23, GINT_FLAG_TUNE bit 32, scratch cap bits 40..59
    from paper_2409_09399_b200.gint import FLAG_TUNE, phi_cap_flag
    assert phi_cap_flag(24) == 24 << 40 and phi_cap_flag((1 << 20) - 1) & (FLAG_TUNE | 0xffffff) == 0
    src = open(os.path.join(ROOT, "include", "gint.h")).read()
    assert "#define GINT_FLAG_TUNE (1ull << 32)" in src and "0xfffffull) << 40)" in src
