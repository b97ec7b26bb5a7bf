"""CPU-only checks of the C-ABI boundary: the library builds, loads without a GPU, exports every symbol
include/retro.h declares, and its host-side validation answers without touching a device."""
import ctypes as C
import os
import re

import pytest

from paper_2508_09001_b200 import binding as rb

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    txt = open(os.path.join(ROOT, "include", "retro.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(retro_[a-z_0-9]+)\s*\(", txt)))


def test_header_symbols_are_exported():
    lib = C.CDLL(rb.library_path())
    names = declared_symbols()
    assert set(names) == set(rb.EXPORTED), (names, rb.EXPORTED)
    for n in names:
        assert hasattr(lib, n), f"libretro.so does not export {n}"


def test_host_side_validation_without_gpu():
    good = rb.make_desc(1, 32, 8, 128, 16, 2304, 64, 2304, 8, "bf16")
    n = rb.retro_workspace_bytes(good)
    assert n > 8 * 2304 * 8 and n % 256 == 0
    assert rb.retro_version() >= 100
    assert "workspace" in rb.retro_error_string(rb.RETRO_ERR_WORKSPACE)
    for bad, code in [
        (rb.make_desc(1, 30, 8, 128, 16, 64, 8, 64, 2, "bf16"), rb.RETRO_ERR_ARG),          # h_q % h_k
        (rb.make_desc(1, 32, 8, 64, 16, 64, 8, 64, 2, "bf16"), rb.RETRO_ERR_UNSUPPORTED),   # bf16 d64
        (rb.make_desc(1, 32, 8, 128, 32, 64, 8, 64, 2, "bf16"), rb.RETRO_ERR_UNSUPPORTED),  # page 32
        (rb.make_desc(1, 32, 8, 128, 16, 64, 8, 64, 40, "bf16"), rb.RETRO_ERR_UNSUPPORTED), # window > 32
        (rb.make_desc(0, 32, 8, 128, 16, 64, 8, 64, 2, "bf16"), rb.RETRO_ERR_ARG),
        (rb.make_desc(1, 32, 8, 128, 16, 64, 0, 64, 2, "bf16"), rb.RETRO_ERR_ARG),
    ]:
        with pytest.raises(rb.RetroError) as e:
            rb.retro_workspace_bytes(bad)
        assert e.value.code == code
    # null pointers are rejected before any launch
    lib = C.CDLL(rb.library_path())
    rc = lib.retro_update_page_bounds(C.byref(good), None, None, None, None, 1, None, None)
    assert rc == rb.RETRO_ERR_ARG
    rc = lib.retro_merge_output_cache(C.byref(good), None, None, None, None, None, None, None, None, None, None)
    assert rc == rb.RETRO_ERR_ARG
    rc = lib.retro_step_diagnostics(C.byref(good), None, None, None, None, None, None, None, None, None, None)
    assert rc == rb.RETRO_ERR_ARG


def test_workspace_grows_with_window_and_batch():
    a = rb.retro_workspace_bytes(rb.make_desc(8, 32, 8, 128, 16, 2064, 256, 8 * 2064, 0, "bf16"))
    b = rb.retro_workspace_bytes(rb.make_desc(8, 32, 8, 128, 16, 2064, 256, 8 * 2064, 32, "bf16"))
    assert b > a
