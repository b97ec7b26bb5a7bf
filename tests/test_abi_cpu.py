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


def test_launch_plan_is_two_kernels_per_layer_step_where_the_fusion_applies():
    """retro_launches_per_step is host logic (no device needed): the bf16 tensor-core path with one row group fuses
    the split combine and S4 into the attend kernel (select + attend = 2 launches); fp32 (C1) and row blocks above
    128 rows (w = 32 with G = 4) run S4 as a third launch."""
    two = {
        "c2": rb.make_desc(1, 32, 8, 128, 16, 2304, 64, 2304, 8, "bf16"),
        "c3": rb.make_desc(16, 32, 8, 128, 16, 1536, 128, 16 * 1536, 16, "bf16"),
        "c4": rb.make_desc(4, 28, 4, 128, 16, 8208, 256, 4 * 8208, 8, "bf16"),
        "c5_w0": rb.make_desc(8, 32, 8, 128, 16, 2064, 256, 8 * 2064, 0, "bf16"),
        "c2_bf16_cache": rb.make_desc(1, 32, 8, 128, 16, 2304, 64, 2304, 8, "bf16", cache_dtype=rb.RETRO_BF16),
    }
    three = {
        "c1_fp32": rb.make_desc(1, 4, 4, 64, 16, 33, 8, 33, 4, "f32"),
        "c5_w32": rb.make_desc(8, 32, 8, 128, 16, 2064, 256, 8 * 2064, 32, "bf16"),
    }
    for name, d in two.items():
        assert rb.retro_launches_per_step(d) == 2, name
    for name, d in three.items():
        assert rb.retro_launches_per_step(d) == 3, name
    # a 16-bit output cache needs bf16 inputs
    with pytest.raises(rb.RetroError) as e:
        rb.retro_workspace_bytes(rb.make_desc(1, 4, 4, 64, 16, 33, 8, 33, 4, "f32", cache_dtype=rb.RETRO_BF16))
    assert e.value.code in (rb.RETRO_ERR_ARG, rb.RETRO_ERR_UNSUPPORTED)


def test_nvtx_build_exports_the_same_abi_and_answers_on_the_host():
    """-DRETRO_NVTX (NVTX ranges around the entry points): same symbols, header-only NVTX 3 inside
    (nothing linked), and a range opened without a tool attached is a no-op."""
    from paper_2508_09001_b200 import build as rbuild
    path = rbuild.build_nvtx()
    lib = C.CDLL(path)
    for n in declared_symbols():
        assert hasattr(lib, n), f"libretro_nvtx.so does not export {n}"
    blob = open(path, "rb").read()
    assert b"nvtxRangePushA" in blob and b"retro_select_pages" in blob
    assert b"nvtxRangePushA" not in open(rb.library_path(), "rb").read()      # the release build has none of it
    # an entry point that opens a range and returns from host-side validation: the range is pushed and popped
    desc = rb.make_desc(1, 32, 8, 128, 16, 64, 8, 64, 2, "bf16")
    lib.retro_workspace_init.restype = C.c_int
    rc = lib.retro_workspace_init(C.byref(desc), C.c_void_p(0), C.c_size_t(0), C.c_void_p(0))
    assert rc == rb.RETRO_ERR_ARG
