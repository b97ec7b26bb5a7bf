"""-m gpu: the -DRETRO_DEBUG_CHECKS build (device-side validation of caller-supplied indices): parity
is unchanged on valid inputs and reports no violation; corrupted selector output is counted and neutralised."""
import numpy as np
import pytest
import torch

from paper_2508_09001_b200 import binding as rb
from paper_2508_09001_b200 import build as rbuild
from paper_2508_09001_b200 import workload as wl
from tests import gpu_harness as GH
from tests import helpers as H

pytestmark = pytest.mark.gpu


@pytest.fixture()
def debug_library():
    H.require_cuda()
    rb.use_library(rbuild.build_debug())
    try:
        yield
    finally:
        rb.use_library(None)


def test_release_build_reports_checks_disabled():
    H.require_cuda()
    cfg = wl.shrink(wl.c2(), (300,), 2, window=2, budget_tokens=64)
    desc, buf = GH.make_device_layer(wl.make_layer_inputs(cfg))
    assert rb.retro_debug_status(desc, buf.workspace) == (0, 0, 0)


@pytest.mark.parametrize("name", ["c1", "c2", "c4", "c5w32"])
def test_parity_under_debug_checks_and_no_violation(debug_library, name):
    cfg = {"c1": wl.c1(),
           "c2": wl.shrink(wl.c2(), (1003,), 12),
           "c4": wl.shrink(wl.c4(), (3001, 2990), 12, batch=2, budget_tokens=512),
           "c5w32": wl.shrink(wl.c5(32, 512), (1500, 1490), 36, batch=2)}[name]
    inp = wl.make_layer_inputs(cfg)
    assert rb.library_path().endswith("libretro_dbg.so")
    GH.lockstep(inp, cfg.n_steps)
    GH.lockstep(inp, cfg.n_steps, use_decode_step=True)
    desc, buf = GH.make_device_layer(inp)
    buf.seq_lens.copy_(inp.seq_lens_at(0))
    buf.rebuild_bounds()
    buf.q_cur.copy_(inp.q_all[0])
    q_win, q_pos = wl.make_q_window(inp, 0)
    buf.q_win.copy_(q_win); buf.q_pos.copy_(q_pos)
    rb.retro_decode_step(desc, buf.state, buf.q_win, buf.q_pos, buf.q_cur, buf.out, buf.out_lse)
    assert rb.retro_debug_status(desc, buf.workspace) == (1, 0, 0)


@pytest.mark.parametrize("dtype_cfg", ["f32", "bf16"])
def test_corrupted_selector_output_is_counted_and_neutralised(debug_library, dtype_cfg):
    """An external selector hands over a page index past the sequence's pages and a block-table
    entry past the pool: the debug build counts both, reads nothing out of bounds, and the rows of every other
    unit are what they are without the corruption."""
    cfg = wl.c1() if dtype_cfg == "f32" else wl.shrink(wl.c2(), (1003, 990), 4, batch=2)
    inp = wl.make_layer_inputs(cfg)
    desc, buf = GH.make_device_layer(inp)
    buf.seq_lens.copy_(inp.seq_lens_at(0))
    buf.rebuild_bounds()
    buf.q_cur.copy_(inp.q_all[0])
    q_win, q_pos = wl.make_q_window(inp, 0)
    buf.q_win.copy_(q_win); buf.q_pos.copy_(q_pos)
    rb.retro_select_pages(desc, buf.q_cur, buf.bounds, buf.seq_lens, buf.budget_pages, buf.last_loaded, buf.sel_pages,
                          buf.sel_prev, buf.sel_count, None, buf.workspace)
    rb.retro_sparse_attend(desc, buf.q_win, buf.q_pos, buf.k_pages, buf.v_pages, buf.block_table, buf.seq_lens,
                           buf.sel_pages, buf.sel_prev, buf.sel_count, buf.part_o, buf.part_lse, buf.workspace)
    torch.cuda.synchronize()
    good_o, good_l = buf.part_o.clone(), buf.part_lse.clone()
    assert rb.retro_debug_status(desc, buf.workspace) == (1, 0, 0)
    hk = cfg.num_kv_heads
    buf.sel_pages[0, 0, 1] = 1_000_000                                    # page index far past the sequence
    j = int(buf.sel_pages[0, hk - 1, 0])
    saved = int(buf.block_table[0, j])
    buf.block_table[0, j] = 2_000_000_000                                 # physical page far past the pool
    rb.retro_sparse_attend(desc, buf.q_win, buf.q_pos, buf.k_pages, buf.v_pages, buf.block_table, buf.seq_lens,
                           buf.sel_pages, buf.sel_prev, buf.sel_count, buf.part_o, buf.part_lse, buf.workspace)
    torch.cuda.synchronize()
    en, n, code = rb.retro_debug_status(desc, buf.workspace)
    assert en == 1 and n >= 2 and code in (1, 2)
    buf.block_table[0, j] = saved
    G = cfg.group
    cur = int(np.argmax(q_pos[0].numpy()))
    for h in range(1, hk):                                                # KV heads of sequence 0 that did not select
        if j in buf.sel_pages[0, h].tolist():                             # the page whose block-table entry was hit
            continue
        for hq in range(h * G, (h + 1) * G):
            # (row sums are accumulated with shared-memory float atomics, the split partials pass through fp16:
            # equal up to the order of the additions amplified to an fp16 ulp)
            assert torch.allclose(buf.part_o[0, cur, hq], good_o[0, cur, hq], atol=2e-3, rtol=2e-3)
            assert torch.allclose(buf.part_lse[0, cur, hq], good_l[0, cur, hq], atol=1e-4, rtol=1e-4)
    if cfg.batch > 1:                                                     # the other sequence is untouched
        assert torch.allclose(buf.part_o[1], good_o[1], atol=2e-3, rtol=2e-3)
    assert torch.isfinite(buf.part_o).all()
