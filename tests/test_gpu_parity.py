"""-m gpu: CUDA path vs the fp64 oracle, element by element, through the C ABI (teacher-forced lock-step).

Shapes are the five BASELINE.json configs: C1 exactly; C2..C5 both shrunk to sizes the oracle finishes in
seconds (several tiles, ragged tails, page roll-over) and at FULL context for a few sampled steps."""
import numpy as np
import pytest
import torch

from oracle import retro_oracle as orc
from paper_2508_09001_b200 import binding as rb
from paper_2508_09001_b200 import workload as wl
from tests import gpu_harness as GH
from tests import helpers as H

pytestmark = pytest.mark.gpu


def test_library_is_loaded_from_tree():
    H.require_cuda()
    assert rb.library_path().endswith("paper_2508_09001_b200/lib/libretro.so")
    assert torch.cuda.get_device_capability()[0] >= 10, "needs sm_100"


def test_c1_tiny_fp32_full_lockstep():
    inp = wl.make_layer_inputs(wl.c1())
    e = GH.lockstep(inp, 16)
    assert e["out"] < 1e-4 and e["part_o"] < 1e-4
    print("c1 errs", e)


def test_c1_whole_step_entry_point():
    """retro_decode_step (S1..S4 back to back) gives the same trajectory without teacher forcing."""
    inp = wl.make_layer_inputs(wl.c1())
    GH.lockstep(inp, 16, use_decode_step=True)


@pytest.mark.parametrize("prompt", [2003, 2048])      # ragged tail / exactly page aligned
def test_c2_shape_shrunk(prompt):
    cfg = wl.shrink(wl.c2(), (prompt,), 40)
    inp = wl.make_layer_inputs(cfg)
    print("c2s errs", GH.lockstep(inp, 40))


def test_c3_shape_shrunk_ragged_batch():
    cfg = wl.shrink(wl.c3(), tuple(700 - 61 * b for b in range(4)), 36, batch=4, budget_tokens=256)
    inp = wl.make_layer_inputs(cfg)
    print("c3s errs", GH.lockstep(inp, 36))


def test_c4_shape_shrunk_gqa7():
    cfg = wl.shrink(wl.c4(), (3001, 2990), 20, batch=2, budget_tokens=512)
    inp = wl.make_layer_inputs(cfg)
    print("c4s errs", GH.lockstep(inp, 20))


@pytest.mark.parametrize("use_step", [False, True])
def test_c2_shape_correlated_queries_high_page_overlap(use_step):
    """Correlated mode: most selected pages repeat from step to step, so most (past row, page)
    pairs are masked (the regime the paper reports on real activations)."""
    cfg = wl.shrink(wl.c2(), (2003,), 30, corr_rho=0.95)
    inp = wl.make_layer_inputs(cfg)
    print("c2 correlated errs", GH.lockstep(inp, 30, use_decode_step=use_step))


@pytest.mark.parametrize("w,budget", [(0, 512), (1, 1024), (32, 512)])
def test_c5_shape_shrunk_sweep_points(w, budget):
    cfg = wl.shrink(wl.c5(w, budget), (1500, 1490), w + 6, batch=2)
    inp = wl.make_layer_inputs(cfg)
    print("c5s errs", w, budget, GH.lockstep(inp, w + 6))


@pytest.mark.parametrize("name,kw", [
    ("c2", dict(prompt_lens=(1003,), n_steps=14)),                                   # 8 splits per unit
    ("c5w8", dict(prompt_lens=(1500, 1490, 1333), n_steps=14, batch=3)),             # 8 KV heads x 3 sequences
    ("c5w0", dict(prompt_lens=(1500, 1490), n_steps=5, batch=2, window=0)),          # plain Quest, no cache
    ("c5w32", dict(prompt_lens=(1500, 1490), n_steps=38, batch=2, window=32, budget_tokens=512)),   # 2 row groups
    ("c4", dict(prompt_lens=(3001, 2990), n_steps=12, batch=2, budget_tokens=512)),  # GQA 7
    ("c5b20", dict(prompt_lens=tuple(600 - 7 * i for i in range(20)), n_steps=11, batch=20)),   # 160 units: one split
])
def test_whole_step_entry_point_bf16(name, kw):
    """retro_decode_step (the call bench.py captures into its graph) against the oracle: selections bit-exact,
    out / out_lse / cache within tolerance, every step, no teacher forcing."""
    base = {"c2": wl.c2(), "c5w8": wl.c5(8, 1024), "c5w0": wl.c5(0, 1024), "c5w32": wl.c5(32, 512), "c4": wl.c4(), "c5b20": wl.c5(8, 512)}[name]
    kw = dict(kw)
    cfg = wl.shrink(base, kw.pop("prompt_lens"), kw.pop("n_steps"), **kw)
    inp = wl.make_layer_inputs(cfg)
    print("whole-step errs", name, GH.lockstep(inp, cfg.n_steps, use_decode_step=True))


def test_multi_block_splits_shrunk():
    """32 units x 128 pages: every attend CTA walks several 128-key blocks (ring reuse, lazy rescale, P buffers)."""
    cfg = wl.shrink(wl.c5(8, 2048), (2500, 2491, 2333, 2100), 12, batch=4)
    inp = wl.make_layer_inputs(cfg)
    print("multi-block errs", GH.lockstep(inp, 12))


def test_edge_budget_covers_whole_cache_is_dense():
    cfg = wl.shrink(wl.c2(), (300,), 12, budget_tokens=16 * 64, window=4)
    inp = wl.make_layer_inputs(cfg)
    GH.lockstep(inp, 12)


def test_edge_single_page_and_budget_one():
    cfg = wl.shrink(wl.c2(), (5,), 14, budget_tokens=16, window=3)     # grows from 1 page to 2; k = 1
    inp = wl.make_layer_inputs(cfg)
    GH.lockstep(inp, 14)


def test_edge_budget_zero_selects_nothing():
    """budget 0: empty page lists, every partial is (0, -inf), outputs are zeros / -inf (window ramp-up included)."""
    cfg = wl.shrink(wl.c2(), (200,), 5, budget_tokens=16, window=2)
    inp = wl.make_layer_inputs(cfg)
    GH.lockstep(inp, 5, budget_pages=0, k_max=4)
    GH.lockstep(inp, 5, budget_pages=0, k_max=16, use_decode_step=True)     # empty splits through combine + merge


def test_edge_max_group_and_window_three_row_groups():
    """G = 8 with w = 32: 264 query rows per KV head = three row groups of 88 rows in the tensor-core kernel."""
    cfg = wl.shrink(wl.c5(32, 512), (900, 890), 36, batch=2, num_q_heads=16, num_kv_heads=2)
    inp = wl.make_layer_inputs(cfg)
    print("G8 w32 errs", GH.lockstep(inp, 36))


def test_edge_dense_budget_above_the_page_list_cap():
    """80 units (a single split each by the one-wave rule) with 1101 selected pages: the 1024-page cap on a
    split's shared-memory page list forces a second split; budget = whole cache, so the result is dense attention."""
    cfg = wl.shrink(wl.c5(1, 17616), (17600,) * 10, 2, batch=10)
    inp = _to_cpu(wl.make_layer_inputs(cfg, device="cuda"))
    print("dense 1101 pages errs", GH.lockstep(inp, 2, check_scores=False))


def test_edge_maximum_pages_per_sequence():
    """262 140-token context = 16 384 pages, the library's page limit (128 KB of top-k keys in shared memory)."""
    cfg = wl.shrink(wl.c4(), (262138,), 2, batch=1, num_q_heads=4, num_kv_heads=2, window=1)
    assert cfg.max_pages_per_seq == 16384
    inp = _to_cpu(wl.make_layer_inputs(cfg, device="cuda"))
    print("max pages errs", GH.lockstep(inp, 2))


def test_edge_pure_topk_and_group_max():
    cfg = wl.shrink(wl.c2(), (777,), 12, budget_tokens=128, window=4)
    inp = wl.make_layer_inputs(cfg)
    GH.lockstep(inp, 12, desc_kw=dict(force_last_page=0), oracle_kw=dict(force_last_page=False))
    GH.lockstep(inp, 12, desc_kw=dict(group_reduce=rb.RETRO_GROUP_MAX), oracle_kw=dict(group_reduce="max"))


def test_edge_exact_score_ties_resolve_to_lower_index():
    """All keys identical => every page has the same score: top-k must be the k-1 lowest indices + newest page."""
    cfg = wl.shrink(wl.c1(), (200,), 3, budget_tokens=64, window=2)
    inp = wl.make_layer_inputs(cfg)
    inp.k_pages[:] = inp.k_pages[0, 0, 0]
    _, buf = GH.make_device_layer(inp)
    # direct call, no oracle needed for the expectation
    buf.seq_lens.fill_(201)
    buf.rebuild_bounds()
    buf.q_cur.copy_(inp.q_all[0])
    desc = buf.desc
    rb.retro_select_pages(desc, buf.q_cur, buf.bounds, buf.seq_lens, buf.budget_pages, buf.last_loaded,
                          buf.sel_pages, buf.sel_prev, buf.sel_count, None, buf.workspace)
    torch.cuda.synchronize()
    assert buf.sel_pages[0, 0].tolist() == [0, 1, 2, 12]
    GH.lockstep(inp, 3)


@pytest.mark.parametrize("base", ["f32", "bf16"])
def test_select_adversarial_near_ties_are_ranked_exactly(base):
    """Scores crowded around the k-th one: every page has the same keys except one channel that is shifted by a
    page-dependent amount, so the Eq. 1 scores differ by gaps from far below to far above the fp32 error of the
    streamed score (fp32: 1e-7 .. 1e-3 relative; bf16: whole ulps on a channel the query weighs lightly, plus
    exact ties).  The selection must be the fp64 oracle's, index for index: the fp32 pre-selection has to notice
    that it cannot decide and rank the undecided pages in fp64."""
    if base == "f32":
        cfg = wl.shrink(wl.c1(), (3000,), 3, budget_tokens=40 * 16, window=2)
    else:
        cfg = wl.shrink(wl.c2(), (3000,), 3, budget_tokens=40 * 16, window=2)
    inp = wl.make_layer_inputs(cfg)
    g = torch.Generator().manual_seed(77)
    npg = inp.k_pages.shape[0]
    row = inp.k_pages[0, :, 0].clone()                               # [h_k][d]: one key row per KV head
    k = row[None, :, None, :].repeat(npg, 1, cfg.page_size, 1).float()
    if base == "f32":
        shift = 10.0 ** (-7.0 + 4.0 * torch.rand(npg, generator=g)) * torch.randint(0, 3, (npg,), generator=g)
        k[:, :, :, 0] += (k[:, :, :, 0].abs() + 1.0) * shift[:, None, None]
    else:
        ulps = torch.randint(0, 4, (npg,), generator=g).float()      # 0..3 bf16 ulps on channel 0: many exact ties
        k[:, :, :, 0] = (k[:, :, :, 0].abs() + 1.0) * (1.0 + ulps[:, None, None] * 2.0 ** -7)
    inp.k_pages[:] = k.to(inp.k_pages.dtype)
    print("near-tie errs", base, GH.lockstep(inp, 3, exact_select=True))
    GH.lockstep(inp, 3, use_decode_step=True)


@pytest.mark.parametrize("base", ["f32", "bf16"])
def test_unwritten_tail_of_newest_page_may_hold_nan_and_inf(base):
    """Slots of the newest page past the last token are unwritten memory in a real paged cache: K there is NaN, V is
    +-Inf / NaN.  Nothing of it may reach a result (the masked weights are 0, and 0 x NaN must never be formed)."""
    if base == "f32":
        cfg = wl.shrink(wl.c1(), (505,), 3)
    else:
        cfg = wl.shrink(wl.c2(), (1003, 771), 3, batch=2)
    inp = wl.make_layer_inputs(cfg)
    P = cfg.page_size
    for b in range(cfg.batch):
        total = cfg.prompt_lens[b] + cfg.n_steps
        assert total % P != 0
        phys = int(inp.block_table[b, total // P])
        inp.k_pages[phys, :, total % P:] = float("nan")
        inp.v_pages[phys, :, total % P:] = float("inf")
        inp.v_pages[phys, :, total % P:, ::2] = float("nan")
        inp.v_pages[phys, :, total % P + 1:, 1::4] = float("-inf")
    print("nan tail errs", base, GH.lockstep(inp, 3))
    GH.lockstep(inp, 3, use_decode_step=True)


def test_c2_full_context_sampled_steps():
    """FULL C2 context (32768-token prompt), the launch configuration bench.py times; first steps + ramp-up."""
    cfg = wl.c2(n_steps=12)
    inp = wl.make_layer_inputs(cfg, device="cuda")
    inp = _to_cpu(inp)
    print("c2 full errs", GH.lockstep(inp, 12))


def test_c2_full_context_whole_step_entry_point():
    """FULL C2 through retro_decode_step, exactly the call bench.py captures into its graph."""
    cfg = wl.c2(n_steps=11)
    inp = _to_cpu(wl.make_layer_inputs(cfg, device="cuda"))
    print("c2 full whole-step errs", GH.lockstep(inp, 11, use_decode_step=True))


# ---- FULL-size configurations, retro window FULL for >= 2 checked steps (Alg. 1's Q_{i:t}).
# The CUDA path runs the whole batch in bench.py's launch configuration; the oracle computes a sample of the
# sequences (the (sequence, KV head) units are independent), every KV head and every window row of them.
def test_c3_full_batch_window_full():
    cfg = wl.c3(n_steps=19)
    inp = _to_cpu(wl.make_layer_inputs(cfg, device="cuda"))
    print("c3 full errs", GH.lockstep(inp, 19, oracle_batch=(0, 7, 15), check_scores=False))


def test_c4_full_context_window_full():
    cfg = wl.c4(n_steps=11)
    inp = _to_cpu(wl.make_layer_inputs(cfg, device="cuda"))
    print("c4 full errs", GH.lockstep(inp, 11, oracle_batch=(0, 3)))


def test_c5_full_point_w8_budget4096_window_full():
    cfg = wl.c5(8, 4096, n_steps=11)
    inp = _to_cpu(wl.make_layer_inputs(cfg, device="cuda"))
    print("c5 full errs", GH.lockstep(inp, 11, oracle_batch=(0, 5), check_scores=False))


@pytest.mark.parametrize("w,budget", [(16, 4096), (32, 2048), (8, 8192), (2, 512), (4, 1024)])
def test_c5_full_sweep_points_whole_step(w, budget):
    """FULL-size C5 sweep points through retro_decode_step (the call bench.py times), no teacher forcing, w + 2
    steps: the window is full on the last two.  (8, 8192) is the bench line's `bandwidth_point`."""
    cfg = wl.c5(w, budget, n_steps=w + 2)
    inp = _to_cpu(wl.make_layer_inputs(cfg, device="cuda"))
    print("c5 sweep errs", w, budget, GH.lockstep(inp, w + 2, oracle_batch=(0, 5), use_decode_step=True))


@pytest.mark.parametrize("use_step", [False, True])
def test_multi_block_wide_rows_window_full(use_step):
    """C3 shape shrunk: 128 units (one split each), 128 selected pages = 16 key blocks per CTA, 68 rows (NT = 80,
    a single P buffer), every step from the empty window to the full one (few live row chunks early on); the last
    sequence is shorter than the budget (dense, 100 pages, a 4-page last block with the partly written newest page)."""
    cfg = wl.shrink(wl.c3(), tuple(2500 - 61 * b for b in range(16)), 18)
    inp = wl.make_layer_inputs(cfg)
    print("multi-block wide errs", GH.lockstep(inp, 18, oracle_batch=(0, 15), use_decode_step=use_step))


def test_multi_block_wide_rows_gqa7_window_full():
    """G = 7 with w = 11: 84 rows (NT = 96), 40 units, several key blocks per CTA, window full at the end."""
    cfg = wl.shrink(wl.c4(), tuple(2700 - 37 * b for b in range(10)), 14, batch=10, budget_tokens=2048, window=11)
    inp = wl.make_layer_inputs(cfg)
    print("multi-block G7 errs", GH.lockstep(inp, 14, oracle_batch=(0, 6), check_from=6))


def test_c2_full_context_late_steps_from_synced_state():
    """C2 near the END of its trajectory (decode steps 4080-4082 of 4096, 36 848-token context): the oracle alone
    runs the 9 steps before, its mask A and output cache are uploaded, then both sides step from that state."""
    cfg = wl.c2()
    inp = _to_cpu(wl.make_layer_inputs(cfg, device="cuda"))
    print("c2 late errs", GH.lockstep(inp, 3, start_step=4080, warm_steps=9))
    print("c2 late whole-step errs", GH.lockstep(inp, 3, start_step=4080, warm_steps=9, use_decode_step=True))


def test_append_kv_and_window_advance_match_pregenerated_pool():
    """retro_append_kv / retro_window_advance (harness + host path plumbing) move bytes exactly."""
    cfg = wl.shrink(wl.c2(), (100,), 6, window=3, budget_tokens=64)
    inp = wl.make_layer_inputs(cfg)
    desc, buf = GH.make_device_layer(inp)
    ref_k = buf.k_pages.clone()
    ref_v = buf.v_pages.clone()
    k_seq, v_seq = H.seq_tokens(inp, 0, 106)
    # wipe the decode-phase tokens, then re-append them one by one
    for pos in range(100, 106):
        phys = int(inp.block_table[0, pos // 16])
        buf.k_pages[phys, :, pos % 16] = 0
        buf.v_pages[phys, :, pos % 16] = 0
    buf.seq_lens.fill_(100)
    for s in range(6):
        pos = 100 + s
        rb.retro_window_advance(desc, inp.q_all[s].cuda().contiguous(), None, 1, buf.seq_lens, buf.q_win, buf.q_pos,
                                buf.q_cur)
        kn = torch.from_numpy(k_seq[pos]).to(torch.bfloat16).cuda().contiguous()[None]
        vn = torch.from_numpy(v_seq[pos]).to(torch.bfloat16).cuda().contiguous()[None]
        rb.retro_append_kv(desc, kn, vn, buf.block_table, buf.seq_lens, buf.k_pages, buf.v_pages)
        torch.cuda.synchronize()
        assert int(buf.seq_lens[0]) == pos + 1
        q_win, q_pos = wl.make_q_window(inp, s)
        assert torch.equal(buf.q_pos.cpu(), q_pos)
        assert torch.equal(buf.q_win.cpu()[q_pos >= 0], q_win[q_pos >= 0])
        assert torch.equal(buf.q_cur.cpu(), inp.q_all[s])
    assert torch.equal(buf.k_pages, ref_k) and torch.equal(buf.v_pages, ref_v)


def test_update_kv_overwrite_and_digest_refresh_match_oracle():
    """NEXT-1: retro_update_kv + retro_update_page_bounds(pos_begin = t - w) against the oracle, bit-exact."""
    cfg = wl.shrink(wl.c2(), (300, 77), 4, window=8, budget_tokens=128, batch=2)
    inp = wl.make_layer_inputs(cfg)
    desc, buf = GH.make_device_layer(inp)
    L = torch.tensor([303, 80], dtype=torch.int32)
    buf.seq_lens.copy_(L)
    buf.rebuild_bounds()
    layer = H.oracle_layer(inp)
    layer.prefill_bounds(L.numpy())
    g = torch.Generator().manual_seed(11)
    w = cfg.window
    positions = torch.stack([torch.arange(int(l) - 1 - w, int(l) - 1, dtype=torch.int32) for l in L])   # t-w .. t-1
    positions[1, 2] = -1
    k_hat = torch.randn((2, w, cfg.num_kv_heads, cfg.head_dim), generator=g).to(torch.bfloat16)
    v_hat = torch.randn((2, w, cfg.num_kv_heads, cfg.head_dim), generator=g).to(torch.bfloat16)
    rb.retro_update_kv(desc, k_hat.cuda(), v_hat.cuda(), positions.cuda(), buf.block_table, buf.seq_lens,
                       buf.k_pages, buf.v_pages)
    pos_begin = (L - 1 - w).to(torch.int32).cuda()
    rb.retro_update_page_bounds(desc, buf.k_pages, buf.block_table, buf.seq_lens, pos_begin, 2, buf.bounds)
    torch.cuda.synchronize()
    orc.update_kv(layer.desc, layer.k_pages, layer.v_pages, layer.block_table, L.numpy(), positions.numpy(),
                  k_hat.double().numpy(), v_hat.double().numpy())
    orc.update_page_bounds(layer.desc, layer.k_pages, layer.block_table, L.numpy(), (L - 1 - w).numpy(), layer.bounds)
    assert np.array_equal(buf.k_pages.double().cpu().numpy(), layer.k_pages)
    assert np.array_equal(buf.v_pages.double().cpu().numpy(), layer.v_pages)
    for b in range(2):
        n = -(-int(L[b]) // 16)
        assert np.array_equal(buf.bounds[b, :, :n].double().cpu().numpy(), layer.bounds[b, :, :n])


@pytest.mark.parametrize("name", ["c1", "c2"])
def test_drift_trajectory_update_kv_inside_the_step_matches_oracle(name):
    """NEXT-4 drift mode inside a trajectory (Alg. 1 lines 2-8): every step the w past window
    tokens are re-embedded - their K / V rows are overwritten (retro_update_kv), the digests of the touched pages
    refreshed (retro_update_page_bounds from t - w), the window queries replaced by their drifted versions - then
    the whole step runs.  The oracle consumes the same arrays; selections bit-exact, outputs within tolerance."""
    cfg = wl.c1() if name == "c1" else wl.shrink(wl.c2(), (1003, 700), 14, batch=2)
    inp = wl.make_layer_inputs(cfg)
    desc, buf = GH.make_device_layer(inp)
    layer = H.oracle_layer(inp)
    B, w, P = cfg.batch, cfg.window, cfg.page_size
    prompt = np.asarray(cfg.prompt_lens)
    layer.prefill_bounds(prompt)
    buf.seq_lens.copy_(torch.from_numpy(prompt.astype(np.int32)))
    buf.rebuild_bounds()
    atol, rtol = GH.TOL[cfg.dtype]
    n_touch = (w + P - 1) // P + 1
    for s in range(cfg.n_steps):
        seq_lens = inp.seq_lens_at(s).numpy()
        dr = wl.drift_step(inp, s)
        # Alg. 1 line 2 (UpdateKV) + digest refresh of the touched pages, both sides
        buf.seq_lens.copy_(torch.from_numpy(seq_lens))
        rb.retro_update_kv(desc, dr["k_hat"].cuda(), dr["v_hat"].cuda(), dr["positions"].cuda(), buf.block_table,
                           buf.seq_lens, buf.k_pages, buf.v_pages)
        pos_begin = torch.from_numpy(np.maximum(seq_lens - 1 - w, 0).astype(np.int32)).cuda()
        rb.retro_update_page_bounds(desc, buf.k_pages, buf.block_table, buf.seq_lens, pos_begin, n_touch, buf.bounds)
        orc.update_kv(layer.desc, layer.k_pages, layer.v_pages, layer.block_table, seq_lens, dr["positions"].numpy(),
                      dr["k_hat"].double().numpy(), dr["v_hat"].double().numpy())
        orc.update_page_bounds(layer.desc, layer.k_pages, layer.block_table, seq_lens,
                               np.maximum(seq_lens - 1 - w, 0), layer.bounds)
        # the window rows use the re-embedded queries (the current row its own query)
        q_win, q_pos = wl.make_q_window(inp, s)
        for b in range(B):
            for i in range(w):
                pos = int(dr["positions"][b, i])
                if pos >= 0:
                    q_win[b, wl.ring_slot(cfg, pos)] = dr["q_hat"][b, i]
        res = layer.step(H.np64(q_win), q_pos.numpy(), H.np64(inp.q_all[s]), seq_lens,
                         np.full(B, cfg.budget_pages, dtype=np.int32))
        buf.q_win.copy_(q_win); buf.q_pos.copy_(q_pos); buf.q_cur.copy_(inp.q_all[s])
        rb.retro_decode_step(desc, buf.state, buf.q_win, buf.q_pos, buf.q_cur, buf.out, buf.out_lse)
        torch.cuda.synchronize()
        assert np.array_equal(buf.k_pages.double().cpu().numpy(), layer.k_pages), f"step {s} K pool after UpdateKV"
        assert np.array_equal(buf.sel_pages.cpu().numpy(), res["sel_pages"]), f"step {s} sel_pages"
        assert np.array_equal(buf.sel_prev.cpu().numpy(), res["sel_prev"]), f"step {s} sel_prev"
        GH.close(buf.out.float().cpu().numpy(), res["out"], atol, rtol, f"drift step {s} out")
        GH.close(buf.out_lse.cpu().numpy(), res["out_lse"], atol, rtol, f"drift step {s} out_lse")
        assert np.array_equal(buf.cache_pos.cpu().numpy(), layer.cache_pos)


@pytest.mark.parametrize("use_step", [False, True])
def test_bf16_output_cache_matches_oracle_with_the_same_rounding(use_step):
    """NEXT-3: 16-bit output cache + fp32 LSE, the paper's footprint (Eq. 12).  Merges run in fp32
    and the row written back to the cache is rounded to bf16; the oracle rounds at the same place (round-to-nearest-
    even), so outputs and cache contents agree within the usual bf16 tolerance over w = 8 consecutive merges."""
    cfg = wl.shrink(wl.c5(8, 1024), (1500, 1490, 1333), 20, batch=3)
    inp = wl.make_layer_inputs(cfg)
    e = GH.lockstep(inp, 20, use_decode_step=use_step, desc_kw=dict(cache_dtype=rb.RETRO_BF16),
                    oracle_kw=dict(cache_round="bf16"))
    print("bf16 cache errs", e)


def test_budget_policy_and_build_mask_match_oracle():
    """NEXT-2: device-side relative budget and Alg. 2 alone (external selector), bit-exact against the oracle."""
    cfg = wl.shrink(wl.c5(8, 1024), (1500, 40, 1714), 4, batch=3)
    inp = wl.make_layer_inputs(cfg)
    desc, buf = GH.make_device_layer(inp)
    layer = H.oracle_layer(inp)
    L = np.array([1503, 43, 1717], dtype=np.int32)
    buf.seq_lens.copy_(torch.from_numpy(L))
    rb.retro_budget_policy(desc, buf.seq_lens, buf.budget_pages, 150, 256)
    torch.cuda.synchronize()
    assert buf.budget_pages.cpu().tolist() == orc.budget_policy(layer.desc, L).tolist() == [16, 16, 16]
    rb.retro_budget_policy(desc, buf.seq_lens, buf.budget_pages, 500, 64)
    torch.cuda.synchronize()
    assert buf.budget_pages.cpu().tolist() == orc.budget_policy(layer.desc, L, 500, 64).tolist()
    # an "external selector": arbitrary distinct pages per (b, h), two rounds so that A carries state
    g = torch.Generator().manual_seed(5)
    k_max = desc.max_sel_pages
    for rnd in range(2):
        sel = torch.full((3, cfg.num_kv_heads, k_max), -1, dtype=torch.int32)
        cnt = torch.zeros((3, cfg.num_kv_heads), dtype=torch.int32)
        for b in range(3):
            npg = -(-int(L[b]) // 16)
            for h in range(cfg.num_kv_heads):
                c = min(npg, int(torch.randint(1, k_max + 1, (1,), generator=g)))
                sel[b, h, :c] = torch.sort(torch.randperm(npg, generator=g)[:c]).values.int()
                cnt[b, h] = c
        buf.sel_pages.copy_(sel); buf.sel_count.copy_(cnt)
        rb.retro_build_mask(desc, buf.sel_pages, buf.sel_count, buf.seq_lens, buf.last_loaded, buf.sel_prev)
        torch.cuda.synchronize()
        want = orc.build_mask(layer.desc, sel.numpy(), cnt.numpy(), L, layer.last_loaded)
        assert np.array_equal(buf.sel_prev.cpu().numpy(), want)
        assert np.array_equal(buf.last_loaded.cpu().numpy(), layer.last_loaded)
        L = L + 1
        buf.seq_lens.copy_(torch.from_numpy(L))


def test_step_diagnostics_match_oracle():
    """NEXT-4: effective-budget page counts (bit-exact) and supplementary attention mass per window row, from the
    oracle's own step outputs (ragged batch, ramp-up rows with q_pos = -1, a page roll-over inside the run)."""
    cfg = wl.shrink(wl.c5(8, 512), (1500, 40, 1714), 12, batch=3, corr_rho=0.8)
    inp = wl.make_layer_inputs(cfg)
    desc, buf = GH.make_device_layer(inp)
    layer, res = H.run_oracle_trajectory(inp, 12)
    R = cfg.window + 1
    supp_pages = torch.full((3, cfg.num_kv_heads, R), -7, dtype=torch.int32, device="cuda")
    supp_mass = torch.full((3, R, cfg.num_q_heads), -7.0, dtype=torch.float32, device="cuda")
    for m, r in enumerate(res):
        k = r["sel_pages"].shape[2]
        buf.sel_pages[:, :, :k].copy_(torch.from_numpy(r["sel_pages"].astype(np.int32)))
        buf.sel_prev[:, :, :k].copy_(torch.from_numpy(r["sel_prev"].astype(np.int32)))
        buf.sel_count.copy_(torch.from_numpy(r["sel_count"].astype(np.int32)))
        buf.seq_lens.copy_(torch.from_numpy(r["seq_lens"].astype(np.int32)))
        q_pos = torch.from_numpy(r["q_pos"].astype(np.int32)).cuda()
        part_lse = torch.from_numpy(r["part_lse"]).float().cuda()
        out_lse = torch.from_numpy(r["out_lse"]).float().cuda()
        rb.retro_step_diagnostics(desc, buf.sel_pages, buf.sel_prev, buf.sel_count, q_pos, buf.seq_lens, part_lse,
                                  out_lse, supp_pages, supp_mass)
        torch.cuda.synchronize()
        want_pages, want_mass = orc.step_diagnostics(layer.desc, r["sel_pages"], r["sel_prev"], r["sel_count"],
                                                     r["q_pos"], r["seq_lens"], r["part_lse"], r["out_lse"])
        assert np.array_equal(supp_pages.cpu().numpy(), want_pages), m
        np.testing.assert_allclose(supp_mass.cpu().numpy(), want_mass, atol=2e-5, rtol=1e-4)


def test_decode_step_host_end_to_end_matches_oracle():
    """retro_decode_step_host (bench.py's e2e leg): pinned host q / k / v of the new token in, window ring and
    KV append on the device, whole step, `out` back on the host - against the oracle, every step."""
    cfg = wl.shrink(wl.c2(), (1003,), 12)
    inp = wl.make_layer_inputs(cfg)
    desc, buf = GH.make_device_layer(inp)
    layer = H.oracle_layer(inp)
    B, w, P = cfg.batch, cfg.window, cfg.page_size
    prompt = np.asarray(cfg.prompt_lens)
    layer.prefill_bounds(prompt)
    buf.seq_lens.copy_(torch.from_numpy(prompt.astype(np.int32)))
    buf.rebuild_bounds()
    dt = torch.bfloat16
    hq_n, hk_n, D = cfg.num_q_heads, cfg.num_kv_heads, cfg.head_dim
    n_q, n_kv = B * hq_n * D, B * hk_n * D
    dqkv = torch.empty(n_q + 2 * n_kv, dtype=dt, device="cuda")
    io = rb.RetroStepIO(dqkv.data_ptr(), buf.q_win.data_ptr(), buf.q_pos.data_ptr(), buf.out.data_ptr())
    hqkv = torch.empty(n_q + 2 * n_kv, dtype=dt).pin_memory()       # [q_new | k_new | v_new], refilled every step
    hout = torch.empty((B, w + 1, hq_n, D), dtype=dt).pin_memory()
    atol, rtol = GH.TOL[cfg.dtype]
    for s in range(12):
        hqkv[:n_q] = inp.q_all[s].cpu().reshape(-1)
        hk = torch.empty((B, hk_n, D), dtype=dt)
        hv = torch.empty_like(hk)
        for b in range(B):
            pos = cfg.prompt_lens[b] + s
            phys = int(inp.block_table[b, pos // P])
            hk[b], hv[b] = inp.k_pages[phys, :, pos % P].cpu(), inp.v_pages[phys, :, pos % P].cpu()
        hqkv[n_q:n_q + n_kv] = hk.reshape(-1)
        hqkv[n_q + n_kv:] = hv.reshape(-1)
        rb.retro_decode_step_host(desc, buf.state, io, hqkv, hout)
        torch.cuda.synchronize()
        q_win, q_pos = wl.make_q_window(inp, s)
        res = layer.step(H.np64(q_win), q_pos.numpy(), H.np64(inp.q_all[s].cpu()), inp.seq_lens_at(s).cpu().numpy(),
                         np.full(B, cfg.budget_pages, dtype=np.int32))
        assert np.array_equal(buf.sel_pages.cpu().numpy(), res["sel_pages"])
        GH.close(hout.float().numpy(), res["out"], atol, rtol, f"e2e step {s} out")


def test_decode_steps_host_two_layers_one_copy_each_way():
    """retro_decode_steps_host: two layers (two independent device states of the same inputs) stepped with ONE
    host->device and ONE device->host copy per step; both layers' outputs against the oracle, every step."""
    cfg = wl.shrink(wl.c5(8, 512), (700, 655), 11, batch=2)
    inp = wl.make_layer_inputs(cfg)
    layers = [GH.make_device_layer(inp) for _ in range(2)]
    desc = layers[0][0]
    layer = H.oracle_layer(inp)
    B, w, P = cfg.batch, cfg.window, cfg.page_size
    hq_n, hk_n, D = cfg.num_q_heads, cfg.num_kv_heads, cfg.head_dim
    prompt = np.asarray(cfg.prompt_lens)
    layer.prefill_bounds(prompt)
    for _, buf in layers:
        buf.seq_lens.copy_(torch.from_numpy(prompt.astype(np.int32)))
        buf.rebuild_bounds()
    dt = torch.bfloat16
    n_q, n_kv = B * hq_n * D, B * hk_n * D
    tok = n_q + 2 * n_kv
    d_in = torch.empty((2, tok), dtype=dt, device="cuda")
    d_out = torch.empty((2, B, w + 1, hq_n, D), dtype=dt, device="cuda")
    ios = [rb.RetroStepIO(d_in[l].data_ptr(), buf.q_win.data_ptr(), buf.q_pos.data_ptr(), d_out[l].data_ptr())
           for l, (_, buf) in enumerate(layers)]
    h_in = torch.empty((2, tok), dtype=dt).pin_memory()
    h_out = torch.empty((2, B, w + 1, hq_n, D), dtype=dt).pin_memory()
    atol, rtol = GH.TOL[cfg.dtype]
    for s in range(11):
        for l in range(2):
            h_in[l, :n_q] = inp.q_all[s].reshape(-1)
            for b in range(B):
                pos = cfg.prompt_lens[b] + s
                phys = int(inp.block_table[b, pos // P])
                h_in[l, n_q + b * hk_n * D:n_q + (b + 1) * hk_n * D] = inp.k_pages[phys, :, pos % P].reshape(-1)
                h_in[l, n_q + n_kv + b * hk_n * D:n_q + n_kv + (b + 1) * hk_n * D] = inp.v_pages[phys, :, pos % P].reshape(-1)
        rb.retro_decode_steps_host(desc, [buf.state for _, buf in layers], ios, h_in, h_out)
        torch.cuda.synchronize()
        q_win, q_pos = wl.make_q_window(inp, s)
        res = layer.step(H.np64(q_win), q_pos.numpy(), H.np64(inp.q_all[s]), inp.seq_lens_at(s).numpy(),
                         np.full(B, cfg.budget_pages, dtype=np.int32))
        for l in range(2):
            assert np.array_equal(layers[l][1].sel_pages.cpu().numpy(), res["sel_pages"])
            GH.close(h_out[l].float().numpy(), res["out"], atol, rtol, f"layers-host step {s} layer {l} out")


def test_sequence_at_capacity_is_not_advanced():
    """A sequence whose block-table row is full is left alone by the window-advance / append helpers (no write
    past its last page, seq_len unchanged); the other sequences of the batch advance normally."""
    cfg = wl.shrink(wl.c2(), (32, 20), 1, window=3, budget_tokens=32, batch=2)
    inp = wl.make_layer_inputs(cfg)
    desc, buf = GH.make_device_layer(inp)
    cap = desc.max_pages_per_seq * cfg.page_size
    buf.seq_lens.copy_(torch.tensor([cap, 21], dtype=torch.int32))
    k_ref, v_ref = buf.k_pages.clone(), buf.v_pages.clone()
    qpos_ref = buf.q_pos.clone()
    q_new = inp.q_all[0].cuda().contiguous()
    rb.retro_window_advance(desc, q_new, None, 1, buf.seq_lens, buf.q_win, buf.q_pos, buf.q_cur)
    kn = torch.ones((2, cfg.num_kv_heads, cfg.head_dim), dtype=torch.bfloat16, device="cuda")
    rb.retro_append_kv(desc, kn, kn, buf.block_table, buf.seq_lens, buf.k_pages, buf.v_pages)
    torch.cuda.synchronize()
    assert buf.seq_lens.cpu().tolist() == [cap, 22]
    assert torch.equal(buf.q_pos[0], qpos_ref[0])
    # sequence 0: (seq_len - 1) is its last valid slot and append rewrites it in place - nothing else moves
    phys1 = int(inp.block_table[1, 21 // 16])
    k_chk = buf.k_pages.clone(); k_chk[phys1, :, 21 % 16] = k_ref[phys1, :, 21 % 16]
    phys0 = int(inp.block_table[0, (cap - 1) // 16])
    k_chk[phys0, :, (cap - 1) % 16] = k_ref[phys0, :, (cap - 1) % 16]
    assert torch.equal(k_chk, k_ref)


def _to_cpu(inp):
    return wl.LayerInputs(inp.cfg, inp.k_pages.cpu(), inp.v_pages.cpu(), inp.block_table.cpu(), inp.q_all.cpu(),
                          inp.prompt_lens.cpu(), inp.outlier_channels.cpu())
