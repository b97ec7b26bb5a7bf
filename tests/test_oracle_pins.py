"""Pins of the fp64 oracle against things other than itself (CPU only).

Each test names the plausible mistake it would catch.  Sources: the hand-worked golden example
(tests/golden/hand_example.*), closed forms, library routines (torch SDPA, numpy stable sort),
brute force on tiny inputs and the invariants the paper states.
"""
import json
import math
import os
from fractions import Fraction

import numpy as np
from dataclasses import replace as dataclasses_replace
import pytest
import torch

from oracle import retro_oracle as orc
from paper_2508_09001_b200 import workload as wl
from tests import helpers as H

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "hand_example.json")


def _val(x, sym):
    """Parse '3/7', 'ln(5)', '2*b', 'a', 0 ... into a float."""
    if isinstance(x, (int, float)):
        return float(x)
    x = x.strip()
    if x.startswith("ln(") and x.endswith(")"):
        return math.log(float(x[3:-1]))
    if "*" in x:
        l, r = x.split("*", 1)
        return _val(l, sym) * _val(r, sym)
    if x in sym:
        return sym[x]
    return float(Fraction(x))


def _hand_setup():
    g = json.load(open(GOLDEN))
    c = g["config"]
    sym = {}
    for k, v in g["symbols"].items():
        sym[k] = _val(v, sym)
    d, P = c["head_dim"], c["page_size"]
    keys = np.array(g["keys"], dtype=np.float64)
    vals = np.array(g["values"], dtype=np.float64)
    n_pages = len(keys) // P
    desc = orc.OracleDesc(batch=1, num_q_heads=1, num_kv_heads=1, head_dim=d, page_size=P,
                          max_pages_per_seq=n_pages, max_sel_pages=c["budget_pages"], window=c["window"],
                          sm_scale=_val(c["sm_scale"], sym))
    # physical pages deliberately permuted: logical j lives at physical (n_pages-1-j)
    bt = np.array([[n_pages - 1 - j for j in range(n_pages)]], dtype=np.int64)
    kp = np.zeros((n_pages, 1, P, d)); vp = np.zeros((n_pages, 1, P, d))
    for j in range(n_pages):
        kp[bt[0, j], 0] = keys[j * P:(j + 1) * P]
        vp[bt[0, j], 0] = vals[j * P:(j + 1) * P]
    layer = orc.OracleLayer(desc, kp, vp, bt)
    layer.prefill_bounds(np.array([c["prompt_len"]]))
    return g, c, sym, desc, layer


def test_hand_worked_example_two_steps():
    """Catches: wrong sign / min-max swap in Eq. 1, budget or forced-page accounting, A/M off-by-one,
    >= vs > in the retrospective mask, missing 1/sqrt(d), wrong merge weights, wrong ring slot."""
    g, c, sym, desc, layer = _hand_setup()
    q0 = np.array([_val(x, sym) for x in g["queries"]["step0"]])
    q1 = np.array([_val(x, sym) for x in g["queries"]["step1"]])
    budget = np.array([c["budget_pages"]], dtype=np.int32)
    t0 = c["prompt_len"]
    R = desc.window + 1

    # ---- step 0
    e = g["step0"]
    q_win = np.zeros((1, R, 1, 4)); q_pos = np.full((1, R), -1, dtype=np.int32)
    q_win[0, t0 % R, 0] = q0; q_pos[0, t0 % R] = t0
    r0 = layer.step(q_win, q_pos, q0[None, None, :], np.array([e["seq_len"]]), budget)
    assert np.array_equal(layer.bounds[0, 0, 3, 0], e["bounds_page3"]["kmax"])
    assert np.array_equal(layer.bounds[0, 0, 3, 1], e["bounds_page3"]["kmin"])
    np.testing.assert_allclose(r0["scores"][0, 0, :3], [_val(x, sym) for x in e["scores"]], atol=1e-14)
    assert r0["sel_pages"][0, 0].tolist() == e["sel_pages"]
    assert r0["sel_prev"][0, 0].tolist() == e["sel_prev"]
    np.testing.assert_allclose(r0["out"][0, t0 % R, 0], [_val(x, sym) for x in e["cur_o"]], atol=1e-14)
    assert abs(r0["out_lse"][0, t0 % R, 0] - _val(e["cur_lse"], sym)) < 1e-14

    # ---- step 1
    e = g["step1"]
    t1 = t0 + 1
    q_win = np.zeros((1, R, 1, 4)); q_pos = np.full((1, R), -1, dtype=np.int32)
    q_win[0, t0 % R, 0] = q0; q_pos[0, t0 % R] = t0
    q_win[0, t1 % R, 0] = q1; q_pos[0, t1 % R] = t1
    r1 = layer.step(q_win, q_pos, q1[None, None, :], np.array([e["seq_len"]]), budget)
    assert np.array_equal(layer.bounds[0, 0, 3, 0], e["bounds_page3"]["kmax"])
    assert np.array_equal(layer.bounds[0, 0, 3, 1], e["bounds_page3"]["kmin"])
    np.testing.assert_allclose(r1["scores"][0, 0, :3], [_val(x, sym) for x in e["scores"]], atol=1e-14)
    assert r1["sel_pages"][0, 0].tolist() == e["sel_pages"]
    assert r1["sel_prev"][0, 0].tolist() == e["sel_prev"]
    np.testing.assert_allclose(r1["part_o"][0, t1 % R, 0], [_val(x, sym) for x in e["cur_o"]], atol=1e-14)
    assert abs(r1["part_lse"][0, t1 % R, 0] - _val(e["cur_lse"], sym)) < 1e-14
    np.testing.assert_allclose(r1["part_o"][0, t0 % R, 0], [_val(x, sym) for x in e["past_sup_o"]], atol=1e-14)
    assert abs(r1["part_lse"][0, t0 % R, 0] - _val(e["past_sup_lse"], sym)) < 1e-14
    np.testing.assert_allclose(r1["out"][0, t0 % R, 0], [_val(x, sym) for x in e["past_up_o"]], atol=1e-14)
    assert abs(r1["out_lse"][0, t0 % R, 0] - _val(e["past_up_lse"], sym)) < 1e-14
    # w = 1: position 6 was popped, the single slot now holds the current row (position 7)
    assert layer.cache_pos[0].tolist() == [t1]
    np.testing.assert_allclose(layer.cache_o[0, 0, 0], [_val(x, sym) for x in e["cur_o"]], atol=1e-14)
    assert layer.last_loaded[0, 0].tolist() == [6, 7, -1, 7]


# ------------------------------------------------------------------------------------------ S1
def test_bounds_bruteforce_and_containment():
    """Catches: digest over invalid slots of a partial page (PAD_VALUE would leak), min/max swapped,
    wrong block-table indirection, wrong head indexing."""
    cfg = wl.shrink(wl.c2(), (37,), 5, window=2, budget_tokens=64, num_q_heads=4, num_kv_heads=2, head_dim=8)
    inp = wl.make_layer_inputs(cfg)
    layer = H.oracle_layer(inp)
    L = 39
    layer.desc  # noqa
    orc.update_page_bounds(layer.desc, layer.k_pages, layer.block_table, np.array([L]), np.array([0]), layer.bounds)
    k, _ = H.seq_tokens(inp, 0, L)
    P = cfg.page_size
    for j in range(-(-L // P)):
        for h in range(cfg.num_kv_heads):
            for c in range(cfg.head_dim):
                col = [k[l, h, c] for l in range(j * P, min((j + 1) * P, L))]
                assert layer.bounds[0, h, j, 0, c] == max(col)
                assert layer.bounds[0, h, j, 1, c] == min(col)
    assert np.all(np.abs(layer.bounds[0, :, :-(-L // P)]) < wl.PAD_VALUE / 2)


def test_bounds_incremental_equals_bulk():
    """pos_begin = seq_len-1 each step must give the same digests as a bulk recompute."""
    cfg = wl.shrink(wl.c2(), (30,), 6, window=2, budget_tokens=64, num_q_heads=4, num_kv_heads=2, head_dim=8)
    inp = wl.make_layer_inputs(cfg)
    a = H.oracle_layer(inp); b = H.oracle_layer(inp)
    a.prefill_bounds(np.array([30]))
    for s in range(6):
        L = np.array([31 + s])
        orc.update_page_bounds(a.desc, a.k_pages, a.block_table, L, L - 1, a.bounds)
    orc.update_page_bounds(b.desc, b.k_pages, b.block_table, np.array([36]), np.array([0]), b.bounds)
    assert np.array_equal(a.bounds[:, :, :3], b.bounds[:, :, :3])


# ------------------------------------------------------------------------------------------ S2a
def test_score_upper_bounds_every_token_logit():
    """Eq. 1 is built from per-channel extrema, so score_j(q) >= q.k_l for every token l of page j
    (PAPER.md:33-42).  Catches min/max swap, wrong sign handling for negative q, wrong page indexing."""
    cfg = wl.shrink(wl.c1(), (75,), 1, num_q_heads=3, num_kv_heads=3, head_dim=16)
    inp = wl.make_layer_inputs(cfg)
    layer = H.oracle_layer(inp)
    L = np.array([76])
    layer.prefill_bounds(L)
    q = H.np64(inp.q_all[0])
    s = orc.page_scores(layer.desc, q, layer.bounds, L)
    k, _ = H.seq_tokens(inp, 0, 76)
    tight = 0
    for h in range(3):
        for j in range(5):
            logits = k[j * 16:min((j + 1) * 16, 76), h] @ q[0, h]
            assert s[0, h, j] >= logits.max() - 1e-12
            tight += s[0, h, j] < logits.max() + 50.0
    assert tight > 0            # not a vacuous bound (e.g. +inf)
    assert np.all(np.isneginf(s[0, :, 5:]))


def test_score_closed_form_and_group_reduce():
    """Closed form: max(q*kmin, q*kmax) = q+ * kmax + q- * kmin (kmax >= kmin), so the group-summed score is
    one dot product [sum q+ ; sum q-].[kmax ; kmin].  Catches a dropped q head in the GQA reduction."""
    cfg = wl.shrink(wl.c2(), (64,), 1, window=0, budget_tokens=32, num_q_heads=8, num_kv_heads=2, head_dim=16)
    inp = wl.make_layer_inputs(cfg)
    for red in ("sum", "max"):
        layer = H.oracle_layer(inp, group_reduce=red)
        L = np.array([65]); layer.prefill_bounds(L)
        q = H.np64(inp.q_all[0])
        s = orc.page_scores(layer.desc, q, layer.bounds, L)
        for h in range(2):
            qg = q[0, h * 4:(h + 1) * 4]
            per = np.stack([np.maximum(x, 0) @ layer.bounds[0, h, :5, 0].T + np.minimum(x, 0) @ layer.bounds[0, h, :5, 1].T
                            for x in qg])
            ref = per.sum(0) if red == "sum" else per.max(0)
            np.testing.assert_allclose(s[0, h, :5], ref, rtol=1e-13, atol=1e-12)


# ------------------------------------------------------------------------------------------ S2b
def _desc_small(n_pages, kmax, window=1, **kw):
    return orc.OracleDesc(batch=1, num_q_heads=1, num_kv_heads=1, head_dim=4, page_size=4,
                          max_pages_per_seq=n_pages, max_sel_pages=kmax, window=window, sm_scale=0.5, **kw)


def test_select_is_argmax_k_set_bruteforce():
    """On tiny inputs S_t = argmax-k set of the exhaustive scores (library stable sort), newest page forced.
    Catches ascending/descending confusion, budget off-by-one, forced page not counted in k."""
    rng = np.random.default_rng(5)
    for trial in range(200):
        n = int(rng.integers(1, 12)); k = int(rng.integers(1, 14))
        seq_len = (n - 1) * 4 + int(rng.integers(1, 5))
        scores = rng.normal(size=(1, 1, n))
        if trial % 3 == 0:
            scores = np.round(scores)       # many exact ties
        desc = _desc_small(n, 16)
        A = np.full((1, 1, n), -1, dtype=np.int32)
        sp, _, sc = orc.select_pages(desc, scores, np.array([seq_len]), np.array([k]), A)
        got = sp[0, 0, :sc[0, 0]].tolist()
        kk = min(k, n)
        if kk == n:
            want = list(range(n))
        else:
            order = np.argsort(-scores[0, 0, :n - 1], kind="stable")[:kk - 1]
            want = sorted(order.tolist() + [n - 1])
        assert got == want and sc[0, 0] == kk
        assert sp[0, 0, kk:].tolist() == [-1] * (16 - kk)
        # pure top-k flag
        desc2 = _desc_small(n, 16, force_last_page=False)
        sp2, _, sc2 = orc.select_pages(desc2, scores, np.array([seq_len]), np.array([k]), A.copy())
        want2 = sorted(np.argsort(-scores[0, 0], kind="stable")[:kk].tolist())
        assert sp2[0, 0, :sc2[0, 0]].tolist() == want2


def test_mask_last_loaded_equals_explicit_seen_sets():
    """Reading Q9: 'page j was loaded at some step in [p, t-1]' <=> 'A[j] >= p' when A holds the last step < t
    that loaded j.  Form A's M list against explicit per-step sets, random selections, 60 steps."""
    rng = np.random.default_rng(11)
    n, k, w = 24, 6, 5
    desc = _desc_small(n, k, window=w)
    A = np.full((1, 1, n), -1, dtype=np.int32)
    history = {}
    t0 = 40
    for t in range(t0, t0 + 60):
        scores = rng.normal(size=(1, 1, n))
        seq_len = t + 1
        n_pages = -(-seq_len // 4)
        if n_pages > n:
            break
        sp, sprev, sc = orc.select_pages(desc, scores, np.array([seq_len]), np.array([k]), A)
        S = sp[0, 0, :sc[0, 0]].tolist()
        for p in range(max(t0, t - w), t):
            seen_before = set().union(*[history[m] for m in range(p, t)])
            for i, j in enumerate(S):
                assert (sprev[0, 0, i] >= p) == (j in seen_before)
        history[t] = set(S)
        assert all(A[0, 0, j] == t for j in S)


# ------------------------------------------------------------------------------------------ S3
def _dense_causal_sdpa(inp, b, pos, step_q):
    cfg = inp.cfg
    k, v = H.seq_tokens(inp, b, pos + 1)
    q = H.np64(inp.q_all[step_q, b])
    qt = torch.from_numpy(q).view(cfg.num_kv_heads, cfg.group, 1, cfg.head_dim)
    kt = torch.from_numpy(k).permute(1, 0, 2)[:, None].expand(-1, cfg.group, -1, -1)
    vt = torch.from_numpy(v).permute(1, 0, 2)[:, None].expand(-1, cfg.group, -1, -1)
    o = torch.nn.functional.scaled_dot_product_attention(qt, kt, vt, scale=cfg.sm_scale)
    return o.reshape(cfg.num_q_heads, cfg.head_dim).numpy()


def test_budget_whole_cache_is_dense_causal_attention():
    """budget >= #pages => every row's FINAL output is textbook dense causal attention,
    checked against torch SDPA in fp64.  The current row is dense at once; a past row already saw everything
    it may see at its own step, so later updates must add nothing (all pages masked)."""
    cfg = wl.shrink(wl.c2(), (45, 33), 7, batch=2, window=3, budget_tokens=16 * 64,
                    num_q_heads=4, num_kv_heads=2, head_dim=16)
    inp = wl.make_layer_inputs(cfg)
    _, res = H.run_oracle_trajectory(inp, 7)
    for s, r in enumerate(res):
        for b in range(2):
            for row in range(cfg.window + 1):
                p = int(r["q_pos"][b, row])
                if p < 0:
                    continue
                ref = _dense_causal_sdpa(inp, b, p, p - cfg.prompt_lens[b])
                np.testing.assert_allclose(r["out"][b, row], ref, rtol=1e-12, atol=1e-13)
                if p < r["seq_lens"][b] - 1:
                    assert np.all(np.isneginf(r["part_lse"][b, row]))


def test_window_zero_is_quest():
    """w = 0 'denotes the model without RetroAttention': the output is attention over the pages
    of S_t only (library SDPA over the gathered tokens) and no cache or mask state is touched."""
    cfg = wl.shrink(wl.c2(), (90,), 4, window=0, budget_tokens=48, num_q_heads=4, num_kv_heads=2, head_dim=16)
    inp = wl.make_layer_inputs(cfg)
    layer, res = H.run_oracle_trajectory(inp, 4)
    assert np.all(layer.last_loaded == -1) and np.all(layer.cache_pos == -1)
    for s, r in enumerate(res):
        p = 90 + s
        k, v = H.seq_tokens(inp, 0, p + 1)
        q = H.np64(inp.q_all[s, 0])
        for h in range(2):
            mask = np.zeros(p + 1, dtype=bool)
            assert r["sel_count"][0, h] == 3
            for j in r["sel_pages"][0, h, :3]:
                mask[j * 16:min((j + 1) * 16, p + 1)] = True
            assert mask[p]                                     # newest page is in S_t
            for g in range(2):
                o, lse = H.sdpa_over_tokens(q[h * 2 + g], k[:, h], v[:, h], mask, cfg.sm_scale)
                np.testing.assert_allclose(r["out"][0, 0, h * 2 + g], o, rtol=1e-12, atol=1e-13)
                assert abs(r["out_lse"][0, 0, h * 2 + g] - lse) < 1e-12


def test_softmax_partial_closed_forms():
    """Uniform logits -> mean of V and lse = x + ln n; shift invariance of o; catches lse = m + l (no log)."""
    v = np.arange(12.0).reshape(4, 3)
    k = np.ones((4, 2)); q = np.array([0.3, -0.1])
    o, lse = orc.softmax_partial(q, k, v, 2.0)
    np.testing.assert_allclose(o, v.mean(0), rtol=1e-15)
    assert abs(lse - (0.4 + math.log(4))) < 1e-15
    o2, lse2 = orc.softmax_partial(q * 1000, k, v, 2.0)        # large logits must not overflow
    np.testing.assert_allclose(o2, v.mean(0), rtol=1e-15)
    assert abs(lse2 - (400 + math.log(4))) < 1e-12
    o3, lse3 = orc.softmax_partial(q, np.zeros((0, 2)), np.zeros((0, 3)), 2.0)
    assert np.all(o3 == 0) and lse3 == -math.inf


# ------------------------------------------------------------------------------------------ S4
def test_merge_partition_property_and_order_independence():
    """'aggregation of two partial softmax outputs can be exactly same as the original softmax output'
    (PAPER.md:444): attention over a token set == merge of attentions over ANY partition, in ANY order;
    merging with the empty partial is the identity."""
    rng = np.random.default_rng(3)
    n, d = 37, 8
    k = rng.normal(size=(n, d)); v = rng.normal(size=(n, d)); q = rng.normal(size=d) * 3
    full_o, full_lse = H.sdpa_over_tokens(q, k, v, np.ones(n, dtype=bool), 0.35)
    for trial in range(20):
        labels = rng.integers(0, 4, size=n)
        parts = [orc.softmax_partial(q, k[labels == c], v[labels == c], 0.35) for c in range(4)]
        parts.append((np.zeros(d), -math.inf))
        order = rng.permutation(len(parts))
        o, lse = parts[order[0]]
        for i in order[1:]:
            o, lse = orc.merge_partials(o, lse, parts[i][0], parts[i][1])
        np.testing.assert_allclose(o, full_o, rtol=1e-12, atol=1e-13)
        assert abs(lse - full_lse) < 1e-12
    o, lse = orc.merge_partials(np.zeros(d), -math.inf, np.zeros(d), -math.inf)
    assert lse == -math.inf and np.all(o == 0)


@pytest.mark.parametrize("force_last,group_reduce", [(True, "sum"), (False, "sum"), (True, "max")])
def test_form_a_equals_plain_definition(force_last, group_reduce):
    """THE main pin.  Form A (digests -> scores -> top-k -> last-loaded mask -> masked attention -> LSE merge
    -> ring) against the plain definition: after step m the output of the query at position p
    is dense attention over tokens l <= p of the pages in the union of S_p..S_m, with every S recomputed
    independently from raw keys by a stable full sort, and the attention done by torch SDPA.
    Ragged batch, GQA 2, page roll-over inside the run, window ramp-up, partial newest page."""
    cfg = wl.shrink(wl.c2(), (61, 50), 12, batch=2, window=3, budget_tokens=16 * 3,
                    num_q_heads=4, num_kv_heads=2, head_dim=16)
    inp = wl.make_layer_inputs(cfg)
    _, res = H.run_oracle_trajectory(inp, 12, force_last_page=force_last, group_reduce=group_reduce)
    for b in range(2):
        fb = H.FormB(inp, b, cfg.budget_pages, force_last, group_reduce)
        for m in range(12):
            S = fb.select(m)
            r = res[m]
            for h in range(2):
                assert set(r["sel_pages"][b, h, :r["sel_count"][b, h]].tolist()) == S[h]
            for s in wl.window_rows(cfg, m, b):
                p = cfg.prompt_lens[b] + s
                row = wl.ring_slot(cfg, p)
                assert r["q_pos"][b, row] == p
                o, lse = fb.out(s, m)
                np.testing.assert_allclose(r["out"][b, row], o, rtol=1e-11, atol=1e-12)
                np.testing.assert_allclose(r["out_lse"][b, row], lse, rtol=1e-12, atol=1e-12)


def test_cache_ring_eviction():
    """A row leaves the cache w steps after its creation; cache_pos holds exactly positions t-w+1..t."""
    cfg = wl.shrink(wl.c1(), (40,), 9, window=3, budget_tokens=32)
    inp = wl.make_layer_inputs(cfg)
    layer = H.oracle_layer(inp)
    layer.prefill_bounds(np.array([40]))
    for s in range(9):
        q_win, q_pos = wl.make_q_window(inp, s)
        layer.step(H.np64(q_win), q_pos.numpy(), H.np64(inp.q_all[s]), inp.seq_lens_at(s).numpy(), np.array([2]))
        t = 40 + s
        want = sorted(p for p in range(t - 2, t + 1) if p >= 40)
        assert sorted(x for x in layer.cache_pos[0].tolist() if x >= 0) == want


def test_effective_budget_grows_with_window():
    """Sanity range only: with retro updates a query is exposed to >= its own budget of pages."""
    cfg = wl.shrink(wl.c2(), (400,), 10, window=4, budget_tokens=16 * 6, num_q_heads=4, num_kv_heads=2, head_dim=16)
    inp = wl.make_layer_inputs(cfg)
    fb = H.FormB(inp, 0, cfg.budget_pages)
    for m in range(10):
        fb.select(m)
    own = len(fb.seen(2, 2, 0)); grown = len(fb.seen(2, 6, 0))
    assert own == 6 and own <= grown <= 6 * 5


# ------------------------------------------------------------------------------- NEXT-1 UpdateKV
def test_update_kv_overwrites_exactly_the_named_rows_and_digests_follow():
    """Catches: wrong block-table indirection or in-page offset, K/V swapped, head stride, skipped -1 entries
    being written, and digests not following the overwrite (incremental refresh == bulk recompute)."""
    cfg = wl.shrink(wl.c2(), (45,), 4, window=3, budget_tokens=64, num_q_heads=4, num_kv_heads=2, head_dim=8)
    inp = wl.make_layer_inputs(cfg)
    layer = H.oracle_layer(inp)
    L = 47
    seq = np.array([L])
    layer.prefill_bounds(seq)
    k0, v0 = H.seq_tokens(inp, 0, L)
    rng = np.random.default_rng(3)
    positions = np.array([[44, -1, 46, 31]], dtype=np.int32)          # two pages, one skipped entry
    # the oracle layer holds the pools as float32 arrays: use float32-representable replacement rows
    k_hat = rng.standard_normal((1, 4, cfg.num_kv_heads, cfg.head_dim)).astype(np.float32).astype(np.float64)
    v_hat = rng.standard_normal((1, 4, cfg.num_kv_heads, cfg.head_dim)).astype(np.float32).astype(np.float64)
    orc.update_kv(layer.desc, layer.k_pages, layer.v_pages, layer.block_table, seq, positions, k_hat, v_hat)
    # plain definition on the logical token sequence
    k1, v1 = k0.copy(), v0.copy()
    for u, pos in enumerate(positions[0]):
        if pos >= 0:
            k1[pos], v1[pos] = k_hat[0, u], v_hat[0, u]
    P = cfg.page_size
    for l in range(L):
        phys = int(layer.block_table[0, l // P])
        assert np.array_equal(layer.k_pages[phys, :, l % P], k1[l])
        assert np.array_equal(layer.v_pages[phys, :, l % P], v1[l])
    # digests: refresh from the oldest overwritten position, compare with brute force over every page
    orc.update_page_bounds(layer.desc, layer.k_pages, layer.block_table, seq, np.array([31]), layer.bounds)
    for j in range(-(-L // P)):
        rows = k1[j * P:min((j + 1) * P, L)]
        assert np.array_equal(layer.bounds[0, :, j, 0], rows.max(axis=0))
        assert np.array_equal(layer.bounds[0, :, j, 1], rows.min(axis=0))
    # overwriting rows with their own values is the identity
    before = layer.k_pages.copy()
    same = np.stack([k1[[44, 46]]])
    orc.update_kv(layer.desc, layer.k_pages, layer.v_pages, layer.block_table, seq, np.array([[44, 46]]),
                  same, np.stack([v1[[44, 46]]]))
    assert np.array_equal(layer.k_pages, before)


# ------------------------------------------------------------------------------- NEXT-2 budget policy, Alg. 2 alone
def test_budget_policy_values_from_the_papers_rule():
    """budget = 0.15 x context length, minimum 256 tokens.  Hand-computed values (page 16):
    32768 -> 4915 tokens -> 307 pages; 1000 -> 150 < 256 -> 16 pages; 1707 -> 256.05 -> 256 -> 16 pages;
    1714 -> 257 tokens -> 16 pages; 131072 -> 19660 -> 1228 pages."""
    desc = dataclasses_replace(_desc_small(4, 4), batch=5, page_size=16)
    got = orc.budget_policy(desc, np.array([32768, 1000, 1707, 1714, 131072]))
    assert got.tolist() == [307, 16, 16, 16, 1228]
    assert orc.budget_policy(desc, np.array([10, 10, 10, 10, 10]), ratio_permille=150, min_tokens=0).tolist() == [1] * 5


def test_build_mask_alone_equals_the_select_epilogue():
    """Alg. 2 run on its own over the S_t that select_pages chose must reproduce select_pages' M and A."""
    cfg = wl.shrink(wl.c2(), (200,), 6, window=3, budget_tokens=64, num_q_heads=4, num_kv_heads=2, head_dim=8)
    inp = wl.make_layer_inputs(cfg)
    a = H.oracle_layer(inp); b = H.oracle_layer(inp)
    a.prefill_bounds(np.array([200])); b.prefill_bounds(np.array([200]))
    budget = np.array([cfg.budget_pages], dtype=np.int32)
    for s in range(6):
        L = np.array([201 + s])
        for lay in (a, b):
            orc.update_page_bounds(lay.desc, lay.k_pages, lay.block_table, L, L - 1, lay.bounds)
        scores = orc.page_scores(a.desc, H.np64(inp.q_all[s]), a.bounds, L)
        sp, sv, sc = orc.select_pages(a.desc, scores, L, budget, a.last_loaded)
        sv2 = orc.build_mask(b.desc, sp, sc, L, b.last_loaded)
        assert np.array_equal(sv, sv2) and np.array_equal(a.last_loaded, b.last_loaded)
    assert (a.last_loaded >= 0).any()


# ------------------------------------------------------------------------------- NEXT-4 correlated workload
def test_correlated_workload_raises_page_overlap_and_keeps_the_main_pin():
    """The correlated query mode (planted keys persist, AR(1) noise) only changes q: K/V and step 0 are the i.i.d.
    ones, the adjacent-step overlap of the oracle's selections goes up (PAPER.md:349 reports ~80 % on real
    activations), and form A still equals the plain definition on these inputs (most pairs are now masked)."""
    cfg = wl.shrink(wl.c2(), (400, 380), 12, batch=2, window=3, budget_tokens=16 * 5,
                    num_q_heads=4, num_kv_heads=2, head_dim=16)
    iid = wl.make_layer_inputs(cfg)
    cor = wl.make_layer_inputs(cfg.replace(corr_rho=0.95))
    assert torch.equal(iid.k_pages, cor.k_pages) and torch.equal(iid.v_pages, cor.v_pages)
    assert torch.equal(iid.q_all[0], cor.q_all[0]) and not torch.equal(iid.q_all[1:], cor.q_all[1:])

    def overlap(inp):
        _, res = H.run_oracle_trajectory(inp, 12)
        same = tot = 0
        for m in range(1, 12):
            for b in range(2):
                for h in range(2):
                    a = set(res[m - 1]["sel_pages"][b, h, :res[m - 1]["sel_count"][b, h]].tolist())
                    c = set(res[m]["sel_pages"][b, h, :res[m]["sel_count"][b, h]].tolist())
                    same += len(a & c); tot += len(c)
        return same / tot, res
    ov_iid, _ = overlap(iid)
    ov_cor, res = overlap(cor)
    assert ov_cor > ov_iid + 0.2 and ov_cor > 0.6, (ov_iid, ov_cor)
    for b in range(2):
        fb = H.FormB(cor, b, cfg.budget_pages)
        for m in range(12):
            fb.select(m)
            for s in wl.window_rows(cfg, m, b):
                row = wl.ring_slot(cfg, cfg.prompt_lens[b] + s)
                o, lse = fb.out(s, m)
                np.testing.assert_allclose(res[m]["out"][b, row], o, rtol=1e-11, atol=1e-12)


def test_step_diagnostics_effective_budget_is_the_union_size_and_mass_identity():
    """Pins for the NEXT-4 counters, against quantities computed another way:
    (i) summed over the steps a query stays in the window, supp_pages is the number of DISTINCT pages (with a token
        at or before the query) in the union of the page sets of those steps (form B's explicit sets): every page
        is counted once, the first time it is loaded (PAPER.md:62 effective KV budget; reading Q9);
    (ii) 1 - supp_mass at step m equals e^{lse(out, step m-1) - lse(out, step m)} for a past row, supp_mass = 1
        for the current row (Eq. 8-9)."""
    cfg = wl.shrink(wl.c2(), (61, 50), 14, batch=2, window=3, budget_tokens=16 * 3,
                    num_q_heads=4, num_kv_heads=2, head_dim=16)
    inp = wl.make_layer_inputs(cfg)
    layer, res = H.run_oracle_trajectory(inp, 14)
    diag = [orc.step_diagnostics(layer.desc, r["sel_pages"], r["sel_prev"], r["sel_count"], r["q_pos"],
                                 r["seq_lens"], r["part_lse"], r["out_lse"]) for r in res]
    P, w = cfg.page_size, cfg.window
    for b in range(2):
        fb = H.FormB(inp, b, cfg.budget_pages)
        for m in range(14):
            fb.select(m)
        for s in range(14 - w):                       # queries whose whole window life is inside the run
            p = cfg.prompt_lens[b] + s
            row = wl.ring_slot(cfg, p)
            for h in range(2):
                total = sum(int(diag[m][0][b, h, row]) for m in range(s, s + w + 1))
                want = len([j for j in fb.seen(s, s + w, h) if j * P <= p])
                assert total == want, (b, s, h, total, want)
            np.testing.assert_allclose(diag[s][1][b, row], 1.0, rtol=0, atol=1e-15)      # current row
            for m in range(s + 1, s + w + 1):
                keep = np.exp(res[m - 1]["out_lse"][b, row] - res[m]["out_lse"][b, row])
                np.testing.assert_allclose(1.0 - diag[m][1][b, row], keep, rtol=0, atol=1e-12)
    # rows that are not in the window report nothing
    for b in range(2):
        empty = [r for r in range(w + 1) if res[0]["q_pos"][b, r] < 0]
        assert len(empty) == w and np.all(diag[0][0][b][:, empty] == 0) and np.all(diag[0][1][b][empty] == 0)


def test_bf16_cache_rounding_is_library_rounding_and_its_error_budget_over_w_merges():
    """NEXT-3 (Eq. 12: 16-bit cached O + fp32 LSE).  (1) round_bf16 == torch's float32 -> bfloat16
    conversion (round-to-nearest-even) on values over 40 binades; (2) error budget: a trajectory with the cache kept
    in bf16 against the same trajectory with the full-precision cache: every merged output within
    (w + 1) roundings of 2^-9 relative to the largest value, far inside the 2e-2 + 1e-2 |x| tolerance."""
    import torch
    rng = np.random.default_rng(3)
    x = rng.standard_normal(200000) * np.exp(rng.uniform(-14, 14, 200000))
    assert np.array_equal(orc.round_bf16(x), torch.from_numpy(x).float().to(torch.bfloat16).double().numpy())
    assert np.array_equal(orc.round_bf16(np.array([0.0, -0.0, 1.0, -2.5])), np.array([0.0, -0.0, 1.0, -2.5]))
    cfg = wl.shrink(wl.c2(), (300,), 14, window=6, budget_tokens=96, num_q_heads=8, num_kv_heads=2)
    inp = wl.make_layer_inputs(cfg)
    _, ref = H.run_oracle_trajectory(inp, 14)
    _, low = H.run_oracle_trajectory(inp, 14, cache_round="bf16")
    worst = 0.0
    for a, b in zip(ref, low):
        assert np.array_equal(a["sel_pages"], b["sel_pages"])
        scale = np.abs(a["out"]).max()
        worst = max(worst, float(np.abs(a["out"] - b["out"]).max() / scale))
        np.testing.assert_allclose(b["out"], a["out"], atol=2e-2, rtol=1e-2)
    assert 0.0 < worst < (cfg.window + 1) * 2.0 ** -9
