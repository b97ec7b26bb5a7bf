"""GPU-vs-oracle lock-step harness with teacher forcing.

State (the mask A and the output cache) depends on the selections, so one tolerated tie would fork the two
trajectories.  At every checked step: (1) run the CUDA select and compare with the oracle under the tie rule;
(2) overwrite the device sel_* / A with the ORACLE's; (3) run the CUDA attend + merge and compare part_*,
out, cache_* within the dtype tolerance.  Everything on the device goes through the C ABI binding.
"""
from __future__ import annotations

import math

import numpy as np
import torch

from oracle import retro_oracle as orc
from paper_2508_09001_b200 import binding as rb
from paper_2508_09001_b200 import workload as wl
from tests import helpers as H

TOL = {"f32": (1e-4, 1e-4), "bf16": (2e-2, 1e-2)}   # (atol, rtol) from BASELINE.json north_star
TIE_TAU = 1e-5                                        # ties within 1e-5 of the k-th score may go either way


def close(got, want, atol, rtol, what):
    got = np.asarray(got, dtype=np.float64)
    want = np.asarray(want, dtype=np.float64)
    both_ninf = np.isneginf(got) & np.isneginf(want)
    g = np.where(both_ninf, 0.0, got)
    w = np.where(both_ninf, 0.0, want)
    assert np.all(np.isfinite(g) == np.isfinite(w)), f"{what}: finiteness pattern differs"
    err = np.abs(g - w)
    bound = atol + rtol * np.abs(w)
    bad = err > bound
    if bad.any():
        i = np.unravel_index(np.argmax(err - bound), err.shape)
        raise AssertionError(f"{what}: {bad.sum()} of {bad.size} outside tol; worst at {i}: got {got[i]} want {want[i]}")
    return float(err.max()) if err.size else 0.0


def make_device_layer(inp: wl.LayerInputs, budget_pages=None, k_max=None, **desc_kw):
    cfg = inp.cfg
    budget = cfg.budget_pages if budget_pages is None else budget_pages
    kmax = max(1, budget if k_max is None else k_max)
    desc = rb.make_desc(cfg.batch, cfg.num_q_heads, cfg.num_kv_heads, cfg.head_dim, cfg.page_size,
                        cfg.max_pages_per_seq, kmax, cfg.num_phys_pages, cfg.window, cfg.dtype,
                        sm_scale=cfg.sm_scale, **desc_kw)
    dev = torch.device("cuda")
    seq_lens = inp.prompt_lens.to(dev).clone()
    bud = torch.full((cfg.batch,), budget, dtype=torch.int32, device=dev)
    buf = rb.LayerBuffers(desc, inp.k_pages.to(dev), inp.v_pages.to(dev), inp.block_table.to(dev), seq_lens, bud)
    return desc, buf


def check_select(cfg, desc, res, g_pages, g_prev, g_count, A_before, A_after_gpu, seq_lens, force_last=True):
    """Tie rule: every candidate with score > s_k + tau selected, none with score < s_k - tau."""
    B, hk = cfg.batch, cfg.num_kv_heads
    for b in range(B):
        L = int(seq_lens[b]); t = L - 1
        n = -(-L // cfg.page_size)
        for h in range(hk):
            k = int(res["sel_count"][b, h])
            assert int(g_count[b, h]) == k, f"sel_count b{b} h{h}: {g_count[b, h]} vs {k}"
            got = g_pages[b, h, :k].tolist()
            assert got == sorted(got) and len(set(got)) == k, "selection must be ascending and unique"
            assert all(0 <= j < n for j in got)
            assert np.all(g_pages[b, h, k:] == -1) and np.all(g_prev[b, h, k:] == -1)
            want = res["sel_pages"][b, h, :k].tolist()
            if got != want:
                s = res["scores"][b, h, :n]
                forced = {n - 1} if (force_last and 0 < k < n) else set()
                cand_sel = [j for j in want if j not in forced]
                s_k = min(s[j] for j in cand_sel) if cand_sel else math.inf
                for j in range(n):
                    if j in forced:
                        assert j in got
                    elif s[j] > s_k + TIE_TAU:
                        assert j in got, f"page {j} (score {s[j]}) must be selected (s_k {s_k})"
                    elif s[j] < s_k - TIE_TAU:
                        assert j not in got, f"page {j} (score {s[j]}) must not be selected (s_k {s_k})"
            if A_before is not None:
                for i, j in enumerate(got):
                    assert int(g_prev[b, h, i]) == int(A_before[b, h, j]), "sel_prev must be A[page] before the update"
                    assert int(A_after_gpu[b, h, j]) == t
                untouched = np.ones(A_before.shape[2], dtype=bool); untouched[got] = False
                assert np.array_equal(A_after_gpu[b, h][untouched], A_before[b, h][untouched])
    return True


def sync_from_oracle(buf, layer, cfg):
    """Upload the oracle's persistent state (mask A, output cache ring) to the device layer: the CUDA path then
    continues a trajectory the oracle ran alone (single-step checks from a synced state)."""
    if cfg.window > 0:
        buf.last_loaded.copy_(torch.from_numpy(layer.last_loaded))
        buf.cache_o.copy_(torch.from_numpy(layer.cache_o).float())
        buf.cache_lse.copy_(torch.from_numpy(layer.cache_lse).float())
        buf.cache_pos.copy_(torch.from_numpy(layer.cache_pos))


def _window(inp, s, first_step):
    cfg = inp.cfg
    B = cfg.batch
    q_win = torch.zeros((B, cfg.window + 1, cfg.num_q_heads, cfg.head_dim), dtype=inp.q_all.dtype)
    q_pos = torch.full((B, cfg.window + 1), -1, dtype=torch.int32)
    for b in range(B):
        for ss in range(max(first_step, s - cfg.window), s + 1):
            pos = cfg.prompt_lens[b] + ss
            q_win[b, wl.ring_slot(cfg, pos)] = inp.q_all[ss, b].cpu()
            q_pos[b, wl.ring_slot(cfg, pos)] = pos
    return q_win, q_pos


def lockstep(inp: wl.LayerInputs, n_steps: int, budget_pages=None, start_step: int = 0, check_scores=True,
             desc_kw=None, oracle_kw=None, k_max=None, use_decode_step=False, warm_steps: int = 0,
             oracle_batch=None, check_from: int = 0, exact_select=False):
    """Run n_steps decode steps on both sides from decode step `start_step`.  With warm_steps = 0 the retro window
    is empty at start_step; with warm_steps > 0 the ORACLE ALONE first runs decode steps start_step - warm_steps ..
    start_step - 1 (from an empty window), its state (A, output cache) is uploaded to the device, and the
    lock-step starts from that synced state with a (partly) filled window.
    oracle_batch: the sequences the oracle computes (sampled outputs at full size: the (sequence, KV head) units
    are independent, the CUDA path always runs the whole batch); default all.  Returns dict of max abs errors."""
    H.require_cuda()
    cfg = inp.cfg
    atol, rtol = TOL[cfg.dtype]
    desc_kw = desc_kw or {}
    oracle_kw = oracle_kw or {}
    budget = cfg.budget_pages if budget_pages is None else budget_pages
    desc, buf = make_device_layer(inp, budget, k_max=k_max, **desc_kw)
    okw = dict(oracle_kw)
    okw["max_sel_pages"] = k_max if k_max is not None else max(1, budget)
    bs = list(range(cfg.batch)) if oracle_batch is None else list(oracle_batch)
    assert warm_steps == 0 or len(bs) == cfg.batch, "a synced start uploads the oracle state of every sequence"
    nb = len(bs)
    sub = cfg.replace(batch=nb, prompt_lens=tuple(cfg.prompt_lens[b] for b in bs))
    layer = H.oracle_layer(inp, batch_rows=bs, **okw)
    dev = buf.seq_lens.device
    B = cfg.batch
    errs = dict(part_o=0.0, part_lse=0.0, out=0.0, cache_o=0.0, scores_rel=0.0)
    bud_o = np.full(nb, budget, dtype=np.int32)
    sub_np = lambda t: t.cpu().numpy()[bs]          # device tensor -> host rows of the oracle's sequences

    # prefill digests on both sides
    first_step = start_step - warm_steps
    assert first_step >= 0
    layer.prefill_bounds(np.asarray(sub.prompt_lens) + first_step)
    for s in range(first_step, start_step):          # oracle alone
        q_win, q_pos = _window(inp, s, first_step)
        layer.step(H.np64(q_win[bs]), q_pos.numpy()[bs], H.np64(inp.q_all[s].cpu()[bs]),
                   inp.seq_lens_at(s).cpu().numpy()[bs], bud_o)
    prompt = np.asarray(cfg.prompt_lens) + start_step
    if warm_steps > 0:                               # digests of the pages the warm steps touched are current
        layer.prefill_bounds(prompt[bs])
        sync_from_oracle(buf, layer, cfg)
    buf.seq_lens.copy_(torch.from_numpy(prompt.astype(np.int32)))
    buf.rebuild_bounds()
    torch.cuda.synchronize()
    for i, b in enumerate(bs):
        npg = -(-int(prompt[b]) // cfg.page_size)
        assert np.array_equal(buf.bounds[b, :, :npg].float().cpu().numpy(),
                              layer.bounds[i, :, :npg].astype(np.float32)), "prefill digests"

    def check_newest_digest(seq_lens):
        for i, b in enumerate(bs):
            j = (int(seq_lens[b]) - 1) // cfg.page_size
            assert np.array_equal(buf.bounds[b, :, j].float().cpu().numpy(),
                                  layer.bounds[i, :, j].astype(np.float32)), "digest of newest page"

    pos_begin = torch.zeros(B, dtype=torch.int32, device=dev)
    scores_out = (torch.zeros((B, cfg.num_kv_heads, cfg.max_pages_per_seq), dtype=torch.float64, device=dev)
                  if check_scores and not use_decode_step else None)
    bs_t = torch.tensor(bs, dtype=torch.long, device=dev)
    for s in range(start_step, start_step + n_steps):
        q_win, q_pos = _window(inp, s, first_step)     # decode steps [max(first_step, s-w), s]
        seq_lens = inp.seq_lens_at(s).cpu().numpy()
        q_cur = inp.q_all[s].cpu()
        A_before = layer.last_loaded.copy() if cfg.window > 0 else None
        res = layer.step(H.np64(q_win[bs]), q_pos.numpy()[bs], H.np64(q_cur[bs]), seq_lens[bs], bud_o)

        buf.seq_lens.copy_(torch.from_numpy(seq_lens))
        buf.q_win.copy_(q_win); buf.q_pos.copy_(q_pos); buf.q_cur.copy_(q_cur)
        if use_decode_step:
            # whole-step entry point: no teacher forcing possible, so only used where selections are tie-free
            rb.retro_decode_step(desc, buf.state, buf.q_win, buf.q_pos, buf.q_cur, buf.out, buf.out_lse)
            torch.cuda.synchronize()
            check_newest_digest(seq_lens)                 # S1 runs inside the select kernel on this path
            assert np.array_equal(sub_np(buf.sel_pages), res["sel_pages"]), f"step {s} sel_pages"
            if cfg.window > 0:      # w = 0: no past rows, the mask list is not used (A is optional there)
                assert np.array_equal(sub_np(buf.sel_prev), res["sel_prev"]), f"step {s} sel_prev"
        else:
            # S1
            pos_begin.copy_(torch.from_numpy((seq_lens - 1).astype(np.int32)))
            rb.retro_update_page_bounds(desc, buf.k_pages, buf.block_table, buf.seq_lens, pos_begin, 1, buf.bounds)
            # S2
            la = buf.last_loaded if cfg.window > 0 else None
            rb.retro_select_pages(desc, buf.q_cur, buf.bounds, buf.seq_lens, buf.budget_pages, la, buf.sel_pages,
                                  buf.sel_prev, buf.sel_count, scores_out, buf.workspace)
            torch.cuda.synchronize()
            check_newest_digest(seq_lens)
            if scores_out is not None:
                gs = sub_np(scores_out)
                for i in range(nb):
                    npg = -(-int(seq_lens[bs[i]]) // cfg.page_size)
                    ref = res["scores"][i, :, :npg]
                    rel = np.abs(gs[i, :, :npg] - ref) / np.maximum(1.0, np.abs(ref))
                    assert rel.max() < 1e-12, f"fp64 scores differ: {rel.max()}"
                    errs["scores_rel"] = max(errs["scores_rel"], float(rel.max()))
                    assert np.all(np.isneginf(gs[i, :, npg:]))
            if exact_select:
                assert np.array_equal(sub_np(buf.sel_pages), res["sel_pages"]), f"step {s} sel_pages (exact)"
            check_select(sub, desc, res, sub_np(buf.sel_pages), sub_np(buf.sel_prev), sub_np(buf.sel_count), A_before,
                         sub_np(buf.last_loaded) if cfg.window > 0 else None, seq_lens[bs],
                         force_last=desc.force_last_page != 0)
            # teacher forcing (the oracle's sequences; the others keep the device's own selection)
            buf.sel_pages[bs_t] = torch.from_numpy(res["sel_pages"]).to(dev)
            buf.sel_prev[bs_t] = torch.from_numpy(res["sel_prev"]).to(dev)
            buf.sel_count[bs_t] = torch.from_numpy(res["sel_count"]).to(dev)
            if cfg.window > 0:
                buf.last_loaded[bs_t] = torch.from_numpy(layer.last_loaded).to(dev)
            # S3
            rb.retro_sparse_attend(desc, buf.q_win, buf.q_pos, buf.k_pages, buf.v_pages, buf.block_table,
                                   buf.seq_lens, buf.sel_pages, buf.sel_prev, buf.sel_count, buf.part_o,
                                   buf.part_lse, buf.workspace)
            # S4
            co = buf.cache_o if cfg.window > 0 else None
            cl = buf.cache_lse if cfg.window > 0 else None
            cp = buf.cache_pos if cfg.window > 0 else None
            rb.retro_merge_output_cache(desc, buf.part_o, buf.part_lse, buf.q_pos, buf.seq_lens, co, cl, cp,
                                        buf.out, buf.out_lse)
            torch.cuda.synchronize()
            if s - start_step >= check_from:
                errs["part_o"] = max(errs["part_o"], close(sub_np(buf.part_o), res["part_o"], atol, rtol, f"step {s} part_o"))
                errs["part_lse"] = max(errs["part_lse"], close(sub_np(buf.part_lse), res["part_lse"], atol, rtol, f"step {s} part_lse"))
        if s - start_step < check_from:
            continue
        errs["out"] = max(errs["out"], close(sub_np(buf.out.float()), res["out"], atol, rtol, f"step {s} out"))
        close(sub_np(buf.out_lse), res["out_lse"], atol, rtol, f"step {s} out_lse")
        if cfg.window > 0:
            assert np.array_equal(sub_np(buf.cache_pos), layer.cache_pos), f"step {s} cache_pos"
            live = layer.cache_pos >= 0
            co_g, cl_g = sub_np(buf.cache_o.float()), sub_np(buf.cache_lse)
            errs["cache_o"] = max(errs["cache_o"], close(co_g[live], layer.cache_o[live], atol, rtol, f"step {s} cache_o"))
            close(cl_g[live], layer.cache_lse[live], atol, rtol, f"step {s} cache_lse")
    return errs
