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


def lockstep(inp: wl.LayerInputs, n_steps: int, budget_pages=None, start_step: int = 0, check_scores=True,
             desc_kw=None, oracle_kw=None, k_max=None, use_decode_step=False):
    """Run n_steps decode steps on both sides from decode step `start_step` (window empty at start).
    Returns dict of max abs errors."""
    H.require_cuda()
    cfg = inp.cfg
    atol, rtol = TOL[cfg.dtype]
    desc_kw = desc_kw or {}
    oracle_kw = oracle_kw or {}
    budget = cfg.budget_pages if budget_pages is None else budget_pages
    desc, buf = make_device_layer(inp, budget, k_max=k_max, **desc_kw)
    okw = dict(oracle_kw)
    if k_max is not None:
        okw["max_sel_pages"] = k_max
    else:
        okw["max_sel_pages"] = max(1, budget)
    layer = H.oracle_layer(inp, **okw)
    dev = buf.seq_lens.device
    B = cfg.batch
    errs = dict(part_o=0.0, part_lse=0.0, out=0.0, cache_o=0.0, scores_rel=0.0)

    # prefill digests on both sides
    prompt = np.asarray(cfg.prompt_lens) + start_step
    layer.prefill_bounds(prompt)
    buf.seq_lens.copy_(torch.from_numpy(prompt.astype(np.int32)))
    buf.rebuild_bounds()
    torch.cuda.synchronize()
    nb = -(-int(prompt.max()) // cfg.page_size)
    g_bounds = buf.bounds.float().cpu().numpy()
    for b in range(B):
        npg = -(-int(prompt[b]) // cfg.page_size)
        assert np.array_equal(g_bounds[b, :, :npg], layer.bounds[b, :, :npg].astype(np.float32)), "prefill digests"

    pos_begin = torch.zeros(B, dtype=torch.int32, device=dev)
    scores_out = torch.zeros((B, cfg.num_kv_heads, cfg.max_pages_per_seq), dtype=torch.float64, device=dev)
    for s in range(start_step, start_step + n_steps):
        # window of decode steps [max(start, s-w), s]
        q_win = torch.zeros_like(buf.q_win, device="cpu")
        q_pos = torch.full((B, cfg.window + 1), -1, dtype=torch.int32)
        for b in range(B):
            for ss in range(max(start_step, s - cfg.window), s + 1):
                pos = cfg.prompt_lens[b] + ss
                q_win[b, wl.ring_slot(cfg, pos)] = inp.q_all[ss, b].cpu()
                q_pos[b, wl.ring_slot(cfg, pos)] = pos
        seq_lens = inp.seq_lens_at(s).cpu().numpy()
        q_cur = inp.q_all[s].cpu()
        A_before = layer.last_loaded.copy() if cfg.window > 0 else None
        res = layer.step(H.np64(q_win), q_pos.numpy(), H.np64(q_cur), seq_lens,
                         np.full(B, budget, dtype=np.int32))

        buf.seq_lens.copy_(torch.from_numpy(seq_lens))
        buf.q_win.copy_(q_win); buf.q_pos.copy_(q_pos); buf.q_cur.copy_(q_cur)
        if use_decode_step:
            # whole-step entry point: no teacher forcing possible, so only used where selections are tie-free
            rb.retro_decode_step(desc, buf.state, buf.q_win, buf.q_pos, buf.q_cur, buf.out, buf.out_lse)
            torch.cuda.synchronize()
            g_bounds = buf.bounds.float().cpu().numpy()      # S1 runs inside the select kernel on this path
            for b in range(B):
                j = (int(seq_lens[b]) - 1) // cfg.page_size
                assert np.array_equal(g_bounds[b, :, j], layer.bounds[b, :, j].astype(np.float32)), "digest of newest page"
            assert np.array_equal(buf.sel_pages.cpu().numpy(), res["sel_pages"])
            if cfg.window > 0:      # w = 0: no past rows, the mask list is not used (A is optional there)
                assert np.array_equal(buf.sel_prev.cpu().numpy(), res["sel_prev"])
        else:
            # S1
            pos_begin.copy_(torch.from_numpy((seq_lens - 1).astype(np.int32)))
            rb.retro_update_page_bounds(desc, buf.k_pages, buf.block_table, buf.seq_lens, pos_begin, 1, buf.bounds)
            # S2
            la = buf.last_loaded if cfg.window > 0 else None
            rb.retro_select_pages(desc, buf.q_cur, buf.bounds, buf.seq_lens, buf.budget_pages, la, buf.sel_pages,
                                  buf.sel_prev, buf.sel_count, scores_out if check_scores else None, buf.workspace)
            torch.cuda.synchronize()
            g_bounds = buf.bounds.float().cpu().numpy()
            for b in range(B):
                j = (int(seq_lens[b]) - 1) // cfg.page_size
                assert np.array_equal(g_bounds[b, :, j], layer.bounds[b, :, j].astype(np.float32)), "digest of newest page"
            if check_scores:
                gs = scores_out.cpu().numpy()
                for b in range(B):
                    npg = -(-int(seq_lens[b]) // cfg.page_size)
                    ref = res["scores"][b, :, :npg]
                    rel = np.abs(gs[b, :, :npg] - ref) / np.maximum(1.0, np.abs(ref))
                    assert rel.max() < 1e-12, f"fp64 scores differ: {rel.max()}"
                    errs["scores_rel"] = max(errs["scores_rel"], float(rel.max()))
                    assert np.all(np.isneginf(gs[b, :, npg:]))
            check_select(cfg, desc, res, buf.sel_pages.cpu().numpy(), buf.sel_prev.cpu().numpy(),
                         buf.sel_count.cpu().numpy(), A_before,
                         buf.last_loaded.cpu().numpy() if cfg.window > 0 else None, seq_lens,
                         force_last=desc.force_last_page != 0)
            # teacher forcing
            buf.sel_pages.copy_(torch.from_numpy(res["sel_pages"]))
            buf.sel_prev.copy_(torch.from_numpy(res["sel_prev"]))
            buf.sel_count.copy_(torch.from_numpy(res["sel_count"]))
            if cfg.window > 0:
                buf.last_loaded.copy_(torch.from_numpy(layer.last_loaded))
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
            errs["part_o"] = max(errs["part_o"], close(buf.part_o.cpu().numpy(), res["part_o"], atol, rtol, f"step {s} part_o"))
            errs["part_lse"] = max(errs["part_lse"], close(buf.part_lse.cpu().numpy(), res["part_lse"], atol, rtol, f"step {s} part_lse"))
        errs["out"] = max(errs["out"], close(buf.out.float().cpu().numpy(), res["out"], atol, rtol, f"step {s} out"))
        close(buf.out_lse.cpu().numpy(), res["out_lse"], atol, rtol, f"step {s} out_lse")
        if cfg.window > 0:
            assert np.array_equal(buf.cache_pos.cpu().numpy(), layer.cache_pos), f"step {s} cache_pos"
            live = layer.cache_pos >= 0
            co_g, cl_g = buf.cache_o.cpu().numpy(), buf.cache_lse.cpu().numpy()
            errs["cache_o"] = max(errs["cache_o"], close(co_g[live], layer.cache_o[live], atol, rtol, f"step {s} cache_o"))
            close(cl_g[live], layer.cache_lse[live], atol, rtol, f"step {s} cache_lse")
    return errs
