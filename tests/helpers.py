"""Shared test helpers: oracle/workload glue and the plain-definition "form B" of the method.

Form B restates what the method is *supposed to reach* (the updated output of a past
query equals softmax(Q K^T/sqrt(d)) V over the pages in the union of the sets loaded while it was in
the window) with explicit per-query seen-page sets and a library softmax-attention
(torch.nn.functional.scaled_dot_product_attention in fp64).  It shares no code with oracle/ form A.
"""
from __future__ import annotations

import math

import numpy as np
import torch

from oracle import retro_oracle as orc
from paper_2508_09001_b200 import workload as wl


def oracle_desc(cfg: wl.RetroConfig, **kw) -> orc.OracleDesc:
    d = dict(batch=cfg.batch, num_q_heads=cfg.num_q_heads, num_kv_heads=cfg.num_kv_heads,
             head_dim=cfg.head_dim, page_size=cfg.page_size, max_pages_per_seq=cfg.max_pages_per_seq,
             max_sel_pages=max(1, cfg.budget_pages), window=cfg.window, sm_scale=cfg.sm_scale)
    d.update(kw)
    return orc.OracleDesc(**d)


def oracle_layer(inp: wl.LayerInputs, batch_rows=None, **kw) -> orc.OracleLayer:
    """batch_rows: the sequences the oracle computes (units are independent; the pools are shared)."""
    bt = inp.block_table.cpu().numpy()
    if batch_rows is not None and list(batch_rows) != list(range(inp.cfg.batch)):
        kw = dict(kw, batch=len(batch_rows))
        bt = bt[list(batch_rows)]
    desc = oracle_desc(inp.cfg, **kw)
    return orc.OracleLayer(desc, inp.k_pages.float().cpu().numpy(), inp.v_pages.float().cpu().numpy(), bt)


def np64(x: torch.Tensor) -> np.ndarray:
    return x.double().cpu().numpy()


def seq_tokens(inp: wl.LayerInputs, b: int, upto: int):
    """K, V of sequence b's tokens 0..upto-1 as [upto][h_k][d] fp64 numpy (gathered through the block table)."""
    cfg = inp.cfg
    P = cfg.page_size
    npg = -(-upto // P)
    phys = inp.block_table[b, :npg].long()
    k = inp.k_pages[phys].double().permute(0, 2, 1, 3).reshape(npg * P, cfg.num_kv_heads, cfg.head_dim)[:upto]
    v = inp.v_pages[phys].double().permute(0, 2, 1, 3).reshape(npg * P, cfg.num_kv_heads, cfg.head_dim)[:upto]
    return k.cpu().numpy(), v.cpu().numpy()


def sdpa_over_tokens(q, k, v, token_mask, sm_scale):
    """Library softmax attention over the tokens where token_mask is True.  q [d], k,v [n][d] -> o [d], lse."""
    if not token_mask.any():
        return np.zeros_like(q), -math.inf
    qt = torch.from_numpy(q)[None, None, None, :]
    kt = torch.from_numpy(k)[None, None]
    vt = torch.from_numpy(v)[None, None]
    m = torch.from_numpy(token_mask)[None, None, None, :]
    o = torch.nn.functional.scaled_dot_product_attention(qt, kt, vt, attn_mask=m, scale=sm_scale)
    x = (kt[0, 0] @ qt[0, 0, 0]) * sm_scale
    lse = torch.logsumexp(x[m[0, 0, 0]], dim=0)
    return o[0, 0, 0].numpy(), float(lse)


class FormB:
    """Plain definition with explicit sets, for one (sequence b) of one layer; all KV heads.

    selections[m][h] = set of pages S_m chosen at decode step m (computed here, independently of form A,
    by a stable full sort of exhaustive Eq. 1 scores on digests recomputed from the raw keys)."""

    def __init__(self, inp: wl.LayerInputs, b: int, budget_pages: int, force_last_page=True, group_reduce="sum"):
        self.inp, self.b, self.cfg = inp, b, inp.cfg
        self.budget = budget_pages
        self.force_last = force_last_page
        self.group_reduce = group_reduce
        self.selections = []   # per step: list over kv heads of python sets
        total = self.cfg.prompt_lens[b] + self.cfg.n_steps
        self.k, self.v = seq_tokens(inp, b, total)

    def scores(self, step: int, h: int):
        cfg = self.cfg
        L = cfg.prompt_lens[self.b] + step + 1
        P, G = cfg.page_size, cfg.group
        n = -(-L // P)
        q = np64(self.inp.q_all[step, self.b])             # [h_q][d]
        s = np.zeros(n)
        for j in range(n):
            keys = self.k[j * P:min((j + 1) * P, L), h, :]
            kmin, kmax = keys.min(0), keys.max(0)
            per = [sum(max(q[h * G + g, c] * kmin[c], q[h * G + g, c] * kmax[c]) for c in range(cfg.head_dim))
                   for g in range(G)]
            s[j] = sum(per) if self.group_reduce == "sum" else max(per)
        return s

    def select(self, step: int):
        cfg = self.cfg
        L = cfg.prompt_lens[self.b] + step + 1
        n = -(-L // cfg.page_size)
        k = min(self.budget, n)
        per_head = []
        for h in range(cfg.num_kv_heads):
            if k == n:
                per_head.append(set(range(n)))
                continue
            s = self.scores(step, h)
            if self.force_last and k > 0:
                order = np.argsort(-s[:n - 1], kind="stable")
                per_head.append(set(order[:k - 1].tolist()) | {n - 1})
            else:
                order = np.argsort(-s, kind="stable")
                per_head.append(set(order[:k].tolist()))
        self.selections.append(per_head)
        return per_head

    def seen(self, step_of_query: int, upto_step: int, h: int):
        u = set()
        for m in range(step_of_query, upto_step + 1):
            u |= self.selections[m][h]
        return u

    def out(self, step_of_query: int, upto_step: int):
        """out(p, m): dense attention of the query born at `step_of_query` over tokens l <= p whose page is in
        the union of the page sets loaded at steps step_of_query..upto_step.  Returns o [h_q][d], lse [h_q]."""
        cfg = self.cfg
        p = cfg.prompt_lens[self.b] + step_of_query
        q = np64(self.inp.q_all[step_of_query, self.b])
        o = np.zeros((cfg.num_q_heads, cfg.head_dim))
        lse = np.full(cfg.num_q_heads, -math.inf)
        for h in range(cfg.num_kv_heads):
            pages = self.seen(step_of_query, upto_step, h)
            mask = np.zeros(p + 1, dtype=bool)
            for j in pages:
                mask[j * cfg.page_size:min((j + 1) * cfg.page_size, p + 1)] = True
            for g in range(cfg.group):
                hq = h * cfg.group + g
                o[hq], lse[hq] = sdpa_over_tokens(q[hq], self.k[:p + 1, h], self.v[:p + 1, h], mask, cfg.sm_scale)
        return o, lse


def run_oracle_trajectory(inp: wl.LayerInputs, n_steps: int, budget_pages=None, **desc_kw):
    """Form A over the first n_steps decode steps.  Returns (layer, list of per-step result dicts with q_pos)."""
    cfg = inp.cfg
    layer = oracle_layer(inp, **desc_kw)
    budget = cfg.budget_pages if budget_pages is None else budget_pages
    layer.prefill_bounds(np.asarray(cfg.prompt_lens))
    results = []
    for s in range(n_steps):
        q_win, q_pos = wl.make_q_window(inp, s)
        seq_lens = inp.seq_lens_at(s).numpy()
        res = layer.step(np64(q_win), q_pos.numpy(), np64(inp.q_all[s]), seq_lens,
                         np.full(cfg.batch, budget, dtype=np.int32))
        res["q_pos"] = q_pos.numpy().copy()
        res["seq_lens"] = seq_lens.copy()
        results.append(res)
    return layer, results


def require_cuda():
    assert torch.cuda.is_available(), "GPU test needs a CUDA device (run through gpurun)"
