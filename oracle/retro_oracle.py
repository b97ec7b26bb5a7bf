"""fp64 CPU oracle for one decode step of retrospective sparse attention (RetroAttention).

TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's `cpu_baseline` /
`--impl reference` legs may import this file.  The product path (paper_2508_09001_b200/) never
imports it and shares no code with it: no kernels, headers, helpers, tables or constants.

It is written from /root/reference/PAPER.md (arxiv 2508.09001) and follows the paper's order and
notation step by step (Alg. 1), in numpy fp64 with explicit loops; nothing is
blocked, fused or reordered beyond what the equations state.  The one notation change (DESIGN.md
reading Q1): `window` w here counts PAST queries, so w_paper = w + 1.

Step            | paper passage                                   | function
----------------|-------------------------------------------------|---------------------------
page digests    | Kmin/Kmax per page, PAPER.md:33 (Sec. 2.1)      | update_page_bounds
page score      | Eq. 1, PAPER.md:35-42                           | page_scores
top-k pages     | PAPER.md:42, 248, 585                           | select_pages
mask A / list M | Alg. 2; Sec. C.2 PAPER.md:448 | select_pages (epilogue)
attention       | Eq. 2 / 6 / 7; Alg.1 l.6  | sparse_attend
merge           | Eq. 8-9; Alg. 1 l.7           | merge_partials, merge_output_cache
output cache    | Sec. 2.3 push/update/pop PAPER.md:83-85; l.8    | merge_output_cache
budget policy   | relative budget 0.15, floor 256 tokens, PAPER.md:122 | budget_policy
external S_t    | Alg. 2 alone (selector-agnostic use)  | build_mask
diagnostics     | effective KV budget PAPER.md:62; suppl. attention :435-456 | step_diagnostics
KV overwrite    | Alg. 1 l.2 UpdateKV PAPER.md:391; Sec. 2.4 :87-93 | update_kv (+ update_page_bounds)

Readings of silent / garbled passages (full list with reasons in DESIGN.md "Readings"):
  Q2  GQA: per-q-head Eq. 1 scores are SUMMED over the q heads of a KV head (flag: max).
  Q3  the newest page is always selected and counts toward the budget (force_last_page=1).
  Q4  digest of a partly filled page = min/max over its valid tokens only.
  Q7  top-k ties: higher score first, then lower page index; emitted in ascending page index.
  Q9  a past query at position p skips page j iff A[j] >= p (the garbled sentence at PAPER.md:448).
  Q10 uniform rule: row at position p attends token l of selected page j iff A_prev[j] < p and
      l <= p (Alg. 2 line 1 is the special case "just-started current page" of this rule).
  Q12 the cache is a ring of w slots, slot = position mod w; the row at position t-w gets its last
      merge at step t, is returned, and its slot then takes the current row.
  Q13 the cache holds the normalised output o and the natural-log LSE (alpha = e^lse in Eq. 8-9).
Parity pins: tests/test_oracle_*.py (closed forms, brute force, hand-worked golden example,
invariants).  What no test can pin is the policy choice itself in Q2/Q3 ("parity unpinned by the
paper": the paper is silent, the reading above is the definition).

Array layouts (all float arrays fp64 here; integer arrays int32/int64):
  k_pages, v_pages [num_phys][h_k][P][d]     block_table [B][max_pages]      seq_lens [B]
  bounds           [B][h_k][max_pages][2][d]  ([..,0,:] = Kmax, [..,1,:] = Kmin)
  last_loaded (A)  [B][h_k][max_pages], -1 = never loaded during decoding
  sel_pages / sel_prev [B][h_k][k_max] (-1 beyond sel_count), sel_count [B][h_k]
  q_win [B][R][h_q][d], q_pos [B][R] (R = w+1 rows in ANY order, -1 = empty row; the row whose
  position equals seq_len-1 is the current query)
  part_o [B][R][h_q][d], part_lse [B][R][h_q]
  cache_o [B][w][h_q][d], cache_lse [B][w][h_q], cache_pos [B][w] (-1 = empty slot)
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

NEG_INF = -math.inf


@dataclasses.dataclass
class OracleDesc:
    batch: int
    num_q_heads: int
    num_kv_heads: int
    head_dim: int
    page_size: int
    max_pages_per_seq: int
    max_sel_pages: int
    window: int                 # number of PAST queries
    sm_scale: float
    group_reduce: str = "sum"   # "sum" | "max"   (reading Q2)
    force_last_page: bool = True  # reading Q3
    cache_round: str = "none"     # "none": the cached O keeps full precision (reading Q13); "bf16": it is stored in 16 bits
                                  # next to an fp32 LSE, the paper's footprint (Eq. 12) with bf16 for FP16

    @property
    def group(self) -> int:
        return self.num_q_heads // self.num_kv_heads

    @property
    def rows(self) -> int:
        return self.window + 1


# --------------------------------------------------------------------------------------------
# S1  page digests: "element-wise minima and maxima of Key vectors within a page"
# --------------------------------------------------------------------------------------------
def update_page_bounds(desc, k_pages, block_table, seq_lens, pos_begin, bounds):
    """Recompute Kmax/Kmin of every logical page touched by positions [pos_begin_b, seq_len_b).

    Only valid tokens (l < seq_len) enter a digest (reading Q4)."""
    P = desc.page_size
    for b in range(desc.batch):
        L = int(seq_lens[b])
        if L <= 0:
            continue
        first = max(0, int(pos_begin[b])) // P
        last = (L - 1) // P
        for j in range(first, last + 1):
            n_valid = min(P, L - j * P)
            phys = int(block_table[b, j])
            for h in range(desc.num_kv_heads):
                keys = k_pages[phys, h, :n_valid, :]          # [n_valid][d]
                bounds[b, h, j, 0, :] = keys.max(axis=0)       # Kmax
                bounds[b, h, j, 1, :] = keys.min(axis=0)       # Kmin
    return bounds


# --------------------------------------------------------------------------------------------
# UpdateKV (Alg. 1 line 2; Sec. 2.4): "overwrite stale KV entries" of the past
# window tokens with their re-embedded K^, V^.  The digests of the touched pages are then stale too: the caller
# refreshes them with update_page_bounds(pos_begin = oldest overwritten position).
# --------------------------------------------------------------------------------------------
def update_kv(desc, k_pages, v_pages, block_table, seq_lens, positions, k_hat, v_hat):
    """positions [B][n_upd] (-1 = skip; must be < seq_len), k_hat / v_hat [B][n_upd][h_k][d].  In place."""
    P = desc.page_size
    for b in range(desc.batch):
        for u in range(positions.shape[1]):
            pos = int(positions[b, u])
            if pos < 0 or pos >= int(seq_lens[b]):
                continue
            phys = int(block_table[b, pos // P])
            for h in range(desc.num_kv_heads):
                k_pages[phys, h, pos % P, :] = k_hat[b, u, h, :]
                v_pages[phys, h, pos % P, :] = v_hat[b, u, h, :]
    return k_pages, v_pages


# --------------------------------------------------------------------------------------------
# S2a  Eq. 1: score_j(Q) = sum_i max(Q_i Kmin_i^j, Q_i Kmax_i^j)
# --------------------------------------------------------------------------------------------
def page_scores(desc, q_cur, bounds, seq_lens):
    """Exhaustive Eq. 1 for the CURRENT query only, one score per (b, KV head, page).

    q_cur [B][h_q][d].  Returns scores [B][h_k][max_pages], -inf for pages that do not exist."""
    P, G = desc.page_size, desc.group
    scores = np.full((desc.batch, desc.num_kv_heads, desc.max_pages_per_seq), NEG_INF, dtype=np.float64)
    for b in range(desc.batch):
        n_pages = -(-int(seq_lens[b]) // P)
        for h in range(desc.num_kv_heads):
            kmax = bounds[b, h, :n_pages, 0, :]               # [n_pages][d]  (all pages j at once)
            kmin = bounds[b, h, :n_pages, 1, :]
            group_score = None
            for g in range(G):
                q = q_cur[b, h * G + g, :][None, :]
                s_g = np.sum(np.maximum(q * kmin, q * kmax), axis=1)      # Eq. 1 for q head g
                if group_score is None:
                    group_score = s_g
                elif desc.group_reduce == "sum":
                    group_score = group_score + s_g
                else:
                    group_score = np.maximum(group_score, s_g)
            scores[b, h, :n_pages] = group_score
    return scores


# --------------------------------------------------------------------------------------------
# S2b/S2c  top-k under the budget and UpdateAndBuildMask (Alg. 2)
# --------------------------------------------------------------------------------------------
def select_count(desc, seq_len, budget_pages):
    n_pages = -(-int(seq_len) // desc.page_size)
    return max(0, min(int(budget_pages), n_pages, desc.max_sel_pages)), n_pages


def select_pages(desc, scores, seq_lens, budget_pages, last_loaded):
    """S_t and the mask list M.

    S_t: k = min(budget, #pages) pages; k == #pages -> all pages; else (force_last_page) the newest
    page plus the k-1 best of the others, ordered by (score desc, index asc) (readings Q3, Q7).
    Alg. 2 lines 3-6: for p in S_t: M.append(A[p]); A[p] <- t, with t = seq_len-1 (position of the
    current query = decode step).  `last_loaded` (A) is updated in place; None iff window == 0."""
    B, hk, kmax = desc.batch, desc.num_kv_heads, desc.max_sel_pages
    sel_pages = np.full((B, hk, kmax), -1, dtype=np.int32)
    sel_prev = np.full((B, hk, kmax), -1, dtype=np.int32)
    sel_count = np.zeros((B, hk), dtype=np.int32)
    for b in range(B):
        t = int(seq_lens[b]) - 1
        k, n_pages = select_count(desc, seq_lens[b], budget_pages[b])
        for h in range(hk):
            if k == n_pages:
                chosen = list(range(n_pages))
            else:
                forced = [n_pages - 1] if (desc.force_last_page and k > 0) else []
                pool = [j for j in range(n_pages) if j not in forced]
                pool.sort(key=lambda j: (-scores[b, h, j], j))
                chosen = sorted(forced + pool[: k - len(forced)])
            sel_count[b, h] = len(chosen)
            for i, p in enumerate(chosen):
                sel_pages[b, h, i] = p
                if last_loaded is not None:
                    sel_prev[b, h, i] = last_loaded[b, h, p]   # M.append(A[p])
                    last_loaded[b, h, p] = t                   # A[p] <- t
    return sel_pages, sel_prev, sel_count


# --------------------------------------------------------------------------------------------
# NEXT-2  relative budget ("relative KV cache budget of 0.15, which dynamically changes the budget to
# context length x 0.15 as decoding continues, with the minimum budget of 256 tokens") and Alg. 2 alone for a page
# set chosen by another selector (the method is selector-agnostic).
# --------------------------------------------------------------------------------------------
def budget_policy(desc, seq_lens, ratio_permille=150, min_tokens=256):
    """budget_pages[b] = floor(max(min_tokens, floor(seq_len * ratio)) / P), at least 1 (integer arithmetic:
    the ratio is given in 1/1000 so both sides take the same integer decision)."""
    out = np.zeros(desc.batch, dtype=np.int32)
    for b in range(desc.batch):
        tokens = max(int(min_tokens), (int(seq_lens[b]) * int(ratio_permille)) // 1000)
        out[b] = max(1, tokens // desc.page_size)
    return out


def build_mask(desc, sel_pages, sel_count, seq_lens, last_loaded):
    """Alg. 2 lines 3-6 for a GIVEN S_t: M.append(A[p]); A[p] <- t.  Returns sel_prev (M)."""
    sel_prev = np.full_like(sel_pages, -1)
    for b in range(desc.batch):
        t = int(seq_lens[b]) - 1
        for h in range(desc.num_kv_heads):
            for i in range(int(sel_count[b, h])):
                p = int(sel_pages[b, h, i])
                sel_prev[b, h, i] = last_loaded[b, h, p]
                last_loaded[b, h, p] = t
    return sel_prev


def step_diagnostics(desc, sel_pages, sel_prev, sel_count, q_pos, seq_lens, part_lse, out_lse):
    """Per step and window row: supp_pages[b][h][r] = selected pages from which the row attends at least one
    token (they enlarge its effective KV budget); supp_mass[b][r][g] = e^{lse_part - lse_merged},
    the share of the merged softmax mass that this step's pages supply."""
    R = desc.window + 1
    G = desc.group
    supp_pages = np.zeros((desc.batch, desc.num_kv_heads, R), dtype=np.int32)
    supp_mass = np.zeros((desc.batch, R, desc.num_q_heads))
    for b in range(desc.batch):
        t = int(seq_lens[b]) - 1
        for r in range(R):
            p = int(q_pos[b, r])
            if p < 0 or p > t or p < t - desc.window:
                continue
            for h in range(desc.num_kv_heads):
                for i in range(int(sel_count[b, h])):
                    one = attend_token_list(desc, p, seq_lens[b], sel_pages[b, h, i:i + 1], sel_prev[b, h, i:i + 1], 1)
                    supp_pages[b, h, r] += 1 if len(one) > 0 else 0
                for g in range(h * G, (h + 1) * G):
                    if part_lse[b, r, g] > NEG_INF:
                        supp_mass[b, r, g] = math.exp(part_lse[b, r, g] - out_lse[b, r, g])
    return supp_pages, supp_mass


# --------------------------------------------------------------------------------------------
# S3  attention of every window row over the selected pages (Eq. 2 / 6 / 7; Alg. 1 line 6)
# --------------------------------------------------------------------------------------------
def attend_token_list(desc, p_row, seq_len, sel_pages_bh, sel_prev_bh, count):
    """Tokens the row at position p_row attends: l in Page_j, j in S_t, M_j < p_row, l <= p_row."""
    P = desc.page_size
    toks = []
    for i in range(int(count)):
        j = int(sel_pages_bh[i])
        if not (int(sel_prev_bh[i]) < p_row):        # page already seen by this query (reading Q9/Q10)
            continue
        for l in range(j * P, min((j + 1) * P, int(seq_len))):
            if l <= p_row:
                toks.append(l)
    return toks


def softmax_partial(q, keys, vals, sm_scale):
    """(o, lse) of softmax(q K^T * sm_scale) V over an explicit token list; empty -> (0, -inf)."""
    d = q.shape[0]
    if keys.shape[0] == 0:
        return np.zeros(d, dtype=np.float64), NEG_INF
    x = (keys @ q) * sm_scale                      # logits Q K_l^T / sqrt(d)
    m = float(np.max(x))
    e = np.exp(x - m)
    l = float(np.sum(e))
    o = (e[:, None] * vals).sum(axis=0) / l        # sum e^x V / sum e^x   (Eq. 2)
    return o, m + math.log(l)                      # lse = ln(alpha), alpha of Eq. 8


def sparse_attend(desc, q_win, q_pos, k_pages, v_pages, block_table, seq_lens,
                  sel_pages, sel_prev, sel_count):
    """O_org for the current row (all of S_t) and O_sup for each past row (unseen pages only)."""
    B, R, hq, d, P, G = desc.batch, q_win.shape[1], desc.num_q_heads, desc.head_dim, desc.page_size, desc.group
    part_o = np.zeros((B, R, hq, d), dtype=np.float64)
    part_lse = np.full((B, R, hq), NEG_INF, dtype=np.float64)
    for b in range(B):
        L = int(seq_lens[b])
        t = L - 1
        for r in range(R):
            p = int(q_pos[b, r])
            if p < 0 or p > t or p < t - desc.window:
                continue                              # empty row
            for h in range(desc.num_kv_heads):
                toks = attend_token_list(desc, p, L, sel_pages[b, h], sel_prev[b, h], sel_count[b, h])
                if toks:
                    phys = [int(block_table[b, l // P]) for l in toks]
                    offs = [l % P for l in toks]
                    keys = np.asarray(k_pages[phys, h, offs, :], dtype=np.float64)
                    vals = np.asarray(v_pages[phys, h, offs, :], dtype=np.float64)
                else:
                    keys = np.zeros((0, d)); vals = np.zeros((0, d))
                for g in range(G):
                    o, lse = softmax_partial(q_win[b, r, h * G + g], keys, vals, desc.sm_scale)
                    part_o[b, r, h * G + g] = o
                    part_lse[b, r, h * G + g] = lse
    return part_o, part_lse


# --------------------------------------------------------------------------------------------
# S4  MergeOutput (Eq. 8-9) and the output cache (Sec. 2.3; Alg. 1 lines 7-8)
# --------------------------------------------------------------------------------------------
def merge_partials(o_a, lse_a, o_b, lse_b):
    """Eq. 8: O_up = (alpha_a O_a + alpha_b O_b) / (alpha_a + alpha_b), alpha_up = alpha_a + alpha_b,
    with alpha = e^lse.  Either side empty (-inf) -> the other side unchanged."""
    if lse_a == NEG_INF:
        return np.array(o_b, dtype=np.float64), lse_b
    if lse_b == NEG_INF:
        return np.array(o_a, dtype=np.float64), lse_a
    m = max(lse_a, lse_b)
    wa, wb = math.exp(lse_a - m), math.exp(lse_b - m)
    return (wa * o_a + wb * o_b) / (wa + wb), m + math.log(wa + wb)


def round_bf16(x):
    """Round-to-nearest-even to bfloat16 (8 significant bits), returned as float64: what a 16-bit output cache stores
    (Eq. 12).  Bit arithmetic on the float32 image; values are finite."""
    f = np.asarray(x, dtype=np.float64).astype(np.float32)
    u = f.view(np.uint32).astype(np.uint64)
    u = (u + 0x7FFF + ((u >> 16) & 1)) & 0xFFFF0000
    return u.astype(np.uint32).view(np.float32).astype(np.float64)


def merge_output_cache(desc, part_o, part_lse, q_pos, seq_lens, cache_o, cache_lse, cache_pos):
    """Update: merge each past row's new partial into its cached (o, lse); Push: store the current
    row; Pop: the row at position t-w is returned after its last merge and its slot is reused.
    Returns out [B][R][h_q][d], out_lse [B][R][h_q]; cache_* updated in place (unused when w == 0)."""
    B, R, hq, d, w = desc.batch, part_o.shape[1], desc.num_q_heads, desc.head_dim, desc.window
    out = np.zeros((B, R, hq, d), dtype=np.float64)
    out_lse = np.full((B, R, hq), NEG_INF, dtype=np.float64)
    for b in range(B):
        t = int(seq_lens[b]) - 1
        new_pos = None if w == 0 else cache_pos[b].copy()
        # Update (and Pop): past rows first, so the oldest row reads its slot before the Push reuses it
        for r in range(R):
            p = int(q_pos[b, r])
            if p < 0 or p >= t or p < t - w:
                continue
            slot = p % w
            cached = int(cache_pos[b, slot]) == p        # else: nothing cached for this position
            for hh in range(hq):
                if cached:
                    o, lse = merge_partials(cache_o[b, slot, hh], float(cache_lse[b, slot, hh]),
                                            part_o[b, r, hh], float(part_lse[b, r, hh]))
                else:
                    o, lse = np.array(part_o[b, r, hh]), float(part_lse[b, r, hh])
                out[b, r, hh] = o
                out_lse[b, r, hh] = lse
                if p != t - w:                           # the oldest row is popped, not written back
                    cache_o[b, slot, hh] = round_bf16(o) if desc.cache_round == "bf16" else o
                    cache_lse[b, slot, hh] = lse
            if p != t - w:
                new_pos[slot] = p
        # Push: the current query's O_org is returned as is and stored in slot t mod w
        for r in range(R):
            if int(q_pos[b, r]) != t:
                continue
            out[b, r] = part_o[b, r]
            out_lse[b, r] = part_lse[b, r]
            if w > 0:
                cache_o[b, t % w] = round_bf16(part_o[b, r]) if desc.cache_round == "bf16" else part_o[b, r]
                cache_lse[b, t % w] = part_lse[b, r]
                new_pos[t % w] = t
        if w > 0:
            cache_pos[b] = new_pos
    return out, out_lse


# --------------------------------------------------------------------------------------------
# One layer's persistent state and one full decode step (Alg. 1 lines 3-8; line 2 is out of scope)
# --------------------------------------------------------------------------------------------
class OracleLayer:
    def __init__(self, desc: OracleDesc, k_pages, v_pages, block_table):
        self.desc = desc
        # pools may be float32 (every bf16 / fp32 input value is exact in it) to halve host memory at full
        # size; all arithmetic upcasts to float64 first (min/max digests are exact in any float type)
        self.k_pages = np.asarray(k_pages)
        self.v_pages = np.asarray(v_pages)
        self.block_table = np.asarray(block_table, dtype=np.int64)
        B, hk, hq, d, w = desc.batch, desc.num_kv_heads, desc.num_q_heads, desc.head_dim, desc.window
        self.bounds = np.zeros((B, hk, desc.max_pages_per_seq, 2, d), dtype=np.float64)
        self.last_loaded = np.full((B, hk, desc.max_pages_per_seq), -1, dtype=np.int32)
        self.cache_o = np.zeros((B, max(w, 1), hq, d), dtype=np.float64)
        self.cache_lse = np.full((B, max(w, 1), hq), NEG_INF, dtype=np.float64)
        self.cache_pos = np.full((B, max(w, 1)), -1, dtype=np.int32)

    def prefill_bounds(self, seq_lens):
        update_page_bounds(self.desc, self.k_pages, self.block_table, seq_lens,
                           np.zeros(self.desc.batch, dtype=np.int64), self.bounds)

    def step(self, q_win, q_pos, q_cur, seq_lens, budget_pages):
        """AppendKV has already made token seq_len-1 valid.  Returns a dict of every intermediate."""
        d = self.desc
        q_win = np.asarray(q_win, dtype=np.float64)
        q_cur = np.asarray(q_cur, dtype=np.float64)
        pos_begin = np.asarray(seq_lens, dtype=np.int64) - 1
        update_page_bounds(d, self.k_pages, self.block_table, seq_lens, pos_begin, self.bounds)
        scores = page_scores(d, q_cur, self.bounds, seq_lens)
        A = self.last_loaded if d.window > 0 else None
        sel_pages, sel_prev, sel_count = select_pages(d, scores, seq_lens, budget_pages, A)
        part_o, part_lse = sparse_attend(d, q_win, q_pos, self.k_pages, self.v_pages, self.block_table,
                                         seq_lens, sel_pages, sel_prev, sel_count)
        out, out_lse = merge_output_cache(d, part_o, part_lse, q_pos, seq_lens,
                                          self.cache_o, self.cache_lse, self.cache_pos)
        return dict(scores=scores, sel_pages=sel_pages, sel_prev=sel_prev, sel_count=sel_count,
                    part_o=part_o, part_lse=part_lse, out=out, out_lse=out_lse)
