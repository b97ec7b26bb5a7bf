"""Synthetic decode harness around the C ABI: L independent attention-layer states stepped in sequence,
the algorithmic byte/flop model of each stage, and the rank plumbing for `bench.py --gpus N`.

Nothing of the method is computed here: every stage of the path runs in libretro's kernels; this module
allocates (torch), enqueues the C-ABI calls in Alg. 1's order and counts bytes."""
from __future__ import annotations

import dataclasses
import os
from typing import Dict, List, Optional

import torch

from . import binding as rb
from . import workload as wl

KERNELS_PER_STEP = 1         # window_advance_layers: every layer's query stream advances in one launch


# ----------------------------------------------------------------------------------------------------
# algorithmic bytes / flops per layer-step (Eq. 3/4, 11-13 terms)
# ----------------------------------------------------------------------------------------------------
def esize(cfg: wl.RetroConfig) -> int:
    return 2 if cfg.dtype == "bf16" else 4


def stage_bytes(cfg: wl.RetroConfig, seq_lens: List[int]) -> Dict[str, float]:
    """Bytes the METHOD must move per layer-step, per stage (what the roofline is judged on).

    digests: n_pages * 2d * e per (b, KV head)           (read by the score stage)
    KV     : k * P * d * 2 * e per (b, KV head)          (read by the attend stage; Eq. 3 term 2)
    q/out  : (w+1) * h_q * d * e per sequence each       (Eq. 3 terms 1 and 4)
    mask   : 16 B per selected page (A gather/scatter, sel_pages, sel_prev; Eq. 3 term 3 is 4 B)
    cache  : 2 * w * h_q * (d+1) * 4 (read + write) + push h_q * (d+1) * 4   (Eq. 12 footprint, moved once)
    """
    e = esize(cfg)
    hq, hk, d, P, w = cfg.num_q_heads, cfg.num_kv_heads, cfg.head_dim, cfg.page_size, cfg.window
    digests = kv = mask = 0.0
    for L in seq_lens:
        n_pages = -(-L // P)
        k = min(cfg.budget_pages, n_pages)
        digests += hk * n_pages * 2 * d * e
        kv += hk * k * P * d * 2 * e
        mask += hk * k * 16
    B = len(seq_lens)
    q = B * (w + 1) * hq * d * e
    part = B * (w + 1) * hq * (d + 1) * 4
    cache = B * (2 * w * hq * (d + 1) * 4 + (hq * (d + 1) * 4 if w > 0 else 0))
    bounds = B * hk * (P * d * e + 2 * d * e)
    return {
        # the two kernels of retro_decode_step: select (S1 of the newest page + S2a-c), attend (S3 + S4)
        "select_step": digests + B * hq * d * e + mask + bounds,
        "attend_step": kv + q + part + mask / 2 + cache + q,
        "bounds": bounds,                                            # newest page in, one record out
        "score": digests + B * hq * d * e + B * hk * (-(-max(seq_lens) // P)) * 8,
        "topk": mask + B * hk * (-(-max(seq_lens) // P)) * 8,
        "attend": kv + q + part + mask / 2,
        "merge": part + cache + q,                                   # q-sized `out` write
        "total": digests + kv + mask + 2 * q + cache,
        "kv": kv, "digests": digests,
    }


def attend_flops(cfg: wl.RetroConfig, seq_lens: List[int]) -> float:
    """Dense rows x keys block: 4 * rows * P * d per (selected page, KV head)."""
    rows = cfg.group * (cfg.window + 1)
    tot = 0.0
    for L in seq_lens:
        k = min(cfg.budget_pages, -(-L // cfg.page_size))
        tot += cfg.num_kv_heads * k * 4.0 * rows * cfg.page_size * cfg.head_dim
    return tot


# ----------------------------------------------------------------------------------------------------
# rank plumbing (one process per GPU; the path shards over sequences with no collective)
# ----------------------------------------------------------------------------------------------------
@dataclasses.dataclass
class RankInfo:
    rank: int
    local_rank: int
    world_size: int


def rank_info() -> RankInfo:
    return RankInfo(int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)),
                    int(os.environ.get("WORLD_SIZE", 1)))


def rank_layer_seed_offset(rank: int) -> int:
    """Each rank owns an independent replica batch (weak scaling): its layers use disjoint seeds."""
    return 100 * rank


def max_over_ranks(value: float, device) -> float:
    """MAX over ranks of a per-rank elapsed time (torch.distributed, any backend); identity when not initialised."""
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, device) -> float:
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


# ----------------------------------------------------------------------------------------------------
# L independent layer states stepped in Alg. 1's order
# ----------------------------------------------------------------------------------------------------
class DecodeStack:
    """`n_layers` attention layers, each with its own K/V pool, digests, mask A, output cache and query
    stream, as in an n_layers-deep model (per-step working sets of different layers do not share L2)."""

    def __init__(self, cfg: wl.RetroConfig, n_layers: int, q_pool_steps: int, device="cuda", seed_offset: int = 0,
                 keep_inputs: bool = False):
        self.cfg, self.n_layers, self.pool_steps = cfg, n_layers, q_pool_steps
        self.device = torch.device(device)
        self.desc = rb.make_desc(cfg.batch, cfg.num_q_heads, cfg.num_kv_heads, cfg.head_dim, cfg.page_size,
                                 cfg.max_pages_per_seq, max(1, cfg.budget_pages), cfg.num_phys_pages, cfg.window,
                                 cfg.dtype, sm_scale=cfg.sm_scale)
        self.layers: List[rb.LayerBuffers] = []
        self.q_pools: List[torch.Tensor] = []
        self.counters: List[torch.Tensor] = []
        self.inputs: List[wl.LayerInputs] = []
        for l in range(n_layers):
            inp = wl.make_layer_inputs(cfg, layer=l + seed_offset, device=self.device, q_steps=q_pool_steps)
            seq_lens = inp.prompt_lens.clone()
            budget = torch.full((cfg.batch,), cfg.budget_pages, dtype=torch.int32, device=self.device)
            buf = rb.LayerBuffers(self.desc, inp.k_pages, inp.v_pages, inp.block_table, seq_lens, budget, self.device)
            buf.rebuild_bounds()
            self.layers.append(buf)
            self.q_pools.append(inp.q_all.contiguous())
            self.counters.append(torch.zeros(1, dtype=torch.int32, device=self.device))
            if keep_inputs:
                self.inputs.append(inp)
        # device table of retro_advance_rec_t records (q_pool, step_counter, seq_lens, q_win, q_pos, q_cur_out)
        self.advance_table = torch.tensor(
            [[pool.data_ptr(), ctr.data_ptr(), buf.seq_lens.data_ptr(), buf.q_win.data_ptr(), buf.q_pos.data_ptr(),
              buf.q_cur.data_ptr()] for buf, pool, ctr in zip(self.layers, self.q_pools, self.counters)],
            dtype=torch.int64, device=self.device)
        torch.cuda.synchronize(self.device)

    def launches_per_layer_step(self) -> int:
        """Kernels retro_decode_step enqueues per layer: select (S1 + S2) and attend (S3 + S4), or three where the
        cache merge is its own launch (fp32 / more than 128 query rows per KV head)."""
        return rb.retro_launches_per_step(self.desc)

    def enqueue_step_part(self, part: int, stream=None):
        """ONE of the step's kernels for every layer back to back (part 0: select, part 1: attend + merge), exactly
        as retro_decode_step launches them (per-kernel timing of the real step; state stays valid for timing)."""
        d = self.desc
        for buf in self.layers:
            rb.retro_decode_step_part(d, buf.state, buf.q_win, buf.q_pos, buf.q_cur, buf.out, part, None, stream)

    def enqueue_step(self, stream=None):
        """One decode step: advance every layer's synthetic query stream (one launch: the stand-in for the QKV
        projections that feed this path), then S1..S4 layer by layer."""
        d = self.desc
        rb.retro_window_advance_layers(d, self.advance_table, self.n_layers, self.pool_steps, stream)
        for buf in self.layers:
            rb.retro_decode_step(d, buf.state, buf.q_win, buf.q_pos, buf.q_cur, buf.out, None, stream)

    def enqueue_stage(self, stage: str, stream=None):
        """One stage of every layer back to back (per-kernel timing; state stays valid for timing purposes)."""
        d = self.desc
        for buf in self.layers:
            if stage == "bounds":
                rb.retro_update_page_bounds(d, buf.k_pages, buf.block_table, buf.seq_lens, None, 1, buf.bounds, stream)
            elif stage == "select":
                la = buf.last_loaded if d.window > 0 else None
                rb.retro_select_pages(d, buf.q_cur, buf.bounds, buf.seq_lens, buf.budget_pages, la, buf.sel_pages,
                                      buf.sel_prev, buf.sel_count, None, buf.workspace, stream)
            elif stage == "attend":
                rb.retro_sparse_attend(d, buf.q_win, buf.q_pos, buf.k_pages, buf.v_pages, buf.block_table,
                                       buf.seq_lens, buf.sel_pages, buf.sel_prev, buf.sel_count, buf.part_o,
                                       buf.part_lse, buf.workspace, stream)
            elif stage == "merge":
                w = d.window > 0
                rb.retro_merge_output_cache(d, buf.part_o, buf.part_lse, buf.q_pos, buf.seq_lens,
                                            buf.cache_o if w else None, buf.cache_lse if w else None,
                                            buf.cache_pos if w else None, buf.out, None, stream)
            else:
                raise ValueError(stage)

    def seq_lens_host(self) -> List[int]:
        return self.layers[0].seq_lens.cpu().tolist()


def capture_graph(fn, warmup: int = 1) -> torch.cuda.CUDAGraph:
    """Capture fn() (which enqueues libretro launches on the current stream) into a CUDA graph."""
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        for _ in range(warmup):
            fn()
    torch.cuda.current_stream().wait_stream(s)
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        fn()
    return g
