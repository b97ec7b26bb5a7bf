"""Seeded synthetic workloads for the RetroAttention decode hot path.

This module is the ONLY code shared by the CUDA path and the CPU oracle, and it
holds none of the method's arithmetic: it produces arrays (paged K/V, block
tables, queries, lengths) and nothing else.  No page bounds, scores, selections,
softmaxes or merges are computed here.

The five configurations are the ones BASELINE.json lists (C1..C5).  They are
synthetic stand-ins for the paper's latency setting (Llama-3.1-8B-shaped
attention at 32k..128k context): no item of any benchmark
dataset is used or needed.  The recipe:

  * K, V ~ N(0,1) per (sequence, token, kv head, channel); `n_outlier` channel
    indices are drawn per (layer, kv head) and K and V are multiplied by
    `outlier_scale` there (a few large-magnitude channels, as in LLM KV caches).
  * Values are drawn in fp32 and rounded ONCE to the config dtype; both sides
    consume the rounded arrays (the oracle upcasts them to fp64).
  * q for (sequence b, decode step i, q head g) = n + beta * sum of `n_planted`
    keys of its kv head at token indices drawn uniformly from [0, t] (C4: one per
    equal stratum of [0, t]), n ~ N(0,1), beta = 2.0 / n_planted: attention is
    peaked on a few pages.  q is rounded to the config dtype.
  * K/V for the WHOLE trajectory (prompt + all decode steps) are written into the
    pages up front; "appending a token" is `seq_len += 1`.
  * Physical pages are interleaved round-robin across the batch
    (phys(b, j) = j * B + b), so block-table rows are non-contiguous.
  * Slots of the last page beyond a sequence's final token hold the finite
    sentinel `PAD_VALUE`; a kernel that leaks them produces visibly wrong output.
  * Seeds: torch.Generator(device).manual_seed(base_seed + 1000*layer + b),
    base_seed = 20250801 + config index.
  * Optional "correlated" mode (`corr_rho` > 0; the default i.i.d. queries are the
    compute-worst case): every planted key persists from the previous step with probability rho and the
    noise is AR(1) with coefficient rho, which raises the adjacent-step page overlap towards what the paper
    reports on real activations (~80 %).

Generators run on whatever torch device is asked for (CPU here, CUDA on the GPU
box); parity tests copy the SAME generated arrays to the other side.
"""
from __future__ import annotations

import dataclasses
import math
from typing import Dict, List, Optional

import torch

PAD_VALUE = 3.0e4  # finite in bf16 and fp32; obviously wrong if it leaks into an output


@dataclasses.dataclass(frozen=True)
class RetroConfig:
    name: str
    index: int                 # BASELINE.json config index (1-based)
    dtype: str                 # "f32" | "bf16"
    batch: int
    num_q_heads: int
    num_kv_heads: int
    head_dim: int
    page_size: int
    prompt_lens: tuple         # per sequence
    n_steps: int               # decode steps in the full trajectory
    budget_tokens: int
    window: int                # number of PAST queries (w_build); w_paper = window + 1
    n_planted: int
    strata: bool = False       # C4: planted keys spread uniformly over the context
    n_outlier: int = 4
    outlier_scale: float = 8.0
    corr_rho: float = 0.0      # "correlated" mode: planted keys persist / noise is AR(1) with this rho

    @property
    def group(self) -> int:
        return self.num_q_heads // self.num_kv_heads

    @property
    def budget_pages(self) -> int:
        return self.budget_tokens // self.page_size

    @property
    def beta(self) -> float:
        return 2.0 / self.n_planted

    @property
    def base_seed(self) -> int:
        return 20250801 + self.index

    @property
    def max_total_len(self) -> int:
        return max(self.prompt_lens) + self.n_steps

    @property
    def max_pages_per_seq(self) -> int:
        return -(-self.max_total_len // self.page_size)

    @property
    def num_phys_pages(self) -> int:
        return self.max_pages_per_seq * self.batch

    @property
    def torch_dtype(self) -> torch.dtype:
        return torch.float32 if self.dtype == "f32" else torch.bfloat16

    @property
    def sm_scale(self) -> float:
        return 1.0 / math.sqrt(self.head_dim)

    def replace(self, **kw) -> "RetroConfig":
        return dataclasses.replace(self, **kw)


def c1() -> RetroConfig:
    """tiny fp32: B1, 4 q = 4 kv heads, d64, 512-token prompt, P16, budget 8 pages, w=4, 16 steps."""
    return RetroConfig("c1_tiny_fp32", 1, "f32", 1, 4, 4, 64, 16, (512,), 16, 8 * 16, 4,
                       n_planted=1, n_outlier=0, outlier_scale=1.0)


def c2(n_steps: int = 4096) -> RetroConfig:
    """Llama-3.1-8B-shaped bf16: B1, 32/8, d128, 32768 prompt + 4096 steps, budget 1024 tok, w=8."""
    return RetroConfig("c2_llama31_8b_32k", 2, "bf16", 1, 32, 8, 128, 16, (32768,), n_steps, 1024, 8,
                       n_planted=8)


def c3(n_steps: int = 16384) -> RetroConfig:
    """batched long generation bf16: B16, 32/8, d128, ragged ~8192 prompts growing by 16384 steps,
    budget 2048 tok, w=16.  Prompt lengths 8192 - 61*b (ragged, not page aligned; DESIGN.md reading)."""
    prompts = tuple(8192 - 61 * b for b in range(16))
    return RetroConfig("c3_batched_longgen", 3, "bf16", 16, 32, 8, 128, 16, prompts, n_steps, 2048, 16,
                       n_planted=8)


def c4(n_steps: int = 256) -> RetroConfig:
    """Qwen2.5-7B-shaped bf16: B4, 28/4 (G7), d128, 131072 context, budget 4096 tok, w=8."""
    return RetroConfig("c4_qwen25_7b_128k", 4, "bf16", 4, 28, 4, 128, 16, (131072,) * 4, n_steps, 4096, 8,
                       n_planted=16, strata=True)


def c5(window: int = 8, budget_tokens: int = 4096, n_steps: int = 256) -> RetroConfig:
    """sweep point bf16: 32768 context, B8, 32/8, d128, P16; w in {0..32} x budget in {512..8192}."""
    return RetroConfig(f"c5_sweep_w{window}_b{budget_tokens}", 5, "bf16", 8, 32, 8, 128, 16,
                       (32768,) * 8, n_steps, budget_tokens, window, n_planted=8)


C5_WINDOWS = (0, 1, 2, 4, 8, 16, 32)
C5_BUDGETS = (512, 1024, 2048, 4096, 8192)


def shrink(cfg: RetroConfig, prompt_lens, n_steps: int, **kw) -> RetroConfig:
    """Same shape family, shorter context: for CPU tests and oracle-sized parity cases."""
    return cfg.replace(prompt_lens=tuple(prompt_lens), n_steps=n_steps, **kw)


@dataclasses.dataclass
class LayerInputs:
    """Everything one attention layer's trajectory needs, as plain tensors.

    k_pages, v_pages : [num_phys][h_k][P][d]  config dtype
    block_table      : [B][max_pages] int32   logical -> physical page
    q_all            : [n_steps][B][h_q][d]   config dtype; q of decode step i (position prompt_len_b + i)
    prompt_lens      : [B] int32
    outlier_channels : [h_k][n_outlier] int64 (diagnostic only)
    """
    cfg: RetroConfig
    k_pages: torch.Tensor
    v_pages: torch.Tensor
    block_table: torch.Tensor
    q_all: torch.Tensor
    prompt_lens: torch.Tensor
    outlier_channels: torch.Tensor

    def seq_lens_at(self, step: int) -> torch.Tensor:
        """Sequence lengths while decode step `step` runs (the current token is included)."""
        return (self.prompt_lens + (step + 1)).to(torch.int32)


def _gen(device, seed: int) -> torch.Generator:
    g = torch.Generator(device=device)
    g.manual_seed(seed)
    return g


def make_layer_inputs(cfg: RetroConfig, layer: int = 0, device="cpu",
                      q_steps: Optional[int] = None) -> LayerInputs:
    """Generate one layer's K/V pages, block table and the queries of the first `q_steps` decode steps."""
    dev = torch.device(device)
    B, hq, hk, d, P = cfg.batch, cfg.num_q_heads, cfg.num_kv_heads, cfg.head_dim, cfg.page_size
    G = cfg.group
    n_q = cfg.n_steps if q_steps is None else min(q_steps, cfg.n_steps)
    maxp = cfg.max_pages_per_seq
    dt = cfg.torch_dtype

    k_pages = torch.full((cfg.num_phys_pages, hk, P, d), PAD_VALUE, dtype=dt, device=dev)
    v_pages = torch.full((cfg.num_phys_pages, hk, P, d), PAD_VALUE, dtype=dt, device=dev)
    block_table = (torch.arange(maxp, device=dev, dtype=torch.int32)[None, :] * B
                   + torch.arange(B, device=dev, dtype=torch.int32)[:, None]).contiguous()

    # outlier channels: per (layer, kv head)
    g_l = _gen(dev, cfg.base_seed + 1000 * layer + 999)
    if cfg.n_outlier > 0:
        outl = torch.stack([torch.randperm(d, generator=g_l, device=dev)[:cfg.n_outlier] for _ in range(hk)])
    else:
        outl = torch.zeros((hk, 0), dtype=torch.int64, device=dev)
    ch_scale = torch.ones((hk, d), dtype=torch.float32, device=dev)
    if cfg.n_outlier > 0:
        ch_scale.scatter_(1, outl, cfg.outlier_scale)

    q_all = torch.zeros((n_q, B, hq, d), dtype=dt, device=dev)
    for b in range(B):
        g_b = _gen(dev, cfg.base_seed + 1000 * layer + b)
        total = cfg.prompt_lens[b] + cfg.n_steps
        npg = -(-total // P)
        k_seq = (torch.randn((total, hk, d), generator=g_b, device=dev, dtype=torch.float32)
                 * ch_scale[None]).to(dt)
        v_seq = (torch.randn((total, hk, d), generator=g_b, device=dev, dtype=torch.float32)
                 * ch_scale[None]).to(dt)
        phys = block_table[b, :npg].long()
        for src, pool in ((k_seq, k_pages), (v_seq, v_pages)):
            pad = torch.full((npg * P, hk, d), PAD_VALUE, dtype=dt, device=dev)
            pad[:total] = src
            pool[phys] = pad.view(npg, P, hk, d).permute(0, 2, 1, 3)
        # queries of decode steps 0..n_q-1; step i sits at position t = prompt + i
        if n_q > 0:
            t = cfg.prompt_lens[b] + torch.arange(n_q, device=dev)                   # [n_q]
            noise = torch.randn((n_q, hq, d), generator=g_b, device=dev, dtype=torch.float32)
            u = torch.rand((n_q, hq, cfg.n_planted), generator=g_b, device=dev, dtype=torch.float64)
            span = (t + 1).to(torch.float64)[:, None, None]                           # tokens 0..t
            if cfg.strata:
                lo = torch.arange(cfg.n_planted, device=dev, dtype=torch.float64)[None, None, :]
                idx = ((lo + u) * span / cfg.n_planted).floor().long()
            else:
                idx = (u * span).floor().long()
            idx = torch.minimum(idx, t[:, None, None])                                # [n_q][hq][n_pl]
            if cfg.corr_rho > 0.0:
                # correlated mode: each planted key is kept from the previous step with probability rho (else the
                # fresh draw above), and the noise is AR(1) with coefficient rho and unit variance.  Extra draws
                # come AFTER the i.i.d. ones, so K/V and the rho = 0 queries are unchanged.
                keep = torch.rand((n_q, hq, cfg.n_planted), generator=g_b, device=dev, dtype=torch.float64) < cfg.corr_rho
                keep[0] = False
                steps_i = torch.arange(n_q, device=dev)[:, None, None].expand_as(idx)
                last_fresh = torch.cummax(torch.where(keep, torch.zeros_like(steps_i), steps_i), dim=0).values
                idx = torch.gather(idx, 0, last_fresh)                                # <= t of that earlier step <= t
                c = math.sqrt(1.0 - cfg.corr_rho ** 2)
                for i in range(1, n_q):
                    noise[i] = cfg.corr_rho * noise[i - 1] + c * noise[i]
            kv_head = (torch.arange(hq, device=dev) // G)[None, :, None].expand_as(idx)
            planted = k_seq.float()[idx, kv_head]                                     # [n_q][hq][n_pl][d]
            q_all[:, b] = (noise + cfg.beta * planted.sum(dim=2)).to(dt)
        del k_seq, v_seq
    prompt = torch.tensor(cfg.prompt_lens, dtype=torch.int32, device=dev)
    return LayerInputs(cfg, k_pages, v_pages, block_table, q_all, prompt, outl)


def window_rows(cfg: RetroConfig, step: int, b: int) -> List[int]:
    """Decode-step indices whose queries are in the window while step `step` runs (oldest first).

    Only decode-phase queries enter the window (reading Q11): at most `window` past steps."""
    first = max(0, step - cfg.window)
    return list(range(first, step + 1))


def ring_slot(cfg: RetroConfig, pos: int) -> int:
    """Row of q_win / out that holds the query at position `pos` (rows form a ring of w+1 slots)."""
    return pos % (cfg.window + 1)


def make_q_window(inp: LayerInputs, step: int):
    """q_win [B][w+1][h_q][d], q_pos [B][w+1] (int32, -1 = empty row) for decode step `step`.

    Row ring_slot(pos) holds the query at position pos; the row whose position is seq_len-1 is the
    current query.  Pure data movement (gather of already generated queries)."""
    cfg = inp.cfg
    B, W1 = cfg.batch, cfg.window + 1
    dev = inp.q_all.device
    q_win = torch.zeros((B, W1, cfg.num_q_heads, cfg.head_dim), dtype=inp.q_all.dtype, device=dev)
    q_pos = torch.full((B, W1), -1, dtype=torch.int32, device=dev)
    for b in range(B):
        for s in window_rows(cfg, step, b):
            pos = cfg.prompt_lens[b] + s
            r = ring_slot(cfg, pos)
            q_win[b, r] = inp.q_all[s, b]
            q_pos[b, r] = pos
    return q_win, q_pos


def tensor_checksum(x: torch.Tensor) -> int:
    """xor-fold of the raw bits, for logging that both sides saw the same array."""
    raw = x.contiguous().view(torch.uint8).flatten()
    pad = (-raw.numel()) % 8
    if pad:
        raw = torch.cat([raw, torch.zeros(pad, dtype=torch.uint8, device=raw.device)])
    import numpy as np
    acc = 0
    for chunk in raw.view(torch.int64).split(1 << 24):
        acc ^= int(np.bitwise_xor.reduce(chunk.cpu().numpy().view(np.uint64)))
    return acc


def drift_step(inp: LayerInputs, step: int, rel_q: float = 0.05, rel_k: float = 0.05, rel_v: float = 0.10):
    """"Drift" mode (in the full model the window tokens are re-embedded every step
    and their Q / K move by < 5 %, V by < 10 % in relative l2 between adjacent steps; Alg. 1 line 2).

    For decode step `step` returns the re-embedded tensors of the w past window tokens, seeded and deterministic:
      positions [B][w] int32   t-w .. t-1, -1 where the position is not a decode-phase token yet
      k_hat, v_hat [B][w][h_k][d], q_hat [B][w][h_q][d]   config dtype:  x_hat = x + rel * rms(x) * n,  n ~ N(0,1),
    x the token's ORIGINAL value (so the drift stays bounded over a trajectory), rms over the head vector.
    Pure data generation: nothing of the method is computed here."""
    cfg = inp.cfg
    B, w, P = cfg.batch, cfg.window, cfg.page_size
    dt = inp.k_pages.dtype
    positions = torch.full((B, max(w, 1)), -1, dtype=torch.int32)
    k_hat = torch.zeros((B, max(w, 1), cfg.num_kv_heads, cfg.head_dim), dtype=dt)
    v_hat = torch.zeros_like(k_hat)
    q_hat = torch.zeros((B, max(w, 1), cfg.num_q_heads, cfg.head_dim), dtype=dt)
    for b in range(B):
        g = _gen("cpu", cfg.base_seed + 7919 * (step + 1) + 31 * b)
        t = cfg.prompt_lens[b] + step
        for i in range(w):
            pos = t - w + i
            s_of = pos - cfg.prompt_lens[b]                 # decode step that produced this token
            if s_of < 0:
                continue
            positions[b, i] = pos
            phys = int(inp.block_table[b, pos // P])
            for src, dst, rel in ((inp.k_pages[phys, :, pos % P].float().cpu(), k_hat, rel_k),
                                  (inp.v_pages[phys, :, pos % P].float().cpu(), v_hat, rel_v),
                                  (inp.q_all[s_of, b].float().cpu(), q_hat, rel_q)):
                n = torch.randn(src.shape, generator=g, dtype=torch.float32)
                rms = src.pow(2).mean(dim=-1, keepdim=True).sqrt()
                dst[b, i] = (src + rel * rms * n).to(dt)
    return dict(positions=positions, k_hat=k_hat, v_hat=v_hat, q_hat=q_hat)
