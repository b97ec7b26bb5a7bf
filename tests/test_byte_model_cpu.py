"""The roofline numerators (harness.stage_bytes / attend_flops) against SURVEY.md 8(d)'s per-config table and its
per-unit formulas: digests n_pages 2 d e, KV k P d 2 e, mask ~16 k per (sequence, KV head); q and out (w+1) h_q d e,
cache 2 w h_q (d+1) 4 + push h_q (d+1) 4 per sequence.  CPU only; no method arithmetic."""
import pytest

from paper_2508_09001_b200 import harness as hs
from paper_2508_09001_b200 import workload as wl

MB = 1e6


def _by_hand(cfg, seq_lens):
    e = 2 if cfg.dtype == "bf16" else 4
    hq, hk, d, P, w = cfg.num_q_heads, cfg.num_kv_heads, cfg.head_dim, cfg.page_size, cfg.window
    tot = 0
    for L in seq_lens:
        n = -(-L // P)
        k = min(cfg.budget_tokens // P, n)
        tot += hk * (n * 2 * d * e + k * P * d * 2 * e + 16 * k)
        tot += 2 * (w + 1) * hq * d * e + 2 * w * hq * (d + 1) * 4 + (hq * (d + 1) * 4 if w else 0)
    return tot


@pytest.mark.parametrize("name,cfg,seq_lens,lo,hi", [
    # (low, high) MB per layer-step: the "Per layer-step algorithmic bytes" column of SURVEY.md 8(d)
    ("c2 start", wl.c2(), [32768 + 1], 13.0, 14.0),
    ("c2 end", wl.c2(), [32768 + 4096], 13.0, 14.6),
    ("c3 start", wl.c3(), [8192 - 61 * b + 1 for b in range(16)], 175.0, 190.0),
    ("c3 end", wl.c3(), [8192 - 61 * b + 16384 for b in range(16)], 240.0, 260.0),
    ("c4", wl.c4(), [131072 + 1] * 4, 100.0, 106.0),
    ("c5 smallest", wl.c5(0, 512), [32768 + 1] * 8, 83.0, 87.0),
    ("c5 largest", wl.c5(32, 8192), [32768 + 1] * 8, 340.0, 360.0),
])
def test_total_bytes_match_the_survey_table(name, cfg, seq_lens, lo, hi):
    sb = hs.stage_bytes(cfg, seq_lens)
    assert sb["total"] == _by_hand(cfg, seq_lens), name
    assert lo * MB <= sb["total"] <= hi * MB, (name, sb["total"] / MB)
    # the two step kernels together move the path's bytes plus what the split between them adds: the fp32 partial
    # rows (written by S3, Eq. 7) and the newest page's digest refresh
    extra = sb["select_step"] + sb["attend_step"] - sb["total"]
    assert 0 <= extra <= 0.08 * sb["total"], (name, extra / MB)


def test_arithmetic_intensity_is_rows_flop_per_kv_byte():
    """Eq. 3: 4 rows P d flop per page of 2 P d e bytes = rows flop / byte in bf16."""
    for cfg in (wl.c2(), wl.c3(), wl.c4(), wl.c5(32, 4096), wl.c5(0, 512)):
        L = [max(cfg.prompt_lens) + 1] * cfg.batch
        ai = hs.attend_flops(cfg, L) / hs.stage_bytes(cfg, L)["kv"]
        assert ai == cfg.group * (cfg.window + 1)
