"""CPU check of the arithmetic the tensor-core attend kernel's tolerance rests on (DESIGN.md sections 7 and 9.4,
attend_umma.cu header).

The kernel departs from "softmax in fp64" in five places: (1) the reference m_ref of a row is LAZY - it is set by the
row's first visible block and raised only when a logit exceeds it by more than 64 (log2 units), so P = 2^(s - m_ref)
ranges up to 2^64; (2) P reaches the tensor core as a bf16 hi + bf16 lo pair; (3) O and the row sums L are fp32;
(4) the normalised partial of a KV split crosses the cluster as an fp16 tile with a base-2 lse; (5) the splits are
combined with weights 2^(lse_s - max) in fp32.  This test restates that ORDER OF OPERATIONS (not the kernel's code)
in numpy float32 with torch's bf16 / fp16 rounding, and compares with the plain definition - softmax(q K^T * scale) V
over the visible keys, in fp64 - on inputs chosen to stress each place: logits that climb just under the rescale
threshold block after block, logits that collapse after the first block, rows whose first visible key sits in a late
block, x8 outlier channels, |v| in the hundreds, thousands of equal logits.  The bar is the bf16 tolerance of the GPU
parity tests (BASELINE.json north_star: atol 2e-2, rtol 1e-2).  No GPU, no oracle: a design claim pinned by
arithmetic.  Tensor-core accumulation is modelled as one fp32 rounding per MMA K step (16 channels or 16 keys)."""
import numpy as np
import pytest
import torch

F32 = np.float32
ATOL, RTOL = 2e-2, 1e-2            # gpu_harness.TOL["bf16"]
THRESH = F32(64.0)                 # kRescaleThreshold
MREF_INIT = F32(-1.0e30)           # kMrefInit
LOG2E = 1.4426950408889634
LN2 = 0.6931471805599453


def _bf16(x):
    return torch.from_numpy(np.ascontiguousarray(x, dtype=np.float32)).to(torch.bfloat16).float().numpy()


def _fp16(x):
    return torch.from_numpy(np.ascontiguousarray(x, dtype=np.float32)).to(torch.float16).float().numpy()


def _exp2_ftz(d):
    with np.errstate(over="ignore", under="ignore"):
        e = np.exp2(d.astype(np.float64)).astype(np.float32)
    e[np.abs(e) < np.finfo(np.float32).tiny] = 0.0      # ex2.approx.ftz
    return e


def _mma_f32(acc, a, b):
    """acc + a @ b with the exact product sum of one K step rounded once into the fp32 accumulator."""
    return (acc.astype(np.float64) + a.astype(np.float64) @ b.astype(np.float64)).astype(np.float32)


def _split_partial(q, k, v, vis, scale_log2):
    """One KV split: blocks of 128 keys.  q [R][128], k / v [n][128] (bf16 values), vis [R][n].
    Returns (o fp16-rounded [R][128], lse2 [R]) or lse2 = -inf for a row that saw nothing."""
    R, n = vis.shape
    mref = np.full(R, MREF_INIT, np.float32)
    L = np.zeros((R, 128), np.float32)                    # per key-thread share of the row sum
    Oh = np.zeros((R, 128), np.float32)
    Ol = np.zeros((R, 128), np.float32)
    for b0 in range(0, n, 128):
        kb, vb, mb = k[b0:b0 + 128], v[b0:b0 + 128], vis[:, b0:b0 + 128]
        nk = kb.shape[0]
        S = np.zeros((R, nk), np.float32)
        for c0 in range(0, 128, 16):                      # S^T = K Q^T: 8 K steps of 16 channels
            S = _mma_f32(S, q[:, c0:c0 + 16], kb[:, c0:c0 + 16].T)
        with np.errstate(over="ignore", invalid="ignore"):
            d = (S.astype(np.float64) * float(scale_log2) - mref[:, None].astype(np.float64)).astype(np.float32)  # fmaf
        d = np.where(mb, d, -np.inf).astype(np.float32)
        if (d > THRESH).any():                            # slow path for the whole block
            xs = np.where(mb, (S * F32(scale_log2)).astype(np.float32), -np.inf).astype(np.float32)
            bm = xs.max(axis=1)
            nw = np.maximum(mref, bm)
            alpha = _exp2_ftz((mref - nw).astype(np.float32))
            mref = nw
            with np.errstate(invalid="ignore"):
                d = (xs - mref[:, None]).astype(np.float32)
            d = np.where(mb, d, -np.inf).astype(np.float32)
            L = (L * alpha[:, None]).astype(np.float32)
            Oh = (Oh * alpha[:, None]).astype(np.float32)
            Ol = (Ol * alpha[:, None]).astype(np.float32)
        e = _exp2_ftz(d)
        assert np.isfinite(e).all() and e.max(initial=0.0) <= 2.0 ** 64 * 1.0001
        L[:, :nk] = (L[:, :nk] + e).astype(np.float32)    # one key per softmax thread
        hi = _bf16(e)
        lo = _bf16((e - hi).astype(np.float32))
        for p0 in range(0, nk, 16):                       # O^T += V^T [P_hi | P_lo]: one page (16 keys) per K step
            Oh = _mma_f32(Oh, hi[:, p0:p0 + 16], vb[p0:p0 + 16])
            Ol = _mma_f32(Ol, lo[:, p0:p0 + 16], vb[p0:p0 + 16])
    Lr = L.copy()
    for s in (64, 32, 16, 8, 4, 2, 1):                    # shuffle tree + shared-memory adds, fp32
        Lr = (Lr[:, :s] + Lr[:, s:2 * s]).astype(np.float32)
    Lr = Lr[:, 0]
    live = Lr > 0
    with np.errstate(divide="ignore", invalid="ignore"):
        inv = (F32(1.0) / Lr).astype(np.float32)
        o = np.where(live[:, None], ((Oh + Ol).astype(np.float32) * inv[:, None]).astype(np.float32), 0.0)
        lse2 = np.where(live, (mref + np.log2(Lr.astype(np.float64)).astype(np.float32)).astype(np.float32), -np.inf)
    return _fp16(o), lse2.astype(np.float32)


def kernel_model(q, k, v, vis, sm_scale, pages_per_split):
    """part_o [R][128], part_lse [R] (natural log) as the kernel's order of operations gives them."""
    scale_log2 = F32(F32(sm_scale) * F32(LOG2E))
    n = k.shape[0]
    step = pages_per_split * 16
    parts = [_split_partial(q, k[s0:s0 + step], v[s0:s0 + step], vis[:, s0:s0 + step], scale_log2)
             for s0 in range(0, n, step)]
    o_s = np.stack([p[0] for p in parts])                 # [S][R][128]
    l_s = np.stack([p[1] for p in parts])                 # [S][R]
    mx = l_s.max(axis=0)
    with np.errstate(invalid="ignore"):
        wgt = np.where(np.isfinite(l_s), _exp2_ftz((l_s - mx[None]).astype(np.float32)), 0.0).astype(np.float32)
    o = np.zeros(o_s.shape[1:], np.float32)
    wsum = np.zeros(o_s.shape[1], np.float32)
    for s in range(o_s.shape[0]):
        use = wgt[s] > 0
        wsum = np.where(use, (wsum + wgt[s]).astype(np.float32), wsum)
        fm = (wgt[s][:, None].astype(np.float64) * o_s[s].astype(np.float64) + o.astype(np.float64)).astype(np.float32)
        o = np.where(use[:, None], fm, o)
    live = wsum > 0
    with np.errstate(divide="ignore", invalid="ignore"):
        o = np.where(live[:, None], (o * (F32(1.0) / wsum)[:, None]).astype(np.float32), 0.0)
        lse = np.where(live, ((mx + np.log2(wsum.astype(np.float64)).astype(np.float32)) * F32(LN2)).astype(np.float32),
                       -np.inf)
    return o.astype(np.float32), lse.astype(np.float32)


def definition(q, k, v, vis, sm_scale):
    """softmax(q K^T * scale) V over the visible keys, fp64 (Eq. 2 / 6)."""
    s = (q.astype(np.float64) @ k.astype(np.float64).T) * float(F32(sm_scale))
    s = np.where(vis, s, -np.inf)
    m = s.max(axis=1, keepdims=True)
    m = np.where(np.isfinite(m), m, 0.0)
    e = np.exp(s - m)
    l = e.sum(axis=1)
    with np.errstate(divide="ignore", invalid="ignore"):
        o = np.where(l[:, None] > 0, (e @ v.astype(np.float64)) / l[:, None], 0.0)
        lse = np.where(l > 0, m[:, 0] + np.log(l), -np.inf)
    return o, lse


def _check(q, k, v, vis, sm_scale, pps, what):
    o, lse = kernel_model(q, k, v, vis, sm_scale, pps)
    o_ref, lse_ref = definition(q, k, v, vis, sm_scale)
    assert np.array_equal(np.isfinite(lse), np.isfinite(lse_ref)), what
    err_o = np.abs(o - o_ref)
    assert np.all(err_o <= ATOL + RTOL * np.abs(o_ref)), (what, float(err_o.max()))
    fin = np.isfinite(lse_ref)
    err_l = np.abs(lse[fin] - lse_ref[fin])
    assert np.all(err_l <= ATOL + RTOL * np.abs(lse_ref[fin])), (what, float(err_l.max(initial=0.0)))
    return float(err_o.max()), float(err_l.max(initial=0.0))


def _kv(rng, n, vscale=1.0, outliers=True):
    k = rng.standard_normal((n, 128))
    v = rng.standard_normal((n, 128)) * vscale
    if outliers:
        ch = rng.choice(128, 4, replace=False)
        k[:, ch] *= 8
        v[:, ch] *= 8
    return _bf16(k), _bf16(v)


def _causal_page_mask(rng, R, n, frac_seen=0.4):
    """Rows = G x window ranks: a later rank sees fewer pages (already seen ones are masked) and a causal cut."""
    vis = np.ones((R, n), dtype=bool)
    for r in range(4, R):
        seen = rng.random(n // 16) < frac_seen
        vis[r] &= ~np.repeat(seen, 16)
        vis[r, n - 1 - (r // 4):] = False
    return vis


@pytest.mark.parametrize("pps", [8, 24, 64])
def test_workload_like_inputs_stay_inside_the_bf16_tolerance(pps):
    rng = np.random.default_rng(509001 + pps)
    n, R = 1024, 36                                     # budget 1024 tokens, G = 4, w = 8
    k, v = _kv(rng, n)
    q = rng.standard_normal((R, 128))
    for r in range(R):                                  # planted alignment: peaked attention
        q[r] += 2.0 * k[rng.integers(n)]
    q = _bf16(q)
    vis = _causal_page_mask(rng, R, n)
    err_o, err_l = _check(q, k, v, vis, 1.0 / np.sqrt(128.0), pps, f"workload pps={pps}")
    assert err_o < 1.5e-2, err_o                        # DESIGN.md 9.4 reports 7.7e-3 against the oracle on the GPU


def test_logits_climbing_just_under_the_rescale_threshold():
    """Every block's best logit beats the previous block's by ~60 log2 units: no block may rescale on its own, P
    reaches ~2^60 .. 2^64 and the early blocks' mass is dwarfed - or the slow path fires; either way the result holds."""
    rng = np.random.default_rng(11)
    n, R = 768, 16
    k, v = _kv(rng, n, outliers=False)
    base = _bf16(rng.standard_normal(128))
    base /= np.linalg.norm(base)
    q = _bf16(np.tile(base, (R, 1)) * 8.0)
    sm = 1.0 / np.sqrt(128.0)
    for blk in range(n // 128):                         # plant one key per block with a prescribed logit
        want_log2 = 10.0 + 60.0 * blk
        j = blk * 128 + int(rng.integers(128))
        k[j] = _bf16(base * (want_log2 / (LOG2E * sm * 8.0)))
    vis = np.ones((R, n), dtype=bool)
    _check(q, k, v, vis, sm, 48, "climbing, one split")
    _check(q, k, v, vis, sm, 16, "climbing, three splits")


def test_logits_collapsing_after_the_first_block_and_late_starting_rows():
    rng = np.random.default_rng(12)
    n, R = 640, 20
    k, v = _kv(rng, n, vscale=3.0)
    q = _bf16(rng.standard_normal((R, 128)) * 2.0)
    k[:128] = _bf16(k[:128] * 6.0)                      # block 0 dominates by hundreds of log2 units for most rows
    vis = np.ones((R, n), dtype=bool)
    vis[10:, :400] = False                              # these rows start in block 3 (mid-block: key 400 = 3 * 128 + 16)
    vis[15:, :] = False
    vis[15:, 639] = True                                # a single visible key: o = v exactly (up to fp16)
    vis[19, :] = False                                  # an empty row: o = 0, lse = -inf
    _check(q, k, v, vis, 1.0 / np.sqrt(128.0), 40, "collapse one split")
    _check(q, k, v, vis, 1.0 / np.sqrt(128.0), 8, "collapse five splits")
    o, lse = kernel_model(q, k, v, vis, 1.0 / np.sqrt(128.0), 8)
    assert np.all(o[19] == 0) and np.isneginf(lse[19])
    assert np.allclose(o[15], v[639], rtol=2.0 ** -10, atol=0)   # fp16 staging: 11 significant bits


def test_large_values_and_thousands_of_equal_logits():
    rng = np.random.default_rng(13)
    n, R = 4096, 8
    k = np.zeros((n, 128), np.float32)                  # all logits equal: uniform attention, L = 4096 exactly
    v = _bf16(rng.standard_normal((n, 128)) * 300.0)    # |v| in the hundreds (the fp16 tile holds up to 65504)
    q = _bf16(rng.standard_normal((R, 128)))
    vis = np.ones((R, n), dtype=bool)
    err_o, err_l = _check(q, k, v, vis, 1.0 / np.sqrt(128.0), 64, "uniform")
    o, lse = kernel_model(q, k, v, vis, 1.0 / np.sqrt(128.0), 64)
    assert np.allclose(lse, np.log(4096.0), atol=1e-5)
    assert err_l < 1e-5


def test_single_bf16_p_would_lose_the_precision_the_pair_keeps():
    """The reason P is a hi + lo pair: with hi alone the rounding error of P (2^-9 relative) survives into O; with
    the pair it drops to the fp32 / fp16 level.  Spread attention over outlier-channel values shows the gap."""
    rng = np.random.default_rng(14)
    n = 512
    k, v = _kv(rng, n)
    q = _bf16(rng.standard_normal((4, 128)) * 0.3)
    s = (q.astype(np.float64) @ k.astype(np.float64).T) / np.sqrt(128.0)
    e = np.exp2((s - s.max(axis=1, keepdims=True)) * LOG2E).astype(np.float32)
    hi = _bf16(e)
    lo = _bf16((e - hi).astype(np.float32))
    exact = e.astype(np.float64) @ v.astype(np.float64)
    err_hi = np.abs(hi.astype(np.float64) @ v.astype(np.float64) - exact).max()
    err_pair = np.abs((hi.astype(np.float64) + lo.astype(np.float64)) @ v.astype(np.float64) - exact).max()
    assert err_pair < err_hi * 2.0 ** -6, (err_pair, err_hi)
