"""CPU check of the error bound the select kernel's exactness rests on (select.cu header).

The kernel ranks pages on fp32 scores and proves its selection exact from |s32_j - s_j| <= eps_j = 2^-20 A_j with
A_j = sum_c |q_c| |K_jc| accumulated next to the score; pages the bound cannot decide are re-scored in fp64.  If the
bound were wrong for the kernel's summation order, a near-tie could be mis-ranked silently.  This test restates that
ORDER (not the kernel's code) in numpy float32 - per lane a chain of fused multiply-adds over its 16 bytes of the
digest record, then a balanced tree over the 32 lanes (strides 16, 8, 4, 2, 1), the same for A_j, eps = A32 * 9.5463e-7
in fp32 - and compares with the exact fp64 score on adversarial digests: heavy cancellation (score ~ 0 at large A_j),
x8 outlier channels, extreme scales, every group size.  fp32 FMA is emulated as round32(a * b + c) in fp64 (the product
of two fp32 values is exact in fp64).  No GPU, no oracle: a design claim pinned by arithmetic."""
import numpy as np
import pytest
import torch

F32 = np.float32
EPS_FACTOR = F32(9.5463e-7)      # 2^-20 (1 + 2^-10), the constant in select.cu


def _bf16(x):
    return torch.from_numpy(np.asarray(x, dtype=np.float32)).to(torch.bfloat16).float().numpy()


def _fma32(a, b, c):
    return (a.astype(np.float64) * b.astype(np.float64) + c.astype(np.float64)).astype(np.float32)


def _tree32(x):
    for s in (16, 8, 4, 2, 1):
        x = (x[:, :s] + x[:, s:2 * s]).astype(np.float32)
    return x[:, 0]


def _model(rec, qcat, vals_per_lane):
    """rec [n][32 * vals_per_lane] (Kmax ; Kmin) as stored, qcat [same] = [sum_g q+ ; sum_g q-] in fp64.
    Returns (s32, eps32, s64, A64)."""
    n = rec.shape[0]
    s64 = (rec.astype(np.float64) * qcat[None, :]).sum(1)
    a64 = (np.abs(rec.astype(np.float64)) * np.abs(qcat)[None, :]).sum(1)
    q32 = qcat.astype(np.float32).reshape(32, vals_per_lane)          # one rounding of q, inside eps
    r = rec.astype(np.float32).reshape(n, 32, vals_per_lane)
    acc = np.zeros((n, 32), np.float32)
    aab = np.zeros((n, 32), np.float32)
    for c in range(vals_per_lane):
        acc = _fma32(np.broadcast_to(q32[:, c], (n, 32)), r[:, :, c], acc)
        aab = _fma32(np.broadcast_to(np.abs(q32[:, c]), (n, 32)), np.abs(r[:, :, c]), aab)
    return _tree32(acc), (_tree32(aab) * EPS_FACTOR).astype(np.float32), s64, a64


def _digests(rng, n, d, kscale, mode, rnd):
    base = rng.standard_normal((n, d)) * kscale
    spread = np.abs(rng.standard_normal((n, d))) * kscale
    kmax, kmin = rnd(base + spread), rnd(base - spread)
    ch = rng.choice(d, 4, replace=False)
    if mode == "outlier":
        kmax[:, ch] = rnd(kmax[:, ch] * 8)
        kmin[:, ch] = rnd(kmin[:, ch] * 8)
    if mode == "cancel":             # Kmin mirrors Kmax: the two halves of the dot product cancel almost exactly
        kmin = -kmax[:, ::-1].copy()
    return kmax, kmin, ch


@pytest.mark.parametrize("dtype", ["bf16", "f32"])
@pytest.mark.parametrize("mode", ["plain", "outlier", "cancel"])
def test_fp32_score_error_stays_inside_the_kernels_bound(dtype, mode):
    rng = np.random.default_rng(20250801 + len(mode))
    d, vals = (128, 8) if dtype == "bf16" else (64, 4)
    rnd = _bf16 if dtype == "bf16" else (lambda x: np.asarray(x, dtype=np.float32))
    worst = 0.0
    for G in (1, 4, 7, 8):
        for qscale, kscale in ((1.0, 1.0), (1e-3, 1e3), (30.0, 1e-2), (1e4, 1e4)):
            q = rnd(rng.standard_normal((G, d)) * qscale)
            kmax, kmin, ch = _digests(rng, 4000, d, kscale, mode, rnd)
            if mode == "outlier":
                q[:, ch] = rnd(q[:, ch] * 8)
            qcat = np.concatenate([np.maximum(q.astype(np.float64), 0).sum(0),
                                   np.minimum(q.astype(np.float64), 0).sum(0)])
            s32, eps, s64, a64 = _model(np.concatenate([kmax, kmin], axis=1), qcat, vals)
            err = np.abs(s32.astype(np.float64) - s64)
            assert np.all(err <= eps.astype(np.float64)), (dtype, mode, G, qscale, kscale)
            worst = max(worst, float((err / np.maximum(eps, 1e-300)).max()))
            # the bound is not vacuous either: eps is within a factor of the true magnitude sum
            assert np.all(eps.astype(np.float64) <= 2.0 ** -19 * a64 + 1e-300)
    # 14 roundings of <= 2^-24 A_j each against a bound of 2^-20 A_j: the observed error sits far inside
    assert worst < 0.5, worst


def test_all_zero_query_gives_zero_bound_and_exact_ties():
    """q = 0: every score and every eps is exactly 0, so T - U = 0 is not > 2 eps and the kernel must take the exact
    (fp64, ties to the lower index) route - the comparison is strict for that reason."""
    rng = np.random.default_rng(7)
    kmax, kmin, _ = _digests(rng, 64, 128, 1.0, "plain", _bf16)
    s32, eps, s64, _ = _model(np.concatenate([kmax, kmin], axis=1), np.zeros(256), 8)
    assert np.all(s32 == 0) and np.all(eps == 0) and np.all(s64 == 0)
    assert not (0.0 - 0.0 > 2.0 * 0.0)
