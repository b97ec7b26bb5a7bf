"""CPU checks of the input generators (no method arithmetic lives there; these only pin their statistics)."""
import numpy as np
import torch

from paper_2508_09001_b200 import workload as wl


def test_drift_step_is_seeded_and_moves_q_k_v_by_the_stated_relative_amounts():
    """Q / K drift < 5 %, V < 10 % in relative l2 between adjacent steps; drift_step's defaults."""
    cfg = wl.shrink(wl.c2(), (100, 77), 12, batch=2)
    inp = wl.make_layer_inputs(cfg)
    a, b = wl.drift_step(inp, 9), wl.drift_step(inp, 9)
    for k in a:
        assert torch.equal(a[k], b[k])
    assert not torch.equal(a["k_hat"], wl.drift_step(inp, 10)["k_hat"])
    pos = a["positions"]
    assert pos[0].tolist() == [101, 102, 103, 104, 105, 106, 107, 108]      # t - w .. t - 1 with t = 109
    early = wl.drift_step(inp, 3)["positions"][0].tolist()
    assert early == [-1, -1, -1, -1, -1, 100, 101, 102]                    # prompt tokens are never re-embedded
    rel = {"k_hat": [], "v_hat": [], "q_hat": []}
    for bb in range(2):
        for i in range(cfg.window):
            p = int(pos[bb, i]); phys = int(inp.block_table[bb, p // 16])
            base = {"k_hat": inp.k_pages[phys, :, p % 16].float(), "v_hat": inp.v_pages[phys, :, p % 16].float(),
                    "q_hat": inp.q_all[p - cfg.prompt_lens[bb], bb].float()}
            for k in rel:
                rel[k].append(float((a[k][bb, i].float() - base[k]).norm() / base[k].norm()))
    assert 0.03 < np.mean(rel["k_hat"]) < 0.06 and 0.03 < np.mean(rel["q_hat"]) < 0.06
    assert 0.07 < np.mean(rel["v_hat"]) < 0.12
