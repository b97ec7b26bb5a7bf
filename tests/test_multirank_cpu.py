"""World-size-2 gloo test of the N>1 plumbing bench.py uses: the path shards over independent sequences with no
data-path collective, so the only cross-rank logic is seed/shard assignment and the MAX-over-ranks timing."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2508_09001_b200 import harness as hs
from paper_2508_09001_b200 import workload as wl


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ri = hs.rank_info()
    assert (ri.rank, ri.world_size) == (rank, world)
    elapsed = 10.0 + 5.0 * rank                       # rank 1 is the slow one
    mx = hs.max_over_ranks(elapsed, "cpu")
    sm = hs.sum_over_ranks(1.0, "cpu")
    # each rank generates ITS OWN replica batch: disjoint seeds, no exchange
    cfg = wl.shrink(wl.c2(), (40,), 2, num_q_heads=4, num_kv_heads=2, head_dim=16)
    inp = wl.make_layer_inputs(cfg, layer=hs.rank_layer_seed_offset(rank))
    out[rank] = (mx, sm, float(inp.k_pages.float().sum()))
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_gloo_max_timing_and_disjoint_shards():
    port = _free_port()
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(2, port, out), nprocs=2, join=True)
    assert out[0][0] == out[1][0] == 15.0             # MAX over ranks, identical on both
    assert out[0][1] == out[1][1] == 2.0
    assert out[0][2] != out[1][2]                      # different data per rank (weak scaling replicas)


def test_single_process_is_identity():
    assert hs.max_over_ranks(3.5, "cpu") == 3.5


def test_byte_model_reduces_to_paper_terms():
    """Eq. 3/4: KV term = 4 k h_k P d bytes in 16-bit, q term = 2 w_p h_q d; ratio vs Quest ~ 1."""
    cfg = wl.c2()
    sb = hs.stage_bytes(cfg, [32768 + 100])
    k, hk, hq, P, d, wp = 64, 8, 32, 16, 128, cfg.window + 1
    assert sb["kv"] == 4 * k * hk * P * d
    q_bytes = 2 * wp * hq * d
    ours = q_bytes + sb["kv"] + 4 * hk * k
    quest = 2 * hq * d + sb["kv"]
    assert 1.0 < ours / quest < 1.02                   # "the ratio stays near 1"
    ai = hs.attend_flops(cfg, [32768 + 100]) / sb["kv"]
    assert ai == wp * hq / hk                          # Eq. 3 simplifies to w h_q / h_k
