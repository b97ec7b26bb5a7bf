#!/usr/bin/env python
"""bench.py — RetroAttention decode hot path on B200: us per decode step per layer, HBM GB/s, overhead vs w=0.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload c2|c5] [--layers L]

A "step" is one decode step of an L-layer stack (default L = 32, Llama-3.1-8B depth): for every layer, in
Alg. 1's order, digest refresh (S1) -> page score + top-k + mask (S2) -> fused multi-query
sparse attention (S3) -> output-cache merge (S4), all through the C ABI (`retro_decode_step`: two launches per
layer - the select kernel with S1 in line, the attend kernel with the split combine and S4 in its epilogue).  Each layer has its own K/V pool,
digests, mask and cache, so consecutive layer-steps do not share L2 (about 13 MB touched per layer-step, 430 MB
per step >> 126 MB L2).  One step is captured in a CUDA graph (every step-varying value lives in device memory)
and replayed K times between CUDA events.  Prints ONE JSON line (rank 0).

`--impl reference` times the fp64 CPU oracle (oracle/retro_oracle.py, as it stands) on the host cores on a
bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import statistics
import subprocess
import sys
import tempfile
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "retro sparse-attn us/step/layer (HBM GB/s vs ~8 TB/s; overhead vs w=0)"
UNIT = "us/step/layer"
NOMINAL_HBM_GBS = 8000.0
FALLBACK_HBM_GBS = 6650.0


def ncu_traffic(workload: str, kernel: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel` ("select" | "attend") from the committed
    `ncu --set full` capture of this workload, exported with `ncu -i <rep> --page raw --csv` to
    profiles/r02_ncu_<workload>_<kernel>.csv (the command is in profiles/r02_summary.md).  None if there is no capture."""
    import csv
    path = os.path.join(ROOT, "profiles", f"r02_ncu_{workload}_{kernel}.csv")
    if not os.path.exists(path):
        return None
    try:
        rows = list(csv.reader(open(path)))
        head = rows[0]
        ir, iw = head.index("dram__bytes_read.sum"), head.index("dram__bytes_write.sum")
        unit_r, unit_w = rows[1][ir], rows[1][iw]
        scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
        vals = [float(r[ir].replace(",", "")) * scale[unit_r] + float(r[iw].replace(",", "")) * scale[unit_w]
                for r in rows[2:] if len(r) > max(ir, iw) and r[ir]]
        return sum(vals) / len(vals) if vals else None
    except Exception:
        return None


def measured_hbm_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


CORR_RHO = 0.0                               # --corr: persistence / AR(1) coefficient of the query stream
C5_POINT = {"window": 8, "budget": 4096}     # the C5 sweep point `--workload c5` runs (see --window / --budget)


def workload_cfg(name: str, n_steps: int, window=None):
    from paper_2508_09001_b200 import workload as wl
    if name == "c2":
        cfg = wl.c2(n_steps=n_steps)
    elif name == "c3":
        cfg = wl.c3(n_steps=n_steps)
    elif name == "c4":
        cfg = wl.c4(n_steps=n_steps)
    elif name == "c5":
        cfg = wl.c5(C5_POINT["window"], C5_POINT["budget"], n_steps=n_steps)
    elif name == "c1":
        cfg = wl.c1()
    else:
        raise SystemExit(f"unknown workload {name}")
    if window is not None:
        cfg = cfg.replace(window=window, name=cfg.name + f"_w{window}")
    if CORR_RHO > 0.0:     # correlated-query mode of the workload generator, separately labelled
        cfg = cfg.replace(corr_rho=CORR_RHO, name=cfg.name + f"_corr{CORR_RHO:g}")
    return cfg


# ------------------------------------------------------------------------------------------------------
class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md clocks line)."""
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.tmp = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.proc = None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={gpu_index}", f"--query-gpu={self.FIELDS}", "--format=csv,noheader,nounits",
                 "-lms", "50"], stdout=self.tmp, stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        self.tmp.flush()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in open(self.tmp.name):
            parts = [x.strip() for x in line.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0])); mx.append(float(parts[1]))
            except ValueError:
                continue
            for n, v in zip(names, parts[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        os.unlink(self.tmp.name)
        if sm:
            out.update(sm_mhz=statistics.median(sm), sm_max_mhz=max(mx), reasons=sorted(reasons), samples=len(sm))
        return out


def time_graph(graph, iters: int):
    import torch
    start, end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    start.record()
    for _ in range(iters):
        graph.replay()
    end.record()
    torch.cuda.synchronize()
    return start.elapsed_time(end)   # ms


def replay_percentiles(graph, n_layers: int, iters: int = 48):
    """p10 / median / p90 of single graph replays (one decode step of the whole stack each), us per layer-step;
    a separate pass after the timed region (per-replay events leave gaps: the headline value is the K-step mean).
    None if anything goes wrong: this is a side figure and must never cost the bench line."""
    try:
        import torch
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(iters)]
        torch.cuda.synchronize()
        for a, b in evs:
            a.record()
            graph.replay()
            b.record()
        torch.cuda.synchronize()
        us = sorted(a.elapsed_time(b) * 1000.0 / n_layers for a, b in evs)
        pick = lambda q: us[min(len(us) - 1, int(q * len(us)))]
        return {"p10": pick(0.10), "p50": pick(0.50), "p90": pick(0.90), "replays": iters,
                "unit": UNIT, "note": "single replays timed one by one (events around each): includes the launch gap "
                                      "between replays that the K-step mean amortises"}
    except Exception:
        return None


def run_stack(cfg, n_layers, steps, warmup, seed_offset, dist_barrier, keep_inputs=False):
    """Build the layer stack, warm up, time `steps` graph replays.  Returns (stack, graph, elapsed_ms)."""
    import torch
    from paper_2508_09001_b200 import harness as hs
    pool = min(warmup + steps, 256)
    stack = hs.DecodeStack(cfg, n_layers, pool, seed_offset=seed_offset, keep_inputs=keep_inputs)
    graph = hs.capture_graph(stack.enqueue_step, warmup=1)      # 1 eager step, then capture
    for _ in range(warmup - 1):
        graph.replay()
    torch.cuda.synchronize()
    dist_barrier()
    ms = time_graph(graph, steps)
    dist_barrier()
    return stack, graph, ms


_ORACLE_JOB = {}


def _oracle_unit(args):
    """One (sequence, KV head) unit of the oracle sample, all steps (the units are independent: SURVEY 8(e))."""
    import numpy as np
    from oracle import retro_oracle as orc
    from paper_2508_09001_b200 import workload as wl
    b, h, n_steps = args
    J = _ORACLE_JOB
    cfg, G = J["cfg"], J["cfg"].group
    desc = orc.OracleDesc(batch=1, num_q_heads=G, num_kv_heads=1, head_dim=cfg.head_dim, page_size=cfg.page_size,
                          max_pages_per_seq=cfg.max_pages_per_seq, max_sel_pages=max(1, cfg.budget_pages),
                          window=cfg.window, sm_scale=cfg.sm_scale)
    layer = orc.OracleLayer(desc, J["k"][:, h:h + 1], J["v"][:, h:h + 1], J["bt"][b:b + 1])
    layer.prefill_bounds(np.asarray(cfg.prompt_lens[b:b + 1]))
    budget = np.full(1, cfg.budget_pages, dtype=np.int32)
    q_all = J["q"]
    t0 = time.perf_counter()
    for s in range(n_steps):
        q_win = np.zeros((1, cfg.window + 1, G, cfg.head_dim))
        q_pos = np.full((1, cfg.window + 1), -1, dtype=np.int32)
        for ss in wl.window_rows(cfg, s, b):
            pos = cfg.prompt_lens[b] + ss
            q_win[0, wl.ring_slot(cfg, pos)] = q_all[ss, b, h * G:(h + 1) * G]
            q_pos[0, wl.ring_slot(cfg, pos)] = pos
        layer.step(q_win, q_pos, q_all[s, b:b + 1, h * G:(h + 1) * G], np.asarray([cfg.prompt_lens[b] + s + 1]), budget)
    return time.perf_counter() - t0


def oracle_sample(cfg, inp, n_steps: int, procs: int = 1):
    """Time the oracle, as it stands, on `n_steps` decode steps of one layer (digest prefill included in the
    multi-process figure, untimed in the single-thread one).  procs > 1: the (sequence, KV head) units are spread
    over `procs` forked worker processes (numpy only), wall clock of the whole pool.  Returns (us per layer-step,
    cores used)."""
    import numpy as np
    from oracle import retro_oracle as orc
    from paper_2508_09001_b200 import workload as wl
    try:
        from threadpoolctl import threadpool_limits
    except Exception:
        threadpool_limits = None
    if procs > 1:
        import multiprocessing as mp
        units = [(b, h, n_steps) for b in range(cfg.batch) for h in range(cfg.num_kv_heads)]
        procs = min(procs, len(units))
        _ORACLE_JOB.update(cfg=cfg, k=inp.k_pages.float().cpu().numpy(), v=inp.v_pages.float().cpu().numpy(),
                           bt=inp.block_table.cpu().numpy(), q=inp.q_all.double().cpu().numpy())
        ctx = mp.get_context("fork")
        t0 = time.perf_counter()
        with ctx.Pool(procs) as pool:
            pool.map(_oracle_unit, units, chunksize=1)
        sec = time.perf_counter() - t0
        _ORACLE_JOB.clear()
        return sec / n_steps * 1e6, procs
    desc = orc.OracleDesc(batch=cfg.batch, num_q_heads=cfg.num_q_heads, num_kv_heads=cfg.num_kv_heads,
                          head_dim=cfg.head_dim, page_size=cfg.page_size, max_pages_per_seq=cfg.max_pages_per_seq,
                          max_sel_pages=max(1, cfg.budget_pages), window=cfg.window, sm_scale=cfg.sm_scale)
    layer = orc.OracleLayer(desc, inp.k_pages.float().cpu().numpy(), inp.v_pages.float().cpu().numpy(),
                            inp.block_table.cpu().numpy())
    layer.prefill_bounds(np.asarray(cfg.prompt_lens))
    budget = np.full(cfg.batch, cfg.budget_pages, dtype=np.int32)
    q_all = inp.q_all.double().cpu()

    def run():
        t0 = time.perf_counter()
        for s in range(n_steps):
            q_win = np.zeros((cfg.batch, cfg.window + 1, cfg.num_q_heads, cfg.head_dim))
            q_pos = np.full((cfg.batch, cfg.window + 1), -1, dtype=np.int32)
            for b in range(cfg.batch):
                for ss in wl.window_rows(cfg, s, b):
                    pos = cfg.prompt_lens[b] + ss
                    q_win[b, wl.ring_slot(cfg, pos)] = q_all[ss, b].numpy()
                    q_pos[b, wl.ring_slot(cfg, pos)] = pos
            layer.step(q_win, q_pos, q_all[s].numpy(), inp.seq_lens_at(s).cpu().numpy(), budget)
        return time.perf_counter() - t0

    if threadpool_limits is not None:
        with threadpool_limits(limits=1):
            sec = run()
    else:
        sec = run()
    return sec / n_steps * 1e6, 1   # us per layer-step


def run_reference(args):
    """--impl reference: the oracle on the host cores, bounded sample, same metric / config / unit.  A "step" of this
    arm is ONE decode step of ONE layer (what is actually timed; the line says so): steps = the sampled decode steps,
    layers_per_step = 1, ms_per_step = one layer-step."""
    ri_rank = int(os.environ.get("RANK", 0))
    if ri_rank != 0:
        return 0
    from paper_2508_09001_b200 import workload as wl
    n_sample = max(1, min(args.steps, 6))
    n_warm = max(0, min(args.warmup, 2))
    cfg = workload_cfg(args.workload, n_steps=n_sample + 2)
    inp = wl.make_layer_inputs(cfg, layer=0, device="cpu", q_steps=n_sample + 2)
    if n_warm:
        oracle_sample(cfg, inp, n_warm)                   # warm-up (numpy import, page cache)
    us, _ = oracle_sample(cfg, inp, n_sample)
    ncpu = os.cpu_count() or 1
    us_all, cores_all = oracle_sample(cfg, inp, n_sample, procs=ncpu) if ncpu > 1 else (us, 1)
    sample = (f"{n_sample} decode steps of 1 layer from the start of decoding (window ramp-up), 1 thread; all-cores: "
              f"{us_all:.0f} us/step/layer on {cores_all} processes over the (sequence, KV head) units, host has {ncpu} cpus")
    line = {
        "impl": "reference", "metric": METRIC, "value": us, "unit": UNIT, "n_gpus": args.gpus, "steps": n_sample,
        "warmup": n_warm, "ms_per_step": us / 1000.0, "higher_is_better": False,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": config_dict(cfg, 1),
        "cpu_baseline": {"value": us, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample,
                         "all_cores": {"value": us_all, "cores": cores_all}},
        "e2e": {"value": us, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
        "note": "steps / warmup / ms_per_step describe what this arm timed: single decode steps of ONE layer "
                f"(requested --steps {args.steps} --warmup {args.warmup}; the sample is bounded)",
    }
    print(json.dumps(line))
    return 0


def config_dict(cfg, n_layers):
    return {"workload": cfg.name, "batch": cfg.batch, "num_q_heads": cfg.num_q_heads,
            "num_kv_heads": cfg.num_kv_heads, "head_dim": cfg.head_dim, "page_size": cfg.page_size,
            "context": max(cfg.prompt_lens), "budget_tokens": cfg.budget_tokens, "window": cfg.window,
            "layers_per_step": n_layers, "query_correlation_rho": cfg.corr_rho,
            "l2": "inputs larger than L2: each layer-step reads its own layer's digests+pages; "
                  f"{n_layers} independent layer states per step"}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=256)
    ap.add_argument("--warmup", type=int, default=16)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c2")
    ap.add_argument("--layers", type=int, default=32)
    ap.add_argument("--no-extras", action="store_true", help="skip w=0 overhead run, stage timing, e2e, cpu baseline")
    ap.add_argument("--oracle-steps", type=int, default=8)
    ap.add_argument("--window", type=int, default=None, help="C5 sweep: retro window w (past queries)")
    ap.add_argument("--budget", type=int, default=None, help="C5 sweep: budget in tokens")
    ap.add_argument("--corr", type=float, default=0.0,
                    help="correlated-query mode: planted keys persist / noise is AR(1) with this rho (default: i.i.d.)")
    ap.add_argument("--no-w0", action="store_true", help="skip the w=0 overhead run (sweeps measure w=0 themselves)")
    ap.add_argument("--lite", action="store_true", help="sweep point: stage timing only (no e2e, cpu baseline, w=0 run)")
    args = ap.parse_args()
    global CORR_RHO
    CORR_RHO = args.corr
    if args.window is not None:
        C5_POINT["window"] = args.window
    if args.budget is not None:
        C5_POINT["budget"] = args.budget
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist
    from paper_2508_09001_b200 import binding as rb
    from paper_2508_09001_b200 import harness as hs

    ri = hs.rank_info()
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(ri.local_rank)
    dev = torch.device("cuda", ri.local_rank)
    if ri.world_size > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if ri.world_size > 1:
            dist.barrier()
        torch.cuda.synchronize()

    warmup = max(args.warmup, 3)
    steps, L = args.steps, args.layers
    w_full = None
    cfg = workload_cfg(args.workload, n_steps=warmup + steps + 160)
    warmup = max(warmup, cfg.window + 2)       # the retro window is full during the timed region
    cfg = workload_cfg(args.workload, n_steps=warmup + steps + 160)
    seed_off = hs.rank_layer_seed_offset(ri.rank)

    sampler = ClockSampler(ri.local_rank) if ri.rank == 0 else None
    stack, graph, ms = run_stack(cfg, L, steps, warmup, seed_off, barrier, keep_inputs=True)
    clocks = sampler.stop() if sampler is not None else None
    ms = hs.max_over_ranks(ms, dev)
    us_layer = ms * 1000.0 / (steps * L)
    # the graph really advanced every layer
    expect = [p + warmup + steps for p in cfg.prompt_lens]
    assert stack.seq_lens_host() == expect, (stack.seq_lens_host(), expect)
    assert torch.isfinite(stack.layers[-1].out.float()).all()

    seq_now = stack.seq_lens_host()
    workload_stats = selection_stats(stack.layers[0], cfg)
    if workload_stats is not None and not args.no_extras and not args.lite:
        workload_stats["device_counters"] = retro_diagnostics(cfg, seed_off)
    bytes_model = hs.stage_bytes(cfg, seq_now)
    peak, peak_src = measured_hbm_peak()
    line = {
        "metric": METRIC, "value": us_layer, "unit": UNIT, "n_gpus": ri.world_size, "steps": steps, "warmup": warmup,
        "ms_per_step": ms / steps, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
        "dtype": cfg.dtype, "data": "synthetic", "config": config_dict(cfg, L), "impl": "ours",
        "gpu_launches": steps * (L * stack.launches_per_layer_step() + hs.KERNELS_PER_STEP),
        "launches_per_layer_step": stack.launches_per_layer_step(),
        "aggregate_layer_steps_per_s": ri.world_size * steps * L / (ms / 1000.0),
        "path_hbm": {"algorithmic_bytes_per_layer_step": bytes_model["total"],
                     "achieved_gbs": bytes_model["total"] / (us_layer * 1e-6) / 1e9,
                     "frac_of_measured": bytes_model["total"] / (us_layer * 1e-6) / 1e9 / peak,
                     "frac_of_nominal_8TBs": bytes_model["total"] / (us_layer * 1e-6) / 1e9 / NOMINAL_HBM_GBS},
        "clocks": clocks, "workload_stats": workload_stats,
    }

    if not args.no_extras:
        line["step_percentiles"] = replay_percentiles(graph, L)
        # ---- device time of the step's OWN kernels (retro_decode_step_part: the select kernel with S1 in line, the
        # attend kernel with the split combine and S4 in its epilogue), each as a CUDA graph of L back-to-back
        # launches (one per layer, different layer state) between CUDA events, from the state the timed steps left
        def time_part(fn):
            g = hs.capture_graph(fn, warmup=1)
            for _ in range(3):
                g.replay()
            it = 20
            return hs.max_over_ranks(time_graph(g, it), dev) * 1000.0 / (it * L)
        # (the attend kernel first: it must see the mask state A / sel_prev the real steps left; replaying the select
        # kernel at a frozen length would mark every selected page as seen by everybody)
        t_att = time_part(lambda: stack.enqueue_step_part(1))
        step_k = {"select_step": time_part(lambda: stack.enqueue_step_part(0)), "attend_step": t_att}
        sb = dict(bytes_model)
        sb["select"] = bytes_model["score"] + bytes_model["topk"]
        dom = max(step_k, key=lambda k: step_k[k])
        ach = sb[dom] / (step_k[dom] * 1e-6) / 1e9
        wl_key = args.workload if (args.window is None and args.budget is None and args.corr == 0.0) else None
        line["step_kernels_us"] = step_k
        line["step_kernels_note"] = ("the kernels retro_decode_step launches per layer, each timed alone (L launches back to "
                                     "back): select_step = S1 of the newest page + page score + top-k + Alg. 2; attend_step = "
                                     "fused multi-query sparse attention + split combine + output-cache merge")
        line["roofline"] = {"bound": "hbm", "kernel": dom, "achieved": ach, "peak": peak, "unit": "GB/s",
                            "frac": ach / peak,
                            "traffic": ncu_traffic(wl_key, dom.split("_")[0]) if wl_key else None,
                            "peak_source": peak_src,
                            "algorithmic_bytes_per_launch": sb[dom], "launch_us": step_k[dom],
                            "frac_of_nominal_8TBs": ach / NOMINAL_HBM_GBS}
        line["step_kernel_rooflines"] = {k: {"achieved_gbs": sb[k] / (step_k[k] * 1e-6) / 1e9,
                                             "frac": sb[k] / (step_k[k] * 1e-6) / 1e9 / peak,
                                             "frac_of_nominal_8TBs": sb[k] / (step_k[k] * 1e-6) / 1e9 / NOMINAL_HBM_GBS,
                                             "algorithmic_bytes_per_launch": sb[k], "launch_us": step_k[k],
                                             "traffic": ncu_traffic(wl_key, k.split("_")[0]) if wl_key else None}
                                         for k in step_k}
        line["attend_arith_intensity_flop_per_byte"] = hs.attend_flops(cfg, seq_now) / bytes_model["kv"]
        # the same counting only the (row, page) pairs the retrospective mask leaves: every pair of the
        # current query's G rows plus the unmasked share of the past rows' pairs (layer 0, last timed step)
        f_unmasked = (workload_stats or {}).get("unmasked_past_row_page_pairs")
        if f_unmasked is not None:
            line["attend_arith_intensity_unmasked_flop_per_byte"] = (
                line["attend_arith_intensity_flop_per_byte"] * (1.0 + cfg.window * f_unmasked) / (cfg.window + 1))
        # ---- the four stand-alone C-ABI entry points (S1, S2, S3, S4 launched alone), for reference ----
        # (they run after the select replays above: their mask state is "every selected page seen", i.e. the
        # stand-alone attend entry point is timed on the current row's work only; the step-kernel figures above are
        # the representative ones)
        stages = {}
        for st in ("bounds", "select", "attend", "merge"):
            stages[st] = time_part(lambda st=st: stack.enqueue_stage(st))
        line["stages_us"] = stages
        line["stages_note"] = ("each stage = its stand-alone C-ABI call launched alone, L times back to back; the step itself "
                               "runs the two kernels of step_kernels_us")
        line["stage_rooflines"] = {k: {"achieved_gbs": sb[k] / (stages[k] * 1e-6) / 1e9,
                                       "frac": sb[k] / (stages[k] * 1e-6) / 1e9 / peak,
                                       "algorithmic_bytes_per_launch": sb[k], "launch_us": stages[k]} for k in stages}
        if args.lite:
            line["e2e"] = None
            if ri.rank == 0:
                print(json.dumps(line))
            return 0
        # ---- end to end through the C ABI with HOST buffers (H2D of the step's inputs, D2H of its result) ----
        e2e_steps = min(steps, 32)
        e2e = run_e2e(stack, cfg, e2e_steps, dev)
        e2e_ms = hs.max_over_ranks(e2e["ms"], dev)
        line["e2e"] = {"value": e2e_ms * 1000.0 / (e2e_steps * L), "unit": UNIT,
                       "h2d_bytes_per_step": e2e["h2d"], "d2h_bytes_per_step": e2e["d2h"], "steps": e2e_steps,
                       "note": "retro_decode_steps_host: one pinned-host copy of all layers' new-token q/k/v in, per layer "
                               "window advance + AppendKV + the step's kernels, one copy of out[L][B][w+1][h_q][d] back "
                               "to pinned host memory; captured once into a CUDA graph, inputs refilled on the CPU and "
                               "the stream synchronised every step; wall clock (host) time"}

        # ---- CPU baseline: the oracle on this box's cores, bounded sample (rank 0, N = 1 only) ----
        if ri.rank == 0 and ri.world_size == 1:
            inp0 = stack.inputs[0]
            n_or = args.oracle_steps
            us_cpu, _ = oracle_sample(cfg, inp0, n_or)
            ncpu = os.cpu_count() or 1
            us_all, cores_all = oracle_sample(cfg, inp0, n_or, procs=ncpu) if ncpu > 1 else (us_cpu, 1)
            line["cpu_baseline"] = {"value": us_cpu, "unit": UNIT, "cores": 1, "kind": "oracle",
                                    "sample": f"{n_or} decode steps of layer 0 from the start of decoding, 1 thread "
                                              f"(host has {ncpu} cpus)",
                                    "all_cores": {"value": us_all, "cores": cores_all,
                                                  "how": "the same sample, (sequence, KV head) units spread over forked "
                                                         "worker processes, wall clock incl. the digest prefill"}}
        # ---- overhead vs w = 0 at the same budget (plain Quest through the same kernels) ----
        del graph
        stack_inputs_free(stack)
        del stack
        torch.cuda.empty_cache()
        # ---- bandwidth point: the same attend kernel where the step is large enough to be HBM-bound rather than
        # launch/latency-bound (C5 sweep point B8, 32k context, budget 8192 tokens, w = 8; 4 layers) ----
        if ri.rank == 0 and ri.world_size == 1 and args.workload == "c2" and args.window is None:
            line["bandwidth_point"] = bandwidth_point(peak, dev)
        if cfg.window > 0 and not args.no_w0:
            cfg0 = workload_cfg(args.workload, n_steps=warmup + steps + 160, window=0)
            stack0, graph0, ms0 = run_stack(cfg0, L, steps, warmup, seed_off, barrier)
            ms0 = hs.max_over_ranks(ms0, dev)
            us0 = ms0 * 1000.0 / (steps * L)
            line["w0_us_per_layer_step"] = us0
            line["overhead_vs_w0"] = us_layer / us0 - 1.0
            del graph0, stack0
            torch.cuda.empty_cache()
        # ---- single layer, hot L2 (SURVEY 8(d) "also report the single-layer hot-L2 number, labelled"): the same
        # step with ONE layer state, so that layer's digests and recurring pages stay in the 126 MB L2 from step to
        # step.  A side figure: never the headline, and never allowed to cost the bench line.
        if ri.world_size == 1:
            try:
                stack1, graph1, ms1 = run_stack(cfg, 1, steps, warmup, seed_off, barrier)
                line["single_layer_hot_l2"] = {
                    "value": ms1 * 1000.0 / steps, "unit": UNIT, "layers_per_step": 1,
                    "note": "one layer state replayed every step: its digests and the pages that stay selected are "
                            "L2 hits; NOT comparable with `value` (32 layer states, inputs larger than L2)"}
                del graph1, stack1
            except Exception as ex:      # noqa: BLE001
                line["single_layer_hot_l2"] = {"value": None, "error": repr(ex)[:200]}
    else:
        line["e2e"] = None

    if ri.rank == 0:
        print(json.dumps(line))
    if ri.world_size > 1:
        dist.destroy_process_group()
    return 0


def selection_stats(buf, cfg):
    """Statistics of the synthetic workload from layer 0's last step (host-side torch ops on the kernel's
    outputs; nothing of the method is computed here): how many selected pages were also selected at the previous
    step (the paper reports ~83 % on real activations) and which fraction of (past row, selected
    page) pairs is unmasked, i.e. supplementary work of the retro rows."""
    import torch
    if cfg.window == 0:
        return None
    cnt = buf.sel_count.cpu()
    prev = buf.sel_prev.cpu()
    qpos = buf.q_pos.cpu()
    seq = buf.seq_lens.cpu()
    tot = ov = pairs = unmasked = 0
    for b in range(cfg.batch):
        t = int(seq[b]) - 1
        past = [int(p) for p in qpos[b].tolist() if 0 <= p < t]
        for h in range(cfg.num_kv_heads):
            pv = prev[b, h, :int(cnt[b, h])]
            tot += pv.numel()
            ov += int((pv == t - 1).sum())
            for p in past:
                pairs += pv.numel()
                unmasked += int((pv < p).sum())
    return {"adjacent_step_page_overlap": ov / max(tot, 1), "unmasked_past_row_page_pairs": unmasked / max(pairs, 1)}


def retro_diagnostics(cfg, seed_offset, n_steps=48):
    """Device-side counters of the retrospective rows (retro_step_diagnostics) over `n_steps` decode
    steps of ONE layer driven through the stand-alone entry points (not timed): the effective KV budget a query
    ends up with, relative to its own budget, and the softmax mass the retro updates add per step."""
    import torch
    from paper_2508_09001_b200 import binding as rb
    from paper_2508_09001_b200 import harness as hs
    if cfg.window == 0:
        return None
    stack = hs.DecodeStack(cfg, 1, n_steps, seed_offset=seed_offset)
    d, buf = stack.desc, stack.layers[0]
    B, hk, hq, R = cfg.batch, cfg.num_kv_heads, cfg.num_q_heads, cfg.window + 1
    supp_pages = torch.zeros((B, hk, R), dtype=torch.int32, device=stack.device)
    supp_mass = torch.zeros((B, R, hq), dtype=torch.float32, device=stack.device)
    pages_acc = torch.zeros((), dtype=torch.float64, device=stack.device)
    mass_acc = torch.zeros((), dtype=torch.float64, device=stack.device)
    mass_n = 0
    counted = 0
    for s in range(n_steps):
        rb.retro_window_advance_layers(d, stack.advance_table, 1, stack.pool_steps)
        for stage in ("bounds", "select", "attend"):
            stack.enqueue_stage(stage)
        rb.retro_merge_output_cache(d, buf.part_o, buf.part_lse, buf.q_pos, buf.seq_lens, buf.cache_o, buf.cache_lse,
                                    buf.cache_pos, buf.out, buf.out_lse)
        rb.retro_step_diagnostics(d, buf.sel_pages, buf.sel_prev, buf.sel_count, buf.q_pos, buf.seq_lens,
                                  buf.part_lse, buf.out_lse, supp_pages, supp_mass)
        if s > cfg.window:                            # window full: every step carries w past rows
            past = (buf.q_pos >= 0) & (buf.q_pos < (buf.seq_lens - 1)[:, None])          # [B][R]
            pages_acc += supp_pages.double().sum()
            mass_acc += (supp_mass.double() * past[:, :, None]).sum()
            mass_n += int(past.sum()) * hq
            counted += 1
    torch.cuda.synchronize()
    k = min(cfg.budget_pages, -(-min(cfg.prompt_lens) // cfg.page_size))
    per_unit_step = float(pages_acc) / max(counted * B * hk, 1)     # = pages one query sees over its window life
    return {"effective_budget_pages_per_query": per_unit_step, "own_budget_pages": k,
            "effective_budget_ratio": per_unit_step / k,
            "supplementary_mass_per_past_row_step": float(mass_acc) / max(mass_n, 1), "steps": counted}


def bandwidth_point(peak, dev):
    """Stage timing of the attend kernel on the C5 point (w = 8, budget 8192 tokens), 4 layers, CUDA events."""
    import torch
    from paper_2508_09001_b200 import harness as hs
    from paper_2508_09001_b200 import workload as wl
    cfg = wl.c5(8, 8192, n_steps=64)
    n_l = 4
    stack = hs.DecodeStack(cfg, n_l, 32)
    for _ in range(cfg.window + 4):          # fill the retro window; leaves valid selections for the stage replay
        stack.enqueue_step()
    torch.cuda.synchronize()
    g = hs.capture_graph(lambda: stack.enqueue_stage("attend"), warmup=1)
    for _ in range(3):
        g.replay()
    it = 20
    us = time_graph(g, it) * 1000.0 / (it * n_l)
    nbytes = hs.stage_bytes(cfg, stack.seq_lens_host())["attend"]
    out = {"workload": cfg.name, "kernel": "attend", "bound": "hbm", "launch_us": us,
           "algorithmic_bytes_per_launch": nbytes, "achieved": nbytes / (us * 1e-6) / 1e9, "peak": peak, "unit": "GB/s",
           "frac": nbytes / (us * 1e-6) / 1e9 / peak,
           "frac_of_nominal_8TBs": nbytes / (us * 1e-6) / 1e9 / NOMINAL_HBM_GBS,
           "l2": "4 layers x 268 MB of selected pages, one launch per layer: every launch reads from HBM"}
    del g, stack
    torch.cuda.empty_cache()
    return out


def stack_inputs_free(stack):
    stack.inputs.clear()


def run_e2e(stack, cfg, n_steps, dev):
    """End to end through retro_decode_steps_host with HOST buffers: per step ONE host->device copy of every layer's
    packed new token [q | k | v] from a pinned buffer, then per layer window advance + AppendKV and the step's
    kernels, then ONE device->host copy of out[L][B][w+1][h_q][d].  The call is captured once into a CUDA graph (the
    C ABI is graph-capturable; the pinned host addresses are baked in), each timed step refills the pinned input
    buffer on the CPU, replays the graph and synchronises: the results are on the host when the step ends."""
    import torch
    from paper_2508_09001_b200 import binding as rb
    d = stack.desc
    B, hq, hk, D, w = cfg.batch, cfg.num_q_heads, cfg.num_kv_heads, cfg.head_dim, cfg.window
    dt = cfg.torch_dtype
    P = cfg.page_size
    L = len(stack.layers)
    seq0 = stack.seq_lens_host()
    n_q, n_kv = B * hq * D, B * hk * D
    tok = n_q + 2 * n_kv
    # host copies of every layer's next n_steps tokens (q from the pool, k/v rows from the trajectory), unpinned
    feed = torch.empty((n_steps + 1, L, tok), dtype=dt)
    for l, buf in enumerate(stack.layers):
        inp = stack.inputs[l]
        ctr = int(stack.counters[l].item())
        for s in range(n_steps + 1):
            feed[s, l, :n_q] = stack.q_pools[l][(ctr + s) % stack.pool_steps].reshape(-1).cpu()
            for b in range(B):
                pos = seq0[b] + s
                phys = int(inp.block_table[b, pos // P])
                feed[s, l, n_q + b * hk * D:n_q + (b + 1) * hk * D] = inp.k_pages[phys, :, pos % P].reshape(-1).cpu()
                feed[s, l, n_q + n_kv + b * hk * D:n_q + n_kv + (b + 1) * hk * D] = inp.v_pages[phys, :, pos % P].reshape(-1).cpu()
    h_in = torch.empty((L, tok), dtype=dt).pin_memory()            # refilled before every step
    h_out = torch.empty((L, B, w + 1, hq, D), dtype=dt).pin_memory()
    d_in = torch.empty((L, tok), dtype=dt, device=dev)
    d_out = torch.empty((L, B, w + 1, hq, D), dtype=dt, device=dev)
    ios = [rb.RetroStepIO(d_in[l].data_ptr(), buf.q_win.data_ptr(), buf.q_pos.data_ptr(), d_out[l].data_ptr())
           for l, buf in enumerate(stack.layers)]
    states = [buf.state for buf in stack.layers]

    def enqueue():
        rb.retro_decode_steps_host(d, states, ios, h_in, h_out)

    from paper_2508_09001_b200 import harness as hs
    h_in.copy_(feed[0])
    graph = hs.capture_graph(enqueue, warmup=1)                    # (the eager warm-up call consumed step 0)
    torch.cuda.synchronize()
    esz = 2 if cfg.dtype == "bf16" else 4
    h2d = L * tok * esz
    d2h = L * B * (w + 1) * hq * D * esz
    t0 = time.perf_counter()
    start, end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    start.record()
    for s in range(1, n_steps + 1):
        h_in.copy_(feed[s])                                        # this step's inputs arrive in host memory
        graph.replay()
        torch.cuda.current_stream().synchronize()                  # the step's results are on the host
    end.record()
    torch.cuda.synchronize()
    wall_ms = (time.perf_counter() - t0) * 1000.0
    assert torch.isfinite(h_out.float()).all()
    return {"ms": max(start.elapsed_time(end), wall_ms), "h2d": h2d, "d2h": d2h}


if __name__ == "__main__":
    sys.exit(main())
