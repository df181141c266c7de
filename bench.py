#!/usr/bin/env python
"""bench.py -- sparse-prefill layer throughput on B200 (BASELINE.json metric), one JSON line on stdout.

A "step" is one pass of the whole hot path (sp_prefill_layer: projection -> scoring (+block max) ->
causal top-k -> gather-sparse GQA attention) over one batch of synthetic input of BASELINE.json's
config 3 (L=32768, Hq=32, Hkv=8, d=128, d_idx=128, k=2048, b_sel=64) -- the 32K / k=2048 configuration
the metric is quoted on (`--workload c5` runs the 128K one).  `value` = tokens/s with inputs resident
in HBM; `e2e` = the same through sp_prefill_layer_host with pinned HOST buffers (copies inside the
timed region).  The dense GQA layer of the same library is timed in the same run.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c3|c5|c2|c1|c4] [--impl reference]
  (--workload c4 prints the oracle-vs-indexer length sweep of BASELINE.json configs[3]: overlap + stage split)

N > 1 (torchrun): the path does not shard (one GPU per layer call, no collectives) -> N independent
replicas, value = N * L / max-over-ranks time ("replicas only").
"""
from __future__ import annotations

import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "sparse_prefill_layer_tokens_per_s"
UNIT = "tokens/s"


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        return dict(hbm=p["hbm_gbs"], tensor_burst=p["bf16_tflops"], tensor=p.get("bf16_tflops_sustained", p["bf16_tflops"]),
                    source="measured")
    return dict(hbm=6650.0, tensor_burst=1590.0, tensor=1400.0, source="fallback")


class ClockSampler(threading.Thread):
    """Samples nvidia-smi clocks / throttle reasons every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        super().__init__(daemon=True)
        self.gpu = gpu_index
        self.samples = []
        self._halt = threading.Event()

    def run(self):
        while not self._halt.is_set():
            try:
                out = subprocess.run(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                      "-i", str(self.gpu)], capture_output=True, text=True, timeout=5).stdout
                f = [x.strip() for x in out.strip().split(",")]
                if len(f) >= 7:
                    self.samples.append(f)
            except Exception:
                pass
            self._halt.wait(0.2)

    def stop(self):
        self._halt.set()
        self.join(timeout=6)

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        sm = sorted(float(s[0]) for s in self.samples)
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(s[3 + i].lower().startswith("active") for s in self.samples)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": float(self.samples[0][1]), "reasons": reasons,
                "samples": len(sm), "power_w_max": max(float(s[2]) for s in self.samples)}


def replicas_aggregate(ms_local, tokens_per_replica, dist=None, device="cpu"):
    """"Replicas only" scaling rule: every rank runs the same layer on its own GPU with no data-path
    collective; the job's step time is the MAX over ranks and the aggregate value is world * tokens / that time."""
    import torch
    world = 1
    ms = float(ms_local)
    if dist is not None:
        t = torch.tensor([ms], dtype=torch.float64, device=device)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
        world = dist.get_world_size()
    return ms, world * tokens_per_replica / (ms * 1e-3)


def kept_pairs(L, k):
    k = min(k, L)
    return k * L - k * (k - 1) // 2


# ------------------------------------------------------------------------------------------------
# CPU oracle leg (cpu_baseline and --impl reference)
# ------------------------------------------------------------------------------------------------

def oracle_sample_rate(cfg, inp, budget_rows=None):
    """Times the oracle, as it stands, on a bounded sample of the workload; returns tokens/s and a
    description.  Indexer mode: full k_idx projection (shared by every row, amortised over L tokens) +
    `rows` support rows done completely (q projection, scores, block max, top-k, sparse attention)."""
    import numpy as np
    from oracle import oracle as orc
    pbo = orc.Problem(L=cfg.L, Hq=cfg.Hq, Hkv=cfg.Hkv, d=cfg.d, k=cfg.k, b_sel=cfg.b_sel, hidden=cfg.hidden,
                      d_idx=cfg.d_idx, local_window=cfg.local_window, local_bias=cfg.local_bias,
                      cu_seqlens=cfg.cu_seqlens)
    n_rows = orc.num_rows(pbo)
    nsel = budget_rows or (96 if cfg.b_sel > 1 else 2048)  # ~10-20 s of host work at the bench workloads
    rows = np.unique(np.linspace(0, n_rows - 1, nsel).astype(np.int64))
    pos = []
    for r in rows:
        s0, t0, t1 = orc.row_info(pbo, int(r))
        pos.extend(range(s0 + t0, s0 + t1 + 1))
    pos = np.array(pos)
    t_shared = 0.0
    kw = {}
    t0 = time.perf_counter()
    if cfg.mode != "oracle":
        ki = orc.project(pbo, inp["X"], inp["Wki"], key=True)
        t_shared = time.perf_counter() - t0
        t1 = time.perf_counter()
        qi = np.zeros((cfg.L, cfg.d_idx), np.uint16)
        qi[pos] = orc.project(pbo, inp["X"], inp["Wqi"], rows=pos)
        kw = dict(q_idx=qi, k_idx=ki)
        mode = orc.MODE_INDEXER
    else:
        t1 = time.perf_counter()
        mode = orc.MODE_ORACLE
    orc.prefill_layer(pbo, mode, inp["Q"], inp["K"], inp["V"], rows=rows, pos=pos, **kw)
    t_rows = time.perf_counter() - t1
    per_token = t_shared / cfg.L + t_rows / len(pos)
    return dict(value=1.0 / per_token, unit=UNIT, cores=orc.max_threads(), kind="oracle",
                sample=(f"{len(rows)} of {n_rows} support rows ({len(pos)} queries, evenly spaced) done completely in "
                        f"{t_rows:.1f} s + the shared k_idx projection of all {cfg.L} tokens in {t_shared:.1f} s "
                        f"amortised over L; extrapolated per token"),
                seconds=t_shared + t_rows)


def run_reference(args, cfg):
    """--impl reference: the fp64 CPU oracle on the host cores, same config / metric / unit.  Each step times the SAME
    bounded sample as the cpu_baseline leg (oracle_sample_rate: at least as many support rows as OpenMP threads, so the
    row-parallel oracle fills the cores) and extrapolates per token; `ms_per_step` is therefore the extrapolated time of
    one whole layer, flagged as such, with the seconds actually spent beside it."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import oracle as orc
    from paper_2606_07703_b200 import inputs as gen
    inp = gen.make_inputs(cfg)
    threads = orc.max_threads()
    rows = max(3 * threads, 48) if cfg.b_sel > 1 else max(32 * threads, 1024)   # a few seconds per step at c3 / c4
    for _ in range(min(args.warmup, 1)):
        oracle_sample_rate(cfg, inp, budget_rows=threads)
    vals, secs = [], 0.0
    last = None
    for _ in range(args.steps):
        last = oracle_sample_rate(cfg, inp, budget_rows=rows)
        vals.append(last["value"])
        secs += last["seconds"]
    v = len(vals) / sum(1.0 / x for x in vals)
    line = {
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * cfg.L / v, "extrapolated": True,
        "measured_seconds_total": secs, "measured_seconds_per_step": secs / max(1, args.steps),
        "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(cfg),
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": last["cores"], "kind": "oracle", "sample": last["sample"]},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def workload_config(cfg):
    return {"workload": f"BASELINE.json configs[{cfg.cfg_id - 1}] ({cfg.name}): one causal GQA layer, {cfg.mode} mode",
            "L": cfg.L, "Hq": cfg.Hq, "Hkv": cfg.Hkv, "d": cfg.d, "k": cfg.k, "b_sel": cfg.b_sel,
            "hidden": cfg.hidden, "d_idx": cfg.d_idx, "local_window": cfg.local_window, "batch": 1,
            "parallelism": "replicas only (no sharding, no collectives)",
            "l2": "no flush: per-step inputs (X+Q+K+V) exceed the 126 MB L2" }


# ------------------------------------------------------------------------------------------------
# GPU leg
# ------------------------------------------------------------------------------------------------

def run_c4_sweep(args, B, torch, gen, peaks):
    """BASELINE.json configs[3]: oracle-vs-indexer length sweep, per-query supports.  For every (L, k) of the sweep:
    the layer in both modes (CUDA events, device-resident inputs), the stage split of each mode (staged C-ABI calls on
    the MIDDLE row panel, scaled by rows / panel rows: per-row cost is linear in the row's prefix length), the support
    overlap |S_oracle & S_indexer| / |S_oracle| (sp_support_overlap) and the mean forward KL(P || softmax(z)) of the
    panel's rows (sp_row_kl).  X is drawn independently of Q/K/V and the indexer weights are random, so the overlap is
    the paper's "untrained indexer" regime (A21): near chance by construction, reported as measured."""
    import numpy as np
    stream = torch.cuda.current_stream()

    def timed(fn, reps, warm=1):
        for _ in range(warm):
            fn()
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        for _ in range(reps):
            fn()
        b.record(stream)
        torch.cuda.synchronize()
        return a.elapsed_time(b) / reps

    out = []
    l0 = B.launch_count()
    reps = max(1, min(args.steps, 3))
    lengths = [int(x) for x in args.c4_lengths.split(",")] if args.c4_lengths else None
    for cfg in gen.C4_SWEEP:
        if lengths is not None and cfg.L not in lengths:
            continue
        inp = gen.make_inputs(cfg, with_indexer=True)
        dv = {n: B.bf16_tensor(inp[n]) for n in ("X", "Wqi", "Wki", "Q", "K", "V")}
        pb = B.Problem.from_config(cfg)
        L, k, n_rows = cfg.L, cfg.k, pb.num_rows
        O = torch.empty(L, cfg.Hq, cfg.d, dtype=torch.bfloat16, device="cuda")
        idx_i = torch.empty(n_rows, k, dtype=torch.int32, device="cuda")
        idx_o = torch.empty_like(idx_i)
        ws = B.alloc_workspace(pb, B.SP_STAGE_LAYER_ORACLE)
        ws_i = B.alloc_workspace(pb, B.SP_STAGE_LAYER_INDEXER)
        t_idx = timed(lambda: B.sp_prefill_layer(pb, B.SP_MODE_INDEXER, dv["X"], dv["Wqi"], dv["Wki"], dv["Q"], dv["K"],
                                                 dv["V"], O, idx_i, ws_i), reps)
        t_orc = timed(lambda: B.sp_prefill_layer(pb, B.SP_MODE_ORACLE, None, None, None, dv["Q"], dv["K"], dv["V"], O,
                                                 idx_o, ws), reps)
        del ws, ws_i
        # ---- support overlap ----
        inter = torch.empty(n_rows, dtype=torch.int32, device="cuda")
        B.sp_support_overlap(pb, idx_o, idx_i, inter)
        cnt = (idx_o >= 0).sum(1)
        beyond = cnt.new_tensor(np.arange(n_rows) + 1 > k, dtype=torch.bool)
        pooled = float(inter.sum().item()) / float(cnt.sum().item())
        pooled_beyond = float(inter[beyond].sum().item()) / max(1.0, float(cnt[beyond].sum().item()))
        chance = float((k / (torch.arange(n_rows, device="cuda")[beyond] + 1).double()).mean().item()) if bool(beyond.any()) else 1.0
        # ---- stage split on the middle panel ----
        ld = (L + 3) // 4 * 4
        panel = min(n_rows, max(1, (1 << 30) // (ld * 4)))
        r0 = (n_rows - panel) // 2
        f = n_rows / panel
        sc = torch.empty(panel, ld, dtype=torch.float32, device="cuda")
        ms = torch.empty(panel, ld, dtype=torch.float32, device="cuda")
        q_idx = torch.empty(L, cfg.d_idx, dtype=torch.bfloat16, device="cuda")
        k_idx = torch.empty_like(q_idx)
        lse = torch.empty(L, cfg.Hq, dtype=torch.float32, device="cuda")
        idx_p = torch.empty(panel, k, dtype=torch.int32, device="cuda")
        wsx = B.alloc_workspace(pb, B.SP_STAGE_INDEXER_SCORES)
        t_both = timed(lambda: B.sp_indexer_scores(pb, dv["X"], dv["Wqi"], dv["Wki"], q_idx, k_idx, False, r0, panel, sc, wsx), reps)
        t_sc = timed(lambda: B.sp_indexer_scores(pb, None, None, None, q_idx, k_idx, True, r0, panel, sc), reps)
        t_p1 = timed(lambda: B.sp_dense_gqa_attn(pb, dv["Q"], dv["K"], dv["V"], None, lse), reps)
        t_p2 = timed(lambda: B.sp_oracle_mass(pb, dv["Q"], dv["K"], lse, True, r0, panel, ms), reps)
        t_tk = timed(lambda: B.sp_topk_support(pb, sc, r0, panel, idx_p), reps)
        # the attention as the layer call runs it (with the SPARSE_ATTN workspace: membership-masked tcgen05 tiles where
        # that plan applies, else the gather kernel), and the gather kernel on its own
        nb_at = B.workspace_bytes(pb, B.SP_STAGE_SPARSE_ATTN)
        ws_at = torch.empty(nb_at, dtype=torch.uint8, device="cuda") if nb_at else None
        t_at_layer = timed(lambda: B.sp_sparse_gqa_attn(pb, dv["Q"], dv["K"], dv["V"], idx_i, O, None, ws_at), reps)
        t_at = timed(lambda: B.sp_sparse_gqa_attn(pb, dv["Q"], dv["K"], dv["V"], idx_i, O), reps)
        del ws_at
        kl = torch.empty(panel, dtype=torch.float32, device="cuda")
        B.sp_row_kl(pb, ms, sc, r0, panel, kl)
        pairs = k * L - k * (k - 1) // 2
        out.append({
            "L": L, "k": k, "indexer_layer_ms": t_idx, "oracle_layer_ms": t_orc,
            "overlap_pooled": pooled, "overlap_pooled_rows_beyond_budget": pooled_beyond, "overlap_chance_level": chance,
            "mean_forward_kl_nats_middle_panel": float(kl.double().mean().item()),
            "stages_ms": {"projection": max(t_both - t_sc, 0.0), "scoring": t_sc * f, "mass_pass1_lse": t_p1,
                          "mass_pass2": t_p2 * f, "topk": t_tk * f, "sparse_attention_per_query": t_at_layer},
            "attention_plan": "membership-masked dense tiles (tcgen05)" if nb_at else "gather (mma.sync + cp.async)",
            "attention_masked_TFLOPs": (4.0 * cfg.d * cfg.Hq * (L * (L + 1) // 2) / (t_at_layer * 1e-3) / 1e12) if nb_at else None,
            "attention_gather_kernel_ms": t_at,
            "gather_GBps": 4.0 * cfg.Hkv * cfg.d * pairs / (t_at * 1e-3) / 1e9,
            "mass_pass2_TFLOPs": 2.0 * cfg.d * cfg.Hq * (L * (L + 1) // 2) / (t_p2 * f * 1e-3) / 1e12,
            "panel_rows": [r0, r0 + panel],
        })
        del dv, O, idx_i, idx_o, sc, ms, inp
        torch.cuda.empty_cache()
    ref = next((e for e in out if e["L"] == 32768), out[-1])
    line = {"metric": METRIC, "value": ref["L"] / (ref["indexer_layer_ms"] * 1e-3), "unit": UNIT, "n_gpus": 1,
            "steps": reps, "warmup": 1, "ms_per_step": ref["indexer_layer_ms"], "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
            "config": {"workload": "BASELINE.json configs[3] (c4): oracle-vs-indexer length sweep, per-query supports; "
                                   "value = the L=32768 indexer-mode layer", "Hq": 32, "Hkv": 8, "d": 128, "d_idx": 128,
                       "b_sel": 1, "parallelism": "replicas only (no sharding, no collectives)"},
            "gpu_launches": int(B.launch_count() - l0), "sweep": out,
            "roofline": ({"bound": "tensor", "achieved": ref["attention_masked_TFLOPs"], "peak": peaks["tensor_burst"],
                          "unit": "TFLOP/s", "frac": ref["attention_masked_TFLOPs"] / peaks["tensor_burst"], "traffic": None,
                          "kernel": "sparse_attention_per_query as membership-masked dense tiles (flops of the causal triangle)",
                          "peak_source": peaks["source"]} if ref["attention_masked_TFLOPs"] else
                         {"bound": "hbm", "achieved": ref["gather_GBps"], "peak": peaks["hbm"], "unit": "GB/s",
                          "frac": ref["gather_GBps"] / peaks["hbm"], "traffic": None,
                          "kernel": "sparse_attention_per_query (gathered K/V rows, mostly L2 hits)",
                          "peak_source": peaks["source"]})}
    print(json.dumps(line))


def run_c3_groups(args, B, torch, gen, peaks):
    """SURVEY.md 8(f) f4 at the c3 shape, ORACLE mode (per-KV-group selection is defined on attention mass only,
    PAPER.md:100, A29): the head-averaged layer (sp_prefill_layer, SP_MODE_ORACLE) beside the per-group
    chain of stage calls -- pass 1 (dense LSE) once, then per KV group sp_oracle_mass_group + sp_topk_support, then
    sp_sparse_gqa_attn under SP_F_GROUP_SUPPORT.  CUDA events on the current stream, device-resident inputs."""
    stream = torch.cuda.current_stream()
    cfg = gen.C3
    inp = gen.make_inputs(cfg, with_indexer=False)
    dv = {n: B.bf16_tensor(inp[n]) for n in ("Q", "K", "V")}
    pb = B.Problem.from_config(cfg)
    L, k, n_rows, Hkv = cfg.L, cfg.k, pb.num_rows, cfg.Hkv

    def timed(fn, reps, warm=3):
        for _ in range(warm):
            fn()
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        for _ in range(reps):
            fn()
        b.record(stream)
        torch.cuda.synchronize()
        return a.elapsed_time(b) / reps

    reps = max(1, args.steps)
    l0 = B.launch_count()
    O = torch.empty(L, cfg.Hq, cfg.d, dtype=torch.bfloat16, device="cuda")
    idx_s = torch.empty(n_rows, k, dtype=torch.int32, device="cuda")
    ws = B.alloc_workspace(pb, B.SP_STAGE_LAYER_ORACLE)
    t_shared = timed(lambda: B.sp_prefill_layer(pb, B.SP_MODE_ORACLE, None, None, None, dv["Q"], dv["K"], dv["V"], O,
                                                idx_s, ws), reps)
    ld = (L + 3) // 4 * 4
    mass = torch.empty(n_rows, ld, dtype=torch.float32, device="cuda")
    lse = torch.empty(L, cfg.Hq, dtype=torch.float32, device="cuda")
    idx_g = torch.empty(Hkv, n_rows, k, dtype=torch.int32, device="cuda")

    def chain():
        B.sp_dense_gqa_attn(pb, dv["Q"], dv["K"], dv["V"], None, lse)
        for r in range(Hkv):
            B.sp_oracle_mass_group(pb, dv["Q"], dv["K"], lse, True, r, 0, n_rows, mass)
            B.sp_topk_support(pb, mass, 0, n_rows, idx_g[r])
        B.sp_sparse_gqa_attn(pb, dv["Q"], dv["K"], dv["V"], idx_g, O)

    t_chain = timed(chain, reps)
    t_p1 = timed(lambda: B.sp_dense_gqa_attn(pb, dv["Q"], dv["K"], dv["V"], None, lse), reps)
    t_ma = timed(lambda: B.sp_oracle_mass(pb, dv["Q"], dv["K"], lse, True, 0, n_rows, mass), reps)
    t_mg = timed(lambda: B.sp_oracle_mass_group(pb, dv["Q"], dv["K"], lse, True, Hkv // 2, 0, n_rows, mass), reps)
    idx_scratch = torch.empty_like(idx_s)   # the stage timings below must not touch the chain's idx_g
    t_tk = timed(lambda: B.sp_topk_support(pb, mass, 0, n_rows, idx_scratch), reps)
    t_ag = timed(lambda: B.sp_sparse_gqa_attn(pb, dv["Q"], dv["K"], dv["V"], idx_g, O), reps)
    t_as = timed(lambda: B.sp_sparse_gqa_attn(pb, dv["Q"], dv["K"], dv["V"], idx_s, O), reps)
    inter = torch.empty(n_rows, dtype=torch.int32, device="cuda")
    agree = []
    for r in range(Hkv):   # how much of the head-averaged support each group's own support keeps
        B.sp_support_overlap(pb, idx_s, idx_g[r], inter)
        agree.append(float(inter.sum().item()) / float((idx_s >= 0).sum().item()))
    mass_flops = 2.0 * cfg.d * cfg.Hq * (L * (L + 1) // 2)
    attn_flops = 4.0 * cfg.d * cfg.Hq * sum(min(k, min(L, (j + 1) * cfg.b_sel)) * min(cfg.b_sel, L - j * cfg.b_sel)
                                            for j in range(n_rows))
    line = {"metric": METRIC, "value": L / (t_chain * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": reps, "warmup": 3,
            "ms_per_step": t_chain, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "bf16",
            "data": "synthetic",
            "config": {"workload": "c3 shape, ORACLE mode, one support per KV group (SURVEY.md 8(f) f4) as stage calls",
                       "L": L, "Hq": cfg.Hq, "Hkv": Hkv, "d": cfg.d, "k": k, "b_sel": cfg.b_sel,
                       "parallelism": "replicas only (no sharding, no collectives)",
                       "l2": "no flush: Q+K+V and the 67 MB mass panel exceed the 126 MB L2"},
            "gpu_launches": int(B.launch_count() - l0),
            "head_averaged_oracle_layer_ms": t_shared,
            "stages_ms": {"mass_pass1_lse": t_p1, "mass_pass2_one_group": t_mg, "mass_pass2_all_heads": t_ma,
                          "topk_one_group": t_tk, "sparse_attention_group_lists": t_ag,
                          "sparse_attention_shared_list": t_as},
            "mass_pass2_TFLOPs": {"all_groups_as_8_calls": mass_flops / (Hkv * t_mg * 1e-3) / 1e12,
                                  "all_heads_one_call": mass_flops / (t_ma * 1e-3) / 1e12},
            "sparse_attention_TFLOPs": {"group_lists": attn_flops / (t_ag * 1e-3) / 1e12,
                                        "shared_list": attn_flops / (t_as * 1e-3) / 1e12},
            "overlap_of_head_averaged_support_with_each_group": agree,
            "roofline": {"bound": "tensor", "achieved": attn_flops / (t_ag * 1e-3) / 1e12, "peak": peaks["tensor_burst"],
                         "unit": "TFLOP/s", "frac": attn_flops / (t_ag * 1e-3) / 1e12 / peaks["tensor_burst"], "traffic": None,
                         "kernel": "sparse_attention (group lists)", "peak_source": peaks["source"]}}
    print(json.dumps(line))


def _timed(torch, stream, fn, reps, warm=1):
    for _ in range(warm):
        fn()
    torch.cuda.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record(stream)
    for _ in range(reps):
        fn()
    b.record(stream)
    torch.cuda.synchronize()
    return a.elapsed_time(b) / reps


def measure_oracle_mode(cfg, B, torch, devt, peaks, reps=2):
    """The same layer in ORACLE mode (Alg.1: dense mass pass 1 + pass 2, top-k, sparse attention) on the tensors
    already resident: layer ms and the two mass passes as TFLOP/s and exp/s (north_star: "indexer and oracle TFLOP/s")."""
    stream = torch.cuda.current_stream()
    pb = B.Problem.from_config(cfg)
    n_rows, L = pb.num_rows, cfg.L
    O = torch.empty(L, cfg.Hq, cfg.d, dtype=torch.bfloat16, device="cuda")
    idx = torch.empty(n_rows, cfg.k, dtype=torch.int32, device="cuda")
    ws = B.alloc_workspace(pb, B.SP_STAGE_LAYER_ORACLE)
    t_layer = _timed(torch, stream, lambda: B.sp_prefill_layer(pb, B.SP_MODE_ORACLE, None, None, None, devt["Q"],
                                                               devt["K"], devt["V"], O, idx, ws), reps)
    del ws
    ld = (pb.max_seqlen + 3) // 4 * 4
    panel = min(n_rows, max(1, (1 << 30) // (ld * 4)))
    r0 = (n_rows - panel) // 2
    mass = torch.empty(panel, ld, dtype=torch.float32, device="cuda")
    lse = torch.empty(L, cfg.Hq, dtype=torch.float32, device="cuda")
    t_p1 = _timed(torch, stream, lambda: B.sp_dense_gqa_attn(pb, devt["Q"], devt["K"], devt["V"], None, lse), reps)
    t_p2 = _timed(torch, stream, lambda: B.sp_oracle_mass(pb, devt["Q"], devt["K"], lse, True, r0, panel, mass), reps)
    t_p2 *= n_rows / panel
    causal = L * (L + 1) // 2
    fl = 2.0 * cfg.d * cfg.Hq * causal
    ex = float(cfg.Hq) * causal
    out = {"layer_ms": t_layer, "tokens_per_s": L / (t_layer * 1e-3),
           "mass_pass1_lse": {"ms": t_p1, "TFLOPs": fl / (t_p1 * 1e-3) / 1e12, "Texp_per_s": ex / (t_p1 * 1e-3) / 1e12,
                              "frac_of_burst_peak": fl / (t_p1 * 1e-3) / 1e12 / peaks["tensor_burst"]},
           "mass_pass2": {"ms": t_p2, "TFLOPs": fl / (t_p2 * 1e-3) / 1e12, "Texp_per_s": ex / (t_p2 * 1e-3) / 1e12,
                          "frac_of_burst_peak": fl / (t_p2 * 1e-3) / 1e12 / peaks["tensor_burst"],
                          "panel_rows": [r0, r0 + panel], "scaled_by_rows": n_rows / panel},
           "config": f"{cfg.name} shape, SP_MODE_ORACLE, b_sel={cfg.b_sel}, k={cfg.k}"}
    # head-axis support granularities: one list per KV group / per query head, selected by
    # the SAME call from one pass 1 (SP_F_GROUP_SUPPORT / SP_F_HEAD_SUPPORT)
    del mass
    for name, flag, units in (("per_kv_group", B.SP_F_GROUP_SUPPORT, cfg.Hkv), ("per_head", B.SP_F_HEAD_SUPPORT, cfg.Hq)):
        pbu = B.Problem.from_config(cfg, flags=flag)
        idx_u = torch.empty(units, n_rows, cfg.k, dtype=torch.int32, device="cuda")
        ws_u = B.alloc_workspace(pbu, B.SP_STAGE_LAYER_ORACLE)
        t_u = _timed(torch, stream, lambda: B.sp_prefill_layer(pbu, B.SP_MODE_ORACLE, None, None, None, devt["Q"], devt["K"],
                                                               devt["V"], O, idx_u, ws_u), 1 if name == "per_head" else reps)
        inter = torch.empty(n_rows, dtype=torch.int32, device="cuda")
        agree = []
        hpl = cfg.Hq // units          # heads per list
        for u in range(0, units, max(1, units // 4)):
            B.sp_support_overlap(pb, idx, idx_u[u], inter)
            agree.append(float(inter.sum().item()) / float((idx >= 0).sum().item()))
        out[name] = {"layer_ms": t_u, "lists": units, "heads_per_list": hpl,
                     "overlap_with_head_averaged_support_sampled_lists": agree,
                     "attention_kernel": "tcgen05 block-shared (a KV group's heads share every gathered row)" if name == "per_kv_group"
                     else "mma.sync per-query tile shape (no two heads share a gathered row)"}
        del ws_u, idx_u
    return out


def measure_per_query_c4(B, torch, gen, peaks, L=32768, reps=2):
    """BASELINE.json configs[3] at L=32768 / k=2048, per-query supports, indexer mode: layer ms, stage split and the
    gather rate of the per-query attention held against (a) the HBM copy peak and (b) the rate a PLAIN gather kernel
    (sp_gather_probe) reaches on the same index stream (256-byte K rows out of L2)."""
    stream = torch.cuda.current_stream()
    cfg = next(c for c in gen.C4_SWEEP if c.L == L)
    inp = gen.make_inputs(cfg, with_indexer=True)
    dv = {n: B.bf16_tensor(inp[n]) for n in ("X", "Wqi", "Wki", "Q", "K", "V")}
    pb = B.Problem.from_config(cfg)
    k, n_rows = cfg.k, pb.num_rows
    O = torch.empty(L, cfg.Hq, cfg.d, dtype=torch.bfloat16, device="cuda")
    idx = torch.empty(n_rows, k, dtype=torch.int32, device="cuda")
    ws = B.alloc_workspace(pb, B.SP_STAGE_LAYER_INDEXER)
    t_layer = _timed(torch, stream, lambda: B.sp_prefill_layer(pb, B.SP_MODE_INDEXER, dv["X"], dv["Wqi"], dv["Wki"],
                                                               dv["Q"], dv["K"], dv["V"], O, idx, ws), reps)
    del ws
    ld = (L + 3) // 4 * 4
    panel = min(n_rows, max(1, (1 << 30) // (ld * 4)))
    r0 = (n_rows - panel) // 2
    f = n_rows / panel
    sc = torch.empty(panel, ld, dtype=torch.float32, device="cuda")
    q_idx = torch.empty(L, cfg.d_idx, dtype=torch.bfloat16, device="cuda")
    k_idx = torch.empty_like(q_idx)
    idx_p = torch.empty(panel, k, dtype=torch.int32, device="cuda")
    wsx = B.alloc_workspace(pb, B.SP_STAGE_INDEXER_SCORES)
    t_both = _timed(torch, stream, lambda: B.sp_indexer_scores(pb, dv["X"], dv["Wqi"], dv["Wki"], q_idx, k_idx, False,
                                                               r0, panel, sc, wsx), reps)
    t_sc = _timed(torch, stream, lambda: B.sp_indexer_scores(pb, None, None, None, q_idx, k_idx, True, r0, panel, sc), reps)
    t_tk = _timed(torch, stream, lambda: B.sp_topk_support(pb, sc, r0, panel, idx_p), reps)
    # per-query attention as the layer runs it: with the SPARSE_ATTN workspace, i.e. the membership-masked tcgen05 tile
    # loop where its plan applies (c4 @ 32K / 64K), else the gather kernel; and the gather kernel on its own
    nb_at = B.workspace_bytes(pb, B.SP_STAGE_SPARSE_ATTN)
    ws_at = torch.empty(max(nb_at, 256), dtype=torch.uint8, device="cuda") if nb_at else None
    t_at_layer = _timed(torch, stream, lambda: B.sp_sparse_gqa_attn(pb, dv["Q"], dv["K"], dv["V"], idx, O, None, ws_at), reps)
    t_at = _timed(torch, stream, lambda: B.sp_sparse_gqa_attn(pb, dv["Q"], dv["K"], dv["V"], idx, O), reps)
    del ws_at
    pairs = kept_pairs(L, k)
    causal = L * (L + 1) // 2
    gather_bytes = 4.0 * cfg.Hkv * cfg.d * pairs
    # plain gather of whole K token rows (all KV heads: Hkv * d * 2 bytes) over the attention's own index stream
    sink = torch.empty(148 * 8 * 256, dtype=torch.int32, device="cuda")
    row_b = pitch = cfg.Hkv * cfg.d * 2
    t_probe = _timed(torch, stream, lambda: B.sp_gather_probe(dv["K"], row_b, pitch, idx, sink), reps)
    probe_GBps = float(pairs) * row_b / (t_probe * 1e-3) / 1e9
    topk_bytes = 4.0 * causal + 4.0 * n_rows * k
    g = gather_bytes / (t_at * 1e-3) / 1e9
    return {"config": f"c4 L={L} k={k} b_sel=1 indexer mode (BASELINE.json configs[3])", "layer_ms": t_layer,
            "tokens_per_s": L / (t_layer * 1e-3),
            "stages_ms": {"projection": max(t_both - t_sc, 0.0), "scoring": t_sc * f, "topk": t_tk * f,
                          "sparse_attention_per_query": t_at_layer},
            "attention_plan": "membership-masked dense tiles (tcgen05)" if nb_at else "gather (mma.sync + cp.async)",
            "attention_masked_TFLOPs": (4.0 * causal * cfg.Hq * cfg.d / (t_at_layer * 1e-3) / 1e12) if nb_at else None,
            "attention_gather_kernel_ms": t_at,
            "scoring_score_write_GBps": 4.0 * causal / (t_sc * f * 1e-3) / 1e9,
            "topk_GBps": topk_bytes / (t_tk * f * 1e-3) / 1e9, "topk_frac_of_hbm": topk_bytes / (t_tk * f * 1e-3) / 1e9 / peaks["hbm"],
            "gather_GBps": g, "gather_frac_of_hbm_copy_peak": g / peaks["hbm"],
            "plain_gather_probe_GBps": probe_GBps, "gather_frac_of_plain_gather": g / probe_GBps,
            "note": "gathered K/V rows are mostly L2 hits (K+V = 134 MB), so the HBM fraction can exceed 1; the plain-gather "
                    "figure is sp_gather_probe on the same index stream (whole 2 KB K token rows, measured in this run)",
            "panel_rows": [r0, r0 + panel]}


def measure_cold_l2(torch, step, n=8):
    """One step at a time with a 256 MB scratch write before each (evicts the 126 MB L2): median / min of n."""
    stream = torch.cuda.current_stream()
    scratch = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    ts = []
    for i in range(n + 1):
        scratch.fill_(i & 0xff)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        step()
        b.record(stream)
        torch.cuda.synchronize()
        if i > 0:
            ts.append(a.elapsed_time(b))
    ts.sort()
    return {"ms_median": ts[len(ts) // 2], "ms_min": ts[0], "n": n,
            "how": "256 MB device scratch fill before every step; each step timed alone with CUDA events"}


def measure_layer_only(cfg, B, torch, gen, steps, chunked=None):
    """Layer latency of another workload (device-resident inputs, CUDA events, 3 warm-up steps) next to the dense
    GQA layer of the same library on the same tensors."""
    inp = gen.make_inputs(cfg)
    indexer = cfg.mode != "oracle"
    gmode = B.SP_MODE_INDEXER if indexer else B.SP_MODE_ORACLE
    names = ("X", "Wqi", "Wki", "Q", "K", "V") if indexer else ("Q", "K", "V")
    devt = {n: B.bf16_tensor(inp[n]) for n in names}
    pb = B.Problem.from_config(cfg)
    O = torch.empty(cfg.L, cfg.Hq, cfg.d, dtype=torch.bfloat16, device="cuda")
    idx = torch.empty(pb.num_rows, cfg.k, dtype=torch.int32, device="cuda")
    ws = B.alloc_workspace(pb, B.SP_STAGE_LAYER_INDEXER if indexer else B.SP_STAGE_LAYER_ORACLE)
    stream = torch.cuda.current_stream()

    def timed(fn, reps, warm):
        for _ in range(warm):
            fn()
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        for _ in range(reps):
            fn()
        b.record(stream)
        torch.cuda.synchronize()
        return a.elapsed_time(b) / reps

    ms = timed(lambda: B.sp_prefill_layer(pb, gmode, devt.get("X"), devt.get("Wqi"), devt.get("Wki"), devt["Q"],
                                          devt["K"], devt["V"], O, idx, ws), steps, 3)
    dense_ms = timed(lambda: B.sp_dense_gqa_attn(pb, devt["Q"], devt["K"], devt["V"], O, None), 2, 1)
    causal = cfg.L * (cfg.L + 1) // 2
    out = {"config": workload_config(cfg), "ms_per_step": ms, "tokens_per_s": cfg.L / (ms * 1e-3), "steps": steps,
           "dense_layer_ms": dense_ms, "dense_tflops": 4.0 * cfg.d * cfg.Hq * causal / (dense_ms * 1e-3) / 1e12,
           "speedup_sparse_vs_dense": dense_ms / ms}
    if chunked:
        B.sp_prefill_layer(pb, gmode, devt.get("X"), devt.get("Wqi"), devt.get("Wki"), devt["Q"], devt["K"], devt["V"],
                           O, idx, ws)   # O again holds the SPARSE layer's output (the dense baseline wrote over it)
        torch.cuda.synchronize()
        del ws
        out["chunked_paged_prefill"] = measure_chunked(cfg, B, torch, devt, O, chunks=chunked)
    return out


def measure_chunked(cfg, B, torch, devt, O_full, chunks=(4096, 8192), page=16):
    """The same layer as a sequence of prefill CHUNKS against a paged KV cache (PAPER.md:292 stage 4, :331, :428:
    max_num_batched_tokens = 4K / 8K): every chunk projects itself, appends K / V / indexer keys to 16-token pages behind
    a shuffled block table, scores against the whole cached prefix, selects and attends THROUGH the block table.
    Reported: the sum over all chunks (CUDA events around the whole sequence of calls) beside the one-call full
    prefill, the last chunk alone, and whether the chunked outputs equal the full prefill bit for bit."""
    import numpy as np
    stream = torch.cuda.current_stream()
    L, b = cfg.L, cfg.b_sel
    n_blocks = (L + page - 1) // page
    n_pages = n_blocks + 3
    rng = np.random.Generator(np.random.Philox(12345))
    bt = torch.from_numpy(rng.permutation(n_pages)[:n_blocks].astype(np.int32)).cuda()
    kv = B.KvPages(torch.zeros(n_pages, page, cfg.Hkv, cfg.d, dtype=torch.bfloat16, device="cuda"),
                   torch.zeros(n_pages, page, cfg.Hkv, cfg.d, dtype=torch.bfloat16, device="cuda"),
                   torch.zeros(n_pages, page, cfg.d_idx, dtype=torch.bfloat16, device="cuda"), bt)
    X, Q = devt["X"].view(L, -1), devt["Q"].view(L, cfg.Hq, cfg.d)
    K, V = devt["K"].view(L, cfg.Hkv, cfg.d), devt["V"].view(L, cfg.Hkv, cfg.d)
    res = {"page_size": page, "block_table": "random permutation"}
    for chunk in chunks:
        plans = []
        for q0 in range(0, L, chunk):
            qc = min(chunk, L - q0)
            pc = B.Problem.from_config(cfg, L=q0 + qc)
            plans.append((pc, q0, qc))
        ws = torch.empty(max(B.chunk_workspace_bytes(pc, q0, qc) for pc, q0, qc in plans), dtype=torch.uint8, device="cuda")
        O_c = torch.empty_like(O_full)

        def run_all():
            for pc, q0, qc in plans:
                B.sp_prefill_chunk(pc, q0, qc, X[q0:q0 + qc], devt["Wqi"], devt["Wki"], Q[q0:q0 + qc], K[q0:q0 + qc],
                                   V[q0:q0 + qc], kv, O_c[q0:q0 + qc], None, ws)

        t_all = _timed(torch, stream, run_all, 2, warm=1)
        pc, q0, qc = plans[-1]
        t_last = _timed(torch, stream, lambda: B.sp_prefill_chunk(pc, q0, qc, X[q0:q0 + qc], devt["Wqi"], devt["Wki"],
                                                                  Q[q0:q0 + qc], K[q0:q0 + qc], V[q0:q0 + qc], kv,
                                                                  O_c[q0:q0 + qc], None, ws), 3, warm=1)
        res[f"chunk_{chunk}"] = {"chunks": len(plans), "all_chunks_ms": t_all, "tokens_per_s": L / (t_all * 1e-3),
                                 "last_chunk_ms": t_last, "equals_full_prefill_bitwise": bool(torch.equal(O_c, O_full))}
        del ws, O_c
    return res


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="c3")
    ap.add_argument("--impl", default="ours")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-long", action="store_true", help="skip the 128K (c5) layer line inside the c3 run")
    ap.add_argument("--c4-lengths", default="", help="--workload c4: comma-separated subset of the sweep's lengths")
    ap.add_argument("--no-extras", action="store_true",
                    help="skip the oracle-mode, per-query (c4 @ 32K) and cold-L2 legs of the c3 run")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl != "reference" else args.warmup

    from paper_2606_07703_b200 import inputs as gen
    if args.workload == "c3-groups" and args.impl != "reference":
        import torch
        from paper_2606_07703_b200 import binding as B
        torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
        B.lib()
        return run_c3_groups(args, B, torch, gen, load_peaks())
    if args.workload == "c4" and args.impl != "reference":
        import torch
        from paper_2606_07703_b200 import binding as B
        torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
        B.lib()
        return run_c4_sweep(args, B, torch, gen, load_peaks())
    cfg = gen.ALL[args.workload]
    if args.impl == "reference":
        return run_reference(args, cfg)

    import numpy as np
    import torch
    from paper_2606_07703_b200 import binding as B

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl")
    B.lib()
    peaks = load_peaks()
    indexer = cfg.mode != "oracle"
    gmode = B.SP_MODE_INDEXER if indexer else B.SP_MODE_ORACLE
    stage = B.SP_STAGE_LAYER_INDEXER if indexer else B.SP_STAGE_LAYER_ORACLE

    inp = gen.make_inputs(cfg)
    names = ("X", "Wqi", "Wki", "Q", "K", "V") if indexer else ("Q", "K", "V")
    host = {n: B.bf16_tensor(inp[n], "cpu").pin_memory() for n in names}
    devt = {n: host[n].cuda(non_blocking=True) for n in names}
    pb = B.Problem.from_config(cfg)
    n_rows = pb.num_rows
    O = torch.empty(cfg.L, cfg.Hq, cfg.d, dtype=torch.bfloat16, device="cuda")
    O_dense = torch.empty_like(O)
    idx = torch.empty(n_rows, cfg.k, dtype=torch.int32, device="cuda")
    ws = B.alloc_workspace(pb, stage)
    stream = torch.cuda.current_stream()

    def step():
        B.sp_prefill_layer(pb, gmode, devt.get("X"), devt.get("Wqi"), devt.get("Wki"), devt["Q"], devt["K"], devt["V"],
                           O, idx, ws)

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
            torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    l0 = B.launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record(stream)
    for _ in range(args.steps):
        step()
    ev1.record(stream)
    barrier()
    launches = B.launch_count() - l0
    ms_step, value = replicas_aggregate(ev0.elapsed_time(ev1) / args.steps, cfg.L, dist, "cuda")

    # ---- CUDA-event timing of a staged call on the launching stream ----
    def time_call(fn, reps):
        fn()
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        for _ in range(reps):
            fn()
        b.record(stream)
        torch.cuda.synchronize()
        return a.elapsed_time(b) / reps

    # ---- per-stage split through the staged C-ABI calls (same stream, CUDA events) ----
    reps = max(1, args.steps)
    ld = (pb.max_seqlen + 3) // 4 * 4
    panel = min(n_rows, max(1, (1 << 30) // (ld * 4)))
    scores = torch.empty(panel, ld, dtype=torch.float32, device="cuda")
    stages = {}
    if indexer:
        q_idx = torch.empty(cfg.L, cfg.d_idx, dtype=torch.bfloat16, device="cuda")
        k_idx = torch.empty_like(q_idx)
        ws_i = B.alloc_workspace(pb, B.SP_STAGE_INDEXER_SCORES)
        t_both = time_call(lambda: B.sp_indexer_scores(pb, devt["X"], devt["Wqi"], devt["Wki"], q_idx, k_idx, False,
                                                       0, panel, scores, ws_i), reps)
        t_sc = time_call(lambda: B.sp_indexer_scores(pb, None, None, None, q_idx, k_idx, True, 0, panel, scores), reps)
        stages["projection"] = max(t_both - t_sc, 0.0)
        stages["scoring"] = t_sc * (n_rows / panel)
    else:
        lse = torch.empty(cfg.L, cfg.Hq, dtype=torch.float32, device="cuda")
        t_both = time_call(lambda: B.sp_oracle_mass(pb, devt["Q"], devt["K"], lse, False, 0, panel, scores), reps)
        t_p2 = time_call(lambda: B.sp_oracle_mass(pb, devt["Q"], devt["K"], lse, True, 0, panel, scores), reps)
        stages["mass_pass1_lse"] = max(t_both - t_p2, 0.0)
        stages["mass_pass2"] = t_p2 * (n_rows / panel)
    idx_p = torch.empty(panel, cfg.k, dtype=torch.int32, device="cuda")
    stages["topk"] = time_call(lambda: B.sp_topk_support(pb, scores, 0, panel, idx_p), reps) * (n_rows / panel)
    stages["sparse_attention"] = time_call(lambda: B.sp_sparse_gqa_attn(pb, devt["Q"], devt["K"], devt["V"], idx, O), reps)

    # ---- dense GQA layer of the same library, same tensors, same run (after the stage split: its 8 ms at
    # full power changes the clock / power state the short sparse kernels would otherwise be timed in) ----
    dense_reps = max(1, min(args.steps, 3))
    dense_ms = time_call(lambda: B.sp_dense_gqa_attn(pb, devt["Q"], devt["K"], devt["V"], O_dense, None), dense_reps)

    # ---- algorithmic work ----
    L, k, d, Hq, Hkv = cfg.L, cfg.k, cfg.d, cfg.Hq, cfg.Hkv
    causal = L * (L + 1) // 2
    # exact useful (query, key) pairs of the sparse attention: support entries with 0 <= s <= t
    b = max(1, cfg.b_sel)
    big = torch.where(idx >= 0, idx, torch.full_like(idx, 2 ** 30))
    if cfg.cu_seqlens is None:
        T = torch.arange(n_rows * b, device="cuda", dtype=torch.int32).view(n_rows, b)
        cnt = torch.searchsorted(big, T.clamp(max=L - 1).contiguous(), right=True)
        pairs = int((cnt * (T < L)).sum().item())
    else:
        pairs = kept_pairs(L, k)  # upper bound for packs; not used for a headline number
    work = {
        "projection": ("tensor", 4.0 * L * cfg.hidden * cfg.d_idx),
        "scoring": ("tensor" if cfg.b_sel > 1 else "hbm", 2.0 * cfg.d_idx * causal if cfg.b_sel > 1 else 4.0 * causal),
        "mass_pass1_lse": ("tensor", 2.0 * d * Hq * causal),
        "mass_pass2": ("tensor", 2.0 * d * Hq * causal),
        "topk": ("hbm", 4.0 * (causal / b if cfg.b_sel == 1 else sum(min(L, (j + 1) * b) for j in range(n_rows))) + 4.0 * n_rows * k),
        "sparse_attention": ("tensor", 4.0 * d * Hq * pairs) if cfg.b_sel > 1 else ("hbm", 4.0 * Hkv * d * pairs),
    }
    dom = max(stages, key=lambda s: stages[s])
    bound, amount = work[dom]
    if bound == "tensor":
        # the stage is timed alone for ~20 ms (burst regime): the burst peak is the denominator, the sustained one beside it
        ach = amount / (stages[dom] * 1e-3) / 1e12
        roof = {"bound": "tensor", "achieved": ach, "peak": peaks["tensor_burst"], "unit": "TFLOP/s",
                "frac": ach / peaks["tensor_burst"], "peak_kind": "burst (kernel timed alone)",
                "frac_of_sustained_peak": ach / peaks["tensor"], "sustained_peak": peaks["tensor"], "traffic": None}
    else:
        ach = amount / (stages[dom] * 1e-3) / 1e9
        roof = {"bound": "hbm", "achieved": ach, "peak": peaks["hbm"], "unit": "GB/s", "frac": ach / peaks["hbm"], "traffic": None}
    roof.update({"kernel": dom, "kernel_ms": stages[dom], "peak_source": peaks["source"],
                 "algorithmic_units": amount})
    stage_rates = {}
    for s, ms in stages.items():
        bd, amt = work[s]
        if ms > 0:
            stage_rates[s] = {"ms": ms, "bound": bd,
                              "rate": amt / (ms * 1e-3) / (1e12 if bd == "tensor" else 1e9),
                              "unit": "TFLOP/s" if bd == "tensor" else "GB/s",
                              "frac": amt / (ms * 1e-3) / ((peaks["tensor_burst"] * 1e12) if bd == "tensor" else (peaks["hbm"] * 1e9)),
                              "frac_of": "burst bf16 peak" if bd == "tensor" else "HBM copy peak"}

    extras = {}
    if cfg.name == "c3" and not args.no_extras and world == 1:
        extras["cold_l2"] = measure_cold_l2(torch, step)
        extras["oracle_mode"] = measure_oracle_mode(cfg, B, torch, devt, peaks)

    # ---- end to end through the C ABI with HOST buffers ----
    arena = torch.empty(B.layer_host_arena_bytes(pb, gmode), dtype=torch.uint8, device="cuda")
    O_host = torch.empty(cfg.L, cfg.Hq, cfg.d, dtype=torch.bfloat16).pin_memory()

    def e2e_step():
        B.sp_prefill_layer_host(pb, gmode, host.get("X"), host.get("Wqi"), host.get("Wki"), host["Q"], host["K"],
                                host["V"], O_host, arena)

    e2e_reps = max(1, min(args.steps, 5))
    e2e_step()
    barrier()
    a, bb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record(stream)
    for _ in range(e2e_reps):
        e2e_step()
    bb.record(stream)
    barrier()
    e2e_serial_ms, _ = replicas_aggregate(a.elapsed_time(bb) / e2e_reps, cfg.L, dist, "cuda")

    # The same call with two steps in flight: step i runs on stream i % 2 with its own device arena and its own
    # pinned output buffer, so the H2D copies of step i + 1 overlap the kernels and the D2H copy of step i (PCIe is
    # full duplex, the B200 has separate copy engines per direction).  Every step still copies all of its inputs in
    # and its output out inside the timed region; this is the throughput a serving loop gets from the host API.
    side = [torch.cuda.Stream(), torch.cuda.Stream()]
    arenas = [arena, torch.empty_like(arena)]
    outs = [O_host, torch.empty_like(O_host).pin_memory()]

    def e2e_pipelined(n):
        for i in range(n):
            with torch.cuda.stream(side[i & 1]):
                B.sp_prefill_layer_host(pb, gmode, host.get("X"), host.get("Wqi"), host.get("Wki"), host["Q"],
                                        host["K"], host["V"], outs[i & 1], arenas[i & 1])

    pipe_reps = 2 * e2e_reps
    for sd in side:
        sd.wait_stream(stream)
    e2e_pipelined(2)
    for sd in side:
        stream.wait_stream(sd)
    barrier()
    a2, b2 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a2.record(stream)
    for sd in side:
        sd.wait_stream(stream)
    e2e_pipelined(pipe_reps)
    for sd in side:
        stream.wait_stream(sd)
    b2.record(stream)
    barrier()
    e2e_ms, _ = replicas_aggregate(a2.elapsed_time(b2) / pipe_reps, cfg.L, dist, "cuda")
    sampler.stop()
    h2d = sum(host[n].numel() * 2 for n in names)
    d2h = O_host.numel() * 2
    # the host path must agree with the device path
    same = bool(torch.equal(outs[0].cuda(), O)) and bool(torch.equal(outs[1].cuda(), O))

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "bf16",
        "data": "synthetic", "config": workload_config(cfg),
        "clocks": sampler.summary(),
        "e2e": {"value": world * cfg.L / (e2e_ms * 1e-3), "unit": UNIT, "ms_per_step": e2e_ms,
                "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "matches_device_path": same,
                "in_flight": "2 steps on 2 streams, double-buffered device arenas and pinned outputs",
                "one_step_at_a_time": {"value": world * cfg.L / (e2e_serial_ms * 1e-3), "ms_per_step": e2e_serial_ms}},
        "gpu_launches": int(launches),
        "roofline": roof,
        "stages": stage_rates,
        "dense_layer": {"ms": dense_ms, "tflops": 4.0 * d * Hq * causal / (dense_ms * 1e-3) / 1e12,
                        "speedup_sparse_vs_dense": dense_ms / ms_step},
        "paper_context": "TTFT ratios in the paper (whole model, other hardware): 1.93x Qwen3.5-9B GPU-80G vs FA2 @256K; "
                         "1.71x Qwen3.5-0.8B NPU-64G vs vLLM-Ascend FA @256K (PAPER.md:434-440); not comparable to a layer",
    }
    # DRAM traffic of the dominant kernel from the committed ncu --set full capture (profiles/): emitted only while the
    # kernel's source file still has the hash recorded with the capture -- a stale figure is worse than none
    tr_path = os.path.join(ROOT, "profiles", "kernel_traffic.txt")
    if os.path.exists(tr_path):
        import hashlib
        with open(tr_path) as f:
            tr = json.load(f).get(cfg.name, {}).get(dom)
        if tr is not None:
            src = os.path.join(ROOT, "paper_2606_07703_b200", "csrc", tr.get("kernel_source", ""))
            sha = hashlib.sha256(open(src, "rb").read()).hexdigest() if os.path.isfile(src) else None
            if sha is not None and sha == tr.get("kernel_source_sha256"):
                line["roofline"]["traffic"] = tr["dram_bytes_per_launch"]
                line["roofline"]["traffic_source"] = tr["source"]
            else:
                line["roofline"]["traffic_source"] = "null: the committed capture predates the current kernel source"
    line.update(extras)
    if cfg.name == "c3" and not args.no_extras and world == 1:
        del devt, host, O, O_dense, idx, ws, arena, scores
        devt = host = O = O_dense = idx = ws = arena = scores = None
        torch.cuda.empty_cache()
        line["per_query_c4_32k"] = measure_per_query_c4(B, torch, gen, peaks)
        torch.cuda.empty_cache()
    if cfg.name == "c3" and not args.no_long and world == 1:
        # the metric is quoted at 32K and 128K: the 128K layer (BASELINE.json configs[4]) timed in the same run
        devt = host = O = O_dense = idx = ws = arena = scores = None
        torch.cuda.empty_cache()
        line["long_context_128k"] = measure_layer_only(gen.ALL["c5"], B, torch, gen, steps=min(args.steps, 5),
                                                       chunked=None if args.no_extras else (4096, 8192))
    if rank == 0 and not args.no_cpu_baseline and world == 1:
        cb = oracle_sample_rate(cfg, inp)
        cb.pop("seconds", None)
        line["cpu_baseline"] = cb
    if rank == 0:
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
