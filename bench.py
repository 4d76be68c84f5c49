#!/usr/bin/env python
"""bench.py -- ART decode-attention benchmark (contract in the task prompt).

One "step" = one pass of the whole hot path (resolve blocks, TMA loads, scores, online softmax,
P.V, probe + criterion + patience, early exit, finalise) over one decode batch of synthetic input.
At N = 1 the workload is BASELINE.json configs[1] (Mistral-7B-shaped decode layer: batch 8,
Hq 32 / Hkv 8, d 128, context 32768, bf16 paged KV, dense policy, paper-default thresholds).

    python bench.py [--gpus N] [--steps K] [--warmup W]          # this repo's CUDA path
    python bench.py --impl reference ...                          # the CPU oracle, as it stands
    python bench.py --report                                       # all five configs (+ variants), one JSON line each
    python bench.py --study                                        # probe-vs-full, ablation, sensitivity

Prints ONE JSON line (rank 0).  `value` is KV tokens/s (sum over sequences of eligible tokens per
step / step time) with inputs resident in HBM; `e2e` is the same through art_decode_attention_host
with pinned HOST q / tables / outputs copied inside the timed region (the KV cache is decode state
and stays in HBM).  Multi-GPU: the path shards by sequence with no exchange, so every rank runs its
own configs[1]-shaped batch (weak scaling) and no data-path collective exists.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "art_decode_attn_kv_tokens_per_s"
UNIT = "KV tok/s"
BLOCK_BYTES = 32768                      # K + V of one 64-token block of one KV head


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def committed_traffic():
    """dram bytes per launch of the dominant kernel from the committed ncu capture (profiles/traffic.csv)."""
    path = os.path.join(ROOT, "profiles", "traffic.csv")
    out = {}
    if os.path.exists(path):
        import csv
        with open(path) as f:
            for row in csv.DictReader(f):
                out[row["key"]] = int(row["bytes_per_launch"])
    return out


class ClockSampler:
    """Samples SM clock and throttle reasons DURING the timed region (NVML)."""
    REASONS = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown",
               0x40: "hw_thermal_slowdown", 0x80: "hw_power_brake_slowdown"}

    def __init__(self, index: int):
        self.samples, self.reasons, self.max_mhz, self._stop = [], set(), None, threading.Event()
        self._h = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self._nv = pynvml
            self._h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self._h = None
        self._t = threading.Thread(target=self._run, daemon=True)

    def _run(self):
        while not self._stop.is_set() and self._h is not None:
            try:
                self.samples.append(int(self._nv.nvmlDeviceGetClockInfo(self._h, self._nv.NVML_CLOCK_SM)))
                r = int(self._nv.nvmlDeviceGetCurrentClocksThrottleReasons(self._h))
                for bit, name in self.REASONS.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(0.001)                 # the timed region is ~10 ms: sample as fast as NVML answers

    def __enter__(self):
        self._t.start(); return self

    def __exit__(self, *a):
        self._stop.set(); self._t.join(timeout=1.0)

    def summary(self):
        s = sorted(self.samples)
        return {"sm_mhz": (s[len(s) // 2] if s else None), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(s)}


def eligible_tokens(w) -> int:
    """Sum over sequences of eligible tokens (sequence level, not multiplied by Hkv)."""
    import torch
    from workloads import generators as gen
    L = w.seq_lens.to(torch.int64)
    if w.policy == gen.POLICY_DENSE:
        return int(L.sum())
    if w.policy == gen.POLICY_SINK_WINDOW:
        s = torch.minimum(L, torch.tensor(w.sink_tokens, device=L.device))
        win = torch.minimum(L, torch.tensor(w.window_tokens, device=L.device))
        return int(torch.minimum(L, s + win).sum())
    # LIST: tokens of the listed blocks, averaged over the KV heads of a sequence
    cnt = w.eligible_counts.to(torch.int64)
    blk = w.eligible_blocks.to(torch.int64)
    idx = torch.arange(blk.shape[2], device=blk.device)[None, None, :] < cnt[:, :, None]
    tok = torch.clamp(L[:, None, None] - blk * 64, min=0, max=64) * idx
    return int(tok.sum() // w.num_kv_heads)


def time_loop(fn, steps: int, warmup: int, barrier=None):
    """W untimed steps, then exactly K steps between CUDA events on the current stream."""
    import torch
    for _ in range(warmup):
        fn()
    torch.cuda.synchronize()
    if barrier:
        barrier()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(steps):
        fn()
    e1.record()
    torch.cuda.synchronize()
    if barrier:
        barrier()
    return e0.elapsed_time(e1)            # ms for K steps


def rank_seed(rank: int) -> int:
    """Every rank draws its own configs[1]-shaped batch: the path shards by sequence, no exchange."""
    from workloads import generators as gen
    return gen.SEED_BASE + 1000 + 17 * rank


def reduce_over_ranks(ms: float, toks: float, device="cpu"):
    """Whole-job numbers: MAX over ranks of the timed region, SUM over ranks of the units processed.
    Works with any initialised process group (nccl on the GPU box, gloo in the CPU tests)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    tk = torch.tensor([float(toks)], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(tk, op=dist.ReduceOp.SUM)
    return float(t), float(tk)


def read_only_ceiling(art, w, steps: int, warmup: int) -> float:
    """GB/s of a read-only stream (art_hbm_read_probe: 32 KiB TMA copies, 3-stage ring, two CTAs per SM, no compute)
    over a 4 GiB device buffer: 32 x L2, and long enough (about 0.6 ms per launch) that launch ramp and tail do not
    count -- streaming the 512 MiB K and V caches of configs[1] in two launches read 1 % lower."""
    import torch
    scratch = torch.empty(4 << 30, dtype=torch.uint8, device=w.k_cache.device)
    ms = time_loop(lambda: art.art_hbm_read_probe(scratch), steps, warmup)
    nbytes = scratch.numel() // BLOCK_BYTES * BLOCK_BYTES
    del scratch
    return nbytes * steps / (ms * 1e-3) / 1e9


def make_runner(art, w, *, art_on: bool, split: int = 0, **th):
    """Pre-marshalled call (descriptors and outputs allocated once); returns (fn, out, stop, loaded)."""
    import torch
    dev = w.q.device
    out = torch.empty(tuple(w.q.shape), dtype=torch.float32, device=dev)        # [B, Hq, d], or [B, m, Hq, d]
    stop = torch.empty((w.batch, w.num_kv_heads), dtype=torch.int32, device=dev)
    loaded = torch.zeros((w.batch, w.num_kv_heads), dtype=torch.int32, device=dev)
    desc = art.make_desc(w, split=split, blocks_loaded=loaded)
    thr = art.ArtThresholds(tau=th.get("tau", w.tau), phi=th.get("phi", w.phi),
                            patience=th.get("patience", w.patience), probe_dim=th.get("probe_dim", w.probe_dim))
    if art_on:
        fn = lambda: art.art_decode_attention(desc, w.q, w.k_cache, w.v_cache, w.block_table, w.eligible_blocks,
                                              w.seq_lens, thr, out, stop)
    else:
        fn = lambda: art.art_decode_attention_off(desc, w.q, w.k_cache, w.v_cache, w.block_table,
                                                  w.eligible_blocks, w.seq_lens, out, stop)
    return fn, out, stop, loaded


def make_host_runner(art, w, *, art_on: bool):
    """art_decode_attention_host: per-step inputs / outputs in pinned host memory."""
    import torch
    pin = lambda t: None if t is None else t.cpu().pin_memory()
    q, bt, sl, el, ec = pin(w.q), pin(w.block_table), pin(w.seq_lens), pin(w.eligible_blocks), pin(w.eligible_counts)
    out = torch.empty(tuple(w.q.shape), dtype=torch.float32).pin_memory()
    stop = torch.empty((w.batch, w.num_kv_heads), dtype=torch.int32).pin_memory()
    desc = art.make_desc(w, eligible_counts=ec)
    ws = torch.empty(art.art_workspace_bytes(desc), dtype=torch.uint8, device=w.q.device)
    thr = art.ArtThresholds(tau=w.tau, phi=w.phi, patience=w.patience, probe_dim=w.probe_dim) if art_on else None
    fn = lambda: art.art_decode_attention_host(desc, q, w.k_cache, w.v_cache, bt, el, sl, thr, out, stop, ws)
    nbytes = lambda t: 0 if t is None else t.numel() * t.element_size()
    h2d = nbytes(q) + nbytes(bt) + nbytes(sl) + nbytes(el) + nbytes(ec)
    d2h = nbytes(out) + nbytes(stop)
    return fn, h2d, d2h, (q, bt, sl, el, ec, out, stop, ws)


def measure(art, w, steps, warmup, barrier=None, *, art_on=True, split=0, **th):
    """Times one configuration; returns a dict of per-step numbers."""
    fn, out, stop, loaded = make_runner(art, w, art_on=art_on, split=split, **th)
    ms = time_loop(fn, steps, warmup, barrier)
    us = ms * 1e3 / steps
    processed = int(stop.sum())
    ld = int(loaded.sum())
    return {"us_per_step": us, "blocks_processed": processed, "blocks_loaded": ld,
            "gbs_processed": processed * BLOCK_BYTES / (us * 1e-6) / 1e9,
            "gbs_loaded": ld * BLOCK_BYTES / (us * 1e-6) / 1e9, "ms_total": ms}


def _oracle_groups(args):
    """Worker (own process): the oracle on the groups of one small carved-out workload, one BLAS thread."""
    mini, art_on = args
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    from helpers import run_oracle                       # imports oracle/: cpu_baseline leg only
    try:
        from threadpoolctl import threadpool_limits
        ctx = threadpool_limits(limits=1)
    except Exception:
        import contextlib
        ctx = contextlib.nullcontext()
    with ctx:
        t0 = time.perf_counter()
        run_oracle(mini, art=art_on)
        return time.perf_counter() - t0


def oracle_sample(w, n_groups: int, art_on: bool = True):
    """The CPU oracle, as it stands, on a bounded sample of groups of workload w (single BLAS thread).
    Returns (seconds, sequence-level KV tokens covered, threads)."""
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    from helpers import extract_groups                   # pure data movement
    import numpy as np
    rng = np.random.default_rng(0)
    B, Hkv = w.batch, w.num_kv_heads
    groups = [(int(rng.integers(B)), int(rng.integers(Hkv))) for _ in range(n_groups)]
    mini = extract_groups(w, groups)
    tokens_all = eligible_tokens(mini)                   # mini has Hkv = 1: per-group tokens
    dt = _oracle_groups((mini, art_on))
    return dt, tokens_all / Hkv, 1


def oracle_sample_all_cores(w, groups_per_core: int = 2, art_on: bool = True):
    """The same oracle, the same way, with the sampled groups spread over every host core (one process per core, one
    BLAS thread each).  Returns (wall seconds of the parallel section, sequence-level KV tokens covered, processes)."""
    import multiprocessing as mp
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    from helpers import extract_groups
    import numpy as np
    n = os.cpu_count() or 1
    rng = np.random.default_rng(1)
    B, Hkv = w.batch, w.num_kv_heads
    jobs, toks = [], 0.0
    for _ in range(n):
        groups = [(int(rng.integers(B)), int(rng.integers(Hkv))) for _ in range(groups_per_core)]
        mini = extract_groups(w, groups)
        toks += eligible_tokens(mini) / Hkv
        jobs.append((mini, art_on))
    os.environ["PYTHONPATH"] = os.pathsep.join([ROOT, os.path.join(ROOT, "tests"), os.environ.get("PYTHONPATH", "")])
    with mp.get_context("spawn").Pool(n) as pool:
        pool.map(_oracle_groups, [(jobs[0][0], art_on)] * n)     # warm-up: imports, page-in (untimed)
        t0 = time.perf_counter()
        pool.map(_oracle_groups, jobs, chunksize=1)
        dt = time.perf_counter() - t0
    return dt, toks, n


def run_reference(args, rank, world):
    """--impl reference: the oracle timed on host cores, bounded sample per step."""
    if rank != 0:
        return
    import torch
    from workloads import generators as gen
    w = gen.config(1, device="cpu", batch=1)             # one sequence of configs[1]; groups sampled from it
    n_groups = 2
    times = []
    for i in range(args.warmup + args.steps):
        dt, toks, cores = oracle_sample(w, n_groups)
        if i >= args.warmup:
            times.append(dt)
    ms = 1e3 * sum(times) / len(times)
    val = toks / (ms * 1e-3)
    sample = f"{n_groups} of 64 (sequence, KV-head) groups of configs[1] per step (context 32768, G=4, d=128)"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "configs[1] mistral7b-shaped decode layer (bounded sample)", "sample": sample},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


def sampled_parity(art, w, art_on: bool, n_groups: int, split: int = 0):
    """GPU vs oracle on a few sampled groups of a full-size workload (tests/parity.py): stop-block mismatches on
    non-fragile / fragile groups, fragile groups, max relative output error."""
    import numpy as np
    import torch
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    from helpers import extract_groups
    from parity import compare
    rng = np.random.default_rng(5)
    groups = sorted({(int(rng.integers(w.batch)), int(rng.integers(w.num_kv_heads))) for _ in range(n_groups)})
    out, stop, _ = art.run_workload(w, art=art_on, split=split)
    torch.cuda.synchronize()
    G = w.group_size
    mini = extract_groups(w, groups)
    o_g = torch.stack([out[b, g * G:(g + 1) * G] for (b, g) in groups])
    s_g = torch.stack([stop[b, g:g + 1] for (b, g) in groups])
    rep = compare(mini, o_g, s_g, art=art_on)
    return {"groups": rep.groups, "stop_mismatch_nonfragile": rep.stop_mismatch_nonfragile,
            "stop_mismatch_fragile": rep.stop_mismatch_fragile, "fragile_groups": rep.fragile_groups,
            "fragile_unreachable": rep.fragile_unreachable, "max_rel_err": rep.max_rel_err}


def needle_report(art, w):
    """configs[4] (the NIAH failure mode of PAPER.md:216-236 Table 2 in synthetic form): per sequence,
    did Algorithm 1 fire, t* against the step at which the needle block is visited (dense order: step T - n_b), and the
    truncation error |out_on - out_off|_inf / |out_off|_inf of the ORACLE for one group of the sequence, next to the
    GPU's stop block for that group."""
    import numpy as np
    import torch
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    from helpers import extract_groups, run_oracle
    out, stop, _ = art.run_workload(w, art=True)
    torch.cuda.synchronize()
    rows = []
    for b in range(w.batch):
        T = (int(w.seq_lens[b]) + 63) // 64
        nb = int(w.notes["needle_block"][b])
        g = b % w.num_kv_heads
        mini = extract_groups(w, [(b, g)])
        _, _, res = run_oracle(mini, art=True)
        r = res[(0, 0)]
        err = float(np.abs(r.out_on - r.out_off).max(axis=-1).max() / np.abs(r.out_off).max())
        st = stop[b].cpu().numpy()
        rows.append({"seq": b, "T": T, "needle_block": nb, "needle_step": T - nb, "gpu_t_star_min": int(st.min()), "gpu_t_star_max": int(st.max()),
                     "groups_that_stop_before_the_needle": int((st < T - nb).sum()), "oracle_group": [b, g],
                     "oracle_t_star": int(r.stop_block), "gpu_t_star_same_group": int(st[g]), "oracle_fired": bool(r.fired),
                     "oracle_rel_trunc_err": err})
    return rows


def run_report(args):
    """All five configs (+ variants R / 0c), ART-on / ART-off / p = inf; one JSON line per row."""
    import torch
    from workloads import generators as gen
    import paper_2606_00024_b200 as art
    peak, which = peaks()
    rows = [(0, "a", ""), (0, "a", "c"), (1, "a", ""), (1, "a", "R"), (2, "a", ""), (2, "a", "R"),
            (3, "a", ""), (3, "a", "R"), (3, "b", ""), (3, "b", "R"), (4, "a", ""), (4, "a", "R")]
    ceiling = None
    for index, sub, variant in rows:
        w = gen.config(index, sub=sub, variant=variant, device="cuda")
        torch.cuda.synchronize()
        if ceiling is None and w.dtype == torch.bfloat16:
            ceiling = read_only_ceiling(art, w, args.steps, args.warmup)
        toks = eligible_tokens(w)
        sp = args.split if w.dtype == torch.bfloat16 else 0
        off = measure(art, w, args.steps, args.warmup, art_on=False, split=sp)
        on = measure(art, w, args.steps, args.warmup, art_on=True, split=sp)
        pinf = measure(art, w, args.steps, args.warmup, art_on=True, split=sp, patience=art.ART_PATIENCE_INF)
        total_blocks = off["blocks_processed"]
        groups = w.batch * w.num_kv_heads
        d_off, d_on = art.make_desc(w, split=sp), art.make_desc(w, split=sp)
        row = {"workload": w.name, "groups": groups,
               "split_on": art.art_query_split(d_on, True), "split_off": art.art_query_split(d_off, False),
               "persistent_clusters_off": art.art_query_clusters(d_off, False) if w.dtype == torch.bfloat16 else 0,
               "eligible_tokens": toks, "blocks_total": total_blocks,
               "off_us": round(off["us_per_step"], 2), "off_gbs": round(off["gbs_processed"], 1),
               "off_frac_of_peak": round(off["gbs_processed"] / peak, 4),
               "on_us": round(on["us_per_step"], 2), "on_gbs_loaded": round(on["gbs_loaded"], 1),
               "on_frac_of_peak_loaded": round(on["gbs_loaded"] / peak, 4),
               "on_gbs_processed": round(on["gbs_processed"], 1),
               "skipped_frac": round(1 - on["blocks_processed"] / max(total_blocks, 1), 4),
               "loaded_frac": round(on["blocks_loaded"] / max(total_blocks, 1), 4),
               "loaded_over_processed": round(on["blocks_loaded"] / max(on["blocks_processed"], 1), 4),
               "discarded_blocks_per_group": round((on["blocks_loaded"] - on["blocks_processed"]) / groups, 2),
               "speedup_on_vs_off": round(off["us_per_step"] / on["us_per_step"], 4),
               "pinf_overhead": round(pinf["us_per_step"] / off["us_per_step"] - 1, 4),
               "kv_tok_s_on": toks / (on["us_per_step"] * 1e-6), "kv_tok_s_off": toks / (off["us_per_step"] * 1e-6),
               "kv_tok_s_on_x_hkv": toks * w.num_kv_heads / (on["us_per_step"] * 1e-6),
               "kv_tok_s_on_physical": on["blocks_processed"] * 64 / (on["us_per_step"] * 1e-6),
               "peak_gbs": peak, "peak_kind": which,
               "read_only_ceiling_gbs": None if ceiling is None else round(ceiling, 1),
               "off_frac_of_read_only_ceiling": None if ceiling is None else round(off["gbs_processed"] / ceiling, 4)}
        if not args.no_parity:
            row["parity_on"] = sampled_parity(art, w, True, 4, sp)
            row["parity_off"] = sampled_parity(art, w, False, 2, sp)
            if index == 4:
                row["needle"] = needle_report(art, w)
        print(json.dumps(row), flush=True)
        del w
        torch.cuda.empty_cache()


def run_study(args):
    """SURVEY 8(f) items 1-2 on the synthetic variant-R workloads: probe (m = 32) vs full-output detector
    (App. B / Table 4 protocol), the ablation switches of Table 3 and the sensitivity
    grid of App. F.  Everything runs through the C ABI; one JSON line per row."""
    import torch
    from workloads import generators as gen
    import paper_2606_00024_b200 as art
    inf = float("inf")
    for index in (1, 4):
        w = gen.config(index, variant="R", device="cuda")
        torch.cuda.synchronize()
        name = w.name
        T = measure(art, w, 3, 3, art_on=False)["blocks_processed"] / (w.batch * w.num_kv_heads)
        o_off, _, _ = art.run_workload(w, art=False)

        def row(kind, **th):
            m = measure(art, w, args.steps, args.warmup, art_on=True, **th)
            out, stop, _ = art.run_workload(w, art=True, **th)
            err = float(((out - o_off).abs().amax(dim=-1) / o_off.abs().amax(dim=-1)).max())
            return {"study": kind, "workload": name, **{k: (str(v) if v == inf else v) for k, v in th.items()},
                    "us": round(m["us_per_step"], 1), "mean_stop_frac": round(float(stop.float().mean()) / T, 4),
                    "fired_frac": round(float((stop.float() < T).float().mean()), 4),
                    "max_rel_trunc_err_vs_off": err}, stop

        # ---- probe vs full output (the paper's "oracle detector" = P = I)
        r32, s32 = row("probe_vs_full", probe_dim=32)
        r0, s0 = row("probe_vs_full", probe_dim=0)
        d = (s32 - s0).float()
        cmp = {"study": "probe_vs_full_summary", "workload": name, "groups": int(s32.numel()),
               "agree_frac": float((d == 0).float().mean()), "probe_earlier_frac(FP)": float((d < 0).float().mean()),
               "probe_later_frac(FN)": float((d > 0).float().mean()), "mean_abs_delta_blocks": float(d.abs().mean()),
               "us_probe32": r32["us"], "us_full": r0["us"]}
        for r in (r32, r0, cmp):
            print(json.dumps(r), flush=True)
        # ---- ablation switches (Table 3): each is a threshold setting
        for label, th in (("default", {}), ("wo_d_scale", {"tau": inf}), ("wo_d_direction", {"phi": inf}),
                          ("wo_patience", {"patience": 1})):
            r, _ = row("ablation:" + label, **th)
            print(json.dumps(r), flush=True)
        # ---- sensitivity (App. F): one parameter at a time around the defaults
        for tau in (1e-6, 1e-5, 1e-4):
            print(json.dumps(row("sensitivity", tau=tau)[0]), flush=True)
        for phi in (1e-4, 1e-3, 1e-2):
            print(json.dumps(row("sensitivity", phi=phi)[0]), flush=True)
        for pt in (1, 2, 5, 10):
            print(json.dumps(row("sensitivity", patience=pt)[0]), flush=True)
        del w, o_off
        torch.cuda.empty_cache()


def run_policy(args):
    """the scored base policy's block list built on the device (art_topk_blocks) on configs[2]
    and configs[3b]: time, K bytes streamed (every K row once: groups x blocks x 16 KiB) against the HBM peak."""
    import torch
    from workloads import generators as gen
    import paper_2606_00024_b200 as art
    peak, which = peaks()
    for index, sub in ((2, "a"), (3, "b")):
        w = gen.config(index, sub=sub, device="cuda")
        torch.cuda.synchronize()
        maxb = int(w.block_table.shape[1]); k = int(w.eligible_blocks.shape[2])
        scores = torch.empty((w.batch, w.num_kv_heads, maxb), dtype=torch.float32, device="cuda")
        lists = torch.empty((w.batch, w.num_kv_heads, k), dtype=torch.int32, device="cuda")
        counts = torch.empty((w.batch, w.num_kv_heads), dtype=torch.int32, device="cuda")
        desc = art.make_desc(w)
        fn = lambda: art.art_topk_blocks(desc, w.q, w.k_cache, w.block_table, w.seq_lens, k, scores, lists, counts)
        ms = time_loop(fn, args.steps, args.warmup)
        us = ms * 1e3 / args.steps
        nblocks = int(((w.seq_lens.to(torch.int64) + 63) // 64).sum()) * w.num_kv_heads
        kbytes = nblocks * 16384
        agree = float((lists == w.eligible_blocks).float().mean())
        print(json.dumps({"policy": "art_topk_blocks", "workload": w.name, "groups": w.batch * w.num_kv_heads, "top_k": k,
                          "us": round(us, 1), "k_bytes": kbytes, "gbs": round(kbytes / (us * 1e-6) / 1e9, 1),
                          "frac_of_peak": round(kbytes / (us * 1e-6) / 1e9 / peak, 4), "peak_gbs": peak, "peak_kind": which,
                          "agrees_with_host_recipe": round(agree, 4)}), flush=True)
        del w
        torch.cuda.empty_cache()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="art", choices=["art", "reference"])
    ap.add_argument("--report", action="store_true")
    ap.add_argument("--policy", action="store_true", help="time art_topk_blocks (SURVEY 8(f).3)")
    ap.add_argument("--study", action="store_true", help="probe-vs-full, ablation and sensitivity sweeps (SURVEY 8(f))")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-parity", action="store_true", help="--report without the oracle columns (timing only)")
    ap.add_argument("--split", type=int, default=0, help="cluster size for --arm / --report (0 = library default = static clusters, -1 - cl = persistent clusters of cl CTAs, detector off only)")
    ap.add_argument("--arm", default=None, choices=["on", "off", "pinf", "R_on", "R_off"],
                    help="time ONLY this arm of one config (short command for ncu captures; prints a small JSON line)")
    ap.add_argument("--q-len", type=int, default=1, help="--arm only: m query tokens per sequence (SURVEY 8(f).4; m * G <= 8)")
    ap.add_argument("--q-heads", type=int, default=0, help="--arm only: override the number of query heads (group size G = Hq / Hkv)")
    ap.add_argument("--config", default="1a", help="config for --arm: index + sub, e.g. 1a, 2a, 3a, 3b, 4a, 0a")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "art" else args.warmup

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
        return
    if args.report:
        run_report(args)
        return
    if args.study:
        run_study(args)
        return
    if args.policy:
        run_policy(args)
        return

    import torch
    import torch.distributed as dist
    from workloads import generators as gen
    import paper_2606_00024_b200 as art           # raises if the CUDA library is not built: no fallback

    torch.cuda.set_device(local)
    barrier = None
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        barrier = dist.barrier
    dev = torch.device("cuda", local)

    if args.arm and args.config != "1a":
        idx, sub = int(args.config[0]), args.config[1:] or "a"
        wa = gen.config(idx, sub=sub, device=dev, variant="R" if args.arm.startswith("R_") else "",
                        **({"num_q_heads": args.q_heads} if args.q_heads else {}))
        if args.q_len > 1:
            wa = gen.with_query_tokens(wa, args.q_len, seed=args.q_len)
        torch.cuda.synchronize()
        kw = {"patience": art.ART_PATIENCE_INF} if args.arm == "pinf" else {}
        sp = args.split if wa.dtype == torch.bfloat16 else 0
        r = measure(art, wa, args.steps, args.warmup, None, art_on=args.arm not in ("off", "R_off"), split=sp, **kw)
        r.update(arm=args.arm, config=wa.name, q_len=args.q_len, split=sp or art.art_query_split(art.make_desc(wa), args.arm not in ("off", "R_off")))
        print(json.dumps(r), flush=True)
        return

    # configs[1]; every rank its own batch (seed offset), no exchange between ranks
    w = gen.config(1, device=dev, seed=rank_seed(rank))
    wR = gen.config(1, device=dev, variant="R", seed=rank_seed(rank))
    torch.cuda.synchronize()
    toks = eligible_tokens(w)
    peak, which = peaks()

    if args.arm:
        wa = wR if args.arm.startswith("R_") else w
        if args.q_heads:
            wa = gen.config(1, device=dev, variant="R" if args.arm.startswith("R_") else "", seed=rank_seed(rank),
                            num_q_heads=args.q_heads)
        if args.q_len > 1:
            wa = gen.with_query_tokens(wa, args.q_len, seed=args.q_len)
        kw = {"patience": art.ART_PATIENCE_INF} if args.arm == "pinf" else {}
        r = measure(art, wa, args.steps, args.warmup, barrier, art_on=args.arm not in ("off", "R_off"),
                    split=args.split, **kw)
        r["arm"] = args.arm
        r["q_len"] = args.q_len
        r["q_heads"] = wa.num_q_heads
        r["split"] = args.split or art.art_query_split(art.make_desc(wa), args.arm not in ("off", "R_off"))
        print(json.dumps(r), flush=True)
        return

    # ---- the timed region of the contract: exactly K ART-on steps on the literal config
    fn, out, stop, loaded = make_runner(art, w, art_on=True)
    with ClockSampler(local) as cs:
        ms = time_loop(fn, args.steps, args.warmup, barrier)
    clocks = cs.summary()
    ms_max, toks_all = reduce_over_ranks(ms, toks, dev)
    ms_per_step = ms_max / args.steps
    value = toks_all / (ms_per_step * 1e-3)
    processed, ld = int(stop.sum()), int(loaded.sum())

    # ---- end to end through the host entry point (H2D of q / tables, D2H of out / stop inside)
    hfn, h2d, d2h, _keep = make_host_runner(art, w, art_on=True)
    for _ in range(args.warmup):
        hfn()
    torch.cuda.synchronize()
    if barrier:
        barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        hfn()                                  # synchronises the stream itself
    e2e_ms = (time.perf_counter() - t0) * 1e3
    e2e_max, _ = reduce_over_ranks(e2e_ms, 0.0, dev)
    e2e_value = toks_all / (e2e_max / args.steps * 1e-3)

    # ---- context numbers (outside the contract's timed region): ART-off, p = inf, variant R
    off = measure(art, w, args.steps, args.warmup, barrier, art_on=False)
    pinf = measure(art, w, args.steps, args.warmup, barrier, art_on=True, patience=art.ART_PATIENCE_INF)
    r_off = measure(art, wR, args.steps, args.warmup, barrier, art_on=False)
    r_on = measure(art, wR, args.steps, args.warmup, barrier, art_on=True)
    # the read-only streaming ceiling of this box, measured here and now: the K and V caches of the
    # workload (512 MiB each, both larger than L2) streamed alternately by art_hbm_read_probe
    ceiling_gbs = read_only_ceiling(art, w, args.steps, args.warmup)

    if rank == 0:
        us = ms / args.steps * 1e3             # this rank's own kernel time per launch
        achieved = ld * BLOCK_BYTES / (us * 1e-6) / 1e9
        traffic = committed_traffic().get("art_on_cfg1_dram_bytes_per_launch")
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "bf16 KV, f32 accumulate", "data": "synthetic",
            "config": {"workload": "configs[1] mistral7b-shaped decode layer: batch 8, Hq 32, Hkv 8, d 128, "
                                   "context 32768, bf16 paged KV (64-token pages, permuted), dense policy, "
                                   "tau 1e-5 phi 1e-3 p 5 (ART on)",
                       "l2": "inputs larger than L2: 1 GiB of KV streamed per step vs 126 MB L2",
                       "cluster_size": art.art_query_split(art.make_desc(w), True), "per_gpu_batch": w.batch},
            "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h},
            "gpu_launches": args.steps,
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s",
                         "frac": achieved / peak, "traffic": traffic, "peak_kind": which,
                         "kernel": "art::tc::art_decode_tc_kernel<4, 1, false>",
                         "bytes_per_launch": ld * BLOCK_BYTES, "frac_of_nominal_8TBs": achieved / 8000.0,
                         "read_only_ceiling_gbs": ceiling_gbs, "frac_of_read_only_ceiling": achieved / ceiling_gbs,
                         "note": "peak is the pool's measured COPY bandwidth (read + write); this kernel only reads, so "
                                 "frac may exceed 1 -- frac_of_read_only_ceiling is against a read-only TMA stream "
                                 "(art_hbm_read_probe over 4 GiB) timed in this run"},
            "art": {"on_us_per_step": us, "off_us_per_step": off["us_per_step"],
                    "off_gbs": off["gbs_processed"], "off_frac_of_peak": off["gbs_processed"] / peak,
                    "pinf_overhead": pinf["us_per_step"] / off["us_per_step"] - 1.0,
                    "skipped_frac": 1.0 - processed / max(off["blocks_processed"], 1),
                    "speedup_on_vs_off": off["us_per_step"] / us,
                    "variant_R": {"on_us_per_step": r_on["us_per_step"], "off_us_per_step": r_off["us_per_step"],
                                  "speedup_on_vs_off": r_off["us_per_step"] / r_on["us_per_step"],
                                  "skipped_frac": 1.0 - r_on["blocks_processed"] / max(r_off["blocks_processed"], 1),
                                  "loaded_frac": r_on["blocks_loaded"] / max(r_off["blocks_processed"], 1),
                                  "on_gbs_loaded": r_on["gbs_loaded"], "on_frac_of_peak_loaded": r_on["gbs_loaded"] / peak,
                                  "loaded_over_processed": r_on["blocks_loaded"] / max(r_on["blocks_processed"], 1),
                                  "discarded_blocks_per_group": (r_on["blocks_loaded"] - r_on["blocks_processed"]) / (wR.batch * wR.num_kv_heads)},
                    "off_frac_of_read_only_ceiling": off["gbs_processed"] / ceiling_gbs},
        }
        line["kv_tok_s_x_hkv"] = value * w.num_kv_heads       # every KV head streams its own copy of the context
        line["kv_tok_s_physical"] = processed * 64 / (us * 1e-6)   # tokens of the blocks actually visited, all heads, this rank
        if world == 1 and not args.no_cpu_baseline:
            dt, ctoks, cores = oracle_sample(w, 16)
            dta, ctoka, ncore = oracle_sample_all_cores(w, 2)
            line["cpu_baseline"] = {"value": ctoks / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
                                    "sample": "16 of 64 (sequence, KV-head) groups of configs[1], one pass, ART on",
                                    "all_cores": {"value": ctoka / dta, "unit": UNIT, "cores": ncore,
                                                  "sample": "2 groups per core, one process per core, one BLAS thread each"},
                                    "host_cores": os.cpu_count()}
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
