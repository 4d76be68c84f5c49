"""Shared GPU-vs-oracle comparison used by the -m gpu parity tests, smoke() and bench.py's checks.

Bars (BASELINE.json north_star): stop_block bit-exact except for groups the ORACLE flags as fragile
(a criterion value within 1e-4 relative of its threshold at a step <= t*), which are reported
separately; outputs within 1e-5 * ||o||_inf (fp32 KV) / 1e-2 * ||o||_inf (bf16 KV, fp32 accumulate).
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np
import torch

from helpers import run_oracle, thresholds_f32

OUT_TOL = {torch.float32: 1e-5, torch.bfloat16: 1e-2}


FRAGILE_REL = 1e-4                # north_star: "within 1e-4 relative of its threshold"


@dataclass
class ParityReport:
    groups: int
    stop_mismatch_nonfragile: int
    stop_mismatch_fragile: int    # stop blocks that differ on groups the oracle flags as fragile (reported separately)
    fragile_groups: int
    max_rel_err: float            # max over compared rows of |gpu - oracle|_inf / |oracle|_inf (fragile mismatches: against
                                  # the oracle's prefix output o^(t) at the GPU's stop block)
    fired_groups: int
    mean_stop_frac: float
    fragile_unreachable: int = 0  # fragile mismatches whose GPU stop block NO outcome of the near-threshold tests gives

    def ok(self, tol: float) -> bool:
        return (self.stop_mismatch_nonfragile == 0 and self.fragile_unreachable == 0 and self.max_rel_err <= tol
                and self.stop_mismatch_fragile <= self.fragile_groups)

    def summary(self) -> str:
        return (f"groups={self.groups} fired={self.fired_groups} stop_mismatch_nonfragile={self.stop_mismatch_nonfragile} "
                f"fragile_groups={self.fragile_groups} stop_mismatch_fragile={self.stop_mismatch_fragile} "
                f"fragile_unreachable={self.fragile_unreachable} max_rel_err={self.max_rel_err:.2e}")


def reachable_stops(d_scale, d_dir, tau: float, phi: float, patience: int) -> set:
    """Stop blocks that Eq. 3 can produce when every test whose value lies within FRAGILE_REL (relative) of its threshold
    may go either way.  d_scale, d_dir: [T, rows] of the oracle's full trace.  Pure bookkeeping over the oracle's numbers."""
    T = d_scale.shape[0]
    def tri(v, thr):                       # 1 surely below, 0 surely not, -1 either
        if not np.isfinite(thr):
            return np.where(np.isnan(v), 0, 1)
        lo, hi = thr * (1 - FRAGILE_REL), thr * (1 + FRAGILE_REL)
        return np.where(v < lo, 1, np.where(v < hi, -1, 0))
    a, b = tri(d_scale, tau), tri(d_dir, phi)
    sure = ((a == 1) & (b == 1)).all(axis=1)
    never = ((a == 0) | (b == 0)).any(axis=1)
    counts, stops = {0}, set()
    for t in range(1, T + 1):
        nxt = set()
        for c in counts:
            outs = [c + 1] if sure[t - 1] else ([0] if never[t - 1] else [c + 1, 0])
            for c2 in outs:
                if c2 >= patience:
                    stops.add(t)
                else:
                    nxt.add(c2)
        counts = nxt
        if not counts:
            break
    if counts:
        stops.add(T)
    return stops


def compare(w_host, out_gpu: torch.Tensor, stop_gpu: torch.Tensor, *, art: bool, groups=None,
            oracle_over: dict | None = None) -> ParityReport:
    """w_host: the workload on the CPU (the payload the GPU saw, bit for bit)."""
    o_ref, s_ref, res = run_oracle(w_host, art=art, groups=groups, **(oracle_over or {}))
    out = out_gpu.detach().cpu().to(torch.float64).numpy()
    stop = stop_gpu.detach().cpu().numpy().astype(np.int64)
    G = w_host.group_size
    mism_nf = mism_f = frag = fired = unreach = 0
    max_rel = 0.0
    fr = []
    d = o_ref.shape[-1]
    thr = {"tau": thresholds_f32(w_host)[0], "phi": thresholds_f32(w_host)[1], "patience": w_host.patience}
    thr.update({k: v for k, v in (oracle_over or {}).items() if k in thr})
    for (b, g), r in res.items():
        frag += int(r.fragile)
        fired += int(r.fired)
        fr.append(r.stop_block / max(r.num_blocks, 1))
        ref_rows = {h: o_ref[b, ..., h, :].reshape(-1, d) for h in range(g * G, (g + 1) * G)}
        if stop[b, g] != s_ref[b, g]:
            if r.fragile and art:
                # The oracle itself says a comparison of this group sits on its threshold: a different stop block is
                # legitimate IF some outcome of those near-threshold tests leads to it; the output must then be the
                # oracle's prefix output at THAT stop block.
                mism_f += 1
                _, _, tr = run_oracle(w_host, art=art, groups=[(b, g)], trace=True, **(oracle_over or {}))
                rt = tr[(b, g)]
                sg = int(stop[b, g])
                if sg not in reachable_stops(rt.d_scale_all, rt.d_direction_all, thr["tau"], thr["phi"], thr["patience"]) or sg < 1:
                    unreach += 1
                    continue
                rows = rt.o[sg - 1]                                   # [m * G, d], row = i * G + h
                m_tok = rows.shape[0] // G
                ref_rows = {g * G + h: rows.reshape(m_tok, G, d)[:, h, :] for h in range(G)}
            else:
                mism_nf += 1
        for h in range(g * G, (g + 1) * G):
            # one row per query token (q [B, m, Hq, d], reading R15), else the head's single row
            for ref, got in zip(ref_rows[h], out[b, ..., h, :].reshape(-1, d)):
                scale = np.abs(ref).max()
                err = np.abs(got - ref).max()
                if not np.isfinite(err):
                    max_rel = float("inf")
                elif scale > 0:
                    max_rel = max(max_rel, err / scale)
                elif err > 0:
                    max_rel = float("inf")
    return ParityReport(len(res), mism_nf, mism_f, frag, max_rel, fired, float(np.mean(fr)) if fr else 0.0, unreach)


# ------------------------------------------------------------------ every group of a full-size config, oracle on all cores

def _compare_chunk(args):
    """Worker of compare_all_groups (own process, one BLAS thread)."""
    mini, o_g, s_g, art, over = args
    try:
        from threadpoolctl import threadpool_limits
        ctx = threadpool_limits(limits=1)
    except Exception:
        import contextlib
        ctx = contextlib.nullcontext()
    with ctx:
        return compare(mini, o_g, s_g, art=art, oracle_over=over)


def compare_all_groups(w, out_gpu: torch.Tensor, stop_gpu: torch.Tensor, *, art: bool, oracle_over: dict | None = None,
                       chunk: int = 2, processes: int | None = None) -> ParityReport:
    """compare() over EVERY (sequence, KV head) group of a (possibly CUDA-resident, full-size) workload: the groups are
    carved out a few at a time (helpers.extract_groups: pure data movement) and handed to the oracle in worker processes,
    one per host core."""
    import multiprocessing as mp
    import os
    import sys
    from helpers import extract_groups
    G = w.group_size
    groups = [(b, g) for b in range(w.batch) for g in range(w.num_kv_heads)]
    jobs = []
    for i in range(0, len(groups), chunk):
        gs = groups[i:i + chunk]
        mini = extract_groups(w, gs)
        o_g = torch.stack([out_gpu[b, ..., g * G:(g + 1) * G, :] for (b, g) in gs]).cpu()
        s_g = torch.stack([stop_gpu[b, g:g + 1] for (b, g) in gs]).cpu()
        jobs.append((mini, o_g, s_g, art, oracle_over))
    here = os.path.dirname(os.path.abspath(__file__))
    os.environ["PYTHONPATH"] = os.pathsep.join([here, os.path.dirname(here), os.environ.get("PYTHONPATH", "")])
    n = processes or min(len(jobs), os.cpu_count() or 1)
    with mp.get_context("spawn").Pool(n) as pool:
        reps = pool.map(_compare_chunk, jobs)
    tot = ParityReport(0, 0, 0, 0, 0.0, 0, 0.0, 0)
    for r in reps:
        tot.mean_stop_frac += r.mean_stop_frac * r.groups
        tot.groups += r.groups; tot.stop_mismatch_nonfragile += r.stop_mismatch_nonfragile
        tot.stop_mismatch_fragile += r.stop_mismatch_fragile; tot.fragile_groups += r.fragile_groups
        tot.max_rel_err = max(tot.max_rel_err, r.max_rel_err); tot.fired_groups += r.fired_groups
        tot.fragile_unreachable += r.fragile_unreachable
    tot.mean_stop_frac /= max(tot.groups, 1)
    return tot
