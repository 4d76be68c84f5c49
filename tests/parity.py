"""Shared GPU-vs-oracle comparison used by the -m gpu parity tests, smoke() and bench.py's checks.

Bars (BASELINE.json north_star): stop_block bit-exact except for groups the ORACLE flags as fragile
(a criterion value within 1e-4 relative of its threshold at a step <= t*), which are reported
separately; outputs within 1e-5 * ||o||_inf (fp32 KV) / 1e-2 * ||o||_inf (bf16 KV, fp32 accumulate).
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np
import torch

from helpers import run_oracle

OUT_TOL = {torch.float32: 1e-5, torch.bfloat16: 1e-2}


@dataclass
class ParityReport:
    groups: int
    stop_mismatch_nonfragile: int
    stop_mismatch_fragile: int
    fragile_groups: int
    max_rel_err: float            # max over compared rows of |gpu - oracle|_inf / |oracle|_inf
    fired_groups: int
    mean_stop_frac: float

    def ok(self, tol: float) -> bool:
        return self.stop_mismatch_nonfragile == 0 and self.max_rel_err <= tol


def compare(w_host, out_gpu: torch.Tensor, stop_gpu: torch.Tensor, *, art: bool, groups=None,
            oracle_over: dict | None = None) -> ParityReport:
    """w_host: the workload on the CPU (the payload the GPU saw, bit for bit)."""
    o_ref, s_ref, res = run_oracle(w_host, art=art, groups=groups, **(oracle_over or {}))
    out = out_gpu.detach().cpu().to(torch.float64).numpy()
    stop = stop_gpu.detach().cpu().numpy().astype(np.int64)
    G = w_host.group_size
    mism_nf = mism_f = frag = fired = 0
    max_rel = 0.0
    fr = []
    for (b, g), r in res.items():
        frag += int(r.fragile)
        fired += int(r.fired)
        fr.append(r.stop_block / max(r.num_blocks, 1))
        if stop[b, g] != s_ref[b, g]:
            if r.fragile:
                mism_f += 1
                continue                       # a legitimately different stop: outputs not comparable
            mism_nf += 1
        d = o_ref.shape[-1]
        for h in range(g * G, (g + 1) * G):
            # one row per query token (q [B, m, Hq, d], reading R15), else the head's single row
            for ref, got in zip(o_ref[b, ..., h, :].reshape(-1, d), out[b, ..., h, :].reshape(-1, d)):
                scale = np.abs(ref).max()
                err = np.abs(got - ref).max()
                if not np.isfinite(err):
                    max_rel = float("inf")
                elif scale > 0:
                    max_rel = max(max_rel, err / scale)
                elif err > 0:
                    max_rel = float("inf")
    return ParityReport(len(res), mism_nf, mism_f, frag, max_rel, fired, float(np.mean(fr)) if fr else 0.0)
