"""Test-side glue: hand a Workload (torch tensors) to the numpy oracle."""
from __future__ import annotations

import numpy as np
import torch

from oracle import art_oracle as ao


def np64(t: torch.Tensor) -> np.ndarray:
    """Exact widening of an fp32 / bf16 payload to float64."""
    return t.detach().to("cpu").to(torch.float64).numpy()


def thresholds_f32(w):
    """The ABI carries tau / phi as fp32; the oracle compares against the same values."""
    return float(np.float32(w.tau)), float(np.float32(w.phi))


def run_oracle(w, *, art: bool = True, groups=None, trace: bool = False, **over):
    tau, phi = thresholds_f32(w)
    kw = dict(num_kv_heads=w.num_kv_heads, policy=w.policy, layout=w.layout,
              sink_tokens=w.sink_tokens, window_tokens=w.window_tokens,
              eligible_blocks=None if w.eligible_blocks is None else w.eligible_blocks.cpu().numpy(),
              eligible_counts=None if w.eligible_counts is None else w.eligible_counts.cpu().numpy(),
              tau=tau, phi=phi, patience=w.patience, probe_dim=w.probe_dim, art=art,
              groups=groups, trace=trace)
    kw.update(over)
    return ao.art_decode_attention_oracle(
        np64(w.q), np64(w.k_cache), np64(w.v_cache), w.block_table.cpu().numpy(),
        w.seq_lens.cpu().numpy(), **kw)
