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


def extract_groups(w, groups):
    """Pure data movement: carve the (b, g) groups out of a (possibly CUDA-resident, full-size)
    workload into a small CPU workload with batch = len(groups), Hkv = 1, Hq = G, identity paging.
    Lets the oracle check sampled outputs of the BASELINE-size configs one by one."""
    from dataclasses import replace
    from workloads.generators import LAYOUT_HND, POLICY_LIST
    G, d = w.group_size, w.head_dim
    qs, ks, vs, lens, tables, lists, counts = [], [], [], [], [], [], []
    page0 = 0
    for (b, g) in groups:
        L = int(w.seq_lens[b]); nb = (L + 63) // 64
        pages = w.block_table[b, :nb].long()
        if w.layout == LAYOUT_HND:
            kb, vb = w.k_cache[pages, g], w.v_cache[pages, g]
        else:
            kb, vb = w.k_cache[pages, :, g], w.v_cache[pages, :, g]
        ks.append(kb.cpu().unsqueeze(1)); vs.append(vb.cpu().unsqueeze(1))      # [nb, 1, 64, d] (HND)
        qs.append(w.q[b, g * G:(g + 1) * G].cpu())
        lens.append(L); tables.append(torch.arange(page0, page0 + nb, dtype=torch.int32)); page0 += nb
        if w.policy == POLICY_LIST:
            lists.append(w.eligible_blocks[b, g].cpu()); counts.append(int(w.eligible_counts[b, g]))
    maxb = max(1, max(len(t) for t in tables))
    bt = torch.zeros((len(groups), maxb), dtype=torch.int32)
    for i, t in enumerate(tables):
        bt[i, :len(t)] = t
    k_cache = torch.cat(ks) if page0 else torch.zeros((1, 1, 64, d), dtype=w.dtype)
    v_cache = torch.cat(vs) if page0 else torch.zeros((1, 1, 64, d), dtype=w.dtype)
    el = ec = None
    if w.policy == POLICY_LIST:
        el = torch.stack(lists).unsqueeze(1); ec = torch.tensor(counts, dtype=torch.int32).unsqueeze(1)
    return replace(w, batch=len(groups), num_q_heads=G, num_kv_heads=1, layout=LAYOUT_HND,
                   q=torch.stack(qs), k_cache=k_cache, v_cache=v_cache, block_table=bt,
                   seq_lens=torch.tensor(lens, dtype=torch.int32), eligible_blocks=el, eligible_counts=ec)
