"""-m gpu: seeded random shapes / policies / thresholds / schedules against the fp64 oracle.  Every case goes
through the same check as the hand-written parity tests (stop blocks exact on non-fragile groups, outputs within
tolerance, loaded >= processed).  ART_FUZZ_EXTRA=N adds N further seeds to each of the two families (a sweep to run by
hand after a kernel change: `ART_FUZZ_EXTRA=1500 python -m pytest tests/test_gpu_fuzz.py -m gpu -x -q`; the default suite
runs the 48 + 32 committed seeds only)."""
import os

import numpy as np
import pytest
import torch

from workloads import generators as gen
from test_gpu_parity import check

pytestmark = pytest.mark.gpu


def random_case(seed):
    rng = np.random.default_rng(1000 + seed)
    bf16 = bool(rng.integers(0, 4) > 0)                      # mostly the bf16 tensor-core path
    dtype, d = (torch.bfloat16, 128) if bf16 else (torch.float32, 64)
    G = int(rng.choice([1, 2, 3, 4, 5, 6, 7, 8]))
    Hkv = int(rng.integers(1, 4))
    B = int(rng.integers(1, 5))
    lens = [int(rng.choice([0, 1, 63, 64, 65, int(rng.integers(100, 6000))], p=[.05, .05, .05, .05, .05, .75])) for _ in range(B)]
    policy = int(rng.choice([gen.POLICY_DENSE, gen.POLICY_SINK_WINDOW, gen.POLICY_LIST]))
    kw = {}
    if policy == gen.POLICY_SINK_WINDOW:
        kw = dict(sink_tokens=int(rng.choice([0, 4, 70, 200])), window_tokens=int(rng.choice([0, 100, 1000, 4096])))
    elif policy == gen.POLICY_LIST:
        kw = dict(topk_blocks=int(rng.integers(1, 40)))
    layout = int(rng.choice([gen.LAYOUT_HND, gen.LAYOUT_NHD])) if bf16 else gen.LAYOUT_HND
    w = gen.make_workload(f"fuzz{seed}", seed=7000 + seed, batch=B, num_q_heads=G * Hkv, num_kv_heads=Hkv, head_dim=d,
                          seq_lens=lens, dtype=dtype, policy=policy, layout=layout,
                          recency_decay=(0.05, 1.0) if rng.integers(0, 4) else None,
                          planted_frac=0.01 if rng.integers(0, 2) else 0.0, **kw)
    th = dict(tau=float(rng.choice([1e-5, 3e-4, 1e-3, 5e-3])), phi=float(rng.choice([1e-3, 1e-2, float("inf")])),
              patience=int(rng.choice([1, 2, 5, 7])), probe_dim=int(rng.choice([32, 32, 0])))
    splits = [0, 1, 2, 4, 8, 16] + ([3, 5, -1, -1] if bf16 else [])
    return w, th, int(rng.choice(splits))


@pytest.mark.parametrize("seed", range(48))
def test_random_case(seed):
    w, th, split = random_case(seed)
    check(w, split=split, **th)
    check(w, art_on=False, split=split)


def random_multi_token_case(seed):
    """q_len = m > 1 (reading R15): m * G <= 8, bf16, cluster schedules."""
    rng = np.random.default_rng(5000 + seed)
    m = int(rng.choice([2, 3, 4, 5, 8]))
    G = int(rng.integers(1, 8 // m + 1))
    Hkv = int(rng.integers(1, 4))
    B = int(rng.integers(1, 5))
    lens = [int(rng.choice([0, 1, 3, 63, 64, 65, 66, 70, 129, int(rng.integers(100, 6000))],
                           p=[.03, .03, .03, .03, .03, .03, .03, .03, .03, .73])) for _ in range(B)]
    policy = int(rng.choice([gen.POLICY_DENSE, gen.POLICY_SINK_WINDOW, gen.POLICY_LIST]))
    kw = {}
    if policy == gen.POLICY_SINK_WINDOW:
        kw = dict(sink_tokens=int(rng.choice([0, 4, 70, 200])), window_tokens=int(rng.choice([0, 3, 100, 1000, 4096])))
    elif policy == gen.POLICY_LIST:
        kw = dict(topk_blocks=int(rng.integers(1, 40)))
    w = gen.make_workload(f"fuzzm{seed}", seed=9000 + seed, batch=B, num_q_heads=G * Hkv, num_kv_heads=Hkv, head_dim=128,
                          seq_lens=lens, policy=policy, layout=int(rng.choice([gen.LAYOUT_HND, gen.LAYOUT_NHD])),
                          recency_decay=(0.05, 1.0) if rng.integers(0, 4) else None,
                          planted_frac=0.01 if rng.integers(0, 2) else 0.0, **kw)
    w = gen.with_query_tokens(w, m, seed=9500 + seed, jitter=float(rng.choice([0.0, 0.3, 1.0])))
    th = dict(tau=float(rng.choice([1e-5, 3e-4, 1e-3, 5e-3])), phi=float(rng.choice([1e-3, 1e-2, float("inf")])),
              patience=int(rng.choice([1, 2, 5, 7])), probe_dim=int(rng.choice([32, 32, 0])))
    return w, th, int(rng.choice([0, 1, 2, 3, 4, 5, 8, 16]))


@pytest.mark.parametrize("seed", range(32))
def test_random_multi_token_case(seed):
    w, th, split = random_multi_token_case(seed)
    check(w, split=split, **th)
    check(w, art_on=False, split=split)


EXTRA = int(os.environ.get("ART_FUZZ_EXTRA", "0"))


@pytest.mark.skipif(EXTRA == 0, reason="ART_FUZZ_EXTRA not set")
@pytest.mark.parametrize("seed", range(48, 48 + max(EXTRA, 1)))
def test_random_case_extra(seed):
    test_random_case(seed)


@pytest.mark.skipif(EXTRA == 0, reason="ART_FUZZ_EXTRA not set")
@pytest.mark.parametrize("seed", range(32, 32 + max(EXTRA, 1)))
def test_random_multi_token_case_extra(seed):
    test_random_multi_token_case(seed)
