"""Pins for the CPU oracle (oracle/art_oracle.py): things the paper and the mathematics
fix, none of which re-type the oracle's own formulae.  CPU only (-m "not gpu").

Each test names the passage it checks (PAPER.md line) or the DESIGN.md reading.
"""
import math
import os

import numpy as np
import pytest
import torch

from oracle import art_oracle as ao

N = ao.BLOCK_TOKENS
GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def rand_group(seed, G=4, d=64, T=10, vscale=1.0, qscale=1.0):
    rng = np.random.default_rng(seed)
    q = rng.standard_normal((G, d)) * qscale
    K = rng.standard_normal((T, N, d))
    V = rng.standard_normal((T, N, d)) * vscale
    return q, K, V, np.ones((T, N), bool)


def decaying_group(seed, G=4, d=64, T=40, lam=0.6):
    """Keys pushed away from q with age so the stream settles and ART can fire."""
    rng = np.random.default_rng(seed)
    q = rng.standard_normal((G, d))
    qs = (q / np.linalg.norm(q, axis=1, keepdims=True)).sum(0)
    K = rng.standard_normal((T, N, d)) - lam * np.arange(T)[:, None, None] * qs[None, None, :] * math.sqrt(d) / G
    V = rng.standard_normal((T, N, d))
    return q, K, V, np.ones((T, N), bool)


# ------------------------------------------------------------------ ART-off == Eq. 1

@pytest.mark.parametrize("seed", range(4))
def test_out_off_is_textbook_softmax_library(seed):
    """Eq. 1: with termination disabled the streamed o^(T) equals
    softmax(q K^T / sqrt(d)) V computed by a LIBRARY routine (torch CPU fp64)."""
    q, K, V, valid = rand_group(seed, G=3, d=32, T=7)
    valid[-1, 40:] = False                      # ragged tail
    r = ao.art_group(q, K, V, valid, tau=0.0, phi=0.0, patience=5)
    assert r.stop_block == 7 and not r.fired
    Kt = torch.from_numpy(K.reshape(-1, 32)); Vt = torch.from_numpy(V.reshape(-1, 32))
    keep = torch.from_numpy(valid.reshape(-1))
    logits = torch.from_numpy(q) @ Kt[keep].T / math.sqrt(32)
    ref = torch.softmax(logits, dim=-1) @ Vt[keep]
    np.testing.assert_allclose(r.out_off, ref.numpy(), rtol=0, atol=1e-13)
    np.testing.assert_allclose(r.out_on, ref.numpy(), rtol=0, atol=1e-13)
    np.testing.assert_allclose(r.out_textbook, ref.numpy(), rtol=0, atol=1e-13)


def test_reordering_invariance_when_untruncated():
    """if all selected blocks are processed, traversal reordering preserves
    the attention output up to floating-point non-associativity."""
    q, K, V, valid = rand_group(11, T=9)
    base = ao.art_group(q, K, V, valid, 0.0, 0.0, 5).out_off
    perm = np.random.default_rng(0).permutation(9)
    other = ao.art_group(q, K[perm], V[perm], valid[perm], 0.0, 0.0, 5).out_off
    np.testing.assert_allclose(other, base, rtol=0, atol=1e-14)


def test_sm_scale_override_and_default():
    """Eq. 1: default scale is 1/sqrt(d); an explicit sm_scale replaces it (R11)."""
    q, K, V, valid = rand_group(5, G=1, d=64, T=2)
    a = ao.art_group(q, K, V, valid, 0.0, 0.0, 5).out_off
    b = ao.art_group(q, K, V, valid, 0.0, 0.0, 5, sm_scale=0.125).out_off     # 1/sqrt(64)
    c = ao.art_group(q * 2, K, V, valid, 0.0, 0.0, 5, sm_scale=0.0625).out_off
    np.testing.assert_allclose(a, b, atol=1e-15)
    np.testing.assert_allclose(a, c, atol=1e-14)


# ------------------------------------------------------------------ brute force on tiny inputs

def brute_prefix_outputs(q, K, V, valid, scale):
    """Softmax over the first t blocks recomputed FROM SCRATCH for every t."""
    G, d = q.shape
    outs = []
    for t in range(1, K.shape[0] + 1):
        k = K[:t].reshape(-1, d)[valid[:t].reshape(-1)]
        v = V[:t].reshape(-1, d)[valid[:t].reshape(-1)]
        if len(k) == 0:
            outs.append(np.zeros((G, d))); continue
        s = q @ k.T * scale
        p = np.exp(s - s.max(axis=1, keepdims=True))
        outs.append((p / p.sum(axis=1, keepdims=True)) @ v)
    return np.array(outs)


def brute_stop(outs, idx, tau, phi, p):
    """First t with p consecutive stable steps, from the from-scratch prefix outputs;
    Eq. 2 / Eq. 3 written independently of the oracle (math.* on python floats)."""
    T, G, _ = outs.shape
    prev = np.zeros((G, len(idx)))
    run = 0
    for t in range(1, T + 1):
        x = outs[t - 1][:, idx]
        ok = True
        for h in range(G):
            ds = math.sqrt(sum((a - b) ** 2 for a, b in zip(x[h], prev[h])))
            na = math.sqrt(sum(a * a for a in x[h])); nb = math.sqrt(sum(b * b for b in prev[h]))
            dd = 1.0 if na == 0.0 or nb == 0.0 else 1.0 - sum(a * b for a, b in zip(x[h], prev[h])) / (na * nb)
            ok = ok and (ds < tau) and (dd < phi)
        run = run + 1 if ok else 0
        if run >= p:
            return t
        prev = x
    return T


@pytest.mark.parametrize("seed", range(6))
def test_prefix_outputs_match_brute_force(seed):
    """App. A recurrence: o^(t) is the softmax output over the first t blocks."""
    q, K, V, valid = rand_group(seed, G=2, d=64, T=6)
    valid[2, ::3] = False
    valid[4, :] = False                          # a fully masked block still counts as a step (R8)
    r = ao.art_group(q, K, V, valid, 0.0, 0.0, 5, trace=True)
    ref = brute_prefix_outputs(q, K, V, valid, 1 / 8.0)
    np.testing.assert_allclose(r.o, ref, rtol=0, atol=1e-12)


@pytest.mark.parametrize("seed,tau,phi,p", [(0, 3e-2, 1e-2, 3), (1, 5e-2, 1e-2, 2), (2, 2e-2, 5e-3, 4),
                                            (3, 1e-1, 1.0, 1), (4, 3e-2, 1e-3, 5), (5, 1e-5, 1e-3, 5)])
def test_stop_block_matches_brute_force(seed, tau, phi, p):
    """Alg. 1 / Eq. 2 / Eq. 3: t* = first step closing p consecutive stable steps."""
    q, K, V, valid = decaying_group(seed, G=3, d=64, T=30)
    r = ao.art_group(q, K, V, valid, tau, phi, p)
    outs = brute_prefix_outputs(q, K, V, valid, 1 / 8.0)
    t_ref = brute_stop(outs, ao.probe_indices(64, 32), tau, phi, p)
    assert r.stop_block == t_ref
    np.testing.assert_allclose(r.out_on, outs[t_ref - 1], atol=1e-12)
    if seed != 5:
        assert r.fired and r.stop_block < 30     # these settings do terminate early


def test_probe_dim_full_uses_all_coordinates():
    """probe_dim = 0 is P = I ("oracle detector")."""
    q, K, V, valid = decaying_group(7, G=2, d=64, T=30)
    r0 = ao.art_group(q, K, V, valid, 3e-2, 1e-2, 3, probe_dim=0)
    outs = brute_prefix_outputs(q, K, V, valid, 1 / 8.0)
    assert r0.stop_block == brute_stop(outs, np.arange(64), 3e-2, 1e-2, 3)
    assert list(ao.probe_indices(128, 32)[:3]) == [0, 4, 8] and list(ao.probe_indices(64, 32)[-2:]) == [60, 62]


# ------------------------------------------------------------------ recurrence identity

def test_recurrence_identity():
    """o^(t) - o^(t-1) = (l_t / A_t)(u^(t) - o^(t-1));
    PAPER.md:361: x^(t) - x^(t-1) = (l_t / A_t) P (u^(t) - o^(t-1))."""
    q, K, V, valid = rand_group(21, G=4, d=64, T=12)
    r = ao.art_group(q, K, V, valid, 0.0, 0.0, 5, trace=True)
    idx = ao.probe_indices(64, 32)
    for t in range(1, 12):
        lhs = r.o[t] - r.o[t - 1]
        rhs = (r.ell[t] / r.A[t])[:, None] * (r.u[t] - r.o[t - 1])
        np.testing.assert_allclose(lhs, rhs, atol=1e-12)
        np.testing.assert_allclose(np.linalg.norm(lhs[:, idx], axis=1), r.d_scale_all[t], atol=1e-12)
    np.testing.assert_allclose(r.o[0], r.u[0], atol=1e-15)        # o^(1) = u^(1)
    np.testing.assert_allclose(np.cumsum(r.ell, axis=0), r.A, rtol=1e-14)


# ------------------------------------------------------------------ closed forms

def test_golden_harmonic_trace():
    """tests/golden/harmonic_trace.txt: closed-form d_scale, d_direction and t* for q = 0,
    one non-zero first block (Eq. 1-3, App. A); catches a wrong norm, a dropped sqrt(m),
    an off-by-one in the patience counter or in x^(0)."""
    rows = [l.split() for l in open(os.path.join(GOLDEN, "harmonic_trace.txt")) if not l.startswith("#")]
    hdr = [l for l in open(os.path.join(GOLDEN, "harmonic_trace.txt")) if l.startswith("# a=")][0]
    meta = dict(kv.split("=") for kv in hdr[2:].split())
    T, tau, p = int(meta["T"]), float(meta["tau"]), int(meta["p"])
    d = 64
    q = np.zeros((2, d)); K = np.random.default_rng(0).standard_normal((T, N, d))
    V = np.zeros((T, N, d)); V[0] = float(meta["a"])
    r = ao.art_group(q, K, V, np.ones((T, N), bool), tau, 1e-3, p, trace=True)
    assert r.stop_block == int(meta["t_star"])
    for t, ds, dd in rows:
        t = int(t)
        np.testing.assert_allclose(r.d_scale_all[t - 1], float(ds), rtol=1e-12)
        np.testing.assert_allclose(r.d_direction_all[t - 1], float(dd), atol=1e-12)


def test_golden_two_direction_trace():
    """tests/golden/two_direction_trace.txt: a closed form whose d_direction is neither 0 nor 1 (block 1 = e_a, block 2 =
    e_b, then e_a again; q = 0): d_direction^(2) = 1 - 1/sqrt(2), d_scale^(t) = sqrt(2) / (t (t - 1)).  Pins Eq. 2's
    cosine with numbers derived by hand, for two heads and two different coordinate pairs."""
    rows = [l.split() for l in open(os.path.join(GOLDEN, "two_direction_trace.txt")) if not l.startswith("#")]
    T, d = len(rows), 64
    idx = ao.probe_indices(d)
    for a, b in ((int(idx[0]), int(idx[5])), (int(idx[31]), int(idx[2]))):
        q = np.zeros((2, d)); K = np.random.default_rng(1).standard_normal((T, N, d))
        V = np.zeros((T, N, d)); V[:, :, a] = 1.0; V[1, :, a] = 0.0; V[1, :, b] = 1.0
        r = ao.art_group(q, K, V, np.ones((T, N), bool), 0.0, 0.0, 5, trace=True)
        assert abs(r.d_direction_all[1, 0] - (1.0 - 1.0 / np.sqrt(2.0))) < 1e-14
        for t, ds, dd in rows:
            t = int(t)
            np.testing.assert_allclose(r.d_scale_all[t - 1], float(ds), rtol=1e-12)
            np.testing.assert_allclose(r.d_direction_all[t - 1], float(dd), rtol=1e-10, atol=1e-14)


@pytest.mark.parametrize("p", [1, 2, 5, 9])
def test_constant_values_stop_at_p_plus_one(p):
    """Closed form (i): all V rows equal v (v[idx] != 0) => o^(t) = v for all t, so
    d_scale = d_dir = 0 from t = 2 and, step 1 being unstable by R4, t* = p + 1 exactly."""
    q, K, V, valid = rand_group(3, G=4, d=64, T=16)
    v = np.random.default_rng(9).standard_normal(64)
    V[:] = v
    r = ao.art_group(q, K, V, valid, 1e-5, 1e-3, p)
    assert r.stop_block == p + 1 and r.fired
    np.testing.assert_allclose(r.out_on, np.tile(v, (4, 1)), atol=1e-13)
    assert r.d_direction[0].tolist() == [1.0] * 4           # R4: x^(0) = 0 => cos := 0


def test_never_fires_cases():
    """Closed forms (ii), (iii): T <= p with phi <= 1 never fires; tau = 0 or phi = 0 or p > T never fires."""
    q, K, V, valid = rand_group(4, T=5)
    V[:] = 1.0
    assert ao.art_group(q, K, V, valid, 1e-5, 1e-3, 5).stop_block == 5        # T <= p
    assert not ao.art_group(q, K, V, valid, 1e-5, 1e-3, 5).fired
    q, K, V, valid = rand_group(4, T=12)
    V[:] = 1.0
    assert ao.art_group(q, K, V, valid, 0.0, 1e-3, 2).stop_block == 12        # tau = 0, strict '<' (R5)
    assert ao.art_group(q, K, V, valid, 1e-5, 0.0, 2).stop_block == 12        # phi = 0
    assert ao.art_group(q, K, V, valid, 1e-5, 1e-3, 13).stop_block == 12      # p > T
    assert ao.art_group(q, K, V, valid, 1e-5, 1e-3, ao.PATIENCE_INF).stop_block == 12


def test_everything_passes_cases():
    """Closed form (iv): tau = phi = +inf, p = 1 => t* = 1 (step 1 has d_dir = 1 < inf);
    tau = +inf, phi = 1, p = 1 => t* >= 2 because d_dir^(1) = 1 is not < 1 (R4, R5)."""
    q, K, V, valid = rand_group(6, T=8)
    assert ao.art_group(q, K, V, valid, np.inf, np.inf, 1).stop_block == 1
    assert ao.art_group(q, K, V, valid, np.inf, 1.0, 1).stop_block >= 2
    assert ao.art_group(q, K, V, valid, np.inf, np.inf, 3).stop_block == 3


def test_dominant_key_analytic_increment():
    """Closed form (v): one key with a dominating logit in block 1 and value v1 =>
    o^(t-1) ~= v1 and d_scale_t ~= (l_t / A_t) ||P(u^(t) - v1)||, with the
    mass ratio l_t / A_t taken straight from Eq. 1's exponentials."""
    d = 64
    q, K, V, valid = rand_group(8, G=1, d=d, T=6)
    K[0, 5] = 14.0 * q[0] / np.linalg.norm(q[0]) ** 2 * math.sqrt(d)          # logit 14
    r = ao.art_group(q, K, V, valid, 0.0, 0.0, 5, trace=True)
    idx = ao.probe_indices(d, 32)
    e = np.exp(np.einsum("tjd,d->tj", K, q[0]) / math.sqrt(d))              # un-shifted weights
    for t in range(1, 6):
        mass_ratio = e[t].sum() / e[:t + 1].sum()
        expect = mass_ratio * np.linalg.norm((r.u[t, 0] - V[0, 5])[idx])
        np.testing.assert_allclose(r.d_scale_all[t, 0], expect, rtol=2e-2)
        np.testing.assert_allclose(r.ell[t, 0] / r.A[t, 0], mass_ratio, rtol=1e-12)


def test_direction_branch_is_exercised_with_tiny_values():
    """R14: with tiny ||x|| the direction test, not the scale test, decides."""
    q, K, V, valid = rand_group(12, G=2, d=64, T=20, vscale=1e-7)
    r = ao.art_group(q, K, V, valid, 1e-5, 1e-3, 3, trace=True)
    assert (r.d_scale_all[1:] < 1e-5).all()                  # scale test always passes
    assert (r.d_direction_all[1:] > 1e-3).any()              # direction test does not
    r2 = ao.art_group(q, K, V, valid, 1e-5, np.inf, 3)
    assert r2.stop_block < r.stop_block or r.stop_block == 20


# ------------------------------------------------------------------ invariants

def test_convex_combination_invariant():
    """Lemma 3: o^(t) is a convex combination of visited V rows."""
    q, K, V, valid = rand_group(31, G=4, d=64, T=8)
    r = ao.art_group(q, K, V, valid, 0.0, 0.0, 5, trace=True)
    Cv = np.linalg.norm(V.reshape(-1, 64), axis=1).max()
    for t in range(8):
        seen = V[:t + 1].reshape(-1, 64)
        assert (r.o[t] <= seen.max(0) + 1e-12).all() and (r.o[t] >= seen.min(0) - 1e-12).all()
        assert (np.linalg.norm(r.o[t], axis=1) <= Cv + 1e-12).all()
        assert (np.linalg.norm(r.u[t], axis=1) <= Cv + 1e-12).all()
        if t:
            assert (np.linalg.norm(r.u[t] - r.o[t - 1], axis=1) <= 2 * Cv).all()   # Lemma 3


def test_stop_block_monotone_in_thresholds():
    """The (d_scale, d_dir) trajectory does not depend on the thresholds before the stop, so
    t* is non-increasing in tau and in phi and non-decreasing in p."""
    q, K, V, valid = decaying_group(41, G=4, d=64, T=40)
    taus = [1e-4, 1e-3, 1e-2, 1e-1]
    stops = [ao.art_group(q, K, V, valid, t, 1e-2, 3).stop_block for t in taus]
    assert stops == sorted(stops, reverse=True) and stops[0] > stops[-1]
    phis = [1e-6, 1e-4, 1e-2, 1.0]
    stops = [ao.art_group(q, K, V, valid, 1e-1, f, 3).stop_block for f in phis]
    assert stops == sorted(stops, reverse=True)
    ps = [1, 2, 5, 10]
    stops = [ao.art_group(q, K, V, valid, 3e-2, 1e-2, p).stop_block for p in ps]
    assert stops == sorted(stops)


def test_group_and_rule_vs_single_heads():
    """R2: AND over heads with one counter == min over heads of per-head counters, so the
    group t* >= max over heads of the single-head t*."""
    q, K, V, valid = decaying_group(43, G=4, d=64, T=40)
    tg = ao.art_group(q, K, V, valid, 3e-2, 1e-2, 3).stop_block
    singles = [ao.art_group(q[h:h + 1], K, V, valid, 3e-2, 1e-2, 3).stop_block for h in range(4)]
    assert tg >= max(singles)
    assert ao.art_group(q[:1], K, V, valid, 3e-2, 1e-2, 3).stop_block == singles[0]   # G = 1 reduces to the paper's rule


# ------------------------------------------------------------------ truncation error (App. A)

@pytest.mark.parametrize("seed", range(8))
def test_truncation_bounds(seed):
    """Skipped-mass bound, telescoped bound (PAPER.md:411 corrected), Thm 2 with mu_emp
     and Thm 1 form with nu_emp."""
    tau, phi, p = 3e-2, 1e-2, 3
    q, K, V, valid = decaying_group(100 + seed, G=2, d=64, T=36, lam=0.35)
    r = ao.art_group(q, K, V, valid, tau, phi, p, trace=True)
    T, ts = r.num_blocks, r.stop_block
    if not r.fired or ts == T:
        pytest.skip("did not fire early")
    idx = ao.probe_indices(64, 32)
    Cv = np.linalg.norm(V.reshape(-1, 64), axis=1).max()
    b = ts - p + 1
    for h in range(2):
        err = np.linalg.norm(r.out_off[h] - r.out_on[h])
        A, ell, u, o = r.A[:, h], r.ell[:, h], r.u[:, h], r.o[:, h]
        # (a) skipped mass
        assert err <= 2 * Cv * (A[-1] - A[ts - 1]) / A[-1] + 1e-12
        # (b) telescoped
        tele = sum(ell[j - 1] / A[j - 1] * np.linalg.norm(u[j - 1] - o[j - 2]) for j in range(ts + 1, T + 1))
        assert err <= tele + 1e-12
        assert tele <= 2 * Cv * sum(ell[j - 1] / A[j - 1] for j in range(ts + 1, T + 1)) + 1e-12
        # (c) Thm 2 with mu_emp = max_{j>=b} j l_j / A_j (Lemma 1 by construction)
        mu = max(j * ell[j - 1] / A[j - 1] for j in range(b, T + 1))
        assert err <= 2 * mu * Cv * math.log(T / ts) + 1e-12
        # (d) Thm 1 form
        incr = [o[j - 1] - o[j - 2] for j in range(ts + 1, T + 1)]
        nu = min(np.linalg.norm(z[idx]) / np.linalg.norm(z) for z in incr if np.linalg.norm(z) > 0)
        pn = lambda j: np.linalg.norm((u[j - 1] - o[j - 2])[idx])
        Delta = max(pn(j) - pn(b) for j in range(b, T + 1))                 # Def. 1
        assert r.d_scale_all[b - 1, h] < tau                                 # Def. 2
        if nu > 0 and ell[b - 1] > 0:                                        # Assumption 2 needs nu > 0
            bound = mu * ((A[b - 1] / ell[b - 1]) * tau + Delta) / nu * math.log(T / ts)
            assert err <= bound + 1e-12


# ------------------------------------------------------------------ traversal, masks, paging

def test_traversal_orders():
    """PAPER.md:171-173 + reading R3."""
    assert ao.traversal_blocks(ao.POLICY_DENSE, 200) == [3, 2, 1, 0]
    assert ao.traversal_blocks(ao.POLICY_DENSE, 0) == []
    assert ao.traversal_blocks(ao.POLICY_DENSE, 64) == [0]
    # sink(4) + window(128) over L = 1000: window covers tokens 872..999 -> blocks 13,14,15
    assert ao.traversal_blocks(ao.POLICY_SINK_WINDOW, 1000, 4, 128) == [0, 15, 14, 13]
    # window reaching into block 0: block 0 still first, visited once
    assert ao.traversal_blocks(ao.POLICY_SINK_WINDOW, 150, 4, 120) == [0, 2, 1]
    assert ao.traversal_blocks(ao.POLICY_SINK_WINDOW, 150, 0, 70) == [2, 1]
    assert ao.traversal_blocks(ao.POLICY_SINK_WINDOW, 150, 0, 0) == []
    assert ao.traversal_blocks(ao.POLICY_SINK_WINDOW, 300, 100, 64) == [0, 4, 3, 1]   # sink spilling into block 1
    assert ao.traversal_blocks(ao.POLICY_LIST, 999, block_list=[7, 2, 9]) == [7, 2, 9]
    m = ao.eligible_token_mask(ao.POLICY_SINK_WINDOW, 1000, 0, 4, 128)
    assert m[:4].all() and not m[4:].any()
    m = ao.eligible_token_mask(ao.POLICY_SINK_WINDOW, 1000, 13, 4, 128)
    assert not m[:40].any() and m[40:].all()                    # 872 = 13*64 + 40
    m = ao.eligible_token_mask(ao.POLICY_DENSE, 1000, 15)
    assert m[:40].all() and not m[40:].any()                    # 1000 = 15*64 + 40


def _paged_problem(seed, B=2, Hkv=2, G=2, d=64, lens=(300, 130), layout=ao.LAYOUT_HND):
    rng = np.random.default_rng(seed)
    nblk = [-(-L // N) for L in lens]
    pages = rng.permutation(sum(nblk) + 3)                       # a few unused pages too
    table = np.zeros((B, max(nblk)), dtype=np.int32); off = 0
    for b in range(B):
        table[b, :nblk[b]] = pages[off:off + nblk[b]]; off += nblk[b]
    shape = (len(pages), Hkv, N, d) if layout == ao.LAYOUT_HND else (len(pages), N, Hkv, d)
    kc = rng.standard_normal(shape); vc = rng.standard_normal(shape)
    q = rng.standard_normal((B, Hkv * G, d))
    return q, kc, vc, table, np.array(lens)


def test_whole_step_matches_dense_library_softmax_and_layouts():
    """The paged driver (block_table, GQA mapping h -> h // G, partial last block, NaN in the
    masked tail) against torch softmax on the gathered logical sequence; HND == NHD."""
    q, kc, vc, table, lens = _paged_problem(3)
    for b in range(2):                                           # poison the masked tail
        L = lens[b]; last = table[b, -(-L // N) - 1]
        kc[last, :, L % N:] = np.nan; vc[last, :, L % N:] = np.nan
    out, stop, _ = ao.art_decode_attention_oracle(q, kc, vc, table, lens, num_kv_heads=2, art=False)
    for b in range(2):
        L = lens[b]; nb = -(-L // N)
        assert (stop[b] == nb).all()
        for h in range(4):
            g = h // 2
            Kl = kc[table[b, :nb], g].reshape(-1, 64)[:L]; Vl = vc[table[b, :nb], g].reshape(-1, 64)[:L]
            ref = torch.softmax(torch.from_numpy(q[b, h] @ Kl.T / 8.0), -1).numpy() @ Vl
            np.testing.assert_allclose(out[b, h], ref, atol=1e-13)
    out2, stop2, _ = ao.art_decode_attention_oracle(
        q, kc.transpose(0, 2, 1, 3).copy(), vc.transpose(0, 2, 1, 3).copy(), table, lens,
        num_kv_heads=2, layout=ao.LAYOUT_NHD, art=False)
    assert np.array_equal(out, out2) and np.array_equal(stop, stop2)


def test_page_permutation_changes_nothing_bitwise():
    """Permuting physical pages (and block_table with them) changes nothing bit-for-bit."""
    q, kc, vc, table, lens = _paged_problem(5)
    a = ao.art_decode_attention_oracle(q, kc, vc, table, lens, num_kv_heads=2, tau=5e-2, phi=1e-2, patience=2)
    perm = np.random.default_rng(1).permutation(kc.shape[0])     # new_page = perm[old_page]
    kc2 = np.empty_like(kc); vc2 = np.empty_like(vc)
    kc2[perm] = kc; vc2[perm] = vc
    b = ao.art_decode_attention_oracle(q, kc2, vc2, perm[table].astype(np.int32), lens, num_kv_heads=2,
                                       tau=5e-2, phi=1e-2, patience=2)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])


def test_sink_window_and_list_policies_against_library_softmax():
    """Token-level eligibility E (R8): sink + window and an explicit list, ART off."""
    q, kc, vc, table, lens = _paged_problem(9, lens=(700, 400))
    out, stop, _ = ao.art_decode_attention_oracle(q, kc, vc, table, lens, num_kv_heads=2, art=False,
                                                  policy=ao.POLICY_SINK_WINDOW, sink_tokens=4, window_tokens=200)
    for b in range(2):
        L = lens[b]; nb = -(-L // N)
        keep = np.r_[0:4, L - 200:L]
        assert stop[b, 0] == len(ao.traversal_blocks(ao.POLICY_SINK_WINDOW, L, 4, 200))
        for h in range(4):
            Kl = kc[table[b, :nb], h // 2].reshape(-1, 64)[keep]; Vl = vc[table[b, :nb], h // 2].reshape(-1, 64)[keep]
            ref = torch.softmax(torch.from_numpy(q[b, h] @ Kl.T / 8.0), -1).numpy() @ Vl
            np.testing.assert_allclose(out[b, h], ref, atol=1e-13)
    lists = np.array([[[5, 0, 10, 3], [1, 2, 0, 0]], [[6, 2, 0, 0], [0, 0, 0, 0]]], dtype=np.int32)
    counts = np.array([[4, 2], [2, 0]], dtype=np.int32)
    out, stop, _ = ao.art_decode_attention_oracle(q, kc, vc, table, lens, num_kv_heads=2, art=False,
                                                  policy=ao.POLICY_LIST, eligible_blocks=lists, eligible_counts=counts)
    assert stop.tolist() == [[4, 2], [2, 0]]
    assert (out[1, 2:] == 0).all()                               # empty list => zero rows, stop 0
    toks = lambda blks, L: np.concatenate([np.arange(b * N, min((b + 1) * N, L)) for b in blks])
    for (b, g, blks) in [(0, 0, [5, 0, 10, 3]), (0, 1, [1, 2]), (1, 0, [6, 2])]:
        L = lens[b]; nb = -(-L // N); keep = toks(blks, L)
        for h in (2 * g, 2 * g + 1):
            Kl = kc[table[b, :nb], g].reshape(-1, 64)[keep]; Vl = vc[table[b, :nb], g].reshape(-1, 64)[keep]
            ref = torch.softmax(torch.from_numpy(q[b, h] @ Kl.T / 8.0), -1).numpy() @ Vl
            np.testing.assert_allclose(out[b, h], ref, atol=1e-13)


def test_empty_and_degenerate_inputs():
    """Edge conventions: seq_len = 0 => zero row, stop 0; a list of blocks wholly
    beyond L => steps counted, output 0, never stable for phi <= 1 (x stays 0, R4)."""
    q, kc, vc, table, lens = _paged_problem(13, lens=(0, 100))
    out, stop, res = ao.art_decode_attention_oracle(q, kc, vc, table, lens, num_kv_heads=2)
    assert (out[0] == 0).all() and (stop[0] == 0).all() and (stop[1] == 2).all()
    lists = np.array([[[0, 0]] * 2, [[7, 9]] * 2], dtype=np.int32); counts = np.array([[0, 0], [2, 2]], np.int32)
    out, stop, res = ao.art_decode_attention_oracle(q, kc, vc, table, lens, num_kv_heads=2, policy=ao.POLICY_LIST,
                                                    eligible_blocks=lists, eligible_counts=counts, patience=1)
    assert (out[1] == 0).all() and (stop[1] == 2).all() and not res[(1, 0)].fired


def test_fragile_flag():
    """north_star: a group is reported separately when a criterion value lies within 1e-4
    relative of its threshold at a step <= t*."""
    q, K, V, valid = decaying_group(51, G=2, d=64, T=30)
    r = ao.art_group(q, K, V, valid, 3e-2, 1e-2, 3, trace=True)
    assert not r.fragile
    v = float(r.d_scale[4, 1])
    assert ao.art_group(q, K, V, valid, v * (1 + 5e-5), 1e-2, 3).fragile
    assert not ao.art_group(q, K, V, valid, v * (1 + 5e-3), 1e-2, 3).fragile
