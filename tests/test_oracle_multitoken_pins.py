"""Pins for the oracle's multi-token queries (reading R15): m query tokens per sequence that
sit at the last m positions, each attending causally, one walk over the blocks and one decision per group.

Pinned against things other than the oracle itself: torch's scaled_dot_product_attention with an explicit causal
mask (library routine), the already pinned single-token path on a shorter sequence, a from-scratch brute force of
the prefix outputs and of Eq. 2 / Eq. 3 on python floats, and the monotonicity the AND rule implies.
"""
import math

import numpy as np
import pytest
import torch

from oracle import art_oracle as ao
from test_oracle_pins import _paged_problem, brute_stop, decaying_group

N = ao.BLOCK_TOKENS


def _multi_problem(seed, m, lens=(300, 130), G=2, Hkv=2, layout=ao.LAYOUT_HND):
    q1, kc, vc, table, lens = _paged_problem(seed, B=len(lens), Hkv=Hkv, G=G, lens=lens, layout=layout)
    rng = np.random.default_rng(seed + 1000)
    q = rng.standard_normal((len(lens), m, Hkv * G, 64))
    return q, kc, vc, table, lens


@pytest.mark.parametrize("m,lens", [(2, (300, 130)), (3, (65, 128)), (4, (66, 7)), (8, (200, 64))])
def test_off_matches_library_sdpa_with_causal_mask(m, lens):
    """ART-off, DENSE: row (i, h) is softmax attention over tokens j <= L - m + i (Eq. 1 + causal mask), against
    torch.nn.functional.scaled_dot_product_attention with a boolean mask.  lens 65/66 with m = 3/4: the first
    query tokens see nothing of the most recent block (a row whose first step is empty)."""
    G, Hkv = (1, 2) if m == 8 else (2, 2)
    q, kc, vc, table, lens = _multi_problem(11 + m, m, lens=lens, G=G, Hkv=Hkv)
    out, stop, _ = ao.art_decode_attention_oracle(q, kc, vc, table, lens, num_kv_heads=Hkv, art=False)
    assert out.shape == q.shape
    for b, L in enumerate(lens):
        nb = -(-L // N)
        assert (stop[b] == nb).all()
        for g in range(Hkv):
            Kl = torch.from_numpy(kc[table[b, :nb], g].reshape(-1, 64)[:L])
            Vl = torch.from_numpy(vc[table[b, :nb], g].reshape(-1, 64)[:L])
            qq = torch.from_numpy(q[b, :, g * G:(g + 1) * G]).permute(1, 0, 2)            # [G, m, d]
            mask = torch.arange(L)[None, :] <= (L - m + torch.arange(m))[:, None]         # [m, L]
            ref = torch.nn.functional.scaled_dot_product_attention(
                qq[None], Kl[None, None].expand(1, G, L, 64), Vl[None, None].expand(1, G, L, 64),
                attn_mask=mask[None, None])[0]                                           # [G, m, d]
            np.testing.assert_allclose(out[b, :, g * G:(g + 1) * G], ref.permute(1, 0, 2).numpy(), atol=1e-13)


def test_each_row_is_the_single_token_path_on_a_shorter_sequence():
    """Row i of an m-token call == the (pinned) single-token oracle with seq_len L - (m - 1 - i), ART-off."""
    m = 4
    q, kc, vc, table, lens = _multi_problem(3, m, lens=(259, 130))
    out, _, _ = ao.art_decode_attention_oracle(q, kc, vc, table, lens, num_kv_heads=2, art=False)
    for i in range(m):
        o1, _, _ = ao.art_decode_attention_oracle(q[:, i], kc, vc, table, lens - (m - 1 - i), num_kv_heads=2, art=False)
        np.testing.assert_allclose(out[:, i], o1, atol=1e-13)


def test_one_query_token_is_the_old_path_bitwise():
    q, kc, vc, table, lens = _multi_problem(5, 1)
    kw = dict(num_kv_heads=2, tau=5e-2, phi=1e-2, patience=2)
    a = ao.art_decode_attention_oracle(q, kc, vc, table, lens, **kw)
    b = ao.art_decode_attention_oracle(q[:, 0], kc, vc, table, lens, **kw)
    assert np.array_equal(a[0][:, 0], b[0]) and np.array_equal(a[1], b[1])


def test_query_tokens_before_the_sequence_start_give_zero_rows():
    """L < m: query tokens at negative positions have no eligible token -> zero rows; the rest still exact."""
    m = 4
    q, kc, vc, table, lens = _multi_problem(9, m, lens=(2, 70))
    out, stop, _ = ao.art_decode_attention_oracle(q, kc, vc, table, lens, num_kv_heads=2, art=False)
    assert np.array_equal(out[0, :2], np.zeros_like(out[0, :2]))            # positions -2, -1
    np.testing.assert_allclose(out[0, 2, 0], vc[table[0, 0], 0, 0], atol=1e-13)   # position 0 sees token 0 only
    assert (stop[0] == 1).all()


def _rows_problem(seed, m=3, G=2, T=24, cut_last=True):
    """A group whose stream settles, as m * G rows with per-row causal masks over the most recent block."""
    q, K, V, valid = decaying_group(seed, G=m * G, d=64, T=T)
    rv = np.repeat(valid[None], m * G, axis=0).copy()
    if cut_last:
        for i in range(m):                                       # traversal step 1 = most recent block
            c = m - 1 - i
            if c:
                rv[i * G:(i + 1) * G, 0, N - c:] = False
    return q, K, V, rv


def _brute_rows(q, K, V, rv, scale):
    """Prefix outputs per row, from scratch for every t, with that row's own mask."""
    R, d = q.shape
    T = K.shape[0]
    outs = np.zeros((T, R, d))
    for t in range(1, T + 1):
        for r in range(R):
            sel = rv[r, :t].reshape(-1)
            k = K[:t].reshape(-1, d)[sel]; v = V[:t].reshape(-1, d)[sel]
            if len(k) == 0:
                continue
            s = k @ q[r] * scale
            p = np.exp(s - s.max())
            outs[t - 1, r] = (p / p.sum()) @ v
    return outs


@pytest.mark.parametrize("seed,tau,phi,p", [(0, 3e-2, 1e-2, 3), (1, 5e-2, 1e-2, 2), (2, 2e-2, 5e-3, 4)])
def test_stop_block_with_row_masks_matches_brute_force(seed, tau, phi, p):
    """One counter for the group, AND over all m * G rows (R15), prefix outputs under per-row masks."""
    q, K, V, rv = _rows_problem(seed)
    r = ao.art_group(q, K, V, rv, tau, phi, p, trace=True)
    outs = _brute_rows(q, K, V, rv, 1 / 8.0)
    np.testing.assert_allclose(r.o, outs, atol=1e-12)
    t_ref = brute_stop(outs, ao.probe_indices(64, 32), tau, phi, p)
    assert r.stop_block == t_ref and r.fired and t_ref < K.shape[0]
    np.testing.assert_allclose(r.out_on, outs[t_ref - 1], atol=1e-12)


def test_a_row_with_an_empty_first_step_cannot_be_stable_there():
    """R4 per row: a row that has seen no token yet has x = 0, d_direction = 1, so step 1 is never stable even with
    huge thresholds on the other rows; brute force agrees."""
    q, K, V, rv = _rows_problem(4, m=2, G=1, T=8)
    rv[0, 0, :] = False                                          # row 0 sees nothing of the most recent block
    r = ao.art_group(q, K, V, rv, 1e9, 0.999, 1, trace=True)
    assert not r.stable[0] and r.d_direction[0, 0] == 1.0 and r.d_scale[0, 0] == 0.0
    outs = _brute_rows(q, K, V, rv, 1 / 8.0)
    assert r.stop_block == brute_stop(outs, ao.probe_indices(64, 32), 1e9, 0.999, 1)


def test_more_rows_never_stop_earlier():
    """AND over rows: the group with all rows stops no earlier than any subset of its rows would."""
    q, K, V, rv = _rows_problem(6, m=4, G=2, T=30)
    full = ao.art_group(q, K, V, rv, 3e-2, 1e-2, 3).stop_block
    for rows in ([0, 1], [2, 3], [4, 5, 6, 7], [0, 7]):
        sub = ao.art_group(q[rows], K, V, rv[rows], 3e-2, 1e-2, 3).stop_block
        assert sub <= full


def test_sink_window_multi_token_against_masked_library_softmax():
    """SINK_WINDOW with m = 2: the policy's set is the group's (relative to L), each row is cut causally."""
    m = 2
    q, kc, vc, table, lens = _multi_problem(21, m, lens=(300, 131))
    out, stop, _ = ao.art_decode_attention_oracle(q, kc, vc, table, lens, num_kv_heads=2, art=False,
                                                  policy=ao.POLICY_SINK_WINDOW, sink_tokens=4, window_tokens=100)
    for b, L in enumerate(lens):
        nb = -(-L // N)
        j = np.arange(L)
        E = (j < 4) | (j >= L - 100)
        for i in range(m):
            Ei = E & (j <= L - m + i)
            for h in range(4):
                g = h // 2
                Kl = kc[table[b, :nb], g].reshape(-1, 64)[:L][Ei]; Vl = vc[table[b, :nb], g].reshape(-1, 64)[:L][Ei]
                ref = torch.softmax(torch.from_numpy(q[b, i, h] @ Kl.T / 8.0), -1).numpy() @ Vl
                np.testing.assert_allclose(out[b, i, h], ref, atol=1e-13)
