"""CPU fp64 oracle for ART decode attention (arXiv 2606.00024).

TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only ``tests/``, ``__graft_entry__.smoke()``
and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import this
module.  It shares no code with the CUDA path under ``paper_2606_00024_b200/`` and
imports nothing from it.

What it is: ART is a heuristic truncation, so the oracle is the paper's algorithm
written out step by step in the paper's order and notation, in float64 (numpy):

* Eq. 1            O = softmax(Q K^T / sqrt(d)) V
* App. A recurrence
      l_t = sum_k exp(q k_{t,k} / sqrt(d)),  A_t = sum_{j<=t} l_j,
      o^(t) = (A_{t-1} o^(t-1) + l_t u^(t)) / A_t
* Algorithm 1 (reconstruction in DESIGN.md)
* Eq. 2           d_scale = ||x^(t) - x^(t-1)||_2,
                                 d_direction = 1 - cos(x^(t), x^(t-1))
* Eq. 3           c^(t) = c^(t-1)+1 if stable else 0; stop when c^(t) >= p
* traversal orders

Readings of the paper taken where it is silent (DESIGN.md "Readings" R1..R11):
R1 probe = coordinate subsample idx_k = k*(d/32) of the NORMALISED output (m = 32;
probe_dim = 0 selects all d coordinates); R2 per-head criterion, logical AND over
the G heads of a GQA group, one patience counter per group; R3 sink block first,
then descending; R4 zero-norm => cos := 0 => d_direction = 1; R5 strict '<' for
both tests, '>=' for the trigger; R6 probe on the normalised o^(t); R8 masked
tokens have weight 0 and a block with no valid token still counts as a step;
R9 stop_block = t* = number of blocks processed; R15 (multi-token
queries: speculative decode / the tail of a chunked prefill): the m query tokens of a
sequence are its LAST m positions, query token i attends causally to the eligible
tokens j <= L - m + i, the group walks its blocks ONCE for all m tokens and the
criterion is the AND over all m * G (token, head) rows -- R2 with more rows.

Parity pins: every function here is pinned by ``tests/test_oracle_*.py`` against
closed forms, brute force, a library softmax, the paper's inequalities and a
hand-derived golden trace (tests/golden/).  The readings R1-R4 themselves are
"parity unpinned" in the sense of DESIGN.md: the paper prints no worked numerical
example of the kernel, so nothing external can confirm them.

No blocking, fusion or reordering beyond what the recurrence states: the global
max M_h is taken in a first pass over all eligible tokens (softmax is shift
invariant), deliberately NOT the running-max rescaling a GPU
kernel uses.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

BLOCK_TOKENS = 64          # n: tokens per KV block = per page (BASELINE.json configs)

POLICY_DENSE = 0           # full KV, reverse temporal order
POLICY_SINK_WINDOW = 1     # StreamingLLM-style sink + recent window
POLICY_LIST = 2            # explicit importance-ordered block list

LAYOUT_HND = 0             # cache[page, kv_head, token, d]
LAYOUT_NHD = 1             # cache[page, token, kv_head, d]

# Paper defaults, PAPER.md:200 (section 4.1)
DEFAULT_TAU = 1e-5
DEFAULT_PHI = 1e-3
DEFAULT_PATIENCE = 5
DEFAULT_PROBE_DIM = 32
PATIENCE_INF = 2**31 - 1   # "p = infinity" mode of App. E

FRAGILE_REL = 1e-4         # north_star's near-threshold band


def probe_indices(head_dim: int, probe_dim: int = DEFAULT_PROBE_DIM) -> np.ndarray:
    """Reading R1: P is a coordinate subsample, idx_k = k * (d / m), k = 0..m-1.

    PAPER.md:99,135 describe a 32-element "deterministic, scattered subsample of
    the full head dimension"; App. A only needs P linear.
    probe_dim = 0 (or = d) selects P = I, the paper's own "oracle detector"
    (PAPER.md:441).
    """
    if probe_dim in (0, head_dim):
        return np.arange(head_dim)
    if head_dim % probe_dim != 0:
        raise ValueError("probe_dim must divide head_dim")
    return np.arange(probe_dim) * (head_dim // probe_dim)


def traversal_blocks(policy: int, seq_len: int, sink_tokens: int = 0,
                     window_tokens: int = 0, block_list=None) -> list[int]:
    """Logical block ids in the order ART walks them.

    DENSE: most recent block first.
    SINK_WINDOW: blocks meeting E = {j < sink} U {j >= L - window}; block 0 first
    if it holds sink tokens (reading R3: "explicitly preserving the sink blocks",
    PAPER.md:172), then the rest in descending index.
    LIST: exactly the list given (caller supplies descending priority).
    """
    n = BLOCK_TOKENS
    L = int(seq_len)
    if policy == POLICY_LIST:
        return [int(b) for b in block_list]
    if L <= 0:
        return []
    nb = -(-L // n)
    if policy == POLICY_DENSE:
        return list(range(nb - 1, -1, -1))
    if policy == POLICY_SINK_WINDOW:
        elig = [blk for blk in range(nb)
                if eligible_token_mask(policy, L, blk, sink_tokens, window_tokens).any()]
        has_sink_block = sink_tokens > 0 and 0 in elig
        rest = sorted((blk for blk in elig if not (has_sink_block and blk == 0)), reverse=True)
        return ([0] if has_sink_block else []) + rest
    raise ValueError("unknown policy")


def eligible_token_mask(policy: int, seq_len: int, blk: int, sink_tokens: int = 0,
                        window_tokens: int = 0) -> np.ndarray:
    """Boolean [64]: which tokens of logical block `blk` are in the eligible set E.

    Reading R8: tokens >= L (partial last block) and tokens outside sink/window are
    excluded (weight 0).
    """
    j = blk * BLOCK_TOKENS + np.arange(BLOCK_TOKENS)
    valid = (j < seq_len) & (j >= 0)
    if policy == POLICY_SINK_WINDOW:
        valid &= (j < sink_tokens) | (j >= seq_len - window_tokens)
    return valid


@dataclass
class GroupResult:
    """Everything the oracle knows about one (sequence, KV head) group."""
    stop_block: int                       # t* (R9): blocks processed; T if never fired
    num_blocks: int                       # T
    out_on: np.ndarray                    # [G, d]  o^(t*)
    out_off: np.ndarray                   # [G, d]  o^(T), streamed
    out_textbook: np.ndarray              # [G, d]  one-shot softmax over E (Eq. 1)
    d_scale: np.ndarray                   # [t*, G] Eq. 2, steps 1..t*
    d_direction: np.ndarray               # [t*, G]
    stable: np.ndarray                    # [t*]   group decision (AND over heads, R2)
    fragile: bool                         # any criterion value within 1e-4 rel. of its threshold
    fired: bool                           # termination triggered (c >= p) at t*
    # optional full trace (trace=True): all T steps, no early break
    ell: np.ndarray | None = None         # [T, G]  l_t
    A: np.ndarray | None = None           # [T, G]  A_t
    u: np.ndarray | None = None           # [T, G, d] block-local outputs u^(t)
    o: np.ndarray | None = None           # [T, G, d] prefix outputs o^(t)
    d_scale_all: np.ndarray | None = None  # [T, G]
    d_direction_all: np.ndarray | None = None
    extras: dict = field(default_factory=dict)


def _criterion(x_new: np.ndarray, x_old: np.ndarray):
    """Eq. 2 per head, with the zero-norm convention R4."""
    d_scale = np.linalg.norm(x_new - x_old, axis=-1)
    n_new = np.linalg.norm(x_new, axis=-1)
    n_old = np.linalg.norm(x_old, axis=-1)
    dots = np.sum(x_new * x_old, axis=-1)
    d_dir = np.ones_like(d_scale)                       # cos := 0 when a norm is 0 (R4)
    ok = (n_new > 0) & (n_old > 0)
    d_dir[ok] = 1.0 - dots[ok] / (n_new[ok] * n_old[ok])
    return d_scale, d_dir


def _stream_step(A, N, w_t, V_t):
    """One application of the App. A recurrence, written on the
    un-normalised pair (A_t, N_t = A_t o^(t)):  A_t = A_{t-1} + l_t,
    N_t = N_{t-1} + sum_k w_{t,k} v_{t,k},  o^(t) = N_t / A_t."""
    ell_t = w_t.sum(axis=1)                                     # l_t
    A = A + ell_t
    N = N + w_t @ V_t
    pos = A > 0                                                 # no valid token seen yet -> o = 0
    o = np.where(pos[:, None], N / np.where(pos, A, 1.0)[:, None], 0.0)
    return ell_t, A, N, o


def art_group(q: np.ndarray, K_blocks: np.ndarray, V_blocks: np.ndarray, valid: np.ndarray,
              tau: float, phi: float, patience: int, probe_dim: int = DEFAULT_PROBE_DIM,
              sm_scale: float | None = None, trace: bool = False) -> GroupResult:
    """ART for one query group, Algorithm 1 step by step.

    q        [G, d]      the G query heads sharing this KV head (R15: the m * G (token, head) rows)
    K_blocks [T, 64, d]  keys of the eligible blocks IN TRAVERSAL ORDER
    V_blocks [T, 64, d]  values, same order
    valid    [T, 64]     token-level eligibility (masked tokens get weight 0, R8); or [G, T, 64], one mask per
                         row (R15: the causal cut differs from query token to query token)
    """
    q = np.asarray(q, dtype=np.float64)
    G, d = q.shape
    T = int(K_blocks.shape[0])
    if patience < 1:
        raise ValueError("patience must be >= 1")
    scale = (1.0 / np.sqrt(d)) if not sm_scale else float(sm_scale)   # Eq. 1 (R11)
    idx = probe_indices(d, probe_dim)
    zeros = np.zeros((G, d))
    if T == 0:
        e = np.zeros((0, G))
        return GroupResult(0, 0, zeros, zeros.copy(), zeros.copy(), e, e.copy(),
                           np.zeros(0, bool), False, False)

    K = np.asarray(K_blocks, dtype=np.float64)
    V = np.asarray(V_blocks, dtype=np.float64)
    valid = np.asarray(valid, dtype=bool)
    row_valid = np.broadcast_to(valid if valid.ndim == 3 else valid[None, :, :], (G, T, BLOCK_TOKENS))
    anyrow = row_valid.any(axis=0)                              # [T, 64] eligible for at least one row
    # masked slots may hold garbage (even NaN) in a paged cache: never let them in
    K = np.where(anyrow[:, :, None], K, 0.0)
    V = np.where(anyrow[:, :, None], V, 0.0)

    # logits s_{h,t,j} = (q_h . k_{t,j}) / sqrt(d)   (Eq. 1)
    S = np.einsum("hd,tjd->htj", q, K) * scale
    S = np.where(row_valid, S, -np.inf)
    has = row_valid.reshape(G, -1).any(axis=1)                  # rows with at least one eligible token
    # first pass: global max over ALL eligible tokens (shift invariance of softmax)
    M = np.where(has, S.reshape(G, -1).max(axis=1), 0.0)
    W = np.where(row_valid, np.exp(S - M[:, None, None]), 0.0)  # w_j = exp(s_j - M_h)

    # one-shot textbook softmax over E (Eq. 1), independent of the streaming below
    Wf = W.reshape(G, -1)
    den = Wf.sum(axis=1, keepdims=True)
    out_textbook = np.where(has[:, None], (Wf / np.where(den > 0, den, 1.0)) @ V.reshape(-1, d), 0.0)

    # ---- Algorithm 1 ----
    A = np.zeros(G)                   # A_0 = 0
    N = np.zeros((G, d))              # A_t o^(t)
    o = np.zeros((G, d))              # l.1  O^(0) <- 0
    x_prev = np.zeros((G, idx.size))  #      x^(0) = PROBE(O^(0)) = 0
    c = 0                             # l.2  c^(0) <- 0
    t_star, fired, fragile = T, False, False
    ds_log, dd_log, st_log = [], [], []
    for t in range(1, T + 1):                                   # l.3
        _, A, N, o = _stream_step(A, N, W[:, t - 1, :], V[t - 1])   # l.4-5
        x = o[:, idx]                                           # l.6  x^(t) = PROBE(O^(t)) (R1, R6)
        d_scale, d_dir = _criterion(x, x_prev)                  # l.7-8 (Eq. 2)
        stable = bool(((d_scale < tau) & (d_dir < phi)).all())  # l.9, strict (R5); AND over heads (R2)
        c = c + 1 if stable else 0                              # l.9-13 (Eq. 3)
        ds_log.append(d_scale); dd_log.append(d_dir); st_log.append(stable)
        with np.errstate(divide="ignore", invalid="ignore"):    # north_star's near-threshold band
            if tau > 0 and np.isfinite(tau):
                fragile |= bool((np.abs(d_scale / tau - 1.0) < FRAGILE_REL).any())
            if phi > 0 and np.isfinite(phi):
                fragile |= bool((np.abs(d_dir / phi - 1.0) < FRAGILE_REL).any())
        x_prev = x
        if c >= patience:                                       # l.14  termination triggered
            t_star, fired = t, True
            break                                               # l.15
    out_on = o.copy()                                           # l.18  return O^(t*)

    # o^(T): keep streaming the blocks ART skipped (no criterion any more)
    for t in range(t_star + 1, T + 1):
        _, A, N, o = _stream_step(A, N, W[:, t - 1, :], V[t - 1])
    out_off = o.copy()

    res = GroupResult(
        stop_block=t_star, num_blocks=T, out_on=out_on, out_off=out_off,
        out_textbook=out_textbook, d_scale=np.array(ds_log).reshape(-1, G),
        d_direction=np.array(dd_log).reshape(-1, G), stable=np.array(st_log, dtype=bool),
        fragile=fragile, fired=fired)
    if trace:
        _full_trace(res, W, V, idx)
    return res


def _full_trace(res: GroupResult, W: np.ndarray, V: np.ndarray, idx: np.ndarray) -> None:
    """All T steps with no termination: l_t, A_t, u^(t), o^(t) and Eq. 2 at every step.
    Used by the pin tests (recurrence identity, bounds, brute force)."""
    G, T, _ = W.shape
    d = V.shape[-1]
    A = np.zeros(G); N = np.zeros((G, d)); x_prev = np.zeros((G, idx.size))
    ell_log, A_log, u_log, o_log, ds, dd = [], [], [], [], [], []
    for t in range(1, T + 1):
        w_t = W[:, t - 1, :]
        ell_t, A, N, o = _stream_step(A, N, w_t, V[t - 1])
        has = ell_t > 0
        u_t = np.where(has[:, None], (w_t @ V[t - 1]) / np.where(has, ell_t, 1.0)[:, None], 0.0)
        x = o[:, idx]
        d_scale, d_dir = _criterion(x, x_prev)
        x_prev = x
        ell_log.append(ell_t); A_log.append(A.copy()); u_log.append(u_t); o_log.append(o.copy())
        ds.append(d_scale); dd.append(d_dir)
    res.ell = np.array(ell_log); res.A = np.array(A_log)
    res.u = np.array(u_log); res.o = np.array(o_log)
    res.d_scale_all = np.array(ds); res.d_direction_all = np.array(dd)


def gather_group_blocks(cache: np.ndarray, layout: int, block_table_row: np.ndarray,
                        kv_head: int, blocks: list[int]) -> np.ndarray:
    """[T, 64, d] tiles of one KV head for the logical blocks `blocks`, through the page table."""
    if len(blocks) == 0:
        d = cache.shape[-1]
        return np.zeros((0, BLOCK_TOKENS, d))
    pages = np.asarray(block_table_row)[np.asarray(blocks, dtype=np.int64)]
    if layout == LAYOUT_HND:
        return np.asarray(cache[pages, kv_head], dtype=np.float64)
    if layout == LAYOUT_NHD:
        return np.asarray(cache[pages, :, kv_head], dtype=np.float64)
    raise ValueError("unknown layout")


def art_decode_attention_oracle(q, k_cache, v_cache, block_table, seq_lens, *,
                                num_kv_heads: int, policy: int = POLICY_DENSE,
                                layout: int = LAYOUT_HND, sink_tokens: int = 0,
                                window_tokens: int = 0, eligible_blocks=None,
                                eligible_counts=None, tau: float = DEFAULT_TAU,
                                phi: float = DEFAULT_PHI, patience: int = DEFAULT_PATIENCE,
                                probe_dim: int = DEFAULT_PROBE_DIM, sm_scale: float | None = None,
                                art: bool = True, groups=None, trace: bool = False):
    """Whole decode step: every (sequence b, KV head g) group, independently.

    q [B, Hq, d], or [B, m, Hq, d] for m query tokens per sequence (R15: they are the last m positions,
    whose K/V are already in the cache and counted in seq_lens; query token i sees tokens j <= L - m + i of
    the policy's eligible set; rows of a group are ordered token-major, row = i * G + h);
    k_cache / v_cache paged (layout above); block_table [B, max_blocks]
    logical block -> physical page; seq_lens [B]; eligible_blocks [B, Hkv, max_eligible]
    and eligible_counts [B, Hkv] for POLICY_LIST.  GQA: query head h belongs to KV head
    h // G (paper silent; standard).  art=False disables termination (ART-off): the
    result is o^(T) and stop_block = T.

    Returns (out [B, Hq, d] (or [B, m, Hq, d]) float64, stop_block [B, Hkv] int64, results dict keyed (b, g)).
    `groups` optionally restricts the work to a list of (b, g) pairs; other rows stay 0.
    """
    q = np.asarray(q, dtype=np.float64)
    multi = q.ndim == 4
    if not multi:
        q = q[:, None]
    B, m, Hq, d = q.shape
    Hkv = int(num_kv_heads)
    assert Hq % Hkv == 0
    G = Hq // Hkv
    out = np.zeros((B, m, Hq, d))
    stop = np.zeros((B, Hkv), dtype=np.int64)
    results = {}
    todo = groups if groups is not None else [(b, g) for b in range(B) for g in range(Hkv)]
    for (b, g) in todo:
        L = int(seq_lens[b])
        if policy == POLICY_LIST:
            cnt = int(eligible_counts[b, g])
            blocks = traversal_blocks(policy, L, block_list=np.asarray(eligible_blocks)[b, g, :cnt])
        else:
            blocks = traversal_blocks(policy, L, sink_tokens, window_tokens)
        valid = np.stack([eligible_token_mask(policy, L, blk, sink_tokens, window_tokens)
                          for blk in blocks]) if blocks else np.zeros((0, BLOCK_TOKENS), bool)
        # a listed block that lies wholly beyond L has no valid token: do not touch its page
        safe_blocks = [blk if valid[i].any() else 0 for i, blk in enumerate(blocks)]
        Kb = gather_group_blocks(k_cache, layout, block_table[b], g, safe_blocks)
        Vb = gather_group_blocks(v_cache, layout, block_table[b], g, safe_blocks)
        if m > 1 and len(blocks):                               # R15: causal cut per query token
            pos = np.asarray(blocks)[:, None] * BLOCK_TOKENS + np.arange(BLOCK_TOKENS)[None, :]     # [T, 64]
            cut = np.stack([pos < L - (m - 1 - i) for i in range(m)])                               # [m, T, 64]
            valid = np.repeat(valid[None] & cut, G, axis=0)     # row i * G + h
        r = art_group(q[b, :, g * G:(g + 1) * G].reshape(m * G, d), Kb, Vb, valid,
                      tau=tau if art else 0.0, phi=phi if art else 0.0,
                      patience=patience if art else PATIENCE_INF,
                      probe_dim=probe_dim, sm_scale=sm_scale, trace=trace)
        out[b, :, g * G:(g + 1) * G] = r.out_on.reshape(m, G, d)
        stop[b, g] = r.stop_block
        results[(b, g)] = r
    return (out if multi else out[:, 0]), stop, results


# --------------------------------------------------------------------------- base-policy block list

def block_scores_oracle(q, k_cache, block_table, seq_lens, *, num_kv_heads: int,
                        layout: int = LAYOUT_HND) -> np.ndarray:
    """Block priority of the scored base policy the paper orders importance-first: for every
    (sequence b, KV head g, logical block) the MEAN over the group's G query heads and the block's valid
    tokens (j < L) of q_h . k_j, in fp64.  (The paper's SnapKV scores need prefill attention maps, which do
    not exist here; this stand-in is BASELINE.json's "mean q.k score".)

    Plain loops over blocks, one dot product per (head, token): the definition written out.
    Returns [B, Hkv, max_blocks] float64; blocks at or beyond ceil(L / 64) get -inf.
    """
    q = np.asarray(q, dtype=np.float64)
    B, Hq, d = q.shape
    Hkv = int(num_kv_heads)
    G = Hq // Hkv
    max_blocks = int(np.asarray(block_table).shape[1])
    scores = np.full((B, Hkv, max_blocks), -np.inf)
    for b in range(B):
        L = int(seq_lens[b])
        nb = -(-L // BLOCK_TOKENS) if L > 0 else 0
        for g in range(Hkv):
            for blk in range(nb):
                tile = gather_group_blocks(k_cache, layout, block_table[b], g, [blk])[0]      # [64, d]
                n_valid = min(BLOCK_TOKENS, L - blk * BLOCK_TOKENS)
                total = 0.0
                for h in range(g * G, (g + 1) * G):
                    total += float((tile[:n_valid] @ q[b, h]).sum())
                scores[b, g, blk] = total / (G * n_valid)
    return scores


def topk_blocks_oracle(scores: np.ndarray, seq_lens, top_k: int):
    """Importance-first list (reading R10): the top_k candidate blocks by DESCENDING score,
    ties -> lower block index first.  Returns (lists [B, Hkv, top_k] int64 padded with -1, counts [B, Hkv])."""
    B, Hkv, _ = scores.shape
    lists = np.full((B, Hkv, max(int(top_k), 0)), -1, dtype=np.int64)
    counts = np.zeros((B, Hkv), dtype=np.int64)
    for b in range(B):
        L = int(seq_lens[b])
        nb = -(-L // BLOCK_TOKENS) if L > 0 else 0
        for g in range(Hkv):
            cand = sorted(range(nb), key=lambda blk: (-scores[b, g, blk], blk))
            k = min(int(top_k), nb)
            lists[b, g, :k] = cand[:k]
            counts[b, g] = k
    return lists, counts
