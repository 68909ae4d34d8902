"""Seeded synthetic input generators (serve BOTH the oracle and the CUDA path).

This module holds none of the method's arithmetic: it only draws tokens, lengths, gaps, features,
metadata and ids from counter-based Philox streams keyed by (seed, stream id).  Shapes follow
BASELINE.json's five configs / SURVEY.md 8(d); the CATraces dataset the paper measures on
 is not available, so these inputs stand in for it.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

VOCAB = 32000
BLOCK = 16

# session_state codes (R4)
TOOL_WAIT, QUEUED, RUNNING, IDLE = 0, 1, 2, 3
REF_VALID = 0x80000000
REF_PINNED = 0x40000000


def rng(seed: int, stream: int) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(key=[seed & 0xFFFFFFFFFFFFFFFF, stream & 0xFFFFFFFFFFFFFFFF]))


def lognormal_int(g: np.random.Generator, median: float, sigma: float, lo: int, hi: int, size=None):
    v = g.lognormal(mean=np.log(median), sigma=sigma, size=size)
    return np.clip(np.floor(v), lo, hi).astype(np.int64)


# --------------------------------------------------------------------------------------------------
# Config 3 — scheduling / eviction stress snapshot (static; no replay)
# --------------------------------------------------------------------------------------------------
@dataclass
class StressSnapshot:
    # request queue (CSR)
    tokens: np.ndarray          # int32[sum T]
    tok_off: np.ndarray         # uint64[R+1]
    need_d: np.ndarray          # uint32[R]  ceil(len/16)
    arrival_seq: np.ndarray     # uint64[R]
    req_id: np.ndarray          # uint32[R]
    req_session: np.ndarray     # uint32[R]
    shared_tokens: np.ndarray   # int64[R] tokens copied from the session stream (closed-form pin for k)
    # resident state
    streams: np.ndarray         # int32[S, L] session token streams
    resident_blocks: int        # RB: blocks [0,RB) of every stream are resident; block id = s*RB + j
    M: int
    table_log2: int
    blk_session: np.ndarray     # uint32[M]
    blk_last_access: np.ndarray  # uint32[M]
    blk_depth: np.ndarray       # uint32[M]
    blk_ref_flags: np.ndarray   # uint32[M]
    hole_ids: np.ndarray        # uint32[...] resident block ids erased in the "holes" variant
    # predictor
    features: np.ndarray        # uint8[S,F]
    weights: np.ndarray         # int16[F]
    bias: int
    session_state: np.ndarray   # uint8[S]
    tick_now: int
    deficit: int
    meta: dict = field(default_factory=dict)


def stress_snapshot(seed: int = 3, S: int = 256, L: int = 131072, RB: int = 4096, req_per_session: int = 16,
                    len_median: float = 16384, len_sigma: float = 1.0, len_min: int = 2048, len_max: int = 131072,
                    F: int = 16, running_frac: float = 52 / 256, idle_frac: float = 24 / 256,
                    deficit_frac: float = 0.05, hole_frac: float = 0.01) -> StressSnapshot:
    """BASELINE.json configs[2] (defaults) or a scaled-down version of the same recipe."""
    assert L % BLOCK == 0 and RB * BLOCK <= L and len_max <= L
    g = rng(seed, 0)
    streams = g.integers(0, VOCAB, size=(S, L), dtype=np.int32)
    R = S * req_per_session
    req_session = np.repeat(np.arange(S, dtype=np.uint32), req_per_session)
    g = rng(seed, 1)
    lens = lognormal_int(g, len_median, len_sigma, len_min, len_max, size=R)
    frac = g.uniform(0.5, 1.0, size=R)
    shared = np.floor(frac * lens).astype(np.int64)
    tok_off = np.zeros(R + 1, np.uint64)
    np.cumsum(lens, out=tok_off[1:].view(np.int64))
    total = int(tok_off[-1])
    tokens = np.empty(total, np.int32)
    g = rng(seed, 2)
    fresh_total = int((lens - shared).sum())
    fresh = g.integers(0, VOCAB, size=fresh_total, dtype=np.int32)
    fo = 0
    for r in range(R):
        o, sh, ln = int(tok_off[r]), int(shared[r]), int(lens[r])
        s = int(req_session[r])
        tokens[o:o + sh] = streams[s, :sh]
        nf = ln - sh
        if nf:
            tokens[o + sh:o + ln] = fresh[fo:fo + nf]
            if sh < L and tokens[o + sh] == streams[s, sh]:  # first fresh token must differ from the stream
                tokens[o + sh] = (tokens[o + sh] + 1) % VOCAB
            fo += nf
    g = rng(seed, 3)
    arrival_seq = g.permutation(R).astype(np.uint64)
    req_id = np.arange(R, dtype=np.uint32)
    need_d = ((lens + BLOCK - 1) // BLOCK).astype(np.uint32)

    M = S * RB
    table_log2 = max(4, int(np.ceil(np.log2(2 * M))))
    n_run, n_idle = int(round(running_frac * S)), int(round(idle_frac * S))
    state = np.full(S, TOOL_WAIT, np.uint8)
    perm = g.permutation(S)
    state[perm[:n_run]] = RUNNING
    state[perm[n_run:n_run + n_idle]] = IDLE
    tick_now = 1_000_000
    sess_access = g.integers(tick_now - 1000, tick_now + 1, size=S).astype(np.uint32)
    blk_session = np.repeat(np.arange(S, dtype=np.uint32), RB)
    blk_depth = np.tile(np.arange(RB, dtype=np.uint32), S)
    blk_last_access = np.repeat(sess_access, RB)
    blk_ref_flags = np.where(state[blk_session] == RUNNING, REF_VALID | 1, REF_VALID).astype(np.uint32)
    n_holes = int(hole_frac * M)
    hole_ids = np.sort(g.choice(M, size=n_holes, replace=False)).astype(np.uint32)

    g = rng(seed, 4)
    features = g.integers(0, 256, size=(S, F), dtype=np.uint8)
    weights = g.integers(-2048, 2048, size=F, dtype=np.int16)
    bias = 1_000_000  # ~1.4 sigma of sum_f w*x for F=16, so that >=90% of raw predictions are > 0
    deficit = int(deficit_frac * M)
    return StressSnapshot(tokens, tok_off, need_d, arrival_seq, req_id, req_session, shared, streams, RB, M,
                          table_log2, blk_session, blk_last_access, blk_depth, blk_ref_flags, hole_ids, features,
                          weights, bias, state, tick_now, deficit,
                          meta=dict(seed=seed, S=S, L=L, RB=RB, R=R, F=F, total_tokens=total))


def stream_tok_off(S: int, L: int) -> np.ndarray:
    return (np.arange(S + 1, dtype=np.uint64) * np.uint64(L))


# --------------------------------------------------------------------------------------------------
# Session traces for the host-driven replays (configs 1, 2, 5)
# --------------------------------------------------------------------------------------------------
@dataclass
class Turn:
    tokens: np.ndarray   # int32[len] full prompt of this turn
    gap_ms: int          # tool / think time after this turn completes, before the next request arrives
    features: np.ndarray  # uint8[F] tool-call metadata features attached when the turn completes
    true_tau_ms: int     # = gap_ms (ground truth for the CacheWise* "Hint" override)
    cluster: int = 0     # metadata cluster of the tool call that follows this turn (paper predictor, L227)


@dataclass
class Trace:
    sessions: list       # list[list[Turn]]
    weights: np.ndarray  # int16[F]
    bias: int
    F: int
    meta: dict


def session_trace(seed: int, n_sessions: int, n_turns: int, F: int, init_len, grow_lo: int, grow_hi: int,
                  keep_frac: float, cap: int, gap_mix) -> Trace:
    """Multi-turn sessions with growing shared prefixes.

    init_len: int, or (median, sigma, lo, hi) lognormal.  Turn t+1 keeps the first floor(keep_frac*len_t)
    tokens of turn t (keep_frac=1: pure append; 0.85: edit/compaction pattern of config 2), then appends
    fresh tokens so that the length grows by U{grow_lo..grow_hi}, capped at ``cap`` tokens.
    gap_mix: list of (prob, median_ms, sigma) lognormal components for the tool-call gap.
    Feature 0 is a bucketed log2 of the true gap (a tool-metadata proxy), the rest are noise.
    """
    sessions = []
    probs = np.array([p for p, _, _ in gap_mix], dtype=np.float64)
    for s in range(n_sessions):
        g = rng(seed, 1000 + s)
        if isinstance(init_len, tuple):
            ln = int(lognormal_int(g, init_len[0], init_len[1], init_len[2], init_len[3]))
        else:
            ln = int(init_len)
        toks = g.integers(0, VOCAB, size=ln, dtype=np.int32)
        turns = []
        for t in range(n_turns):
            comp = int(g.choice(len(gap_mix), p=probs / probs.sum()))
            gap = int(lognormal_int(g, gap_mix[comp][1], gap_mix[comp][2], 1, 10_000_000))
            feat = g.integers(0, 256, size=F, dtype=np.uint8)
            feat[0] = min(255, int(np.log2(gap + 1) * 10))
            turns.append(Turn(toks.copy(), gap, feat, gap))
            keep = int(np.floor(keep_frac * toks.size)) if keep_frac < 1.0 else toks.size
            new_len = min(cap, toks.size + int(g.integers(grow_lo, grow_hi + 1)))
            if new_len <= keep:
                keep = max(0, new_len - 1)
            fresh = g.integers(0, VOCAB, size=new_len - keep, dtype=np.int32)
            if keep < toks.size and fresh.size and fresh[0] == toks[keep]:
                fresh[0] = (fresh[0] + 1) % VOCAB
            toks = np.concatenate([toks[:keep], fresh])
        sessions.append(turns)
    weights = np.zeros(F, np.int16)
    weights[0] = 400  # tau grows with the gap bucket; other features get small weights
    gw = rng(seed, 999)
    weights[1:] = gw.integers(-8, 9, size=F - 1).astype(np.int16)
    return Trace(sessions, weights, -20000, F, dict(seed=seed, n_sessions=n_sessions, n_turns=n_turns))


def tool_clusters(seed: int, C: int = 20, n_lo: int = 9, n_hi: int = 64):
    """Synthetic per-cluster tool-duration history, shaped like PAPER.md Table 3 (L241-248) / Fig. 9 (L137-169):
    cluster medians log-spaced from ~50 ms to ~80 s, heavy right tails (P90/P50 between 2x and ~100x), 9..64 samples
    per cluster.  Returns (median_ms[C], sigma[C], sample_off u64[C+1], samples u32[sum n], sorted inside a cluster)."""
    g = rng(seed, 500)
    med = np.exp(np.linspace(np.log(50.0), np.log(80000.0), C))
    sig = g.uniform(0.5, 2.0, size=C)
    n = g.integers(n_lo, n_hi + 1, size=C)
    off = np.zeros(C + 1, np.uint64)
    np.cumsum(n, out=off[1:].view(np.int64))
    samples = np.concatenate([np.sort(lognormal_int(g, med[c], sig[c], 1, 10_000_000, size=int(n[c]))) for c in range(C)])
    return med, sig, off, samples.astype(np.uint32)


def cluster_trace(seed: int, n_sessions: int, n_turns: int, C: int = 20, init_len=(6000.0, 0.6, 1024, 24000),
                  grow_lo: int = 128, grow_hi: int = 1024, cap: int = 40000) -> Trace:
    """Sessions whose tool gaps are drawn from the per-cluster distributions of tool_clusters(seed): every turn ends
    with a tool call of a random cluster (fast clusters more often, as in Fig. 9), whose duration is a fresh draw from
    that cluster's lognormal — the replay only sees the cluster id and the HISTORICAL samples (a separate draw)."""
    med, sig, off, samples = tool_clusters(seed, C)
    tr = session_trace(seed, n_sessions, n_turns, 8, init_len, grow_lo, grow_hi, 1.0, cap, [(1.0, 1000.0, 1.0)])
    w = 1.0 / np.arange(1, C + 1)
    w /= w.sum()
    for s, turns in enumerate(tr.sessions):
        g = rng(seed, 700 + s)
        for t in turns:
            c = int(g.choice(C, p=w))
            t.cluster = c
            t.gap_ms = int(lognormal_int(g, med[c], sig[c], 1, 10_000_000))
            t.true_tau_ms = t.gap_ms
            t.features[0] = min(255, int(np.log2(t.gap_ms + 1) * 10))  # the linear predictor's proxy feature
    tr.meta.update(sample_off=off, samples=samples, C=C)
    return tr


def tiny_trace(seed: int = 0) -> Trace:
    """BASELINE.json configs[0]: 4 sessions x 8 turns, 512-token first prompt, +U{64..256} per turn."""
    return session_trace(seed, 4, 8, 4, 512, 64, 256, 1.0, 1 << 30, [(1.0, 2000.0, 1.0)])


def llama8b_trace(seed: int = 1, n_sessions: int = 64, n_turns: int = 40) -> Trace:
    """BASELINE.json configs[1]: initial prefix lognormal median 8k capped 64k, 85% shared with prior turn."""
    return session_trace(seed, n_sessions, n_turns, 8, (8192.0, 1.0, 512, 65536), 256, 2048, 0.85, 65536,
                         [(1.0, 2000.0, 1.0)])


def long_agent_trace(seed: int = 5, n_sessions: int = 512, n_turns: int = 200, cap: int = 200_000) -> Trace:
    """BASELINE.json configs[4]: contexts grow to 200k tokens, bimodal gaps (70% ~1 s, 30% ~60 s)."""
    grow = max(64, cap // max(n_turns, 1))
    return session_trace(seed, n_sessions, n_turns, 8, (4096.0, 0.5, 512, cap), grow // 2, grow * 3 // 2, 1.0,
                         cap, [(0.7, 1000.0, 1.0), (0.3, 60000.0, 1.0)])


# --------------------------------------------------------------------------------------------------
# Config 4 — swap sweep, and page content
# --------------------------------------------------------------------------------------------------
def swap_victims(seed: int, M: int, n: int) -> np.ndarray:
    """n random distinct block ids out of M, in the (unsorted) order drawn."""
    return rng(seed, 40).choice(M, size=n, replace=False).astype(np.uint32)


def page_bytes(tag: np.ndarray, page: int) -> np.ndarray:
    """Procedural page content: uint8[len(tag), page], a function of the 64-bit tag and the offset only, so
    that neither side has to store 100+ GB of expected KV bytes.  (Harness arithmetic, not the method's.)"""
    tag = np.asarray(tag, np.uint64).reshape(-1, 1)
    off = np.arange(page // 8, dtype=np.uint64).reshape(1, -1)
    with np.errstate(over="ignore"):
        w = (tag + off * np.uint64(0x9E3779B97F4A7C15)) * np.uint64(0xD6E8FEB86659FD93)
        w ^= w >> np.uint64(29)
    return w.view(np.uint8).reshape(tag.shape[0], page)
