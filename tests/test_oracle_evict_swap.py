"""Pins for the oracle's stage 3 (predictor, score, victim selection) and stage 4 (swap).  CPU only.

Selection is pinned by an exhaustive Python sort, by the invariants of PAPER.md L252 (unreferenced blocks
only) / L181 (never the requesting = RUNNING/QUEUED session first), and by the special cases that reduce to
textbook policies: all tau equal => LRU (L281), tau = true next use => Belady furthest-in-future (L215),
idle sessions first (L277).  Swap is pinned by numpy fancy indexing on both pool layouts.
"""
import numpy as np
import pytest

import oracle
from harness import gen

TAU_MAX = (1 << 24) - 1
V, P = 0x80000000, 0x40000000


def py_tau(features, weights, bias, state, override=None):
    raw = bias + (features.astype(np.int64) * weights.astype(np.int64)[None, :]).sum(axis=1)
    tau = np.clip(raw, 0, TAU_MAX - 1)
    if override is not None:
        tau = np.minimum(np.asarray(override, np.int64), TAU_MAX - 1)
    tau = np.where((state == 1) | (state == 2), 0, tau)
    tau = np.where(state >= 3, TAU_MAX, tau)
    return tau.astype(np.uint32)


def py_select(tau, tick, sess, last, depth, rf, deficit):
    cands = []
    for b in range(len(sess)):
        if not (rf[b] & V) or (rf[b] & P) or (rf[b] & 0x3FFFFFFF):
            continue
        t = int(tau[sess[b]]) if sess[b] < len(tau) else TAU_MAX
        age = min(max(int(tick) - int(last[b]), 0), 0xFFFFF)
        score = ((TAU_MAX - t) << 40) | ((0xFFFFF - age) << 20) | (0xFFFFF - min(int(depth[b]), 0xFFFFF))
        cands.append((score, b))
    cands.sort()
    return cands[:deficit], len(cands)


def random_pool(g, M, S, F=4):
    sess = g.integers(0, S + 2, size=M).astype(np.uint32)          # some ids >= S (unknown session)
    last = g.integers(900, 1010, size=M).astype(np.uint32)         # some in the future (age clamps to 0)
    depth = g.integers(0, 50, size=M).astype(np.uint32)
    rf = np.where(g.random(M) < 0.85, V, 0).astype(np.uint32)
    rf |= np.where(g.random(M) < 0.2, g.integers(1, 4, size=M), 0).astype(np.uint32)
    rf |= np.where(g.random(M) < 0.1, P, 0).astype(np.uint32)
    feats = g.integers(0, 256, size=(S, F), dtype=np.uint8)
    w = g.integers(-300, 300, size=F).astype(np.int16)
    state = g.integers(0, 5, size=S).astype(np.uint8)
    return sess, last, depth, rf, feats, w, state


def test_predictor_equals_numpy_int64_dot_product():
    g = np.random.default_rng(40)
    for F in (1, 4, 16):
        feats = g.integers(0, 256, size=(200, F), dtype=np.uint8)
        w = g.integers(-32768, 32768, size=F).astype(np.int16)
        state = g.integers(0, 5, size=200).astype(np.uint8)
        for bias in (0, -(1 << 30), 1 << 30, 123456):
            assert (oracle.session_tau(feats, w, bias, state) == py_tau(feats, w, bias, state)).all()
        ov = g.integers(0, 1 << 26, size=200).astype(np.uint32)
        assert (oracle.session_tau(feats, w, 5, state, ov) == py_tau(feats, w, 5, state, ov)).all()
    with pytest.raises(ValueError):
        oracle.session_tau(feats, w, (1 << 30) + 1, state)


def test_score_bit_layout():
    assert oracle.block_score(0, 100, 100, 0) == (1 << 64) - 1
    assert oracle.block_score(TAU_MAX, 5, 5, 0) == (0xFFFFF << 20) | 0xFFFFF
    assert oracle.block_score(TAU_MAX, 1 << 21, 0, 1 << 21) == 0
    assert oracle.block_score(7, 50, 60, 3) == ((TAU_MAX - 7) << 40) | (0xFFFFF << 20) | (0xFFFFF - 3)
    # larger tau, older access, deeper block  =>  strictly lower score (evicted earlier)
    assert oracle.block_score(9, 50, 40, 3) < oracle.block_score(8, 50, 0, 99)
    assert oracle.block_score(9, 50, 39, 3) < oracle.block_score(9, 50, 40, 99)
    assert oracle.block_score(9, 50, 40, 4) < oracle.block_score(9, 50, 40, 3)


def test_selection_equals_exhaustive_sort_and_invariants():
    g = np.random.default_rng(41)
    for trial in range(30):
        M, S = int(g.integers(1, 300)), int(g.integers(1, 9))
        sess, last, depth, rf, feats, w, state = random_pool(g, M, S)
        deficit = int(g.integers(0, M + 5))
        tau = py_tau(feats, w, 1000, state)
        expect, n_ev = py_select(tau, 1000, sess, last, depth, rf, deficit)
        vic, sc, st = oracle.score_evict(1000, feats, w, 1000, state, None, deficit, sess, last, depth, rf)
        assert vic.tolist() == [b for _, b in expect] and sc.tolist() == [s for s, _ in expect]
        assert len(vic) == min(deficit, n_ev) and st == (0 if deficit <= n_ev else -2)
        assert all((rf[b] & V) and not (rf[b] & P) and not (rf[b] & 0x3FFFFFFF) for b in vic)
        keys = list(zip(sc.tolist(), vic.tolist()))
        assert keys == sorted(keys) and len(set(vic.tolist())) == len(vic)


def test_all_tau_equal_reduces_to_lru():
    g = np.random.default_rng(42)
    M, S = 400, 5
    sess = g.integers(0, S, size=M).astype(np.uint32)
    last = g.permutation(M).astype(np.uint32) + 10           # distinct access ticks
    depth = g.integers(0, 100, size=M).astype(np.uint32)
    rf = np.full(M, V, np.uint32)
    feats = np.zeros((S, 4), np.uint8)
    vic, _, st = oracle.score_evict(1000, feats, np.zeros(4, np.int16), 500, np.zeros(S, np.uint8), None, 123,
                                    sess, last, depth, rf)
    assert st == 0 and vic.tolist() == np.argsort(last, kind="stable")[:123].tolist()   # least recent first


def test_true_tau_override_reduces_to_belady():
    g = np.random.default_rng(43)
    S, per = 7, 20
    next_use = g.permutation(S).astype(np.uint32) * 1000 + 5          # distinct true times-to-next-use
    sess = np.repeat(np.arange(S, dtype=np.uint32), per)
    depth = np.tile(np.arange(per, dtype=np.uint32), S)
    last = np.full(S * per, 77, np.uint32)
    rf = np.full(S * per, V, np.uint32)
    feats = g.integers(0, 256, size=(S, 4), dtype=np.uint8)
    w = g.integers(-100, 100, size=4).astype(np.int16)
    vic, _, _ = oracle.score_evict(100, feats, w, 0, np.zeros(S, np.uint8), next_use, 3 * per, sess, last, depth, rf)
    far = np.argsort(-next_use.astype(np.int64))[:3]                  # furthest-in-future sessions first
    assert [int(sess[b]) for b in vic] == np.repeat(far, per).tolist()
    assert depth[vic[:per]].tolist() == list(range(per - 1, -1, -1))  # deepest block first within a session


def test_idle_sessions_go_first_then_tool_wait_never_running_before_them():
    S, per = 4, 10
    state = np.array([0, 3, 2, 1], np.uint8)      # TOOL_WAIT, IDLE, RUNNING, QUEUED
    sess = np.repeat(np.arange(S, dtype=np.uint32), per)
    depth = np.tile(np.arange(per, dtype=np.uint32), S)
    rf = np.full(S * per, V, np.uint32)
    feats = np.full((S, 4), 10, np.uint8)
    w = np.full(4, 100, np.int16)
    vic, _, st = oracle.score_evict(10, feats, w, 0, state, None, 4 * per, sess, np.full(S * per, 3, np.uint32),
                                    depth, rf)
    order = [int(sess[b]) for b in vic]
    assert st == 0 and order[:per] == [1] * per and order[per:2 * per] == [0] * per
    assert set(order[2 * per:]) == {2, 3}          # tau = 0: last resort, tie broken by depth then id


@pytest.mark.parametrize("layout", ["layer_major", "block_major"])
def test_swap_equals_fancy_indexing_and_round_trips(layout):
    g = np.random.default_rng(44)
    M, n_chunks, chunk = 37, 6, 48
    page = n_chunks * chunk
    if layout == "layer_major":
        chunk_stride, block_stride = M * chunk, chunk
        view = lambda p: p[:M * page].reshape(n_chunks, M, chunk).transpose(1, 0, 2)
    else:
        chunk_stride, block_stride = chunk, page
        view = lambda p: p[:M * page].reshape(M, n_chunks, chunk)
    pool = g.integers(0, 256, size=M * page + 64, dtype=np.uint8)
    pool[M * page:] = 0xA5                                            # guard bytes
    orig = pool.copy()
    vic = g.choice(M, size=9, replace=False).astype(np.uint32)
    stage = np.zeros((9, page), np.uint8)
    oracle.swap_out(pool, n_chunks, chunk, chunk_stride, block_stride, vic, stage.reshape(-1))
    assert (stage.reshape(9, n_chunks, chunk) == view(orig)[vic]).all() and (pool == orig).all()
    slots = np.array([4, 0, 11, 2, 7, 9, 1, 3, 5], np.uint32)
    tier = np.zeros((12, page), np.uint8)
    oracle.swap_out(pool, n_chunks, chunk, chunk_stride, block_stride, vic, tier.reshape(-1), slots=slots)
    assert (tier[slots] == stage).all()
    free = np.setdiff1d(np.arange(M), vic)
    dst = g.choice(free, size=9, replace=False).astype(np.uint32)     # restore into DIFFERENT block ids
    oracle.swap_in(pool, n_chunks, chunk, chunk_stride, block_stride, tier.reshape(-1), dst, slots=slots)
    assert (view(pool)[dst] == view(orig)[vic]).all()
    untouched = np.setdiff1d(np.arange(M), dst)
    assert (view(pool)[untouched] == view(orig)[untouched]).all() and (pool[M * page:] == 0xA5).all()
    before = pool.copy()
    oracle.swap_in(pool, n_chunks, chunk, chunk_stride, block_stride, stage.reshape(-1), dst[:0])
    assert (pool == before).all()                                     # n = 0 is a no-op


def test_generators_are_seeded_and_shaped():
    a, b = gen.stress_snapshot(seed=9, S=4, L=1024, RB=32, req_per_session=3, len_median=300, len_min=64,
                               len_max=1024), None
    b = gen.stress_snapshot(seed=9, S=4, L=1024, RB=32, req_per_session=3, len_median=300, len_min=64,
                            len_max=1024)
    assert (a.tokens == b.tokens).all() and (a.features == b.features).all() and a.M == 128
    assert a.tokens.dtype == np.int32 and 0 <= a.tokens.min() and a.tokens.max() < 32000
    t = gen.tiny_trace(0)
    assert len(t.sessions) == 4 and all(len(s) == 8 for s in t.sessions)
    for s in t.sessions:
        assert s[0].tokens.size == 512
        for u, v in zip(s, s[1:]):
            assert 64 <= v.tokens.size - u.tokens.size <= 256 and (v.tokens[:u.tokens.size] == u.tokens).all()
    pb = gen.page_bytes(np.array([1, 2, 1], np.uint64), 64)
    assert pb.shape == (3, 64) and (pb[0] == pb[2]).all() and (pb[0] != pb[1]).any()
