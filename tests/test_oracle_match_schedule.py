"""Pins for the oracle's stage 2 (table + prefix match, schedule).  CPU only.

Match is pinned by brute-force token-by-token prefix comparison against every resident chain (PAPER.md
L173 "contiguous ... prefix", L177 k_i(t)); schedule by Python's sorted() on tuples plus a literal
admission loop and the textbook special cases (FCFS, L281).
"""
import numpy as np
import pytest

import oracle
from harness import gen

MISS = 0xFFFFFFFF
HOST = 0x80000000


def brute_force_match(resident, req_tokens):
    """resident: list of (tokens, {block j: loc}) ; returns (k_total, n_gpu, locs) by token comparison."""
    n = len(req_tokens) // 16
    k, g, locs = 0, 0, []
    for j in range(n):
        found = None
        for toks, blocks in resident:
            if j in blocks and len(toks) >= 16 * (j + 1) and np.array_equal(toks[:16 * (j + 1)],
                                                                           req_tokens[:16 * (j + 1)]):
                found = blocks[j] if found is None else min(found, blocks[j])
        if found is None:
            break
        k += 1
        g += 0 if found & HOST else 1
        locs.append(found)
    return k, g, locs


@pytest.mark.parametrize("holes", [False, True])
def test_match_equals_brute_force_prefix_comparison(holes):
    g = np.random.default_rng(10 + holes)
    # 3 resident session chains, the third forks off the first after 5 blocks
    s0 = g.integers(0, 32000, size=16 * 20, dtype=np.int32)
    s1 = g.integers(0, 32000, size=16 * 11 + 3, dtype=np.int32)
    s2 = np.concatenate([s0[:16 * 5 + 4], g.integers(0, 32000, size=16 * 9, dtype=np.int32)])
    table = oracle.Table(8)
    resident, next_loc = [], 0
    for toks, nb in ((s0, 14), (s1, 11), (s2, 12)):
        h, _ = oracle.hash_blocks(toks, [0, toks.size])
        blocks = {}
        for j in range(nb):
            if holes and g.random() < 0.15:
                continue
            loc = next_loc | (HOST if g.random() < 0.3 else 0)
            next_loc += 1
            win, st = table.insert([h[j]], [loc])
            assert st == 0
            blocks[j] = int(win[0])   # a block shared with an earlier chain keeps the earlier loc
        resident.append((toks, blocks))
    reqs = [s0[:16 * 20], s0[:16 * 9 + 7], s1, s2[:16 * 8], np.concatenate([s1[:40], s0[:100]]),
            g.integers(0, 32000, size=50, dtype=np.int32), s0[:5], s2]
    off = np.concatenate([[0], np.cumsum([len(r) for r in reqs])]).astype(np.uint64)
    h, hoff = oracle.hash_blocks(np.concatenate(reqs), off)
    k_total, n_gpu, hit_loc = table.match_prefix(h, hoff)
    for r, toks in enumerate(reqs):
        k, gg, locs = brute_force_match(resident, toks)
        assert (int(k_total[r]), int(n_gpu[r])) == (k, gg), r
        lo, hi = int(hoff[r]), int(hoff[r + 1])
        assert hit_loc[lo:lo + k].tolist() == locs
        assert (hit_loc[lo + k:hi] == MISS).all()     # past the run = MISS even if the key is present
    if holes:  # the holes variant must contain a request whose hit count exceeds its leading run
        assert any((table.lookup(h[int(hoff[r]):int(hoff[r + 1])]) != MISS).sum() > k_total[r]
                   for r in range(len(reqs)))


def test_stress_recipe_closed_form_overlap():
    snap = gen.stress_snapshot(seed=3, S=6, L=2048, RB=64, req_per_session=5, len_median=600, len_min=64,
                               len_max=2048)
    S, L, RB = 6, 2048, 64
    hs, _ = oracle.hash_blocks(snap.streams.reshape(-1), gen.stream_tok_off(S, L))
    hs = hs.reshape(S, L // 16)[:, :RB].reshape(-1)
    table = oracle.Table(snap.table_log2)
    win, st = table.insert(hs, np.arange(S * RB, dtype=np.uint32))
    assert st == 0 and (win == np.arange(S * RB)).all()
    h, hoff = oracle.hash_blocks(snap.tokens, snap.tok_off)
    k_total, n_gpu, _ = table.match_prefix(h, hoff)
    expect = np.minimum(snap.shared_tokens // 16, RB)   # first fresh token differs from the stream token
    assert (k_total == expect).all() and (n_gpu == expect).all()
    assert (snap.need_d >= k_total).all()


def test_table_insert_erase_retag_semantics():
    t = oracle.Table(4)
    win, st = t.insert([5, 9, 5, 0, 1, (1 << 64) - 1, (1 << 64) - 2], [50, 90, 51, 100, 101, 102, 103])
    # duplicates: lowest input index wins; reserved keys 0 -> 1 and 2^64-1 -> 2^64-2 are remapped
    assert st == 0 and win.tolist() == [50, 90, 50, 100, 100, 102, 102] and len(t) == 4
    win, _ = t.insert([9, 7], [99, 70])
    assert win.tolist() == [90, 70]                       # already-present entry wins
    assert t.lookup([5, 9, 7, 8, 0, 1]).tolist() == [50, 90, 70, MISS, 100, 100]
    t.erase([9, 12345])                                   # erasing an absent key is a no-op
    assert t.lookup([9]).tolist() == [MISS] and len(t) == 4
    t.retag([5, 9], [HOST | 3, 77])                        # retag of an absent key is a no-op
    assert t.lookup([5, 9]).tolist() == [HOST | 3, MISS]
    win, _ = t.insert([9], [91])                          # slot reuse after erase
    assert win.tolist() == [91]
    # capacity: 16 slots
    keys = np.arange(1000, 1020, dtype=np.uint64)
    win, st = t.insert(keys, np.arange(20, dtype=np.uint32))
    assert st == -2 and len(t) == 16 and (win[:11] == np.arange(11)).all() and (win[11:] == MISS).all()


def py_schedule(d, n_gpu, arr, rid, policy, free, evictable, max_admit):
    R = len(d)
    a = [max(int(d[i]) - int(n_gpu[i]), 0) for i in range(R)]
    if policy == 0:
        key = lambda i: (a[i], -int(n_gpu[i]), int(arr[i]), int(rid[i]), i)
    elif policy == 1:
        key = lambda i: (-int(n_gpu[i]), a[i], int(arr[i]), int(rid[i]), i)
    else:
        key = lambda i: (int(arr[i]), int(rid[i]), i)
    order = sorted(range(R), key=key)
    need = count = 0
    for i in order:
        if count >= max_admit or need + a[i] > free + evictable:
            break
        need += a[i]
        count += 1
    return order, count, max(0, need - free)


@pytest.mark.parametrize("policy", [0, 1, 2])
def test_schedule_equals_sorted_tuples_and_literal_admission(policy):
    g = np.random.default_rng(20 + policy)
    for trial in range(40):
        R = int(g.integers(0, 60))
        d = g.integers(1, 40, size=R).astype(np.uint32)
        n_gpu = np.minimum(g.integers(0, 40, size=R), d).astype(np.uint32)
        arr = g.integers(0, 8, size=R).astype(np.uint64)          # many ties
        rid = g.integers(0, 6, size=R).astype(np.uint32)          # even duplicate ids -> input index
        free, ev, mx = int(g.integers(0, 100)), int(g.integers(0, 200)), int(g.integers(0, 70))
        order, na, de = oracle.schedule(d, n_gpu, arr, rid, policy, free, ev, mx)
        eo, ena, ede = py_schedule(d, n_gpu, arr, rid, policy, free, ev, mx)
        assert order.tolist() == eo and (na, de) == (ena, ede)
        assert sorted(order.tolist()) == list(range(R))
        adm = order[:na]
        assert (d[adm].astype(int) - n_gpu[adm]).sum() <= free + ev and na <= mx


def test_schedule_special_cases():
    g = np.random.default_rng(30)
    R = 50
    arr = g.permutation(R).astype(np.uint64)
    rid = np.arange(R, dtype=np.uint32)
    d = np.full(R, 17, np.uint32)
    n_gpu = g.integers(0, 17, size=R).astype(np.uint32)
    o0, *_ = oracle.schedule(d, n_gpu, arr, rid, 0, 10, 10, R)
    o1, *_ = oracle.schedule(d, n_gpu, arr, rid, 1, 10, 10, R)
    assert o0.tolist() == o1.tolist()                    # all d equal: min-additional == overlap-first
    z = np.zeros(R, np.uint32)
    o0, *_ = oracle.schedule(d, z, arr, rid, 0, 10, 10, R)
    o2, *_ = oracle.schedule(d, z, arr, rid, 2, 10, 10, R)
    assert o0.tolist() == o2.tolist() == np.argsort(arr).tolist()    # no overlap, equal d: FCFS (L281)
    # the request needing the fewest additional blocks is dispatched first (L207)
    d = g.integers(1, 100, size=R).astype(np.uint32)
    n_gpu = np.minimum(g.integers(0, 100, size=R), d).astype(np.uint32)
    o0, na, de = oracle.schedule(d, n_gpu, arr, rid, 0, 1 << 20, 0, R)
    assert (d - n_gpu)[o0[0]] == (d - n_gpu).min() and na == R and de == 0
    # stop at the first misfit: no back-filling with a smaller later request
    d = np.array([5, 9, 1], np.uint32)
    o, na, de = oracle.schedule(d, np.zeros(3, np.uint32), [0, 1, 2], [0, 1, 2], 2, 4, 6, 3)
    assert o.tolist() == [0, 1, 2] and na == 1 and de == 1


# ---------------------------------------------------------------------------------------------- NEXT-3: chunked prefill
def _admit_chunked_brute(order, need, n_gpu, new_tokens, free, evictable, max_admit, budget):
    """PAPER.md L271 / DESIGN.md R8 restated as the literal loop, in Python integers."""
    chunk = [0] * len(need)
    used = blocks = count = 0
    for i in order:
        a = max(int(need[i]) - int(n_gpu[i]), 0)
        if count >= max_admit or blocks + a > free + evictable or used >= budget:
            break
        chunk[i] = min(int(new_tokens[i]), budget - used)
        used += chunk[i]
        blocks += a
        count += 1
    return chunk, count, max(0, blocks - free)


def test_admit_chunked_matches_the_literal_loop_and_its_special_cases():
    g = gen.rng(77, 0)
    for R in (1, 2, 17, 300):
        need = g.integers(1, 400, size=R).astype(np.uint32)
        n_gpu = np.minimum(need, g.integers(0, 400, size=R)).astype(np.uint32)
        new_tok = ((need - n_gpu).astype(np.int64) * 16 - g.integers(0, 16, size=R)).clip(0).astype(np.uint32)
        arr, rid = g.permutation(R).astype(np.uint64), np.arange(R, dtype=np.uint32)
        for policy in (0, 2):
            order, na0, de0 = oracle.schedule(need, n_gpu, arr, rid, policy, 50, 3000, R)
            for budget in (0, 1, 512, 2048, 10**7, 1 << 40):
                for max_admit in (1, 5, R):
                    ch, na, de = oracle.admit_chunked(order, need, n_gpu, new_tok, 50, 3000, max_admit, budget)
                    ech, ena, ede = _admit_chunked_brute(order, need, n_gpu, new_tok, 50, 3000, max_admit, budget)
                    assert ch.tolist() == ech and (na, de) == (ena, ede), (R, policy, budget, max_admit)
                    # invariants: the budget is never exceeded; only the LAST admitted request can get a partial chunk
                    assert int(ch.sum()) <= budget or budget == 0
                    adm = [int(i) for i in order[:na]]
                    assert all(ch[i] == new_tok[i] for i in adm[:-1])
                    assert all(ch[int(i)] == 0 for i in order[na:])
            # an unlimited budget admits exactly what cwo_schedule admits
            ch, na, de = oracle.admit_chunked(order, need, n_gpu, new_tok, 50, 3000, R, 1 << 62)
            assert (na, de) == (na0, de0) and (ch[order[:na]] == new_tok[order[:na]]).all()
    # requests with nothing to prefill (full hits) cost no budget and do not stop the walk
    order = np.arange(4, dtype=np.uint32)
    ch, na, de = oracle.admit_chunked(order, [5, 5, 5, 5], [5, 5, 1, 0], [0, 0, 600, 80], 0, 100, 4, 512)
    assert ch.tolist() == [0, 0, 512, 0] and na == 3 and de == 4     # the 4th finds the budget used up
