"""GPU parity — stage 2 (table, cw_match_prefix, cw_schedule) against the oracle, bit-exact."""
import numpy as np
import pytest

import oracle
from harness import gen

pytestmark = pytest.mark.gpu
MISS, HOST = 0xFFFFFFFF, 0x80000000


def _match(ctx, h, hoff, want_loc=True):
    from gpu_util import dev, host, zeros
    R = hoff.size - 1
    k, g, loc = zeros(R, np.uint32), zeros(R, np.uint32), zeros(h.size, np.uint32)
    ctx.match_prefix(dev(h), dev(hoff), R, k, g, loc if want_loc else None)
    assert ctx.sync(check=False) == 0
    return host(k, np.uint32)[:R], host(g, np.uint32)[:R], host(loc, np.uint32)[:h.size]


def _insert(ctx, keys, loc):
    from gpu_util import dev, host, zeros
    keys, loc = np.asarray(keys, np.uint64), np.asarray(loc, np.uint32)
    win = zeros(keys.size, np.uint32)
    ctx.table_insert(dev(keys), dev(loc), keys.size, win)
    st = ctx.sync(check=False)
    return host(win, np.uint32)[:keys.size], st


def _lookup(ctx, keys):
    from gpu_util import dev, host, zeros
    keys = np.asarray(keys, np.uint64)
    out = zeros(keys.size, np.uint32)
    ctx.table_lookup(dev(keys), keys.size, out)
    ctx.sync()
    return host(out, np.uint32)[:keys.size]


def test_table_insert_erase_retag_semantics():
    from gpu_util import dev, small_ctx
    ctx = small_ctx(num_blocks=8, table_log2_slots=4)
    ot = oracle.Table(4)
    M64 = (1 << 64) - 1
    keys, locs = [5, 9, 5, 0, 1, M64, M64 - 1], [50, 90, 51, 100, 101, 102, 103]
    win, st = _insert(ctx, keys, locs)
    ewin, est = ot.insert(keys, locs)
    assert st == est == 0 and (win == ewin).all()
    win, _ = _insert(ctx, [9, 7], [99, 70])
    ewin, _ = ot.insert([9, 7], [99, 70])
    assert (win == ewin).all()
    q = [5, 9, 7, 8, 0, 1, M64, M64 - 1]
    assert (_lookup(ctx, q) == ot.lookup(q)).all()
    ctx.table_erase(dev(np.array([9, 12345], np.uint64)), 2)
    ot.erase([9, 12345])
    ctx.table_retag(dev(np.array([5, 9], np.uint64)), dev(np.array([HOST | 3, 77], np.uint32)), 2)
    ot.retag([5, 9], [HOST | 3, 77])
    assert (_lookup(ctx, q) == ot.lookup(q)).all()
    win, _ = _insert(ctx, [9], [91])  # tombstone reuse
    ot.insert([9], [91])
    assert win.tolist() == [91] and _lookup(ctx, [9]).tolist() == [91]
    # capacity: 16 slots, 5 live -> the FIRST 11 of 20 new keys (by input index) fit, as in the oracle
    keys = np.arange(1000, 1020, dtype=np.uint64)
    win, st = _insert(ctx, keys, np.arange(20, dtype=np.uint32))
    ewin, est = ot.insert(keys, np.arange(20, dtype=np.uint32))
    assert st == est == -2 and (win == ewin).all() and (win != MISS).sum() == 11
    got = _lookup(ctx, keys)
    assert (got == win).all()
    ctx.close()


def test_insert_is_deterministic_under_heavy_duplication():
    from gpu_util import small_ctx
    g = gen.rng(21, 0)
    ctx = small_ctx(num_blocks=1 << 15, table_log2_slots=16)
    ot = oracle.Table(16)
    for rnd in range(3):
        keys = g.integers(1, 3000 * (rnd + 1), size=20000, dtype=np.uint64)  # ~7x duplication, clustered homes
        locs = g.integers(0, 1 << 20, size=keys.size, dtype=np.uint32)
        win, st = _insert(ctx, keys, locs)
        ewin, est = ot.insert(keys, locs)
        assert st == est == 0
        assert (win == ewin).all()
        kill = keys[g.integers(0, keys.size, size=500)]
        from gpu_util import dev
        ctx.table_erase(dev(kill), kill.size)
        ot.erase(kill)
        allk = np.arange(0, 9100, dtype=np.uint64)
        assert (_lookup(ctx, allk) == ot.lookup(allk)).all()
    ctx.close()


@pytest.mark.parametrize("holes", [False, True])
def test_match_prefix_scaled_stress_with_holes_and_host_tier(holes):
    from gpu_util import dev, small_ctx
    S, L, RB = 8, 16384, 512
    snap = gen.stress_snapshot(seed=6, S=S, L=L, RB=RB, req_per_session=24, len_median=3000, len_min=0 + 16,
                               len_max=L, hole_frac=0.02)
    ctx = small_ctx(num_blocks=snap.M, table_log2_slots=snap.table_log2, max_hashed_blocks=1 << 20)
    hs, _ = oracle.hash_blocks(snap.streams.reshape(-1), gen.stream_tok_off(S, L))
    hs = hs.reshape(S, L // 16)[:, :RB].reshape(-1)
    loc = np.arange(S * RB, dtype=np.uint32)
    loc[::7] |= HOST  # every 7th resident block lives in the host tier
    ot = oracle.Table(snap.table_log2)
    ot.insert(hs, loc)
    win, st = _insert(ctx, hs, loc)
    assert st == 0 and (win == loc).all()
    if holes:
        ot.erase(hs[snap.hole_ids])
        ctx.table_erase(dev(hs[snap.hole_ids]), snap.hole_ids.size)
    h, hoff = oracle.hash_blocks(snap.tokens, snap.tok_off)
    ek, eg, eloc = ot.match_prefix(h, hoff)
    k, g, gl = _match(ctx, h, hoff)
    assert (k == ek).all() and (g == eg).all() and (gl == eloc).all()
    if holes:
        assert (ot.lookup(h) != MISS).sum() > ek.sum()  # leading run != hit count somewhere
    k2, g2, _ = _match(ctx, h, hoff, want_loc=False)    # second call: scratch re-armed; NULL hit_loc
    assert (k2 == ek).all() and (g2 == eg).all()
    ctx.close()


def test_match_edge_cases_empty_requests_and_total_miss():
    from gpu_util import small_ctx
    ctx = small_ctx()
    ot = oracle.Table(12)
    g = gen.rng(22, 0)
    lens = [0, 3, 16 * 40, 0, 0, 16 * 3 + 1, 15, 16 * 70, 0]
    tok_off = np.concatenate([[0], np.cumsum(lens)]).astype(np.uint64)
    tokens = g.integers(0, gen.VOCAB, size=int(tok_off[-1]), dtype=np.int32)
    h, hoff = oracle.hash_blocks(tokens, tok_off)
    ek, eg, eloc = ot.match_prefix(h, hoff)
    k, gg, gl = _match(ctx, h, hoff)
    assert (k == 0).all() and (k == ek).all() and (gg == eg).all() and (gl == eloc).all()
    # make request 2 fully resident and request 7 resident except its first block
    keys = np.concatenate([h[int(hoff[2]):int(hoff[3])], h[int(hoff[7]) + 1:int(hoff[8])]])
    loc = np.arange(keys.size, dtype=np.uint32)
    ot.insert(keys, loc)
    _insert(ctx, keys, loc)
    ek, eg, eloc = ot.match_prefix(h, hoff)
    k, gg, gl = _match(ctx, h, hoff)
    assert ek[2] == 40 and ek[7] == 0
    assert (k == ek).all() and (gg == eg).all() and (gl == eloc).all()
    ctx.close()


def _schedule(ctx, d, n_gpu, arr, rid, policy, free, evictable, max_admit):
    from gpu_util import dev, host, zeros
    R = len(d)
    order, na, de = zeros(R, np.uint32), zeros(1, np.uint32), zeros(1, np.uint32)
    ctx.schedule(R, dev(d, np.uint32), dev(n_gpu, np.uint32), dev(arr, np.uint64), dev(rid, np.uint32), policy, free,
                 evictable, max_admit, order, na, de)
    assert ctx.sync(check=False) == 0
    return host(order, np.uint32)[:R], int(host(na, np.uint32)[0]), int(host(de, np.uint32)[0])


@pytest.mark.parametrize("policy", [0, 1, 2])
def test_schedule_random_queues(policy):
    from gpu_util import small_ctx
    ctx = small_ctx(max_requests=8192)
    g = gen.rng(23, policy)
    for R in [1, 2, 3, 31, 32, 33, 1000, 1024, 1025, 4096, 5000, 8192]:
        d = g.integers(0, 50, size=R).astype(np.uint32)             # many ties
        n_gpu = np.minimum(d, g.integers(0, 50, size=R)).astype(np.uint32)
        arr = g.integers(0, max(2, R // 4), size=R).astype(np.uint64)  # ties in arrival_seq too
        rid = g.integers(0, max(2, R // 2), size=R).astype(np.uint32)  # and in req_id: input index decides
        free, evictable = int(g.integers(0, 25 * R + 1)), int(g.integers(0, 10 * R + 1))
        max_admit = int(g.integers(0, R + 2))
        eo, ena, ede = oracle.schedule(d, n_gpu, arr, rid, policy, free, evictable, max_admit)
        o, na, de = _schedule(ctx, d, n_gpu, arr, rid, policy, free, evictable, max_admit)
        assert (o == eo).all() and (na, de) == (ena, ede), R
    ctx.close()


def test_schedule_more_requests_than_one_key_tile():
    """R > 8192: the leading key words are staged tile by tile; heavy ties force the second pass in every tile."""
    from gpu_util import small_ctx
    R = 20000
    ctx = small_ctx(max_requests=R)
    g = gen.rng(24, 0)
    for policy in (0, 1, 2):
        d = g.integers(0, 20, size=R).astype(np.uint32)
        n_gpu = np.minimum(d, g.integers(0, 20, size=R)).astype(np.uint32)
        arr = g.integers(0, 50, size=R).astype(np.uint64)
        rid = g.integers(0, 100, size=R).astype(np.uint32)
        eo, ena, ede = oracle.schedule(d, n_gpu, arr, rid, policy, 1000, 50000, R)
        o, na, de = _schedule(ctx, d, n_gpu, arr, rid, policy, 1000, 50000, R)
        assert (o == eo).all() and (na, de) == (ena, ede), policy
    ctx.close()


def test_schedule_wide_key_ranges_and_tie_groups():
    """Leading words whose ranges do not fit the compressed 30-bit key (64-bit path), and tie groups on the leading
    word of every size around the per-warp tie list (128): the remaining key words decide inside a group."""
    from gpu_util import small_ctx
    ctx = small_ctx(max_requests=8192)
    g = gen.rng(25, 0)
    for policy in (0, 1, 2):
        for R in (100, 4096, 6000):
            d = g.integers(0, 2**32, size=R, dtype=np.uint64).astype(np.uint32)
            n_gpu = (g.random(R) * d).astype(np.uint32)
            arr = g.integers(0, 2**63, size=R, dtype=np.uint64) * np.uint64(2) + np.uint64(1)
            rid = g.integers(0, 2**32, size=R, dtype=np.uint64).astype(np.uint32)
            eo, ena, ede = oracle.schedule(d, n_gpu, arr, rid, policy, 10**9, 10**9, R)
            o, na, de = _schedule(ctx, d, n_gpu, arr, rid, policy, 10**9, 10**9, R)
            assert (o == eo).all() and (na, de) == (ena, ede), (policy, R)
    for policy in (0, 1, 2):
        R = 4096
        grp = np.repeat(np.arange(16), [1, 2, 3, 31, 32, 33, 127, 128, 129, 130, 255, 256, 257, 500, 1000, 1342])[:R]
        perm = g.permutation(R)
        d = (1000 + 3 * grp[perm]).astype(np.uint32)
        n_gpu = (grp[perm] % 5).astype(np.uint32)
        arr = np.where(policy == 2, grp[perm], g.integers(0, 7, size=R)).astype(np.uint64)
        rid = g.integers(0, 4, size=R).astype(np.uint32)
        eo, ena, ede = oracle.schedule(d, n_gpu, arr, rid, policy, 5000, 100000, R)
        o, na, de = _schedule(ctx, d, n_gpu, arr, rid, policy, 5000, 100000, R)
        assert (o == eo).all() and (na, de) == (ena, ede), policy
    ctx.close()


def test_schedule_edges():
    import paper_2606_16824_b200 as cw
    from gpu_util import small_ctx
    ctx = small_ctx(max_requests=8192)
    # R = 0
    o, na, de = _schedule(ctx, [], [], [], [], 0, 5, 5, 5)
    assert (na, de) == (0, 0)
    # huge needs: 64-bit running sums, deficit exact
    R = 4096
    d = np.full(R, 0xFFFFFFFF, np.uint32)
    z = np.zeros(R, np.uint32)
    arr = np.arange(R, dtype=np.uint64)[::-1].copy()
    eo, ena, ede = oracle.schedule(d, z, arr, z, 2, 0xFFFFFFFF, 0xFFFFFFFF, R)
    o, na, de = _schedule(ctx, d, z, arr, z, 2, 0xFFFFFFFF, 0xFFFFFFFF, R)
    assert (o == eo).all() and (na, de) == (ena, ede) and na == 2
    # n_gpu > d clamps a to 0; everything admitted, no deficit
    eo, ena, ede = oracle.schedule(z, d, arr, z, 0, 0, 0, R)
    o, na, de = _schedule(ctx, z, d, arr, z, 0, 0, 0, R)
    assert (o == eo).all() and (na, de) == (ena, ede) == (R, 0)
    with pytest.raises(cw.CwError):
        _schedule(ctx, [1], [0], [0], [0], 3, 1, 1, 1)
    ctx.close()
