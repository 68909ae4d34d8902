"""GPU parity — cw_match_prefix_shared (the shared part of a request is looked up once, through its leader) against
the oracle's plain per-request definition, bit-exact, on CHAIN hashes (the call's precondition), and against
cw_match_prefix on the same inputs.  Hints of every kind: the longest request of the session, a random request of the
session, a request of ANOTHER session (shares nothing), itself, a non-leader, an index out of range."""
import numpy as np
import pytest

import oracle
from harness import gen

pytestmark = pytest.mark.gpu
MISS, HOST = 0xFFFFFFFF, 0x80000000


def _shared(ctx, h, hoff, leader, want_loc=True):
    from gpu_util import dev, host, zeros
    R = hoff.size - 1
    G = 32                                                  # guard words around every output
    k, g, loc = zeros(R + 2 * G, np.uint32), zeros(R + 2 * G, np.uint32), zeros(h.size + 2 * G, np.uint32)
    for t in (k, g, loc):
        t.fill_(0x5A5A5A5A)                                 # every position must be written, nothing beside them
    ctx.match_prefix_shared(dev(h), dev(hoff), R, dev(np.asarray(leader, np.uint32)), k[G:], g[G:],
                            loc[G:] if want_loc else None)
    assert ctx.sync(check=False) == 0
    hk, hg, hl = host(k, np.uint32), host(g, np.uint32), host(loc, np.uint32)
    for a, n in ((hk, R), (hg, R), (hl, h.size)):
        assert (a[:G] == 0x5A5A5A5A).all() and (a[G + n:] == 0x5A5A5A5A).all(), "write outside an output array"
    return hk[G:G + R], hg[G:G + R], hl[G:G + h.size]


def _flat(ctx, h, hoff):
    from gpu_util import dev, host, zeros
    R = hoff.size - 1
    k, g, loc = zeros(R, np.uint32), zeros(R, np.uint32), zeros(h.size, np.uint32)
    ctx.match_prefix(dev(h), dev(hoff), R, k, g, loc)
    assert ctx.sync(check=False) == 0
    return host(k, np.uint32)[:R], host(g, np.uint32)[:R], host(loc, np.uint32)[:h.size]


def _longest_of_session(req_session, n):
    lead = np.arange(req_session.size, dtype=np.uint32)
    for s in np.unique(req_session):
        idx = np.nonzero(req_session == s)[0]
        lead[idx] = idx[np.argmax(n[idx])]
    return lead


def _hints(snap, n, g):
    R = n.size
    longest = _longest_of_session(snap.req_session, n)
    yield "longest of the session", longest
    yield "itself", np.arange(R, dtype=np.uint32)
    rnd = longest.copy()                                    # a random request of the session as the session's leader
    for s in np.unique(snap.req_session):
        idx = np.nonzero(snap.req_session == s)[0]
        rnd[idx] = idx[g.integers(0, idx.size)]
    yield "random request of the session", rnd
    other = np.roll(longest, 24 * 3)                        # leaders of another session: nothing is shared
    other[other == np.arange(R)] = 0
    yield "another session", other.astype(np.uint32)
    mixed = longest.copy()                                  # non-leaders, out-of-range indices, chains of hints
    mixed[::5] = (np.arange(R, dtype=np.uint32)[::5] + 1) % R
    mixed[3::11] = R + 7
    mixed[4::13] = 0xFFFFFFFF
    yield "mixed and invalid", mixed


@pytest.mark.parametrize("holes", [False, True])
def test_shared_match_scaled_stress_all_hint_kinds(holes):
    from gpu_util import dev, small_ctx
    S, L, RB = 8, 16384, 512
    snap = gen.stress_snapshot(seed=6, S=S, L=L, RB=RB, req_per_session=24, len_median=3000, len_min=0 + 16,
                               len_max=L, hole_frac=0.02)
    ctx = small_ctx(num_blocks=snap.M, table_log2_slots=snap.table_log2, max_hashed_blocks=1 << 20)
    hs, _ = oracle.hash_blocks(snap.streams.reshape(-1), gen.stream_tok_off(S, L))
    hs = hs.reshape(S, L // 16)[:, :RB].reshape(-1)
    loc = np.arange(S * RB, dtype=np.uint32)
    loc[::7] |= HOST                                        # every 7th resident block lives in the host tier
    ot = oracle.Table(snap.table_log2)
    ot.insert(hs, loc)
    from test_gpu_match_schedule import _insert
    win, st = _insert(ctx, hs, loc)
    assert st == 0 and (win == loc).all()
    if holes:
        ot.erase(hs[snap.hole_ids])
        ctx.table_erase(dev(hs[snap.hole_ids]), snap.hole_ids.size)
    h, hoff = oracle.hash_blocks(snap.tokens, snap.tok_off)
    n = (hoff[1:] - hoff[:-1]).astype(np.int64)
    ek, eg, eloc = ot.match_prefix(h, hoff)
    g = gen.rng(77, 0)
    for name, lead in _hints(snap, n, g):
        k, gg, gl = _shared(ctx, h, hoff, lead)
        assert (k == ek).all() and (gg == eg).all(), name
        bad = np.nonzero(gl != eloc)[0]
        assert bad.size == 0, (name, bad[:5], gl[bad[:5]], eloc[bad[:5]])
        k2, g2, _ = _shared(ctx, h, hoff, lead, want_loc=False)          # NULL hit_loc; scratch re-armed
        assert (k2 == ek).all() and (g2 == eg).all(), name
        fk, fg, fl = _flat(ctx, h, hoff)                                   # the plain call right after: scratch is armed
        assert (fk == ek).all() and (fg == eg).all() and (fl == eloc).all(), name
    ctx.close()


def test_shared_match_followers_longer_than_the_leader_and_resident_tails():
    """A follower that goes on matching BEHIND the shared prefix (its own tail is resident), a follower that is a
    strict prefix of its leader, identical requests, empty requests, a leader whose run ends inside the shared part."""
    from gpu_util import small_ctx
    from test_gpu_match_schedule import _insert
    g = gen.rng(31, 0)
    base = g.integers(0, gen.VOCAB, size=16 * 700, dtype=np.int32)
    alt = g.integers(0, gen.VOCAB, size=16 * 300, dtype=np.int32)
    reqs = [base[:16 * 400],                                              # 0 leader (hint target)
            np.concatenate([base[:16 * 250], alt]),                       # 1 shares 250, own tail of 300 (resident)
            base[:16 * 130 + 5],                                          # 2 strict prefix of the leader
            base[:16 * 400],                                              # 3 identical to the leader
            np.zeros(0, np.int32),                                        # 4 empty
            base[:16 * 700],                                              # 5 LONGER than its leader
            np.concatenate([base[:16 * 390], alt[:16 * 9 + 3]]),          # 6 shares 390
            alt[:7]]                                                      # 7 no full block
    tok_off = np.concatenate([[0], np.cumsum([r.size for r in reqs])]).astype(np.uint64)
    tokens = np.concatenate(reqs)
    h, hoff = oracle.hash_blocks(tokens, tok_off)
    lead = np.zeros(len(reqs), np.uint32)
    for resident_upto in (700, 300, 260, 0):                             # the leader's run ends at min(400, this)
        ctx = small_ctx()
        ot = oracle.Table(12)
        keys = np.concatenate([h[int(hoff[5]):int(hoff[5]) + resident_upto],          # base blocks [0, upto)
                               h[int(hoff[1]) + 250:int(hoff[2])][:280]])             # request 1's own tail, 280 of 300
        locs = np.arange(keys.size, dtype=np.uint32)
        locs[5::9] |= HOST
        ot.insert(keys, locs)
        _insert(ctx, keys, locs)
        ek, eg, eloc = ot.match_prefix(h, hoff)
        k, gg, gl = _shared(ctx, h, hoff, lead)
        assert (k == ek).all() and (gg == eg).all() and (gl == eloc).all(), resident_upto
        if resident_upto == 700:
            assert ek.tolist() == [400, 530, 130, 400, 0, 700, 390, 0]
        ctx.close()


def test_shared_match_on_a_slice_of_a_longer_csr():
    """hash_off may be a slice of a longer CSR array (absolute offsets), as for cw_match_prefix: requests [a, b) of the
    queue, leader indices relative to the slice, outputs at the absolute positions of d_hit_loc."""
    from gpu_util import dev, host, small_ctx, zeros
    from test_gpu_match_schedule import _insert
    S, L, RB = 6, 8192, 256
    snap = gen.stress_snapshot(seed=9, S=S, L=L, RB=RB, req_per_session=10, len_median=2500, len_min=16, len_max=L)
    ctx = small_ctx(num_blocks=snap.M, table_log2_slots=snap.table_log2, max_hashed_blocks=1 << 20)
    hs, _ = oracle.hash_blocks(snap.streams.reshape(-1), gen.stream_tok_off(S, L))
    hs = hs.reshape(S, L // 16)[:, :RB].reshape(-1)
    loc = np.arange(S * RB, dtype=np.uint32)
    ot = oracle.Table(snap.table_log2)
    ot.insert(hs, loc)
    _insert(ctx, hs, loc)
    h, hoff = oracle.hash_blocks(snap.tokens, snap.tok_off)
    n = (hoff[1:] - hoff[:-1]).astype(np.int64)
    ek, eg, eloc = ot.match_prefix(h, hoff)
    lead = _longest_of_session(snap.req_session, n)
    a, b = 13, 47                                           # cuts sessions 1 and 4 in two
    sl = lead[a:b].astype(np.int64) - a
    sl[(sl < 0) | (sl >= b - a)] = np.arange(b - a)[(sl < 0) | (sl >= b - a)]      # leader outside the slice: own
    R = b - a
    k, gg = zeros(R, np.uint32), zeros(R, np.uint32)
    d_loc = zeros(h.size, np.uint32)
    d_loc.fill_(0x5A5A5A5A)
    d_hoff = dev(hoff)
    ctx.match_prefix_shared(dev(h), d_hoff[a:], R, dev(sl.astype(np.uint32)), k, gg, d_loc)
    assert ctx.sync(check=False) == 0
    assert (host(k, np.uint32)[:R] == ek[a:b]).all() and (host(gg, np.uint32)[:R] == eg[a:b]).all()
    got = host(d_loc, np.uint32)[:h.size]
    lo, hi = int(hoff[a]), int(hoff[b])
    assert (got[lo:hi] == eloc[lo:hi]).all()
    assert (got[:lo] == 0x5A5A5A5A).all() and (got[hi:] == 0x5A5A5A5A).all()
    ctx.close()
