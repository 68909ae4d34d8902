"""GPU parity — stage 3 (cw_score_evict) and stage 4 (cw_gather/scatter_pages, cw_swap_out/in) against the
oracle, bit-exact, through the C ABI."""
import numpy as np
import pytest

import oracle
from harness import gen

pytestmark = pytest.mark.gpu
V, P = 0x80000000, 0x40000000
TAU_MAX = (1 << 24) - 1


def _load_meta(ctx, tier, sess, last, depth, rf):
    from gpu_util import dev
    M = len(sess)
    ctx.blocks_update(tier, dev(np.arange(M, dtype=np.uint32)), M, session=dev(sess, np.uint32),
                      depth=dev(depth, np.uint32), last_access=dev(last, np.uint32), ref_flags=dev(rf, np.uint32))


def _evict(ctx, tick, feats, w, bias, state, override, deficit, cap, tier=0, want_scores=True):
    from gpu_util import dev, host, zeros
    S, F = feats.shape
    vic, sc, nv = zeros(cap, np.uint32), zeros(cap, np.uint64), zeros(1, np.uint32)
    ctx.score_evict(tick, S, F, dev(feats, np.uint8), dev(w, np.int16), bias, dev(state, np.uint8),
                    None if override is None else dev(override, np.uint32), dev(np.array([deficit], np.uint32)), tier,
                    vic, sc if want_scores else None, nv, cap)
    st = ctx.sync(check=False)
    n = int(host(nv, np.uint32)[0])
    return host(vic, np.uint32)[:n], host(sc, np.uint64)[:n], st


def _random_pool(g, M, S, F):
    sess = g.integers(0, S + 2, size=M).astype(np.uint32)
    last = g.integers(900, 1010, size=M).astype(np.uint32)
    depth = g.integers(0, 50, size=M).astype(np.uint32)
    rf = np.where(g.random(M) < 0.85, V, 0).astype(np.uint32)
    rf |= np.where(g.random(M) < 0.2, g.integers(1, 4, size=M), 0).astype(np.uint32)
    rf |= np.where(g.random(M) < 0.1, P, 0).astype(np.uint32)
    feats = g.integers(0, 256, size=(S, F), dtype=np.uint8)
    w = g.integers(-300, 300, size=F).astype(np.int16)
    state = g.integers(0, 5, size=S).astype(np.uint8)
    return sess, last, depth, rf, feats, w, state


@pytest.mark.parametrize("M", [1, 7, 2048, 2049, 4096, 4097, 30000, 70001])
def test_score_evict_random_pools_many_ties(M):
    """Few distinct scores (heavy ties => the block-id tie-break decides), every deficit regime: 0, small,
    below / at / above one sort run, all evictable, more than evictable (CW_E_CAPACITY)."""
    from gpu_util import small_ctx
    g = gen.rng(31, M)
    S, F = 6, 4
    ctx = small_ctx(num_blocks=M, table_log2_slots=max(4, int(np.ceil(np.log2(2 * M)))), max_sessions=S)
    sess, last, depth, rf, feats, w, state = _random_pool(g, M, S, F)
    _load_meta(ctx, 0, sess, last, depth, rf)
    for deficit in sorted({0, 1, 2, M // 3, 4095, 4096, 4097, 9000, M - 1, M, M + 5}):
        if deficit < 0:
            continue
        ev, es, est = oracle.score_evict(1000, feats, w, 1000, state, None, deficit, sess, last, depth, rf, cap=M)
        gv, gs, gst = _evict(ctx, 1000, feats, w, 1000, state, None, deficit, M)
        assert gst == est, (deficit, gst, est)
        assert gv.tolist() == ev.tolist() and gs.tolist() == es.tolist(), deficit
    ctx.close()


def test_score_evict_cap_override_null_scores_and_repeat():
    from gpu_util import small_ctx
    g = gen.rng(32, 0)
    M, S, F = 50000, 40, 16
    ctx = small_ctx(num_blocks=M, table_log2_slots=17, max_sessions=S)
    sess, last, depth, rf, feats, w, state = _random_pool(g, M, S, F)
    depth = g.integers(0, 1 << 22, size=M).astype(np.uint32)   # beyond the 20-bit clamp
    last = g.integers(0, 1 << 22, size=M).astype(np.uint32)
    w = g.integers(-32768, 32768, size=F).astype(np.int16)
    _load_meta(ctx, 0, sess, last, depth, rf)
    ov = g.integers(0, 1 << 25, size=S).astype(np.uint32)
    tick = 1 << 21
    for override, bias, deficit, cap in [(None, -(1 << 30), 777, M), (None, 1 << 30, 20000, 5000), (ov, 0, 12345, M),
                                         (None, 3_000_000, 6000, M)]:
        ev, es, est = oracle.score_evict(tick, feats, w, bias, state, override, deficit, sess, last, depth, rf, cap=cap)
        for _ in range(2):  # second call: the kernel re-zeroed its own scratch
            gv, gs, gst = _evict(ctx, tick, feats, w, bias, state, override, deficit, cap)
            assert gst == est and gv.tolist() == ev.tolist() and gs.tolist() == es.tolist()
        gv, _, _ = _evict(ctx, tick, feats, w, bias, state, override, deficit, cap, want_scores=False)
        assert gv.tolist() == ev.tolist()
    ctx.close()


def test_score_evict_scaled_stress_snapshot_and_host_tier():
    from gpu_util import small_ctx
    snap = gen.stress_snapshot(seed=7, S=32, L=32768, RB=2048, req_per_session=2, len_median=4096, len_min=64,
                               len_max=32768)
    M, S = snap.M, 32
    ctx = small_ctx(num_blocks=M, host_slots=M, table_log2_slots=snap.table_log2 + 1, max_sessions=S)
    args = (snap.blk_session, snap.blk_last_access, snap.blk_depth, snap.blk_ref_flags)
    _load_meta(ctx, 0, *args)
    ev, es, est = oracle.score_evict(snap.tick_now, snap.features, snap.weights, snap.bias, snap.session_state, None,
                                     snap.deficit, *args)
    gv, gs, gst = _evict(ctx, snap.tick_now, snap.features, snap.weights, snap.bias, snap.session_state, None,
                         snap.deficit, M)
    assert gst == est == 0 and gv.tolist() == ev.tolist() and gs.tolist() == es.tolist()
    # invariants (PAPER.md L252 unreferenced only, L277 idle sessions first)
    assert (snap.blk_ref_flags[gv] == V).all()
    n_idle_blocks = int((snap.session_state[snap.blk_session] == gen.IDLE).sum())
    k = min(n_idle_blocks, gv.size)
    assert (snap.session_state[snap.blk_session[gv[:k]]] == gen.IDLE).all()
    # tier 1 has its own metadata: empty until updated -> nothing evictable -> CW_E_CAPACITY, 0 victims
    gv1, _, st1 = _evict(ctx, snap.tick_now, snap.features, snap.weights, snap.bias, snap.session_state, None, 10, M,
                         tier=1)
    assert gv1.size == 0 and st1 == -2
    rev = (snap.blk_session[::-1].copy(), snap.blk_last_access[::-1].copy(), snap.blk_depth[::-1].copy(),
           snap.blk_ref_flags[::-1].copy())
    _load_meta(ctx, 1, *rev)
    ev, es, est = oracle.score_evict(snap.tick_now, snap.features, snap.weights, snap.bias, snap.session_state, None,
                                     1000, *rev)
    gv1, gs1, st1 = _evict(ctx, snap.tick_now, snap.features, snap.weights, snap.bias, snap.session_state, None, 1000,
                           M, tier=1)
    assert st1 == est and gv1.tolist() == ev.tolist() and gs1.tolist() == es.tolist()
    ctx.close()


@pytest.mark.parametrize("bulks", [(10000,), (3000, 3000), (5000, 40, 4500)])
def test_score_evict_ordering_paths_medium_and_large_buckets(bulks):
    """Keys built to defeat the 16-bit bucket split of the ordering phase: 16 - log2(#bulks) outlier sessions
    own the top varying bits, so every bulk session (equal tau, thousands of blocks) lands in ONE bucket —
    medium buckets (CTA sort) and buckets above 4096 keys (grid-wide bitonic fallback) must both agree with
    the oracle, and so must a repeat of the call (self-cleaning scratch)."""
    from gpu_util import small_ctx
    g = gen.rng(33, sum(bulks))
    nb = len(bulks)
    low = {1: 0, 2: 1, 3: 2}[nb]                      # tau bits used to tell the bulks apart
    n_out = 16 - low
    S = nb + n_out
    tau = np.zeros(S, np.uint32)
    for b in range(nb):
        tau[b] = TAU_MAX - 1 - (b << 8)               # v = TAU_MAX - tau = 1 + (b << 8)
    for o in range(n_out):
        tau[nb + o] = TAU_MAX - 1 - (1 << (8 + low + o))
    sess = np.concatenate([np.full(n, b, np.uint32) for b, n in enumerate(bulks)] +
                          [np.arange(nb, S, dtype=np.uint32)])
    M = sess.size
    perm = g.permutation(M)
    sess = sess[perm]
    depth = g.integers(0, 6000, size=M).astype(np.uint32)        # ties inside a bulk: the id decides
    last = np.full(M, 500, np.uint32)
    rf = np.full(M, V, np.uint32)
    feats = np.zeros((S, 4), np.uint8)
    w = np.zeros(4, np.int16)
    state = np.zeros(S, np.uint8)
    ctx = small_ctx(num_blocks=M, table_log2_slots=max(4, int(np.ceil(np.log2(2 * M)))), max_sessions=S)
    _load_meta(ctx, 0, sess, last, depth, rf)
    for deficit in (M, M - 7, 4097):
        ev, es, est = oracle.score_evict(1000, feats, w, 0, state, tau, deficit, sess, last, depth, rf, cap=M)
        for _ in range(2):
            gv, gs, gst = _evict(ctx, 1000, feats, w, 0, state, tau, deficit, M)
            assert gst == est == 0 and gv.tolist() == ev.tolist() and gs.tolist() == es.tolist(), deficit
    ctx.close()


def test_score_evict_more_sessions_than_the_shared_memory_table():
    """S > 4096: tau goes through global memory (one more grid barrier) instead of the per-CTA table."""
    from gpu_util import small_ctx
    g = gen.rng(34, 0)
    M, S, F = 60000, 5000, 8
    ctx = small_ctx(num_blocks=M, table_log2_slots=17, max_sessions=S)
    sess, last, depth, rf, feats, w, state = _random_pool(g, M, S, F)
    _load_meta(ctx, 0, sess, last, depth, rf)
    for deficit in (100, 5000, 30000):
        ev, es, est = oracle.score_evict(1000, feats, w, 500, state, None, deficit, sess, last, depth, rf, cap=M)
        gv, gs, gst = _evict(ctx, 1000, feats, w, 500, state, None, deficit, M)
        assert gst == est and gv.tolist() == ev.tolist() and gs.tolist() == es.tolist(), deficit
    ctx.close()


def test_score_evict_host_side_argument_checks():
    import paper_2606_16824_b200 as cw
    from gpu_util import dev, small_ctx, zeros
    ctx = small_ctx(num_blocks=64, table_log2_slots=8, max_sessions=4)
    f, w, s = dev(np.zeros((4, 4), np.uint8)), dev(np.zeros(4, np.int16)), dev(np.zeros(4, np.uint8))
    d, v, n = dev(np.array([1], np.uint32)), zeros(64, np.uint32), zeros(1, np.uint32)
    bad = [dict(bias=(1 << 30) + 1), dict(S=5), dict(F=17), dict(tier=2), dict(deficit=None), dict(victims=None)]
    for kw in bad:
        a = dict(tick_now=1, S=4, F=4, features=f, weights=w, bias=0, session_state=s, tau_override=None, deficit=d,
                 tier=0, victims=v, victim_scores=None, num_victims=n, cap=64)
        a.update(kw)
        with pytest.raises(cw.CwError) as e:
            ctx.score_evict(**a)
        assert e.value.code == cw.CW_E_INVAL, kw
    with pytest.raises(cw.CwError) as e:  # tier 1 without host slots
        ctx.score_evict(1, 4, 4, f, w, 0, s, None, d, 1, v, None, n, 64)
    assert e.value.code == cw.CW_E_STATE
    ctx.close()


# ------------------------------------------------------------------------------------------------ stage 4
LAYOUTS = ["layer_major", "block_major"]


def _pool_cfg(layout, M, n_chunks, chunk_bytes):
    if layout == "layer_major":   # vLLM-like: one [M, chunk] array per (layer, K|V)
        return dict(chunk_stride=M * chunk_bytes, block_stride=chunk_bytes)
    return dict(chunk_stride=chunk_bytes, block_stride=n_chunks * chunk_bytes)


def _swap_ctx(layout, M, n_chunks, chunk_bytes, staging_pages, pool_np):
    import torch
    from gpu_util import small_ctx
    pool = torch.from_numpy(pool_np.copy()).cuda()
    page = n_chunks * chunk_bytes
    ctx = small_ctx(num_blocks=M, table_log2_slots=max(4, int(np.ceil(np.log2(2 * M)))), n_chunks=n_chunks,
                    chunk_bytes=chunk_bytes, pool=pool, staging_bytes=2 * staging_pages * page,
                    **_pool_cfg(layout, M, n_chunks, chunk_bytes))
    return ctx, pool


@pytest.mark.parametrize("layout", LAYOUTS)
@pytest.mark.parametrize("n_chunks,chunk_bytes", [(4, 4096), (3, 16), (2, 16384 + 48), (5, 40000)])
def test_gather_scatter_pages_equal_memcpy_loop(layout, n_chunks, chunk_bytes):
    """C1-shaped page (2 layers x {K,V} x 2 heads x 64 x 16 fp16 = 4 chunks of 4 KiB) and odd shapes: a chunk
    of one 16-byte unit, a chunk just over one TMA piece, a chunk of several pieces with a ragged tail."""
    import torch
    from gpu_util import dev, host
    M = 97
    g = gen.rng(33, n_chunks)
    page = n_chunks * chunk_bytes
    pool_np = g.integers(0, 256, size=M * page, dtype=np.uint8)
    ctx, pool = _swap_ctx(layout, M, n_chunks, chunk_bytes, 4, pool_np)
    cfg = _pool_cfg(layout, M, n_chunks, chunk_bytes)
    for n in (0, 1, 2, 40, 97):
        ids = g.permutation(M)[:n].astype(np.uint32)
        exp = oracle.swap_out(pool_np, n_chunks, chunk_bytes, cfg["chunk_stride"], cfg["block_stride"], ids,
                              np.zeros(max(n, 1) * page, np.uint8))
        staged = torch.full((max(n, 1) * page + 64,), 0xAB, dtype=torch.uint8, device="cuda")
        ctx.gather_pages(dev(ids) if n else dev(np.zeros(1, np.uint32)), None, n, staged)
        assert ctx.sync(check=False) == 0
        got = staged.cpu().numpy()
        assert (got[:n * page] == exp[:n * page]).all()
        assert (got[n * page:] == 0xAB).all()   # nothing written past the last page
        # scatter into DIFFERENT block ids and compare with the oracle's swap_in on a copy of the pool
        dst = g.permutation(M)[:n].astype(np.uint32)
        exp_pool = oracle.swap_in(host(pool, np.uint8).copy(), n_chunks, chunk_bytes, cfg["chunk_stride"],
                                  cfg["block_stride"], exp, dst)
        ctx.scatter_pages(dev(dst) if n else dev(np.zeros(1, np.uint32)), None, n, staged)
        assert ctx.sync(check=False) == 0
        assert (host(pool, np.uint8) == exp_pool).all()   # every other pool byte untouched
        pool_np = exp_pool                                # the next round gathers from the scattered pool
        # device-side count smaller than cap
        if n >= 2:
            staged.fill_(0xCD)
            ctx.gather_pages(dev(ids), dev(np.array([n - 1], np.uint32)), n, staged)
            ctx.sync()
            got = staged.cpu().numpy()
            exp2 = oracle.swap_out(host(pool, np.uint8), n_chunks, chunk_bytes, cfg["chunk_stride"],
                                   cfg["block_stride"], ids[:n - 1], np.zeros(n * page, np.uint8))
            assert (got[:(n - 1) * page] == exp2[:(n - 1) * page]).all() and (got[(n - 1) * page:] == 0xCD).all()
    ctx.close()


@pytest.mark.parametrize("layout", LAYOUTS)
def test_swap_out_swap_in_round_trip_through_pinned_host(layout):
    """Staging ring of 3 pages per half => 20 victims take 7 slices (ragged last slice); contiguous and
    slot-addressed host layouts; swap-in into different block ids; byte-identical (SURVEY 8c stage-4 pins)."""
    import torch
    from gpu_util import dev, host
    M, n_chunks, chunk_bytes = 64, 4, 4096
    page = n_chunks * chunk_bytes
    g = gen.rng(34, 0)
    pool_np = g.integers(0, 256, size=M * page, dtype=np.uint8)
    ctx, pool = _swap_ctx(layout, M, n_chunks, chunk_bytes, 3, pool_np)
    cfg = _pool_cfg(layout, M, n_chunks, chunk_bytes)
    n = 20
    vic = g.permutation(M)[:n].astype(np.uint32)
    # (a) contiguous host buffer
    h = torch.zeros(n * page, dtype=torch.uint8).pin_memory()
    ctx.swap_out(dev(vic), None, n, None, h)
    assert ctx.sync(check=False) == 0
    exp = oracle.swap_out(pool_np, n_chunks, chunk_bytes, cfg["chunk_stride"], cfg["block_stride"], vic,
                          np.zeros(n * page, np.uint8))
    assert (h.numpy() == exp).all()
    # (b) slot-addressed host tier, some slots consecutive (coalesced copies) and some not
    slots = np.array([5, 6, 7, 30, 2, 3, 40, 41, 42, 43, 0, 20, 21, 9, 11, 10, 50, 51, 52, 1], np.uint32)
    tier = torch.zeros(64 * page, dtype=torch.uint8).pin_memory()
    ctx.swap_out(dev(vic), None, n, slots, tier)
    assert ctx.sync(check=False) == 0
    exp_tier = oracle.swap_out(pool_np, n_chunks, chunk_bytes, cfg["chunk_stride"], cfg["block_stride"], vic,
                               np.zeros(64 * page, np.uint8), slots=slots)
    assert (tier.numpy() == exp_tier).all()
    # (c) swap-in from the tier into different blocks
    dst = g.permutation(M)[:n].astype(np.uint32)
    exp_pool = oracle.swap_in(pool_np.copy(), n_chunks, chunk_bytes, cfg["chunk_stride"], cfg["block_stride"],
                              exp_tier, dst, slots=slots)
    ctx.swap_in(slots, tier, dev(dst), n)
    assert ctx.sync(check=False) == 0
    assert (host(pool, np.uint8) == exp_pool).all()
    # (d) contiguous swap-in restores the victims' original bytes in place
    pool.copy_(torch.from_numpy(np.zeros(M * page, np.uint8)))
    ctx.swap_in(None, h, dev(vic), n)
    ctx.sync()
    now = host(pool, np.uint8)
    back = oracle.swap_out(now, n_chunks, chunk_bytes, cfg["chunk_stride"], cfg["block_stride"], vic,
                           np.zeros(n * page, np.uint8))
    assert (back == exp).all()
    ctx.swap_out(dev(vic), None, 0, None, h)  # n = 0 is a no-op
    assert ctx.sync(check=False) == 0
    ctx.close()


@pytest.mark.parametrize("layout", LAYOUTS)
@pytest.mark.parametrize("tp", [2, 4])
def test_tp_sharded_swap_equals_the_unsharded_page(layout, tp):
    """SURVEY 8(e) / PAPER.md L271 (TP=2): stage 4 shards by KV head with no exchange.  Rank t holds bytes
    [t*cb/tp, (t+1)*cb/tp) of every chunk (chunk = [kv_head][token][dim]) in its own pool and runs the SAME victim
    list (decisions are replicated); the rank pages, re-interleaved per chunk, must equal the oracle's page of the
    unsharded pool, and swapping them back in must restore every rank's pool bytes."""
    import torch
    from gpu_util import dev, host
    M, n_chunks, cb = 48, 6, 8192
    g = gen.rng(36, tp)
    full = g.integers(0, 256, size=(n_chunks, M, cb), dtype=np.uint8)       # [chunk][block][byte]
    full_cfg = _pool_cfg("layer_major", M, n_chunks, cb)
    n = 17
    vic = g.permutation(M)[:n].astype(np.uint32)
    exp = oracle.swap_out(full.reshape(-1).copy(), n_chunks, cb, full_cfg["chunk_stride"], full_cfg["block_stride"], vic,
                          np.zeros(n * n_chunks * cb, np.uint8)).reshape(n, n_chunks, cb)
    from harness import tp as htp
    sb = cb // tp
    pages, ctxs = [], []
    for t in range(tp):
        assert htp.head_slice(cb, tp, t) == (t * sb, sb)
        pool_np = htp.shard_pool(full, tp, t, "layer" if layout == "layer_major" else "block")  # rank t's head slice
        ctx, pool = _swap_ctx(layout, M, n_chunks, sb, 4, pool_np)
        h = torch.zeros(n * n_chunks * sb, dtype=torch.uint8).pin_memory()
        ctx.swap_out(dev(vic), None, n, None, h)
        assert ctx.sync(check=False) == 0
        pages.append(h.numpy().reshape(n, n_chunks, sb).copy())
        ctxs.append((ctx, pool, pool_np, h))
    assert (htp.interleave_pages(pages, n, n_chunks) == exp).all()
    for ctx, pool, pool_np, h in ctxs:                                        # restore into wiped pools
        pool.zero_()
        ctx.swap_in(None, h, dev(vic), n)
        assert ctx.sync(check=False) == 0
        cfg = _pool_cfg(layout, M, n_chunks, sb)
        want = oracle.swap_in(np.zeros_like(pool_np), n_chunks, sb, cfg["chunk_stride"], cfg["block_stride"],
                              h.numpy().copy(), vic)
        assert (host(pool, np.uint8) == want).all()
        ctx.close()


def test_out_of_range_block_id_is_reported_and_touches_nothing():
    import torch
    from gpu_util import dev
    M, n_chunks, chunk_bytes = 8, 2, 256
    pool_np = np.arange(M * n_chunks * chunk_bytes, dtype=np.uint32).astype(np.uint8)
    ctx, pool = _swap_ctx("block_major", M, n_chunks, chunk_bytes, 2, pool_np)
    staged = torch.zeros(2 * n_chunks * chunk_bytes, dtype=torch.uint8, device="cuda")
    ctx.gather_pages(dev(np.array([3, 8], np.uint32)), None, 2, staged)
    assert ctx.sync(check=False) == -1
    ctx.close()


def _c3_words(b, c, n_words, n_chunks):
    """Procedural content of chunk c of block b as uint64 words (harness arithmetic: a counter through a mixer)."""
    base = (np.asarray(b, np.uint64).reshape(-1, 1) * np.uint64(n_chunks) + np.uint64(c)) * np.uint64(n_words)
    with np.errstate(over="ignore"):
        w = (base + np.arange(n_words, dtype=np.uint64).reshape(1, -1)) * np.uint64(0xD6E8FEB86659FD93)
        w ^= w >> np.uint64(29)
    return w


def test_swap_config3_shape_llama70b_pages_layer_major_60gib_pool():
    """BASELINE.json configs[3] at its own shape: 160 chunks x 32 KiB = 5 MiB pages scattered over a 60 GiB
    LAYER-MAJOR pool (12,288 blocks); 512 random victims gathered to pinned host and restored into 512 other blocks.
    cw_swap_out / cw_swap_in against cwo_swap_out / cwo_swap_in, every byte of every page; the oracle's 60 GiB pool is
    a lazily mapped zero array in which only the blocks the test touches are filled."""
    import torch
    from gpu_util import dev
    torch.cuda.empty_cache()
    if torch.cuda.mem_get_info()[0] < 70 << 30:
        pytest.skip("needs 70 GiB of free HBM")
    n_chunks, chunk, M, n = 160, 32768, 12288, 512
    page, n_words = n_chunks * chunk, chunk // 8
    cs, bs = M * chunk, chunk
    pool = torch.empty(M * page, dtype=torch.uint8, device="cuda")
    pv = pool.view(torch.int64).view(n_chunks, M, n_words)
    wi = torch.arange(n_words, dtype=torch.int64, device="cuda").unsqueeze(0)
    bi = torch.arange(M, dtype=torch.int64, device="cuda").unsqueeze(1)
    for c in range(n_chunks):                                    # the same words as _c3_words, computed by torch
        w = ((bi * n_chunks + c) * n_words + wi) * (-2960836687051489901)   # 0xD6E8FEB86659FD93 as int64
        w ^= (w >> 29) & ((1 << 35) - 1)
        pv[c] = w
    ctx = __import__("paper_2606_16824_b200").Context(
        num_blocks=M, table_log2_slots=15, max_requests=1, max_hashed_blocks=1, n_chunks=n_chunks, chunk_bytes=chunk,
        chunk_stride=cs, block_stride=bs, pool=pool, staging_bytes=2 * (320 << 20))
    g = gen.rng(35, 0)
    perm = g.permutation(M)
    vic, dst, bystanders = perm[:n].astype(np.uint32), perm[n:2 * n].astype(np.uint32), perm[2 * n:2 * n + 64]
    # the oracle's pool: 60 GiB of lazily mapped zeros, filled only where the test looks
    opool = np.zeros(M * page, np.uint8)
    ov = opool.view(np.uint64).reshape(n_chunks, M, n_words)
    touched = np.concatenate([vic, dst, bystanders.astype(np.uint32)])
    for c in range(n_chunks):
        ov[c, touched] = _c3_words(touched, c, n_words, n_chunks)
    # ---- swap-out
    h = torch.zeros(n * page, dtype=torch.uint8).pin_memory()
    ctx.swap_out(dev(vic), None, n, None, h)
    assert ctx.sync(check=False) == 0
    exp = oracle.swap_out(opool, n_chunks, chunk, cs, bs, vic, np.zeros(n * page, np.uint8))
    assert np.array_equal(h.numpy(), exp), "swap-out bytes (512 x 5 MiB pages)"
    # ---- the device-count form (TMA stores straight to pinned host) at the same shape
    h2 = torch.zeros(64 * page, dtype=torch.uint8).pin_memory()
    ctx.swap_out(dev(vic), dev(np.array([37], np.uint32)), 64, None, h2)
    assert ctx.sync(check=False) == 0
    assert np.array_equal(h2.numpy()[:37 * page], exp[:37 * page]) and not h2.numpy()[37 * page:].any()
    # ---- swap-in into other blocks
    ctx.swap_in(None, h, dev(dst), n)
    assert ctx.sync(check=False) == 0
    oracle.swap_in(opool, n_chunks, chunk, cs, bs, exp, dst)
    look = np.concatenate([dst.astype(np.int64), vic.astype(np.int64), bystanders.astype(np.int64)])
    got = pool.view(n_chunks, M, chunk)[:, torch.from_numpy(look).cuda(), :].cpu().numpy()
    want = opool.reshape(n_chunks, M, chunk)[:, look, :]
    assert np.array_equal(got, want), "pool bytes after swap-in (destinations, sources and bystanders)"
    ctx.close()
    del pool, pv
    torch.cuda.empty_cache()


@pytest.mark.parametrize("with_idle", [False, True])
def test_score_evict_rank_mode_with_unknown_sessions(with_idle):
    """Level 0 of the select uses the RANK of a session's tau (S <= 512).  Blocks whose session id is >= S count as
    tau = TAU_MAX; they must share a level-0 digit with idle sessions (same tau) and with nobody else — also when NO
    real session sits at TAU_MAX.  Large pool (the grid-wide path), deficits that cut inside the unknown group,
    inside the next tau group, and across several."""
    from gpu_util import small_ctx
    g = gen.rng(37, int(with_idle))
    M, S, F = 60000, 40, 8
    ctx = small_ctx(num_blocks=M, table_log2_slots=17, max_sessions=S)
    sess = g.integers(0, S + 6, size=M).astype(np.uint32)              # ~13% of the blocks name a session >= S
    last = g.integers(500, 1000, size=M).astype(np.uint32)
    depth = g.integers(0, 3000, size=M).astype(np.uint32)
    rf = np.full(M, V, np.uint32)
    feats = g.integers(0, 256, size=(S, F), dtype=np.uint8)
    w = g.integers(50, 300, size=F).astype(np.int16)
    state = np.zeros(S, np.uint8)                                       # everybody TOOL_WAIT: every tau < TAU_MAX ...
    if with_idle:
        state[[3, 17]] = 3                                              # ... unless two sessions are idle
    _load_meta(ctx, 0, sess, last, depth, rf)
    n_unknown = int((sess >= S).sum())
    for deficit in (1, n_unknown // 2, n_unknown, n_unknown + 700, n_unknown + 9000, M // 2, M):
        ev, es, est = oracle.score_evict(1000, feats, w, 100, state, None, deficit, sess, last, depth, rf, cap=M)
        gv, gs, gst = _evict(ctx, 1000, feats, w, 100, state, None, deficit, M)
        assert gst == est and gv.tolist() == ev.tolist() and gs.tolist() == es.tolist(), (with_idle, deficit)
    ctx.close()
