"""GPU parity — round-2 additions to the boundary, all through the C ABI and against the oracle:

* table robustness: insert/erase churn of fresh keys (tombstone reclamation + compaction), a completely full table
  (absent keys answer MISS, the winners of an overflowing insert are the oracle's), the 2^32-hash limit;
* cw_score_evict_begin / cw_score_evict_end (speculative selection beside the rest of the step) = cw_score_evict;
* cw_swap_out with a device-side victim count moves exactly n pages;
* debug build: duplicate victims are rejected.
"""
import os
import subprocess
import sys

import numpy as np
import pytest

import oracle
from harness import gen

pytestmark = pytest.mark.gpu
MISS, HOST = 0xFFFFFFFF, 0x80000000
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


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


def _match(ctx, h, hoff):
    from gpu_util import dev, host, zeros
    R = hoff.size - 1
    k, g, loc = zeros(R, np.uint32), zeros(R, np.uint32), zeros(h.size, np.uint32)
    ctx.match_prefix(dev(h), dev(hoff), R, k, g, loc)
    st = ctx.sync(check=False)
    return host(k, np.uint32)[:R], host(g, np.uint32)[:R], host(loc, np.uint32)[:h.size], st


def test_table_churn_of_fresh_keys_reclaims_tombstones():
    """36% live load, 24 N fresh-key insert/erase rounds.  Without reclamation every EMPTY slot
    ends up a tombstone and miss probes walk the whole table; with it the table keeps answering like the oracle's
    map, tombstones stay bounded and probes stay short."""
    from gpu_util import dev, small_ctx
    log2, N = 12, 4096
    ctx = small_ctx(num_blocks=N // 2, table_log2_slots=log2)
    ot = oracle.Table(log2)
    g = gen.rng(41, 0)
    live = np.zeros(0, np.uint64)
    next_key = 1000
    target = int(0.36 * N)
    for rnd in range(96):                                   # 96 rounds x N/4 fresh keys = 24 N inserts
        fresh = (np.arange(N // 4, dtype=np.uint64) + np.uint64(next_key)) * np.uint64(0x9E3779B97F4A7C15)
        next_key += N // 4
        room = target - live.size
        if room < fresh.size:                               # erase the oldest keys to make room
            kill, live = live[:fresh.size - room], live[fresh.size - room:]
            ctx.table_erase(dev(kill), kill.size)
            ot.erase(kill)
        locs = g.integers(0, 1 << 20, size=fresh.size, dtype=np.uint32)
        win, st = _insert(ctx, fresh, locs)
        ewin, est = ot.insert(fresh, locs)
        assert st == est == 0 and (win == ewin).all(), rnd
        live = np.concatenate([live, fresh])
        if rnd % 8 == 7:
            probe = np.concatenate([live[::3], fresh + np.uint64(12345)])   # residents and absent keys
            assert (_lookup(ctx, probe) == ot.lookup(probe)).all(), rnd
            s = ctx.table_stats()
            assert s["live"] == len(ot) == live.size
            assert s["live"] + s["tombstones"] <= 0.36 * N + N // 4 + N // 4 + 1, s   # bounded by the compaction rule
            assert s["probe_p99"] <= 128, s
    s = ctx.table_stats()
    assert s["compactions"] >= 10, s
    # a leading-run match over residents followed by absent keys, after all that churn
    h = np.concatenate([live[:500], live[:3] + np.uint64(1)])
    hoff = np.array([0, h.size], np.uint64)
    ek, eg, eloc = ot.match_prefix(h, hoff)
    k, gg, loc, st = _match(ctx, h, hoff)
    assert st == 0 and (k == ek).all() and (gg == eg).all() and (loc == eloc).all()
    ctx.table_compact()
    s2 = ctx.table_stats()
    assert s2["tombstones"] == 0 and s2["live"] == live.size and s2["compactions"] == s["compactions"] + 1
    assert (_lookup(ctx, live) == ot.lookup(live)).all()
    ctx.close()


def test_full_table_answers_miss_and_overflow_winners_are_the_oracles():
    from gpu_util import dev, small_ctx
    ctx = small_ctx(num_blocks=8, table_log2_slots=4)
    ot = oracle.Table(4)
    win, st = _insert(ctx, [5, 9, 7, 1, 3], [50, 90, 70, 10, 30])
    ewin, est = ot.insert([5, 9, 7, 1, 3], [50, 90, 70, 10, 30])
    assert st == est == 0 and (win == ewin).all()
    # 16 slots, 5 live: the FIRST 11 new keys by input index fit (duplicates and present keys take no slot)
    keys = np.concatenate([np.arange(1000, 1008), [9, 1003], np.arange(1008, 1020)]).astype(np.uint64)
    locs = np.arange(keys.size, dtype=np.uint32) + 200
    win, st = _insert(ctx, keys, locs)
    ewin, est = ot.insert(keys, locs)
    assert st == est == -2 and (win == ewin).all() and (win == MISS).sum() == 9
    assert (_lookup(ctx, keys) == ot.lookup(keys)).all()
    s = ctx.table_stats()
    assert s["live"] == s["slots"] == 16 and s["tombstones"] == 0
    # every slot is occupied: absent keys must come back MISS (bounded probe), present ones still resolve
    q = np.array([5, 4242, 1000, 77777, 1010, 1019, 31337], np.uint64)
    assert (_lookup(ctx, q) == ot.lookup(q)).all()
    for h in (np.array([5, 1000, 4242, 9], np.uint64), np.arange(4000, 4200, dtype=np.uint64),
              np.concatenate([keys[:8], np.arange(5000, 5300, dtype=np.uint64)])):
        hoff = np.array([0, 2, h.size], np.uint64)
        ek, eg, eloc = ot.match_prefix(h, hoff)
        k, g, loc, st = _match(ctx, h, hoff)
        assert st == 0 and (k == ek).all() and (g == eg).all() and (loc == eloc).all()
    # erase -> tombstones only (no EMPTY slot anywhere): absent keys still terminate; insert reuses a tombstone
    ctx.table_erase(dev(np.array([1001, 1002], np.uint64)), 2)
    ot.erase([1001, 1002])
    assert (_lookup(ctx, q) == ot.lookup(q)).all()
    win, st = _insert(ctx, [4242, 4243, 4244], [1, 2, 3])
    ewin, est = ot.insert([4242, 4243, 4244], [1, 2, 3])
    assert st == est == -2 and (win == ewin).all()
    ctx.close()


def test_match_rejects_more_than_2_pow_32_hashes_and_leaves_outputs_untouched():
    from gpu_util import dev, host, small_ctx
    ctx = small_ctx()
    hoff = np.array([0, (1 << 32) + 5], np.uint64)           # never dereferenced: the call is rejected on the device
    k, g = dev(np.array([123], np.uint32)), dev(np.array([456], np.uint32))
    loc = dev(np.full(8, 789, np.uint32))
    ctx.match_prefix(dev(np.zeros(8, np.uint64)), dev(hoff), 1, k, g, loc)
    assert ctx.sync(check=False) == -1
    assert host(k, np.uint32)[0] == 123 and host(g, np.uint32)[0] == 456 and (host(loc, np.uint32) == 789).all()
    # the scratch is still armed: a normal call afterwards is correct
    win, st = _insert(ctx, [11, 12], [1, 2])
    kk, gg, ll, st = _match(ctx, np.array([11, 12, 13], np.uint64), np.array([0, 3], np.uint64))
    assert st == 0 and kk.tolist() == [2] and ll.tolist() == [1, 2, MISS]
    ctx.close()


# ---------------------------------------------------------------------------------------------- speculative evict
def _load_meta(ctx, tier, sess, last, depth, rf):
    from gpu_util import dev
    M = len(sess)
    ctx.blocks_update(tier, dev(np.arange(M, dtype=np.uint32)), M, session=dev(sess, np.uint32),
                      depth=dev(depth, np.uint32), last_access=dev(last, np.uint32), ref_flags=dev(rf, np.uint32))


@pytest.mark.parametrize("n_ctas", [0, 1, 3])
def test_speculative_evict_equals_serial_evict_and_the_oracle(n_ctas):
    """victims for any deficit are a prefix of the budget's sorted victims.  begin/end must give
    exactly cw_score_evict's outputs (victims, scores, count, CW_E_CAPACITY) for deficit in {0, 1, budget/3,
    budget, > evictable}, with other work queued on stream_main in between, and again when captured in a graph."""
    import torch
    from gpu_util import dev, host, small_ctx, zeros
    snap = gen.stress_snapshot(seed=8, S=32, L=32768, RB=2048, req_per_session=2, len_median=4096, len_min=64,
                               len_max=32768)
    M, S, F = snap.M, 32, snap.features.shape[1]
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        ctx = small_ctx(num_blocks=M, table_log2_slots=snap.table_log2, max_sessions=S, stream_main=stream)
        args = (snap.blk_session, snap.blk_last_access, snap.blk_depth, snap.blk_ref_flags)
        _load_meta(ctx, 0, *args)
        n_ev = int((snap.blk_ref_flags == gen.REF_VALID).sum())
        budget = snap.deficit
        d_f, d_w, d_s = dev(snap.features), dev(snap.weights), dev(snap.session_state)
        filler = torch.zeros(1 << 20, dtype=torch.int32, device="cuda")
        for cap, deficits in ((budget, [0, 1, budget // 3, budget, budget + 7]), (M, [n_ev - 1, n_ev, n_ev + 9])):
            vic, sc, nv = zeros(cap, np.uint32), zeros(cap, np.uint64), zeros(1, np.uint32)
            d_def = zeros(1, np.uint32)

            def spec():
                ctx.score_evict_begin(snap.tick_now, S, F, d_f, d_w, snap.bias, d_s, None, 0, vic, sc, cap, n_ctas)
                filler.add_(1)                      # stands for hash -> match -> schedule on stream_main
                ctx.score_evict_end(d_def, nv)

            g = torch.cuda.CUDAGraph()
            d_def.fill_(1)
            spec()
            ctx.sync(check=False)
            with torch.cuda.graph(g, stream=stream):
                spec()
            for deficit in deficits:
                ev, es, est = oracle.score_evict(snap.tick_now, snap.features, snap.weights, snap.bias,
                                                 snap.session_state, None, deficit, *args, cap=cap)
                for mode in ("eager", "graph"):
                    d_def.fill_(int(np.int32(np.uint32(deficit))))
                    nv.fill_(-1)
                    if mode == "eager":
                        spec()
                    else:
                        g.replay()
                    st = ctx.sync(check=False)
                    n = int(host(nv, np.uint32)[0])
                    assert st == est and n == ev.size, (cap, deficit, mode, st, est, n, ev.size)
                    assert host(vic, np.uint32)[:n].tolist() == ev.tolist(), (cap, deficit, mode)
                    assert host(sc, np.uint64)[:n].tolist() == es.tolist(), (cap, deficit, mode)
        # misuse: end without begin, begin twice, serial call while a speculative one is open
        import paper_2606_16824_b200 as cw
        with pytest.raises(cw.CwError) as e:
            ctx.score_evict_end(d_def, nv)
        assert e.value.code == cw.CW_E_STATE
        ctx.score_evict_begin(snap.tick_now, S, F, d_f, d_w, snap.bias, d_s, None, 0, vic, sc, cap, n_ctas)
        for bad in (lambda: ctx.score_evict_begin(snap.tick_now, S, F, d_f, d_w, snap.bias, d_s, None, 0, vic, sc, cap),
                    lambda: ctx.score_evict(snap.tick_now, S, F, d_f, d_w, snap.bias, d_s, None, d_def, 0, vic, sc, nv,
                                            cap)):
            with pytest.raises(cw.CwError) as e:
                bad()
            assert e.value.code == cw.CW_E_STATE
        ctx.score_evict_end(d_def, nv)
        ctx.sync(check=False)
        ctx.close()


# ---------------------------------------------------------------------------------------------- swap-out, device count
@pytest.mark.parametrize("layout", ["block", "layer"])
def test_swap_out_with_a_device_count_moves_exactly_n_pages(layout):
    import torch
    import paper_2606_16824_b200 as cw
    from gpu_util import dev, small_ctx
    M, n_chunks, chunk = 96, 6, 4096 + 16
    page = n_chunks * chunk
    cs, bs = (chunk, page) if layout == "block" else (M * chunk, chunk)
    pool_np = gen.page_bytes(np.arange(M, dtype=np.uint64) + 77, page).reshape(M, n_chunks, chunk)
    if layout == "layer":
        pool_np = pool_np.transpose(1, 0, 2)
    pool_np = np.ascontiguousarray(pool_np).reshape(-1)
    pool = torch.from_numpy(pool_np.copy()).cuda()
    ctx = small_ctx(num_blocks=M, n_chunks=n_chunks, chunk_bytes=chunk, chunk_stride=cs, block_stride=bs, pool=pool,
                    staging_bytes=2 * 4 * page)
    cap = 40
    vic = gen.rng(44, 0).permutation(M)[:cap].astype(np.uint32)
    h_dst = torch.full((cap * page,), 0xAB, dtype=torch.uint8).pin_memory()
    for n in (0, 1, 17, cap, cap + 5):
        h_dst.fill_(0xAB)
        ctx.swap_out(dev(vic), dev(np.array([n], np.uint32)), cap, None, h_dst)
        assert ctx.sync(check=False) == 0
        m = min(n, cap)
        want = oracle.swap_out(pool_np, n_chunks, chunk, cs, bs, vic[:m], np.full(cap * page, 0xAB, np.uint8))
        assert np.array_equal(h_dst.numpy(), want), (layout, n)          # pages >= n keep the guard pattern
    # a slot list with a device count is refused (it would overwrite live host-tier pages), so is pageable memory
    slots = np.arange(cap, dtype=np.uint32)
    assert cw.lib().cw_swap_out(ctx._h, dev(vic).data_ptr(), dev(np.array([3], np.uint32)).data_ptr(), cap,
                                slots.ctypes.data, h_dst.data_ptr()) == cw.CW_E_INVAL
    pageable = np.zeros(cap * page, np.uint8)
    assert cw.lib().cw_swap_out(ctx._h, dev(vic).data_ptr(), dev(np.array([3], np.uint32)).data_ptr(), cap, None,
                                pageable.ctypes.data) == cw.CW_E_INVAL
    # the host-count form still goes through the staging ring and the copy engine
    h_dst.fill_(0xAB)
    ctx.swap_out(dev(vic), None, 23, slots[::-1][:23].copy(), h_dst)
    assert ctx.sync(check=False) == 0
    want = oracle.swap_out(pool_np, n_chunks, chunk, cs, bs, vic[:23], np.full(cap * page, 0xAB, np.uint8),
                           slots=slots[::-1][:23].copy())
    assert np.array_equal(h_dst.numpy(), want)
    ctx.close()


# ---------------------------------------------------------------------------------------------- debug build
_DEBUG_PROG = r"""
import os, sys
sys.path.insert(0, {root!r}); sys.path.insert(0, os.path.join({root!r}, "tests"))
import numpy as np, torch
import paper_2606_16824_b200 as cw
from gpu_util import dev, small_ctx
assert cw.DEBUG and cw.LIB_PATH.endswith("libcachewise_debug.so")
M, page = 32, 4096
pool = torch.zeros(M * page, dtype=torch.uint8, device="cuda")
ctx = small_ctx(num_blocks=M, n_chunks=1, chunk_bytes=page, chunk_stride=page, block_stride=page, pool=pool,
                staging_bytes=2 * 8 * page)
staged = torch.zeros(8 * page, dtype=torch.uint8, device="cuda")
ctx.gather_pages(dev(np.array([3, 9, 4, 30], np.uint32)), None, 4, staged)
assert ctx.sync(check=False) == 0
ctx.gather_pages(dev(np.array([3, 9, 4, 9], np.uint32)), None, 4, staged)      # block 9 twice
assert ctx.sync(check=False) == cw.CW_E_INVAL
ctx.gather_pages(dev(np.array([9, 3], np.uint32)), None, 2, staged)            # the bitmap was cleared again
assert ctx.sync(check=False) == 0
h = torch.zeros(8 * page, dtype=torch.uint8).pin_memory()
ctx.swap_out(dev(np.array([1, 2, 1], np.uint32)), None, 3, None, h)
assert ctx.sync(check=False) == cw.CW_E_INVAL
ctx.close()
print("debug ok")
"""


def test_debug_build_rejects_duplicate_victims(tmp_path):
    """SURVEY.md 8c stage 4: duplicates in `victims` -> CW_E_INVAL in debug builds (libcachewise_debug.so, -DCW_DEBUG)."""
    from paper_2606_16824_b200 import build
    build.build(debug=True)
    script = tmp_path / "dbg.py"
    script.write_text(_DEBUG_PROG.format(root=ROOT))
    out = subprocess.run([sys.executable, str(script)], env=dict(os.environ, CACHEWISE_DEBUG="1"), capture_output=True,
                         text=True, timeout=600)
    assert out.returncode == 0 and "debug ok" in out.stdout, out.stdout + out.stderr


# ---------------------------------------------------------------------------------------------- NEXT-3: chunked prefill
@pytest.mark.parametrize("R", [1, 2, 33, 1025, 5000])
def test_admit_chunked_matches_the_oracle(R):
    """PAPER.md L271 (chunked prefill, 512 tokens per chunk) as an admission budget: cw_schedule -> cw_admit_chunked
    against cwo_schedule -> cwo_admit_chunked, every output, budgets from 0 to unlimited, both block regimes."""
    from gpu_util import dev, host, small_ctx, zeros
    g = gen.rng(78, R)
    ctx = small_ctx(max_requests=max(R, 8))
    need = g.integers(1, 3000, size=R).astype(np.uint32)
    n_gpu = np.minimum(need, g.integers(0, 3000, size=R)).astype(np.uint32)
    n_gpu[::7] = need[::7]                                                  # full hits: nothing to prefill
    new_tok = ((need - n_gpu).astype(np.int64) * 16 - g.integers(0, 16, size=R)).clip(0).astype(np.uint32)
    arr, rid = g.permutation(R).astype(np.uint64), np.arange(R, dtype=np.uint32)
    d_need, d_g, d_t = dev(need), dev(n_gpu), dev(new_tok)
    d_order, d_na, d_de = zeros(R, np.uint32), zeros(1, np.uint32), zeros(1, np.uint32)
    d_chunk = zeros(R, np.uint32)
    for policy in (0, 1, 2):
        for free, evictable in ((0, 50_000), (1_000, 4_000_000_000), (7, 0)):
            ctx.schedule(R, d_need, d_g, dev(arr), dev(rid), policy, free, evictable, R, d_order, d_na, d_de)
            eorder, _, _ = oracle.schedule(need, n_gpu, arr, rid, policy, free, evictable, R)
            for budget in (0, 1, 512, 8192, (1 << 32) + 5, (1 << 63)):
                for max_admit in (1, 8, R):
                    d_chunk.fill_(-1)
                    ctx.admit_chunked(R, d_order, d_need, d_g, d_t, free, evictable, max_admit, budget, d_chunk, d_na,
                                      d_de)
                    assert ctx.sync(check=False) == 0
                    ech, ena, ede = oracle.admit_chunked(eorder, need, n_gpu, new_tok, free, evictable, max_admit, budget)
                    assert host(d_order, np.uint32)[:R].tolist() == eorder.tolist()
                    assert host(d_chunk, np.uint32)[:R].tolist() == ech.tolist(), (policy, free, budget, max_admit)
                    assert (int(host(d_na, np.uint32)[0]), int(host(d_de, np.uint32)[0])) == (ena, ede)
    # a corrupt order is reported, not followed
    bad = np.arange(R, dtype=np.uint32)
    bad[0] = R + 3
    ctx.admit_chunked(R, dev(bad), d_need, d_g, d_t, 0, 10, R, 512, d_chunk, d_na, d_de)
    assert ctx.sync(check=False) == -1
    ctx.close()
