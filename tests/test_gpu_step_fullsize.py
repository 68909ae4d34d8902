"""GPU parity at BASELINE.json configs[2] FULL size, in the launch configuration bench.py times
(harness.stress.StressStep: the same object, the same six C-ABI calls, the same grids).

The oracle finishes the whole step in about a second, so nothing is sampled except the KV bytes: every hash
(6.6 M), every overlap length and location, the queue order, admission, and all 52 k victims with their scores are
compared element by element; staged pages are compared on 256 sampled victims against the pool content, and the
pool must be byte-identical after gather + scatter.  The steady-state step (only the 256 newest requests hashed)
must reproduce the same outputs."""
import numpy as np
import pytest

import oracle
from harness import gen

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("shared_match", [True, False])
def test_full_size_step_matches_the_oracle_everywhere(shared_match):
    """shared_match: stage 2a through cw_match_prefix_shared (the bench's step: the queue carries session ids, the
    leader hint is the longest queued request of the session) or through the plain cw_match_prefix."""
    import torch

    from harness import stress
    snap = gen.stress_snapshot(seed=3)
    stream = torch.cuda.Stream()
    st = stress.StressStep(snap, stream, shared_match=shared_match)
    S, L = snap.streams.shape
    with torch.cuda.stream(stream):
        pool_sum = int(st.pool.view(torch.int64).sum().item())
        st.step()
        res = st.results()
        assert st.ctx.sync(check=False) == 0
    # ---- oracle: resident table from its own stream hashes, then the step
    sh, _ = oracle.hash_blocks(snap.streams.reshape(-1), np.arange(S + 1, dtype=np.uint64) * np.uint64(L))
    assert np.array_equal(stress.host(st.d_stream_hashes, np.uint64), sh), "stream hashes"
    table = oracle.Table(snap.table_log2)
    table.insert(sh.reshape(S, L // 16)[:, :snap.resident_blocks].reshape(-1), np.arange(snap.M, dtype=np.uint32))
    o_h, ho = oracle.hash_blocks(snap.tokens, snap.tok_off)
    assert np.array_equal(res["hashes"], o_h), "hashes"
    ek, eg, eloc = table.match_prefix(o_h, ho)
    assert np.array_equal(res["k_total"], ek) and np.array_equal(res["n_gpu"], eg), "overlap lengths"
    assert np.array_equal(ek, np.minimum(snap.shared_tokens // 16, snap.resident_blocks)), "closed form of the recipe"
    assert np.array_equal(res["hit_loc"], eloc), "hit locations"
    eo, ena, ede = oracle.schedule(snap.need_d, eg, snap.arrival_seq, snap.req_id, st.policy, st.free_blocks,
                                   st.evict_budget, st.R)
    assert np.array_equal(res["order"], eo) and (res["num_admit"], res["deficit"]) == (ena, ede), "queue order / admission"
    ev, es, est = oracle.score_evict(snap.tick_now, snap.features, snap.weights, snap.bias, snap.session_state, None,
                                     ede, snap.blk_session, snap.blk_last_access, snap.blk_depth, snap.blk_ref_flags,
                                     cap=st.cap)
    assert est == 0 and res["num_victims"] == ev.size > 50000
    assert np.array_equal(res["victims"], ev) and np.array_equal(res["victim_scores"], es), "victims"
    # ---- stage 4 at full size: sampled staged pages = pool pages of the victims; pool untouched by the round trip
    page = st.page
    with torch.cuda.stream(stream):
        idx = gen.rng(3, 77).choice(ev.size, size=256, replace=False)
        staged = st.d_staged.view(-1, page)[torch.from_numpy(idx).cuda()].cpu().numpy()
        pool_pages = st.pool.view(-1, page)[torch.from_numpy(ev[idx].astype(np.int64)).cuda()].cpu().numpy()
        assert np.array_equal(staged, pool_pages), "staged KV bytes"
        assert int(st.pool.view(torch.int64).sum().item()) == pool_sum, "pool changed by gather + scatter"
        # ---- steady-state step: hashes persist, only the newest requests are re-hashed
        st.d_hashes[int(st.hash_off[st.R - st.new_requests]):].zero_()
        st.step(steady=True)
        res2 = st.results()
    for k in ("hashes", "k_total", "n_gpu", "hit_loc", "order", "victims", "victim_scores"):
        assert np.array_equal(res[k], res2[k]), f"steady step: {k}"
    st.close()


def test_repeated_steps_are_deterministic_and_self_cleaning():
    """300 back-to-back steps (cold / steady alternating, hashes cleared in between) on a 1/16 snapshot must give the
    same outputs every time: the kernels' scratch (tickets, epochs, histograms, barrier words) cleans itself, and
    nothing depends on the order in which CTAs or atomics happen to run."""
    import torch

    from harness import stress
    snap = gen.stress_snapshot(seed=5, S=16)
    stream = torch.cuda.Stream()
    st = stress.StressStep(snap, stream)

    def digest():
        w = torch.arange(1, st.cap + 1, device="cuda")
        return (int(st.d_hashes.sum().item()), int(st.d_k.sum().item()), int(st.d_g.sum().item()),
                int(st.d_loc.to(torch.int64).sum().item()),
                int((st.d_order.to(torch.int64) * torch.arange(1, st.R + 1, device="cuda")).sum().item()),
                int((st.d_vic.to(torch.int64) * w).sum().item()), int(st.d_sc.sum().item()), int(st.d_nv.item()),
                int(st.d_def.item()), int(st.d_na.item()))

    with torch.cuda.stream(stream):
        st.step()
        first = digest()
        assert first[7] > 0
        for i in range(300):
            if i % 3 == 0:
                st.d_hashes.zero_()
            st.step(steady=(i % 3 == 1))
            assert digest() == first, i
    assert st.ctx.sync(check=False) == 0
    st.close()
