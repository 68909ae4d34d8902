"""Host-driven replay of a seeded synthetic session trace (R6, SURVEY.md 8c "Replay").

The DRIVER below is backend-agnostic harness code: virtual time, queue, free lists, reference counts, logging.
Every decision of the block-management pass comes from the backend it is given:

  * ``GpuBackend`` (this file)        -> ``paper_2606_16824_b200`` (libcachewise.so), the product path
  * ``oracle.backend.OracleBackend``  -> the CPU oracle (imported by tests / bench only; never from here)

Both are driven by the same trace and their per-step logs are compared element by element (hashes, overlap
lengths, queue order, admission, victims + scores, staged KV bytes, eviction / drop / swap-in counts).
The driver holds none of the method's arithmetic: it never hashes, probes, sorts, scores or copies pages.

  python -m harness.replay --config 0|1|4 [--scale K]      run the GPU backend and print the totals
"""
from __future__ import annotations

import heapq
from dataclasses import dataclass, field

import numpy as np

from harness import gen

MISS = 0xFFFFFFFF
HOST_BIT = 0x80000000
REF_VALID = 0x80000000


@dataclass
class ReplayConfig:
    name: str
    num_blocks: int                 # M: HBM pool capacity in blocks
    host_slots: int                 # host-tier capacity in blocks
    n_chunks: int
    chunk_bytes: int
    layout: str = "block"           # "block" (page contiguous) or "layer" (vLLM-like, chunk-major)
    policy: int = 0                 # cw_schedule policy
    max_admit: int = 2
    use_hint: bool = False          # CacheWise* (PAPER.md L285): tau_override = true gap
    evict_policy: str = "cachewise"  # "cachewise" (per-session linear predictor), "hint" (= use_hint), "lru" (vLLM,
                                     # L281: every tau equal), "infercept" (L283: session moving average of tool time),
                                     # "cluster" (the paper's predictor, L219-227: cw_predict_tau over per-cluster history)
    c0_ms: int = 20                 # integer service model: c0 + ceil(c_tok*new_tokens/1000) + c_blk*swapped_in
    c_tok_us: int = 250
    c_blk_ms: int = 1
    token_budget: int = 0           # chunked prefill (512 tokens per chunk): new tokens an engine
                                    # iteration may prefill; admission goes through cw_admit_chunked; 0 = unlimited
    offload: str = "swap"           # service cost of a host-tier hit: "swap" = PCIe swap-in (c_blk_ms per
                                    # block), "auto" = the cheaper of swap-in and recomputing those 16 tokens per block
    store_bytes: bool = True        # log the staged bytes of every swap-out (tiny configs only)
    max_steps: int = 1_000_000

    @property
    def page(self):
        return self.n_chunks * self.chunk_bytes

    def strides(self):
        if self.layout == "block":
            return self.chunk_bytes, self.page                       # chunk_stride, block_stride
        return self.num_blocks * self.chunk_bytes, self.chunk_bytes


@dataclass
class Request:
    session: int
    turn: int
    tokens: np.ndarray
    arrival_seq: int
    req_id: int
    hashes: np.ndarray = None       # u64[n_full]
    need: int = 0                   # d_r = ceil(len/16)


@dataclass
class StepLog:
    step: int
    now_ms: int
    queued: list
    new_hashes: np.ndarray
    k_total: np.ndarray
    n_gpu: np.ndarray
    order: np.ndarray
    num_admit: int
    deficit: int
    admitted: list
    victims: np.ndarray
    victim_scores: np.ndarray
    host_drops: np.ndarray
    staged: np.ndarray
    swapped_in: int
    chunk: np.ndarray = None        # cw_admit_chunked: tokens each queued request may prefill this iteration


@dataclass
class ReplayResult:
    steps: list = field(default_factory=list)
    evictions: int = 0
    drops: int = 0
    swap_ins: int = 0
    hit_blocks: int = 0
    new_blocks: int = 0
    completed: int = 0
    end_ms: int = 0
    session_done_ms: dict = field(default_factory=dict)
    page_bytes: int = 0
    swap_outs: int = 0              # pages that physically crossed PCIe device -> host
    prefill_iterations: int = 0     # engine iterations spent on prefill chunks (token_budget > 0)
    new_tokens: int = 0             # tokens prefilled (token goodput numerator)

    def totals(self):
        return dict(steps=len(self.steps), evictions=self.evictions, drops=self.drops, swap_ins=self.swap_ins,
                    hit_blocks=self.hit_blocks, new_blocks=self.new_blocks, completed=self.completed,
                    end_ms=self.end_ms)

    def metrics(self):
        """The paper's session-level metrics (PAPER.md 6.1 L287, 6.4 L337) in the replay's virtual time."""
        done = list(self.session_done_ms.values())
        return dict(
            transfer_volume_bytes=self.evictions * self.page_bytes,          # L337: eviction count x KV block size
            pcie_bytes=(self.swap_outs + self.swap_ins) * self.page_bytes,   # what the offload tier really moved (L345)
            mean_session_ms=int(np.mean(done)) if done else 0,               # L287 (3): request latencies, no tool time
            token_goodput_per_s=round(self.new_tokens * 1000.0 / max(self.end_ms, 1), 1),     # L287 (1)
            requests_per_s=round(self.completed * 1000.0 / max(self.end_ms, 1), 3),
            prefill_iterations=self.prefill_iterations)


def tail_tag(session: int, turn: int) -> int:
    """Content tag of a request's private partial tail block (never hashed, never shared)."""
    return (0x7A11 << 48) | (session << 20) | turn


def lcp_blocks(a: np.ndarray, b: np.ndarray) -> int:
    """Full 16-token blocks shared by two token arrays (queue bookkeeping: which blocks need hashing at all)."""
    n = min(a.size, b.size)
    if n == 0:
        return 0
    neq = np.nonzero(a[:n] != b[:n])[0]
    first = int(neq[0]) if neq.size else n
    return first // 16


def run(trace: gen.Trace, cfg: ReplayConfig, be) -> ReplayResult:
    """Replays `trace` against backend `be`.  Deterministic given the backend's answers."""
    S, F, M, HS = len(trace.sessions), trace.F, cfg.num_blocks, cfg.host_slots
    res = ReplayResult(page_bytes=cfg.page)
    free_hbm = list(range(M))
    free_host = list(range(HS))
    heapq.heapify(free_hbm)
    heapq.heapify(free_host)
    b_hash = np.zeros(M, np.uint64)
    b_sess, b_depth, b_last = np.zeros(M, np.uint32), np.zeros(M, np.uint32), np.zeros(M, np.uint32)
    b_ref = np.zeros(M, np.int64)
    b_valid = np.zeros(M, bool)
    h_hash = np.zeros(max(HS, 1), np.uint64)
    h_sess, h_depth, h_last = (np.zeros(max(HS, 1), np.uint32) for _ in range(3))
    h_valid, h_pin = np.zeros(max(HS, 1), bool), np.zeros(max(HS, 1), np.int64)
    turn_idx = np.zeros(S, np.int64)
    state = np.full(S, gen.TOOL_WAIT, np.uint8)
    next_arrival = np.arange(S, dtype=np.int64) * 5          # first prompts arrive 5 ms apart
    waiting = np.ones(S, bool)                               # has a turn that has not been enqueued yet
    features = np.zeros((S, F), np.uint8)
    prev_tokens = [np.zeros(0, np.int32) for _ in range(S)]
    prev_hashes = [np.zeros(0, np.uint64) for _ in range(S)]
    queue: list[Request] = []
    now, tick, seq, rid = 0, 1, 0, 0
    gap_avg = np.zeros(S, np.int64)      # InferCept baseline: what the session's tool calls took so far
    last_done = np.zeros(S, np.int64)
    sess_cluster = np.zeros(S, np.uint32)  # cluster of the tool call each session is waiting on

    def flags(ids):
        return (np.where(b_valid[ids], REF_VALID, 0) | b_ref[ids]).astype(np.uint32)

    def hflags(ids):
        return (np.where(h_valid[ids], REF_VALID, 0) | h_pin[ids]).astype(np.uint32)

    for step in range(cfg.max_steps):
        # ---- 1. arrivals
        arr = [s for s in np.nonzero(waiting & (next_arrival <= now))[0]]
        if not queue and not arr:
            if not waiting.any():
                break
            now = int(next_arrival[waiting].min())
            continue
        arr.sort(key=lambda s: (int(next_arrival[s]), int(s)))
        new_reqs = []
        for s in arr:
            t = trace.sessions[s][turn_idx[s]]
            q = Request(int(s), int(turn_idx[s]), t.tokens, seq, rid, need=(t.tokens.size + 15) // 16)
            seq += 1
            rid += 1
            waiting[s] = False
            state[s] = gen.QUEUED
            queue.append(q)
            new_reqs.append(q)
        # ---- 2. hash the new requests from the first block that differs from the session's previous turn
        new_hashes = np.zeros(0, np.uint64)
        if new_reqs:
            tok_off = np.zeros(len(new_reqs) + 1, np.uint64)
            sb = np.zeros(len(new_reqs), np.uint32)
            ss = np.zeros(len(new_reqs), np.uint64)
            parts = []
            for i, q in enumerate(new_reqs):
                tok_off[i + 1] = tok_off[i] + np.uint64(q.tokens.size)
                k = min(lcp_blocks(q.tokens, prev_tokens[q.session]), prev_hashes[q.session].size)
                q.hashes = np.zeros(q.tokens.size // 16, np.uint64)
                q.hashes[:k] = prev_hashes[q.session][:k]
                sb[i] = k
                ss[i] = q.hashes[k - 1] if k else 0
                parts.append(q.hashes)
            hashes = np.concatenate(parts) if parts else np.zeros(0, np.uint64)
            hashes = be.hash_blocks(np.concatenate([q.tokens for q in new_reqs]), tok_off, sb, ss, hashes)
            o = 0
            for q in new_reqs:
                q.hashes = hashes[o:o + q.hashes.size].copy()
                o += q.hashes.size
            new_hashes = hashes
        # ---- 3. match every queued request
        R = len(queue)
        hoff = np.zeros(R + 1, np.uint64)
        for i, q in enumerate(queue):
            hoff[i + 1] = hoff[i] + np.uint64(q.hashes.size)
        allh = np.concatenate([q.hashes for q in queue]) if R else np.zeros(0, np.uint64)
        k_total, n_gpu, hit_loc = be.match(allh, hoff)
        # ---- 4. schedule
        need = np.array([q.need for q in queue], np.uint32)
        evictable = int(np.count_nonzero(b_valid & (b_ref == 0)))
        order, num_admit, deficit = be.schedule(need, n_gpu, np.array([q.arrival_seq for q in queue], np.uint64),
                                                np.array([q.req_id for q in queue], np.uint32), cfg.policy,
                                                len(free_hbm), evictable, cfg.max_admit)
        chunk = None
        if cfg.token_budget:   # chunked prefill: the iteration's token budget bounds the admitted prefix (L271)
            new_tok = np.array([q.tokens.size - 16 * int(k_total[i]) for i, q in enumerate(queue)], np.uint32)
            chunk, num_admit, deficit = be.admit_chunked(order, need, n_gpu, new_tok, len(free_hbm), evictable,
                                                         cfg.max_admit, cfg.token_budget)
        # ---- 5. pin + touch the hits of the admitted requests (a request whose own hits use up the evictable
        #         blocks it was counting on stays queued)
        admitted, need_sum, pinned = [], 0, 0
        touch_ids, touch_slots = [], []
        for p in range(num_admit):
            qi = int(order[p])
            q = queue[qi]
            if q.need > M:
                continue
            locs = hit_loc[int(hoff[qi]):int(hoff[qi]) + int(k_total[qi])]
            hbm = locs[(locs & HOST_BIT) == 0].astype(np.int64)
            host = (locs[(locs & HOST_BIT) != 0] & ~np.uint32(HOST_BIT)).astype(np.int64)
            newly = int(np.count_nonzero(b_ref[hbm] == 0))
            a = q.need - int(n_gpu[qi])
            if need_sum + a > len(free_hbm) + evictable - pinned - newly:
                break
            b_ref[hbm] += 1
            b_last[hbm] = tick
            h_pin[host] += 1
            pinned += newly
            need_sum += a
            touch_ids.append(hbm)
            touch_slots.append(host)
            admitted.append((qi, q, locs, hbm, host))
            state[q.session] = gen.RUNNING
        if touch_ids and sum(x.size for x in touch_ids):
            ids = np.unique(np.concatenate(touch_ids)).astype(np.uint32)
            be.blocks_update(0, ids, last_access=b_last[ids], ref_flags=flags(ids))
        if touch_slots and sum(x.size for x in touch_slots):
            sl = np.unique(np.concatenate(touch_slots)).astype(np.uint32)
            be.blocks_update(1, sl, ref_flags=hflags(sl))
        # ---- 6. evict the shortfall, swap the victims out to the host tier (drop host entries if it is full)
        victims, vscores = np.zeros(0, np.uint32), np.zeros(0, np.uint64)
        host_drops, staged = np.zeros(0, np.uint32), np.zeros(0, np.uint8)
        short = max(0, need_sum - len(free_hbm))
        if short:
            tau_ov = None
            if cfg.use_hint or cfg.evict_policy == "hint":
                tau_ov = np.clip(next_arrival - now, 0, 0xFFFFFF).astype(np.uint32)
            elif cfg.evict_policy == "lru":
                tau_ov = np.full(S, 1000, np.uint32)
            elif cfg.evict_policy == "cluster":     # E[remaining | still running] from the cluster's history
                tau_ov = be.predict_tau(sess_cluster, np.clip(now - last_done, 0, 0xFFFFFFFF).astype(np.uint32),
                                        trace.meta["sample_off"], trace.meta["samples"])
            elif cfg.evict_policy == "infercept":   # moving average of the session's past gaps minus the elapsed time
                tau_ov = np.clip(gap_avg - (now - last_done), 0, 0xFFFFFF).astype(np.uint32)
            victims, vscores, st = be.score_evict(tick, features, trace.weights, trace.bias, state, tau_ov, short, 0,
                                                  short)
            assert victims.size == short, (victims.size, short, st)
            n_sw = min(short, HS)
            lack = n_sw - len(free_host)
            if lack > 0:
                host_drops, _, _ = be.score_evict(tick, features, trace.weights, trace.bias, state, tau_ov, lack, 1,
                                                  lack)
                if host_drops.size:
                    be.table_erase(h_hash[host_drops])
                    h_valid[host_drops] = False
                    be.blocks_update(1, host_drops, ref_flags=hflags(host_drops))
                    for sl in host_drops:
                        heapq.heappush(free_host, int(sl))
                    res.drops += int(host_drops.size)
                n_sw = min(n_sw, len(free_host))
            vs, vd = victims[:n_sw], victims[n_sw:]
            if vs.size:
                slots = np.array([heapq.heappop(free_host) for _ in range(vs.size)], np.uint32)
                staged = be.swap_out(vs, slots, cfg.store_bytes, b_hash[vs])
                res.swap_outs += int(vs.size)
                be.table_retag(b_hash[vs], slots | np.uint32(HOST_BIT))
                h_hash[slots], h_sess[slots], h_depth[slots], h_last[slots] = b_hash[vs], b_sess[vs], b_depth[vs], b_last[vs]
                h_valid[slots] = True
                h_pin[slots] = 0
                be.blocks_update(1, slots, session=h_sess[slots], depth=h_depth[slots], last_access=h_last[slots],
                                 ref_flags=hflags(slots))
            if vd.size:  # no room left in the host tier: these are dropped (recomputed later)
                be.table_erase(b_hash[vd])
                res.drops += int(vd.size)
            b_valid[victims] = False
            be.blocks_update(0, victims, ref_flags=flags(victims))
            for b in victims:
                heapq.heappush(free_hbm, int(b))
            res.evictions += int(victims.size)
        # ---- 7. swap the host-tier hits of the admitted requests back in; 8. allocate + "prefill" the misses
        swapped_in = 0
        svc_max = 0
        done_reqs = []
        for qi, q, locs, hbm, host in admitted:
            s = q.session
            shared = list(hbm)                     # shared (table-resident) blocks this request holds a ref on
            private = []
            if host.size:
                dst = np.array([heapq.heappop(free_hbm) for _ in range(host.size)], np.uint32)
                be.swap_in(host.astype(np.uint32), dst)
                pos = np.nonzero((locs & HOST_BIT) != 0)[0]          # depth of every host hit inside the run
                be.table_retag(q.hashes[pos], dst)
                b_hash[dst], b_sess[dst], b_depth[dst] = q.hashes[pos], h_sess[host], h_depth[host]
                b_last[dst], b_ref[dst], b_valid[dst] = tick, 1, True
                be.blocks_update(0, dst, session=b_sess[dst], depth=b_depth[dst], last_access=b_last[dst],
                                 ref_flags=flags(dst))
                h_valid[host], h_pin[host] = False, 0
                be.blocks_update(1, host.astype(np.uint32), ref_flags=hflags(host))
                for sl in host:
                    heapq.heappush(free_host, int(sl))
                shared += [int(b) for b in dst]
                swapped_in += int(host.size)
            k = int(k_total[qi])
            n_full = q.hashes.size
            n_new = q.need - k
            if n_new:
                ids = np.array([heapq.heappop(free_hbm) for _ in range(n_new)], np.uint32)
                tags = np.empty(n_new, np.uint64)
                tags[:n_full - k] = q.hashes[k:]
                if q.need > n_full:
                    tags[-1] = tail_tag(s, q.turn)
                be.write_pages(ids, tags)
                full_ids = ids[:n_full - k]
                if full_ids.size:
                    win = be.table_insert(q.hashes[k:], full_ids)
                    mine = win == full_ids
                    own = full_ids[mine]
                    depth = np.arange(k, n_full, dtype=np.uint32)[mine]
                    b_hash[own], b_sess[own], b_depth[own] = q.hashes[k:][mine], s, depth
                    b_last[own], b_ref[own], b_valid[own] = tick, 1, True
                    if own.size:
                        be.blocks_update(0, own, session=b_sess[own], depth=b_depth[own], last_access=b_last[own],
                                         ref_flags=flags(own))
                    shared += [int(b) for b in own]
                    private += [int(b) for b in full_ids[~mine]]     # the key was already resident elsewhere
                private += [int(b) for b in ids[n_full - k:]]        # partial tail block
                res.new_blocks += n_new
            res.hit_blocks += k
            new_tokens = q.tokens.size - 16 * k
            res.new_tokens += new_tokens
            # chunked prefill: the request occupies ceil(new_tokens / budget) engine iterations of c0 each
            iters = max(1, -(-new_tokens // cfg.token_budget)) if cfg.token_budget else 1
            res.prefill_iterations += iters
            swap_ms = cfg.c_blk_ms * int(host.size)
            if cfg.offload == "auto":   # L345: PCIe swap-in vs recomputing the same blocks, whichever is cheaper
                swap_ms = min(swap_ms, (cfg.c_tok_us * 16 * int(host.size) + 999) // 1000)
            svc = cfg.c0_ms * iters + (cfg.c_tok_us * new_tokens + 999) // 1000 + swap_ms
            svc_max = max(svc_max, svc)
            done_reqs.append((q, shared, private))
        res.swap_ins += swapped_in
        # a request that can never fit (needs more blocks than the pool has) is rejected so that time moves on
        rejected = None
        if not admitted and queue:
            rejected = queue[int(order[0])]
            done_reqs.append((rejected, [], []))
        # ---- 9. service + completion
        now += max(1, svc_max)
        gone = set()
        for q, shared, private in done_reqs:
            s = q.session
            if shared:
                ids = np.array(shared, np.int64)
                b_ref[ids] -= 1
                idu = np.unique(ids).astype(np.uint32)
                be.blocks_update(0, idu, ref_flags=flags(idu))
            for b in private:
                heapq.heappush(free_hbm, b)
            t = trace.sessions[s][q.turn]
            features[s] = t.features
            prev_tokens[s], prev_hashes[s] = q.tokens, q.hashes
            turn_idx[s] += 1
            res.completed += 1
            res.session_done_ms[s] = res.session_done_ms.get(s, 0) + (now - int(next_arrival[s]))
            if turn_idx[s] < len(trace.sessions[s]):
                state[s] = gen.TOOL_WAIT
                next_arrival[s] = now + t.gap_ms
                last_done[s] = now
                sess_cluster[s] = t.cluster
                if q.turn > 0:  # the previous gap is known by now: exponential moving average (alpha = 1/2)
                    prev_gap = trace.sessions[s][q.turn - 1].gap_ms
                    gap_avg[s] = prev_gap if q.turn == 1 else (gap_avg[s] + prev_gap) // 2
                waiting[s] = True
            else:
                state[s] = gen.IDLE
                next_arrival[s] = np.iinfo(np.int64).max // 2
            gone.add(q.req_id)
        res.steps.append(StepLog(step, now, [q.req_id for q in queue], new_hashes, k_total, n_gpu, order, num_admit,
                                 deficit, [q.req_id for q, _, _ in done_reqs], victims, vscores, host_drops, staged,
                                 swapped_in, chunk if chunk is not None else np.zeros(0, np.uint32)))
        queue = [q for q in queue if q.req_id not in gone]
        tick += 1
    res.end_ms = now
    return res


SYSTEMS = {  # the paper's comparison systems as (schedule policy, eviction policy) pairs — PAPER.md L281-285
    "vLLM (FCFS + LRU)": (2, "lru"),
    "InferCept (FCFS + moving average)": (2, "infercept"),
    "vLLM (prefix-aware)": (0, "lru"),
    "CacheWise (prefix-aware + predictor)": (0, "cachewise"),
    "CacheWise (prefix-aware + cluster predictor)": (0, "cluster"),
    "CacheWise* (prefix-aware + true tau)": (0, "hint"),
}


def policy_sweep(trace: gen.Trace, base: ReplayConfig, make_backend):
    """Runs the same trace under every system of SYSTEMS; returns {name: totals + mean session time}."""
    import dataclasses
    out = {}
    for name, (sched, ev) in SYSTEMS.items():
        if ev == "cluster" and "samples" not in trace.meta:
            continue
        cfg = dataclasses.replace(base, policy=sched, evict_policy=ev, use_hint=False)
        r = run(trace, cfg, make_backend(cfg))
        t = r.totals()
        t.update(r.metrics())
        out[name] = t
    return out


def compare(a: ReplayResult, b: ReplayResult):
    """Element-by-element comparison of two replays; returns a list of differences (empty = identical)."""
    diffs = []
    if a.totals() != b.totals():
        diffs.append(("totals", a.totals(), b.totals()))
    if a.metrics() != b.metrics():
        diffs.append(("metrics", a.metrics(), b.metrics()))
    for x, y in zip(a.steps, b.steps):
        for f in ("now_ms", "queued", "num_admit", "deficit", "admitted", "swapped_in"):
            if getattr(x, f) != getattr(y, f):
                diffs.append((x.step, f, getattr(x, f), getattr(y, f)))
        for f in ("new_hashes", "k_total", "n_gpu", "order", "victims", "victim_scores", "host_drops", "staged", "chunk"):
            u, v = getattr(x, f), getattr(y, f)
            if u.shape != v.shape or not np.array_equal(u, v):
                diffs.append((x.step, f, u.shape, v.shape))
        if len(diffs) > 20:
            break
    return diffs


# --------------------------------------------------------------------------------------------------
# The product backend: every call goes through libcachewise.so (no oracle import here, no CPU fallback)
# --------------------------------------------------------------------------------------------------
class GpuBackend:
    def __init__(self, cfg: ReplayConfig, S: int, F: int, max_requests: int = 4096, max_hashed: int = 1 << 22,
                 verify_pages: int = 0):
        import torch

        import paper_2606_16824_b200 as cw
        from harness import stress
        self.torch, self.cw, self.st, self.cfg = torch, cw, stress, cfg
        self.verify_pages, self.pages_verified = verify_pages, 0
        self.stream = torch.cuda.Stream()
        cs, bs = cfg.strides()
        M, HS, page = cfg.num_blocks, cfg.host_slots, cfg.page
        with torch.cuda.stream(self.stream):
            self.pool = torch.zeros(M * page, dtype=torch.uint8, device="cuda")
            self.tier = torch.zeros(max(HS, 1) * page, dtype=torch.uint8).pin_memory()
            log2 = max(4, int(np.ceil(np.log2(2 * (M + HS)))))
            self.ctx = cw.Context(num_blocks=M, host_slots=HS, table_log2_slots=log2, max_requests=max_requests,
                                  max_hashed_blocks=max_hashed, max_sessions=max(S, 1), max_features=16,
                                  n_chunks=cfg.n_chunks, chunk_bytes=cfg.chunk_bytes, chunk_stride=cs, block_stride=bs,
                                  pool=self.pool, staging_bytes=2 * max(page, min(64 * page, 256 << 20)),
                                  stream_main=self.stream)
        self.stream.synchronize()

    def _dev(self, a, dt=None):
        return self.st.dev(a, dt)

    def hash_blocks(self, tokens, tok_off, sb, ss, hashes):
        with self.torch.cuda.stream(self.stream):
            ho = self.st.hash_off_of(tok_off)
            d_h = self._dev(np.concatenate([hashes, np.zeros(1, np.uint64)]))
            self.ctx.hash_blocks(self._dev(np.concatenate([tokens, np.zeros(4, np.int32)])), self._dev(tok_off),
                                 self._dev(ho), tok_off.size - 1, d_h, start_block=self._dev(sb), start_state=self._dev(ss))
            self.ctx.sync()
            return self.st.host(d_h, np.uint64)[:hashes.size].copy()

    def match(self, allh, hoff):
        R = hoff.size - 1
        if R == 0 or allh.size == 0:
            return np.zeros(R, np.uint32), np.zeros(R, np.uint32), np.zeros(0, np.uint32)
        t = self.torch
        with t.cuda.stream(self.stream):
            d_k, d_g = t.zeros(R, dtype=t.int32, device="cuda"), t.zeros(R, dtype=t.int32, device="cuda")
            d_loc = t.zeros(allh.size, dtype=t.int32, device="cuda")
            self.ctx.match_prefix(self._dev(allh), self._dev(hoff), R, d_k, d_g, d_loc)
            self.ctx.sync()
            return self.st.host(d_k, np.uint32), self.st.host(d_g, np.uint32), self.st.host(d_loc, np.uint32)

    def schedule(self, need, n_gpu, arr, rid, policy, free, evictable, max_admit):
        t, R = self.torch, need.size
        with t.cuda.stream(self.stream):
            d_o = t.zeros(max(R, 1), dtype=t.int32, device="cuda")
            d_s = t.zeros(2, dtype=t.int32, device="cuda")
            self.ctx.schedule(R, self._dev(need), self._dev(n_gpu), self._dev(arr), self._dev(rid), policy, free,
                              evictable, max_admit, d_o, d_s[0:1], d_s[1:2])
            self.ctx.sync()
            sc = self.st.host(d_s, np.uint32)
            return self.st.host(d_o, np.uint32)[:R], int(sc[0]), int(sc[1])

    def admit_chunked(self, order, need, n_gpu, new_tokens, free, evictable, max_admit, token_budget):
        t, R = self.torch, need.size
        with t.cuda.stream(self.stream):
            d_c = t.zeros(max(R, 1), dtype=t.int32, device="cuda")
            d_s = t.zeros(2, dtype=t.int32, device="cuda")
            self.ctx.admit_chunked(R, self._dev(order, np.uint32), self._dev(need), self._dev(n_gpu),
                                   self._dev(new_tokens, np.uint32), free, evictable, max_admit, token_budget, d_c,
                                   d_s[0:1], d_s[1:2])
            self.ctx.sync()
            sc = self.st.host(d_s, np.uint32)
            return self.st.host(d_c, np.uint32)[:R].copy(), int(sc[0]), int(sc[1])

    def blocks_update(self, tier, ids, session=None, depth=None, last_access=None, ref_flags=None):
        if ids.size == 0:
            return
        f = lambda x: None if x is None else self._dev(x, np.uint32)
        with self.torch.cuda.stream(self.stream):
            self.ctx.blocks_update(tier, self._dev(ids, np.uint32), ids.size, session=f(session), depth=f(depth),
                                   last_access=f(last_access), ref_flags=f(ref_flags))
            self.ctx.sync()

    def score_evict(self, tick, features, weights, bias, state, tau_ov, deficit, tier, cap):
        t = self.torch
        S, F = features.shape
        with t.cuda.stream(self.stream):
            d_v = t.zeros(max(cap, 1), dtype=t.int32, device="cuda")
            d_s = t.zeros(max(cap, 1), dtype=t.int64, device="cuda")
            d_n = t.zeros(1, dtype=t.int32, device="cuda")
            self.ctx.score_evict(tick, S, F, self._dev(features), self._dev(weights), int(bias), self._dev(state),
                                 None if tau_ov is None else self._dev(tau_ov), self._dev(np.array([deficit], np.uint32)),
                                 tier, d_v, d_s, d_n, cap)
            st = self.ctx.sync(check=False)
            n = int(self.st.host(d_n, np.uint32)[0])
            return self.st.host(d_v, np.uint32)[:n].copy(), self.st.host(d_s, np.uint64)[:n].copy(), st

    def table_insert(self, keys, locs):
        with self.torch.cuda.stream(self.stream):
            d_w = self.torch.zeros(keys.size, dtype=self.torch.int32, device="cuda")
            self.ctx.table_insert(self._dev(keys, np.uint64), self._dev(locs, np.uint32), keys.size, d_w)
            self.ctx.sync()
            return self.st.host(d_w, np.uint32)

    def table_erase(self, keys):
        with self.torch.cuda.stream(self.stream):
            self.ctx.table_erase(self._dev(keys, np.uint64), keys.size)
            self.ctx.sync()

    def table_retag(self, keys, locs):
        with self.torch.cuda.stream(self.stream):
            self.ctx.table_retag(self._dev(keys, np.uint64), self._dev(locs, np.uint32), keys.size)
            self.ctx.sync()

    def swap_out(self, victims, slots, want_bytes, tags):
        page = self.cfg.page
        with self.torch.cuda.stream(self.stream):
            self.ctx.swap_out(self._dev(victims, np.uint32), None, victims.size, np.ascontiguousarray(slots, np.uint32),
                              self.tier)
            self.ctx.sync()
        tier = self.tier.numpy().reshape(-1, page)
        for j in list(range(victims.size))[:self.verify_pages] + list(range(victims.size))[-self.verify_pages:]:
            if self.verify_pages:  # KV bytes of sampled victims = the procedural content of their block
                assert np.array_equal(tier[int(slots[j])], gen.page_bytes(tags[j:j + 1], page)[0]), "swap-out bytes"
                self.pages_verified += 1
        if want_bytes:
            return tier[slots.astype(np.int64)].reshape(-1).copy()
        return np.zeros(0, np.uint8)

    def predict_tau(self, cluster, elapsed_ms, sample_off, samples):
        t = self.torch
        with t.cuda.stream(self.stream):
            d_out = t.zeros(cluster.size, dtype=t.int32, device="cuda")
            self.ctx.predict_tau(cluster.size, self._dev(cluster, np.uint32), self._dev(elapsed_ms, np.uint32),
                                 sample_off.size - 1, self._dev(sample_off, np.uint64), self._dev(samples, np.uint32), d_out)
            self.ctx.sync()
            return self.st.host(d_out, np.uint32)

    def swap_in(self, slots, dst):
        with self.torch.cuda.stream(self.stream):
            self.ctx.swap_in(np.ascontiguousarray(slots, np.uint32), self.tier, self._dev(dst, np.uint32), dst.size)
            self.ctx.sync()

    def write_pages(self, ids, tags):
        """"Prefill": procedural page content g(tag, offset) (same function as gen.page_bytes, evaluated on the
        device), placed with the library's own scatter kernel."""
        t, page = self.torch, self.cfg.page
        step = max(1, (256 << 20) // page)
        with t.cuda.stream(self.stream):
            off = t.arange(page // 8, dtype=t.int64, device="cuda").unsqueeze(0) * (-7046029254386353131)  # 0x9E37..15
            for i in range(0, ids.size, step):
                tg = self._dev(tags[i:i + step], np.uint64).unsqueeze(1)
                w = (tg + off) * (-2960836687051489901)                                                 # 0xD6E8..93
                w ^= (w >> 29) & ((1 << 35) - 1)
                self.ctx.scatter_pages(self._dev(ids[i:i + step], np.uint32), None, tg.shape[0], w.contiguous())
            self.ctx.sync()

    def read_pool(self):
        self.stream.synchronize()
        return self.pool.cpu().numpy()

    def close(self):
        self.ctx.close()
        self.pool = self.tier = None


# --------------------------------------------------------------------------------------------------
# Full-size configurations (BASELINE.json configs[0], [1], [4]) scaled to the box by rule
# --------------------------------------------------------------------------------------------------
def full_config(which: int, hbm_budget_gib: float = 120.0, host_budget_gib: float = 48.0, scale: int = 1):
    """Returns (trace, cfg, note).  Pools are sized by the config's rule, then capped by the memory budgets
    (page count shrinks, page size never does); the applied scale is stated in `note`."""
    if which == 0:
        return gen.tiny_trace(0), ReplayConfig("configs[0]", 256, 64, 4, 4096, max_admit=2), "as specified"
    if which == 1:
        tr = gen.llama8b_trace(1, n_sessions=64 // scale, n_turns=40)
        n_chunks, chunk = 64, 32768
        frac, max_admit = 0.6, 8
    elif which == 4:
        tr = gen.long_agent_trace(5, n_sessions=512 // scale, n_turns=200 // scale, cap=200_000)
        n_chunks, chunk = 56, 16384
        frac, max_admit = None, 16
    else:
        raise ValueError("replay configs are 0, 1 and 4")
    page = n_chunks * chunk
    ws = sum(max((t.tokens.size + 15) // 16 for t in s) for s in tr.sessions)
    want_m = int(frac * ws) if frac else int(120e9 // page)
    want_h = ws if which == 1 else int(512e9 // page)
    m = min(want_m, int(hbm_budget_gib * 2**30 // page))
    h = min(want_h, int(host_budget_gib * 2**30 // page))
    note = (f"working set {ws} blocks; pool {m} of {want_m} blocks ({m * page / 2**30:.1f} GiB), host tier {h} of {want_h} "
            f"slots ({h * page / 2**30:.1f} GiB); sessions/turns scale 1/{scale}")
    cfg = ReplayConfig(f"configs[{which}]", m, h, n_chunks, chunk, layout="layer" if which == 1 else "block",
                       max_admit=max_admit, store_bytes=False)
    return tr, cfg, note


def main():
    import argparse
    import json
    import time
    ap = argparse.ArgumentParser(description="host-driven replay on the CUDA path")
    ap.add_argument("--config", type=int, default=0, choices=[0, 1, 4])
    ap.add_argument("--scale", type=int, default=1, help="divide the number of sessions (and turns of config 4)")
    ap.add_argument("--hbm-gib", type=float, default=120.0)
    ap.add_argument("--host-gib", type=float, default=48.0)
    ap.add_argument("--sweep", action="store_true", help="run the paper's comparison systems on a synthetic trace")
    a = ap.parse_args()
    if a.sweep:
        tr = gen.cluster_trace(31, 48, 24)   # tool gaps drawn from 20 per-cluster distributions (Table 3 shaped)
        ws = sum(max((t.tokens.size + 15) // 16 for t in s) for s in tr.sessions)
        base = ReplayConfig("sweep", int(0.3 * ws), 0, 4, 4096, max_admit=8, store_bytes=False)
        print(json.dumps(policy_sweep(tr, base, lambda c: GpuBackend(c, 48, 8)), indent=1))
        return
    tr, cfg, note = full_config(a.config, a.hbm_gib, a.host_gib, a.scale)
    be = GpuBackend(cfg, len(tr.sessions), tr.F, verify_pages=1)
    t0 = time.time()
    r = run(tr, cfg, be)
    out = dict(config=cfg.name, note=note, wall_s=round(time.time() - t0, 1), pages_verified=be.pages_verified,
               kernel_launches=be.ctx.launches, **r.totals())
    be.close()
    print(json.dumps(out))


if __name__ == "__main__":
    main()
