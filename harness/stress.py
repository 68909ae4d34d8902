"""Config-3 step driver (BASELINE.json configs[2]) on the CUDA path: device state + the six C-ABI calls.

Serves ``bench.py`` and the full-size ``-m gpu`` parity tests so that both run the SAME launch configuration.
Marshalling only: every result comes out of ``paper_2606_16824_b200`` (libcachewise.so).  This module never
imports ``oracle``.
"""
from __future__ import annotations

import numpy as np
import torch

import paper_2606_16824_b200 as cw
from harness import gen

_SIGNED = {np.dtype(np.uint64): np.int64, np.dtype(np.uint32): np.int32, np.dtype(np.uint16): np.int16}


def as_torch(a, dtype=None, pin=False):
    """numpy -> host torch tensor holding the same bytes (unsigned dtypes travel as their signed twins)."""
    a = np.ascontiguousarray(a, dtype=dtype)
    if a.dtype in _SIGNED:
        a = a.view(_SIGNED[a.dtype])
    t = torch.from_numpy(a)
    return t.pin_memory() if pin else t


def dev(a, dtype=None):
    return as_torch(a, dtype).cuda()


def host(t, dtype):
    return t.cpu().numpy().view(dtype)


def session_leaders(req_session, hash_off):
    """The hint cw_match_prefix_shared takes: for every queued request the index of the LONGEST queued request of its
    session (what a scheduler that keeps its queue per session knows; none of the method's arithmetic)."""
    n = (hash_off[1:] - hash_off[:-1]).astype(np.int64)
    order = np.lexsort((np.arange(n.size), -n, req_session))      # per session: longest first, lowest index on ties
    first = np.ones(n.size, bool)
    first[1:] = req_session[order][1:] != req_session[order][:-1]
    lead_of_session = {int(s): int(i) for s, i in zip(req_session[order][first], order[first])}
    return np.array([lead_of_session[int(s)] for s in req_session], np.uint32)


def hash_off_of(tok_off):
    tok_off = np.asarray(tok_off, np.uint64)
    n = (tok_off[1:] - tok_off[:-1]) // np.uint64(16)
    ho = np.zeros(tok_off.size, np.uint64)
    np.cumsum(n, out=ho[1:])
    return ho


# KV page of the step pool: config 3 names no KV shape, and a 2^20-block pool only fits one B200 with a small
# page, so the step uses config 1's page (2 layers x {K,V} x 2 heads x 64 dim x 16 tokens fp16 = 4 x 4 KiB).
STEP_N_CHUNKS = 4
STEP_CHUNK_BYTES = 4096


class StressStep:
    """Device-resident state of one config-3 snapshot and the calls of one block-management step."""

    STAGES = ("hash", "match", "schedule", "score_evict", "gather", "scatter")

    def __init__(self, snap: gen.StressSnapshot, stream: torch.cuda.Stream, with_pool: bool = True,
                 layout: str = "block", n_chunks: int = STEP_N_CHUNKS, chunk_bytes: int = STEP_CHUNK_BYTES,
                 staging_bytes: int = 128 << 20, policy: int = cw.POLICY_MIN_ADDITIONAL, free_blocks: int = 0,
                 holes: bool = False, new_requests: int = 256, spec_ctas: int = 0, stream_copy=None,
                 shared_match: bool = True):
        self.snap, self.stream = snap, stream
        S, L = snap.streams.shape
        self.S, self.L, self.RB, self.M = S, L, snap.resident_blocks, snap.M
        self.R = snap.tok_off.size - 1
        self.F = snap.features.shape[1]
        self.policy, self.free_blocks = policy, free_blocks
        self.spec_ctas = spec_ctas                # CTAs of the speculative selection (0 = library default)
        self.shared_match = shared_match          # stage 2a through cw_match_prefix_shared (leader = longest of the session)
        self.evict_budget = snap.deficit          # "eviction deficit 5% of the pool per step"
        self.cap = max(snap.deficit, 1)
        self.page = n_chunks * chunk_bytes
        self.hash_off = hash_off_of(snap.tok_off)
        self.n_hashed = int(self.hash_off[-1])
        with torch.cuda.stream(stream):
            self.pool = None
            kw = {}
            if with_pool:
                self.pool = torch.empty(self.M * self.page, dtype=torch.uint8, device="cuda")
                # cheap deterministic fill (content is irrelevant to timing; parity tests overwrite it)
                v = self.pool.view(torch.int64)
                torch.arange(v.numel(), dtype=torch.int64, device="cuda", out=v)
                v.mul_(-7046029254386353131)
                if layout == "block":
                    cs, bs = chunk_bytes, self.page
                else:  # layer-major (vLLM-like)
                    cs, bs = self.M * chunk_bytes, chunk_bytes
                kw = dict(n_chunks=n_chunks, chunk_bytes=chunk_bytes, chunk_stride=cs, block_stride=bs, pool=self.pool,
                          staging_bytes=staging_bytes)
            self.chunk_stride, self.block_stride = kw.get("chunk_stride", 0), kw.get("block_stride", 0)
            self.n_chunks, self.chunk_bytes = n_chunks, chunk_bytes
            self.ctx = cw.Context(num_blocks=self.M, table_log2_slots=snap.table_log2, max_requests=max(self.R, S),
                                  max_hashed_blocks=max(self.n_hashed, S * (L // 16), 1), max_sessions=S,
                                  max_features=16, stream_main=stream, stream_copy=stream_copy, **kw)
            c = self.ctx
            # resident set: blocks [0,RB) of every session stream, hashed by the CUDA path itself
            d_stream = dev(np.concatenate([snap.streams.reshape(-1), np.zeros(4, np.int32)]))
            sho = np.arange(S + 1, dtype=np.uint64) * np.uint64(L // 16)
            self.d_stream_hashes = torch.zeros(S * (L // 16), dtype=torch.int64, device="cuda")
            c.hash_blocks(d_stream, dev(gen.stream_tok_off(S, L)), dev(sho), S, self.d_stream_hashes)
            keys = self.d_stream_hashes.view(S, L // 16)[:, :self.RB].contiguous().view(-1)
            loc = torch.arange(self.M, dtype=torch.int32, device="cuda")
            c.table_insert(keys, loc, self.M)
            if holes and snap.hole_ids.size:
                hid = dev(snap.hole_ids.astype(np.int64))
                c.table_erase(keys[hid].contiguous(), int(snap.hole_ids.size))
            c.blocks_update(0, loc, self.M, session=dev(snap.blk_session), depth=dev(snap.blk_depth),
                            last_access=dev(snap.blk_last_access), ref_flags=dev(snap.blk_ref_flags))
            c.sync()
            del d_stream
            # the request queue
            self.d_tok = dev(np.concatenate([snap.tokens, np.zeros(4, np.int32)]))
            self.d_tok_off, self.d_hash_off = dev(snap.tok_off), dev(self.hash_off)
            self.d_need, self.d_arr, self.d_rid = dev(snap.need_d), dev(snap.arrival_seq), dev(snap.req_id)
            self.d_leader = dev(session_leaders(snap.req_session, self.hash_off))
            self.d_feat, self.d_w = dev(snap.features), dev(snap.weights)
            self.d_state = dev(snap.session_state)
            R = self.R
            i32 = dict(dtype=torch.int32, device="cuda")
            self.d_hashes = torch.zeros(max(self.n_hashed, 1), dtype=torch.int64, device="cuda")
            self.d_k, self.d_g = torch.zeros(R, **i32), torch.zeros(R, **i32)
            self.d_loc = torch.zeros(max(self.n_hashed, 1), **i32)
            self.d_order = torch.zeros(R, **i32)
            self.d_na, self.d_def, self.d_nv = torch.zeros(1, **i32), torch.zeros(1, **i32), torch.zeros(1, **i32)
            self.d_vic = torch.zeros(self.cap, **i32)
            self.d_vic_prev = torch.zeros(self.cap, **i32)   # victims whose pages are still on their way back
            self.d_sc = torch.zeros(self.cap, dtype=torch.int64, device="cuda")
            self.d_staged = torch.empty(self.cap * self.page, dtype=torch.uint8, device="cuda") if with_pool else None
            # steady state: hashes persist, only the last `new_requests` requests of the queue are new arrivals
            self.new_requests = min(new_requests, R)
            r0 = R - self.new_requests
            self.d_tok_off_new = self.d_tok_off[r0:]
            self.d_hash_off_new = self.d_hash_off[r0:]
            self.n_hashed_new = int(self.hash_off[-1] - self.hash_off[r0])
            stream.synchronize()

    # ---- one call per stage (each asynchronous on `stream`)
    def hash(self, steady: bool = False):
        if steady:
            self.ctx.hash_blocks(self.d_tok, self.d_tok_off_new, self.d_hash_off_new, self.new_requests, self.d_hashes)
        else:
            self.ctx.hash_blocks(self.d_tok, self.d_tok_off, self.d_hash_off, self.R, self.d_hashes)

    def match(self):
        if self.shared_match:
            self.ctx.match_prefix_shared(self.d_hashes, self.d_hash_off, self.R, self.d_leader, self.d_k, self.d_g,
                                         self.d_loc)
        else:
            self.ctx.match_prefix(self.d_hashes, self.d_hash_off, self.R, self.d_k, self.d_g, self.d_loc)

    def schedule(self):
        self.ctx.schedule(self.R, self.d_need, self.d_g, self.d_arr, self.d_rid, self.policy, self.free_blocks,
                          self.evict_budget, self.R, self.d_order, self.d_na, self.d_def)

    def score_evict(self):
        s = self.snap
        self.ctx.score_evict(s.tick_now, self.S, self.F, self.d_feat, self.d_w, s.bias, self.d_state, None,
                             self.d_def, 0, self.d_vic, self.d_sc, self.d_nv, self.cap)

    def gather(self):
        self.ctx.gather_pages(self.d_vic, self.d_nv, self.cap, self.d_staged)

    def scatter(self):
        self.ctx.scatter_pages(self.d_vic, self.d_nv, self.cap, self.d_staged)

    def score_evict_begin(self):
        s = self.snap
        self.ctx.score_evict_begin(s.tick_now, self.S, self.F, self.d_feat, self.d_w, s.bias, self.d_state, None, 0,
                                   self.d_vic, self.d_sc, self.cap, self.spec_ctas)

    def score_evict_end(self):
        self.ctx.score_evict_end(self.d_def, self.d_nv)

    def decide(self, steady: bool = False, overlap: bool = True):
        """Stages 1-3 (the <=100 us target of BASELINE.json).  overlap: the selection of the eviction budget runs on
        the ctx's side stream beside hash -> match -> schedule (cw_score_evict_begin / _end); otherwise the four
        calls run in series."""
        # the fork comes first in both kinds of step: the round-2 hash kernel (4 + 1 warps, 3 CTAs per SM) no longer
        # loses more to the selection's 37 SMs than the match gains from the earlier start (cold: 211-215 us against
        # 215-221 us with the fork after the hash; with the round-1 hash kernel it was the other way round)
        if overlap:
            self.score_evict_begin()
        self.hash(steady)
        self.match()
        self.schedule()
        if overlap:
            self.score_evict_end()
        else:
            self.score_evict()

    def step(self, steady: bool = False):
        """One pass of the whole hot path with everything resident in HBM (device halves of stage 4)."""
        self.decide(steady)
        if self.pool is not None:
            self.gather()
            self.scatter()

    def stage_fns(self, steady: bool = False):
        fns = [lambda: self.hash(steady), self.match, self.schedule, self.score_evict]
        if self.pool is not None:
            fns += [self.gather, self.scatter]
        return fns

    # ---- algorithmic bytes per launch (per-unit figure x units of one launch)
    def algorithmic_bytes(self, n_victims: int, steady: bool = False):
        nh = self.n_hashed_new if steady else self.n_hashed
        return {
            "hash": 72 * nh,                                   # 64 B tokens read + 8 B hash written per block
            "match": 28 * self.n_hashed,                       # 8 B hash + 16 B slot read + 4 B hit_loc written
            "schedule": 16 * self.R + 4 * self.R,              # d, n_gpu, arrival, req_id read + order written
            "score_evict": 16 * self.M + 12 * n_victims,       # 4 x u32 metadata per block + victim id/score
            "gather": 2 * self.page * n_victims,               # read + write of every victim page
            "scatter": 2 * self.page * n_victims,
        }

    def results(self):
        self.stream.synchronize()
        n = int(host(self.d_nv, np.uint32)[0])
        return dict(hashes=host(self.d_hashes, np.uint64)[:self.n_hashed], k_total=host(self.d_k, np.uint32),
                    n_gpu=host(self.d_g, np.uint32), hit_loc=host(self.d_loc, np.uint32)[:self.n_hashed],
                    order=host(self.d_order, np.uint32), num_admit=int(host(self.d_na, np.uint32)[0]),
                    deficit=int(host(self.d_def, np.uint32)[0]), num_victims=n,
                    victims=host(self.d_vic, np.uint32)[:n], victim_scores=host(self.d_sc, np.uint64)[:n])

    def close(self):
        self.ctx.close()
        self.pool = self.d_staged = None
