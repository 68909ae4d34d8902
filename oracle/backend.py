"""ORACLE — test infrastructure, not the product.

Replay backend over the CPU oracle (``oracle/cw_oracle.cpp``): the same interface as
``harness.replay.GpuBackend`` so that the shared host-driven replay driver (R6) can run either.
Only ``tests/``, ``bench.py``'s CPU legs and ``__graft_entry__.smoke()`` import this module.
"""
from __future__ import annotations

import numpy as np

import oracle
from harness import gen


class OracleBackend:
    def __init__(self, cfg, S: int, F: int):
        self.cfg = cfg
        M, HS = cfg.num_blocks, cfg.host_slots
        self.cs, self.bs = cfg.strides()
        self.table = oracle.Table(max(4, int(np.ceil(np.log2(2 * (M + HS))))))
        self.meta = [dict(session=np.zeros(n, np.uint32), depth=np.zeros(n, np.uint32),
                          last_access=np.zeros(n, np.uint32), ref_flags=np.zeros(n, np.uint32))
                     for n in (M, max(HS, 1))]
        self.pool = self.tier = None
        if cfg.store_bytes:
            self.pool = np.zeros(M * cfg.page, np.uint8)
            self.tier = np.zeros(max(HS, 1) * cfg.page, np.uint8)

    def hash_blocks(self, tokens, tok_off, sb, ss, hashes):
        h, _ = oracle.hash_blocks(tokens, tok_off, start_block=sb, start_state=ss, hashes=hashes.copy())
        return h

    def match(self, allh, hoff):
        R = hoff.size - 1
        if R == 0 or allh.size == 0:
            return np.zeros(R, np.uint32), np.zeros(R, np.uint32), np.zeros(0, np.uint32)
        return self.table.match_prefix(allh, hoff)

    def schedule(self, need, n_gpu, arr, rid, policy, free, evictable, max_admit):
        return oracle.schedule(need, n_gpu, arr, rid, policy, free, evictable, max_admit)

    def admit_chunked(self, order, need, n_gpu, new_tokens, free, evictable, max_admit, token_budget):
        return oracle.admit_chunked(order, need, n_gpu, new_tokens, free, evictable, max_admit, token_budget)

    def blocks_update(self, tier, ids, session=None, depth=None, last_access=None, ref_flags=None):
        m = self.meta[tier]
        for name, v in (("session", session), ("depth", depth), ("last_access", last_access), ("ref_flags", ref_flags)):
            if v is not None:
                m[name][ids] = v

    def score_evict(self, tick, features, weights, bias, state, tau_ov, deficit, tier, cap):
        m = self.meta[tier]
        n = self.cfg.num_blocks if tier == 0 else self.cfg.host_slots
        return oracle.score_evict(tick, features, weights, bias, state, tau_ov, deficit, m["session"][:n],
                                  m["last_access"][:n], m["depth"][:n], m["ref_flags"][:n], cap=cap)

    def table_insert(self, keys, locs):
        win, _ = self.table.insert(keys, locs)
        return win

    def table_erase(self, keys):
        self.table.erase(keys)

    def table_retag(self, keys, locs):
        self.table.retag(keys, locs)

    def swap_out(self, victims, slots, want_bytes, tags):
        if self.pool is None:
            return np.zeros(0, np.uint8)
        c = self.cfg
        oracle.swap_out(self.pool, c.n_chunks, c.chunk_bytes, self.cs, self.bs, victims, self.tier, slots=slots)
        if want_bytes:
            return self.tier.reshape(-1, c.page)[slots.astype(np.int64)].reshape(-1).copy()
        return np.zeros(0, np.uint8)

    def predict_tau(self, cluster, elapsed_ms, sample_off, samples):
        return oracle.predict_tau(cluster, elapsed_ms, sample_off, samples)[0]

    def swap_in(self, slots, dst):
        if self.pool is None:
            return
        c = self.cfg
        oracle.swap_in(self.pool, c.n_chunks, c.chunk_bytes, self.cs, self.bs, self.tier, dst, slots=slots)

    def write_pages(self, ids, tags):
        if self.pool is None:
            return
        c = self.cfg
        content = gen.page_bytes(tags, c.page).reshape(-1)
        oracle.swap_in(self.pool, c.n_chunks, c.chunk_bytes, self.cs, self.bs, content, ids)

    def read_pool(self):
        return self.pool

    def close(self):
        pass
