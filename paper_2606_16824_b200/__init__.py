"""paper_2606_16824_b200 — thin Python binding of libcachewise.so (include/cachewise.h).

Argument marshalling only: every step of the block-management pass (hash -> match -> schedule ->
score/select -> swap; BASELINE.json north_star) runs in the sm_100a CUDA kernels of
``csrc/``.  PyTorch supplies device memory and streams.  There is no CPU fallback: if the shared library
is missing or cannot be loaded, importing ``lib()`` raises.
"""
from __future__ import annotations

import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
# CACHEWISE_DEBUG=1 selects the -DCW_DEBUG build (phase timestamps, duplicate-victim check; `build.build(debug=True)`)
DEBUG = os.environ.get("CACHEWISE_DEBUG", "0") not in ("", "0")
LIB_PATH = os.path.join(_HERE, "libcachewise_debug.so" if DEBUG else "libcachewise.so")

CW_OK, CW_E_INVAL, CW_E_CAPACITY, CW_E_CUDA, CW_E_STATE = 0, -1, -2, -3, -4
CW_MISS = 0xFFFFFFFF
CW_HOST_BIT = 0x80000000
CW_TAU_MAX = 0x00FFFFFF
CW_REF_VALID = 0x80000000
CW_REF_PINNED = 0x40000000
POLICY_MIN_ADDITIONAL, POLICY_OVERLAP_FIRST, POLICY_FCFS = 0, 1, 2

EXPORTS = ["cw_create", "cw_destroy", "cw_sync", "cw_join_copy", "cw_last_error", "cw_launch_count", "cw_hash_blocks",
           "cw_match_prefix", "cw_schedule", "cw_admit_chunked", "cw_score_evict", "cw_score_evict_begin", "cw_score_evict_end",
           "cw_predict_tau", "cw_swap_out", "cw_swap_in", "cw_gather_pages", "cw_scatter_pages", "cw_table_insert",
           "cw_table_erase", "cw_table_retag", "cw_table_lookup", "cw_table_compact", "cw_table_stats",
           "cw_blocks_update", "cw_hash_blocks_static", "cw_match_prefix_shared"]
DEBUG_EXPORTS = ["cw_debug_evict_times", "cw_debug_stamp", "cw_debug_stamps"]  # libcachewise_debug.so only


class CwConfig(C.Structure):
    _fields_ = [("num_blocks", C.c_uint32), ("host_slots", C.c_uint32), ("table_log2_slots", C.c_uint32),
                ("block_tokens", C.c_uint32), ("n_chunks", C.c_uint32), ("chunk_bytes", C.c_uint64),
                ("chunk_stride", C.c_uint64), ("block_stride", C.c_uint64), ("d_pool", C.c_void_p),
                ("max_requests", C.c_uint32), ("max_sessions", C.c_uint32), ("max_features", C.c_uint32),
                ("max_hashed_blocks", C.c_uint64), ("staging_bytes", C.c_uint64), ("stream_main", C.c_void_p),
                ("stream_copy", C.c_void_p)]


class CwError(RuntimeError):
    def __init__(self, code, where, text=""):
        super().__init__(f"{where}: status {code} {text}".strip())
        self.code = code


_lib = None


def lib():
    """Loads libcachewise.so (built by ``paper_2606_16824_b200.build``).  Fails loudly if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} not built: run `python -m paper_2606_16824_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        P, U32, U64, I32 = C.c_void_p, C.c_uint32, C.c_uint64, C.c_int32
        L.cw_create.argtypes = [C.POINTER(CwConfig), C.POINTER(P)]
        L.cw_destroy.argtypes = [P]
        L.cw_sync.argtypes = [P]
        L.cw_join_copy.argtypes = [P]
        if DEBUG:
            L.cw_debug_evict_times.argtypes = [P, P]
            L.cw_debug_evict_times.restype = I32
            L.cw_debug_stamp.argtypes = [P, U32]
            L.cw_debug_stamp.restype = I32
            L.cw_debug_stamps.argtypes = [P, P]
            L.cw_debug_stamps.restype = I32
        L.cw_last_error.argtypes = [P]
        L.cw_last_error.restype = C.c_char_p
        L.cw_launch_count.argtypes = [P]
        L.cw_launch_count.restype = U64
        L.cw_hash_blocks.argtypes = [P, P, P, P, P, P, P, U32, P]
        L.cw_hash_blocks_static.argtypes = [P, P, P, P, P, P, U32, U64, P, P, P]
        L.cw_match_prefix.argtypes = [P, P, P, U32, P, P, P]
        L.cw_match_prefix_shared.argtypes = [P, P, P, U32, P, P, P, P]
        L.cw_schedule.argtypes = [P, U32, P, P, P, P, U32, U32, U32, U32, P, P, P]
        L.cw_admit_chunked.argtypes = [P, U32, P, P, P, P, U32, U32, U32, U64, P, P, P]
        L.cw_score_evict.argtypes = [P, U32, U32, U32, P, P, I32, P, P, P, U32, P, P, P, U32]
        L.cw_score_evict_begin.argtypes = [P, U32, U32, U32, P, P, I32, P, P, U32, P, P, U32, U32]
        L.cw_score_evict_end.argtypes = [P, P, P]
        L.cw_table_compact.argtypes = [P]
        L.cw_table_stats.argtypes = [P, P]
        L.cw_predict_tau.argtypes = [P, U32, P, P, U32, P, P, P]
        L.cw_swap_out.argtypes = [P, P, P, U32, P, P]
        L.cw_swap_in.argtypes = [P, P, P, P, U32]
        L.cw_gather_pages.argtypes = [P, P, P, U32, P]
        L.cw_scatter_pages.argtypes = [P, P, P, U32, P]
        L.cw_table_insert.argtypes = [P, P, P, U32, P]
        L.cw_table_erase.argtypes = [P, P, U32]
        L.cw_table_retag.argtypes = [P, P, P, U32]
        L.cw_table_lookup.argtypes = [P, P, U32, P]
        L.cw_blocks_update.argtypes = [P, U32, P, U32, P, P, P, P]
        for name in EXPORTS:
            if name not in ("cw_last_error", "cw_launch_count"):
                getattr(L, name).restype = I32
        _lib = L
    return _lib


HASH_STATIC_MAX_REQUESTS = 16384


def hash_blocks_static(tokens, tok_off, hash_off, R, hashes, max_hashed_blocks, start_block=None, start_state=None,
                       salt=None, status=None, stream=None):
    """cw_hash_blocks_static: stage 1 with no ctx and no allocation (fixed static device scratch; at most
    HASH_STATIC_MAX_REQUESTS requests per call; calls that overlap on the GPU race).  `stream` = raw cudaStream_t
    (int) or None for the legacy default stream; asynchronous on it."""
    rc = lib().cw_hash_blocks_static(_ptr(tokens), _ptr(tok_off), _ptr(start_block), _ptr(start_state), _ptr(salt),
                                     _ptr(hash_off), R, max_hashed_blocks, _ptr(hashes), _ptr(status), stream)
    if rc != CW_OK:
        raise CwError(rc, "cw_hash_blocks_static")


def _ptr(x):
    """torch tensor (device or pinned host) / numpy array / int / None -> address."""
    if x is None:
        return None
    if isinstance(x, int):
        return x
    if hasattr(x, "data_ptr"):
        return x.data_ptr()
    return x.ctypes.data


class Context:
    """One cw_ctx.  Methods mirror the C entry points one to one and are asynchronous on ``stream_main``;
    ``sync()`` waits and returns the latched device status (raises on CW_E_CUDA)."""

    def __init__(self, num_blocks, table_log2_slots, max_requests, max_hashed_blocks, max_sessions=1, max_features=16,
                 host_slots=0, n_chunks=0, chunk_bytes=0, chunk_stride=0, block_stride=0, pool=None, staging_bytes=0,
                 stream_main=None, stream_copy=None):
        self._h = None
        cfg = CwConfig(num_blocks, host_slots, table_log2_slots, 16, n_chunks, chunk_bytes, chunk_stride, block_stride,
                       _ptr(pool), max_requests, max_sessions, max_features, max_hashed_blocks, staging_bytes,
                       _stream(stream_main), _stream(stream_copy))
        self.page_bytes = n_chunks * chunk_bytes
        self._pool = pool  # keep alive
        h = C.c_void_p()
        st = lib().cw_create(C.byref(cfg), C.byref(h))
        if st != CW_OK:
            text = lib().cw_last_error(h).decode() if h else ""
            if h:
                lib().cw_destroy(h)
            raise CwError(st, "cw_create", text)
        self._h = h

    def close(self):
        if self._h:
            lib().cw_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _ck(self, st, where):
        if st != CW_OK:
            raise CwError(st, where, lib().cw_last_error(self._h).decode())

    def sync(self, check=True):
        st = lib().cw_sync(self._h)
        if st == CW_E_CUDA or (check and st != CW_OK):
            raise CwError(st, "cw_sync", lib().cw_last_error(self._h).decode())
        return st

    def join_copy(self):
        self._ck(lib().cw_join_copy(self._h), "cw_join_copy")

    def debug_evict_times(self):
        """Phase timestamps (ns) of the last score_evict, relative to its first one (CACHEWISE_DEBUG=1 only)."""
        if not DEBUG:
            raise CwError(CW_E_STATE, "cw_debug_evict_times", "needs the debug library (CACHEWISE_DEBUG=1)")
        buf = (C.c_uint64 * 32)()
        self._ck(lib().cw_debug_evict_times(self._h, buf), "cw_debug_evict_times")
        n = min(int(buf[31]), 31)
        return [int(buf[i]) - int(buf[0]) for i in range(n)]

    def debug_timeline(self, fn_list):
        """Debug build: runs the callables in order with a %globaltimer stamp on stream_main before the first and after
        each; returns (main-stream stamps in ns, absolute stamps of the last evict kernel in ns)."""
        if not DEBUG:
            raise CwError(CW_E_STATE, "debug_timeline", "needs the debug library (CACHEWISE_DEBUG=1)")
        L = lib()
        self._ck(L.cw_debug_stamp(self._h, 0), "cw_debug_stamp")
        for i, f in enumerate(fn_list):
            f()
            self._ck(L.cw_debug_stamp(self._h, i + 1), "cw_debug_stamp")
        buf, ev = (C.c_uint64 * 32)(), (C.c_uint64 * 32)()
        self._ck(L.cw_debug_stamps(self._h, buf), "cw_debug_stamps")
        self._ck(L.cw_debug_evict_times(self._h, ev), "cw_debug_evict_times")
        n = min(int(ev[31]), 31)
        return [int(buf[i]) for i in range(len(fn_list) + 1)], [int(ev[i]) for i in range(n)]

    @property
    def launches(self):
        return int(lib().cw_launch_count(self._h))

    def hash_blocks(self, tokens, tok_off, hash_off, R, hashes, start_block=None, start_state=None, salt=None):
        self._ck(lib().cw_hash_blocks(self._h, _ptr(tokens), _ptr(tok_off), _ptr(start_block), _ptr(start_state),
                                      _ptr(salt), _ptr(hash_off), R, _ptr(hashes)), "cw_hash_blocks")

    def match_prefix(self, hashes, hash_off, R, k_total, n_gpu, hit_loc=None):
        self._ck(lib().cw_match_prefix(self._h, _ptr(hashes), _ptr(hash_off), R, _ptr(k_total), _ptr(n_gpu),
                                       _ptr(hit_loc)), "cw_match_prefix")

    def match_prefix_shared(self, hashes, hash_off, R, leader, k_total, n_gpu, hit_loc=None):
        self._ck(lib().cw_match_prefix_shared(self._h, _ptr(hashes), _ptr(hash_off), R, _ptr(leader), _ptr(k_total),
                                              _ptr(n_gpu), _ptr(hit_loc)), "cw_match_prefix_shared")

    def schedule(self, R, need, n_gpu, arrival_seq, req_id, policy, free_blocks, evictable, max_admit, order,
                 num_admit, deficit):
        self._ck(lib().cw_schedule(self._h, R, _ptr(need), _ptr(n_gpu), _ptr(arrival_seq), _ptr(req_id), policy,
                                   free_blocks, evictable, max_admit, _ptr(order), _ptr(num_admit), _ptr(deficit)),
                 "cw_schedule")

    def admit_chunked(self, R, order, need, n_gpu, new_tokens, free_blocks, evictable, max_admit, token_budget,
                      chunk_tokens, num_admit, deficit):
        self._ck(lib().cw_admit_chunked(self._h, R, _ptr(order), _ptr(need), _ptr(n_gpu), _ptr(new_tokens), free_blocks,
                                        evictable, max_admit, token_budget, _ptr(chunk_tokens), _ptr(num_admit),
                                        _ptr(deficit)), "cw_admit_chunked")

    def score_evict(self, tick_now, S, F, features, weights, bias, session_state, tau_override, deficit, tier, victims,
                    victim_scores, num_victims, cap):
        self._ck(lib().cw_score_evict(self._h, tick_now, S, F, _ptr(features), _ptr(weights), bias,
                                      _ptr(session_state), _ptr(tau_override), _ptr(deficit), tier, _ptr(victims),
                                      _ptr(victim_scores), _ptr(num_victims), cap), "cw_score_evict")

    def score_evict_begin(self, tick_now, S, F, features, weights, bias, session_state, tau_override, tier, victims,
                          victim_scores, cap, n_ctas=0):
        self._ck(lib().cw_score_evict_begin(self._h, tick_now, S, F, _ptr(features), _ptr(weights), bias,
                                            _ptr(session_state), _ptr(tau_override), tier, _ptr(victims),
                                            _ptr(victim_scores), cap, n_ctas), "cw_score_evict_begin")

    def score_evict_end(self, deficit, num_victims):
        self._ck(lib().cw_score_evict_end(self._h, _ptr(deficit), _ptr(num_victims)), "cw_score_evict_end")

    def predict_tau(self, S, cluster, elapsed_ms, C, sample_off, samples, tau_out):
        self._ck(lib().cw_predict_tau(self._h, S, _ptr(cluster), _ptr(elapsed_ms), C, _ptr(sample_off), _ptr(samples),
                                      _ptr(tau_out)), "cw_predict_tau")

    def swap_out(self, victims, num_victims, cap, host_slots, h_dst):
        self._ck(lib().cw_swap_out(self._h, _ptr(victims), _ptr(num_victims), cap, _ptr(host_slots), _ptr(h_dst)),
                 "cw_swap_out")

    def swap_in(self, host_slots, h_src, dst_blocks, n):
        self._ck(lib().cw_swap_in(self._h, _ptr(host_slots), _ptr(h_src), _ptr(dst_blocks), n), "cw_swap_in")

    def gather_pages(self, ids, num, cap, staged):
        self._ck(lib().cw_gather_pages(self._h, _ptr(ids), _ptr(num), cap, _ptr(staged)), "cw_gather_pages")

    def scatter_pages(self, ids, num, cap, staged):
        self._ck(lib().cw_scatter_pages(self._h, _ptr(ids), _ptr(num), cap, _ptr(staged)), "cw_scatter_pages")

    def table_insert(self, keys, loc, n, winner_loc=None):
        self._ck(lib().cw_table_insert(self._h, _ptr(keys), _ptr(loc), n, _ptr(winner_loc)), "cw_table_insert")

    def table_erase(self, keys, n):
        self._ck(lib().cw_table_erase(self._h, _ptr(keys), n), "cw_table_erase")

    def table_retag(self, keys, new_loc, n):
        self._ck(lib().cw_table_retag(self._h, _ptr(keys), _ptr(new_loc), n), "cw_table_retag")

    def table_lookup(self, keys, n, loc):
        self._ck(lib().cw_table_lookup(self._h, _ptr(keys), n, _ptr(loc)), "cw_table_lookup")

    def table_compact(self):
        self._ck(lib().cw_table_compact(self._h), "cw_table_compact")

    def table_stats(self):
        """dict(live, tombstones, slots, probe_max, probe_p50, probe_p99, compactions, probe_sum); synchronises."""
        buf = (C.c_uint64 * 8)()
        self._ck(lib().cw_table_stats(self._h, buf), "cw_table_stats")
        keys = ("live", "tombstones", "slots", "probe_max", "probe_p50", "probe_p99", "compactions", "probe_sum")
        return {k: int(buf[i]) for i, k in enumerate(keys)}

    def blocks_update(self, tier, ids, n, session=None, depth=None, last_access=None, ref_flags=None):
        self._ck(lib().cw_blocks_update(self._h, tier, _ptr(ids), n, _ptr(session), _ptr(depth), _ptr(last_access),
                                        _ptr(ref_flags)), "cw_blocks_update")


def _stream(s):
    if s is None:
        return None
    if isinstance(s, int):
        return s
    return s.cuda_stream  # torch.cuda.Stream
