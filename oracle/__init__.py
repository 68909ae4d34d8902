"""ORACLE — test infrastructure, not the product.

ctypes binding of ``oracle/cw_oracle.cpp`` (plain single-threaded C++17, host pointers only).  Only
``tests/``, ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs and ``__graft_entry__.smoke()``
may import this package; ``paper_2606_16824_b200`` never does.  Every wrapper takes and returns numpy
arrays; the arithmetic lives in the C++ file, each function citing the PAPER.md passage it follows.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "cw_oracle.cpp")
_LIB = os.path.join(_HERE, "libcw_oracle.so")

MISS = 0xFFFFFFFF
HOST_BIT = 0x80000000
TAU_MAX = (1 << 24) - 1
REF_VALID = 0x80000000
REF_PINNED = 0x40000000


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (no CUDA).  Building the checker is not using it."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".{os.getpid()}.tmp"
        subprocess.check_call(["g++", "-std=c++17", "-O2", "-fPIC", "-shared", "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.cwo_fin.restype = C.c_uint64
        _lib.cwo_fin.argtypes = [C.c_uint64]
        _lib.cwo_block_digest.restype = C.c_uint64
        _lib.cwo_block_digest.argtypes = [C.c_void_p]
        _lib.cwo_block_score.restype = C.c_uint64
        _lib.cwo_block_score.argtypes = [C.c_uint32] * 4
        _lib.cwo_table_create.restype = C.c_void_p
        _lib.cwo_table_create.argtypes = [C.c_uint32]
        _lib.cwo_table_destroy.argtypes = [C.c_void_p]
        _lib.cwo_table_size.restype = C.c_uint64
        _lib.cwo_table_size.argtypes = [C.c_void_p]
    return _lib


def _p(a):
    return None if a is None else C.c_void_p(a.ctypes.data)


def _arr(a, dtype):
    if a is None:
        return None
    return np.ascontiguousarray(a, dtype=dtype)


def fin(x: int) -> int:
    return int(lib().cwo_fin(C.c_uint64(x & 0xFFFFFFFFFFFFFFFF)))


def block_digest(tok16) -> int:
    t = _arr(tok16, np.int32)
    assert t.size == 16
    return int(lib().cwo_block_digest(_p(t)))


def hash_blocks(tokens, tok_off, start_block=None, start_state=None, salt=None, hashes=None):
    """Returns (hashes u64[sum N], hash_off u64[R+1]).  ``hashes`` may be passed in (in-out)."""
    tokens = _arr(tokens, np.int32)
    tok_off = _arr(tok_off, np.uint64)
    R = tok_off.size - 1
    n = (tok_off[1:] - tok_off[:-1]) // np.uint64(16)
    hash_off = np.zeros(R + 1, np.uint64)
    np.cumsum(n, out=hash_off[1:])
    if hashes is None:
        hashes = np.zeros(int(hash_off[-1]), np.uint64)
    assert hashes.dtype == np.uint64 and hashes.size == int(hash_off[-1]) and hashes.flags.c_contiguous
    sb, ss, sl = _arr(start_block, np.uint32), _arr(start_state, np.uint64), _arr(salt, np.uint64)
    st = lib().cwo_hash_blocks(_p(tokens), _p(tok_off), _p(sb), _p(ss), _p(sl), _p(hash_off), C.c_uint32(R),
                               _p(hashes))
    if st:
        raise ValueError(f"cwo_hash_blocks status {st}")
    return hashes, hash_off


class Table:
    """Exact hash -> loc map (std::unordered_map)."""

    def __init__(self, log2_slots: int):
        self._h = C.c_void_p(lib().cwo_table_create(C.c_uint32(log2_slots)))

    def __del__(self):
        if getattr(self, "_h", None) and _lib is not None:
            _lib.cwo_table_destroy(self._h)
            self._h = None

    def __len__(self):
        return int(lib().cwo_table_size(self._h))

    def insert(self, keys, loc):
        keys, loc = _arr(keys, np.uint64), _arr(loc, np.uint32)
        win = np.empty(keys.size, np.uint32)
        st = lib().cwo_table_insert(self._h, _p(keys), _p(loc), C.c_uint32(keys.size), _p(win))
        return win, st

    def erase(self, keys):
        keys = _arr(keys, np.uint64)
        lib().cwo_table_erase(self._h, _p(keys), C.c_uint32(keys.size))

    def retag(self, keys, new_loc):
        keys, new_loc = _arr(keys, np.uint64), _arr(new_loc, np.uint32)
        lib().cwo_table_retag(self._h, _p(keys), _p(new_loc), C.c_uint32(keys.size))

    def lookup(self, keys):
        keys = _arr(keys, np.uint64)
        loc = np.empty(keys.size, np.uint32)
        lib().cwo_table_lookup(self._h, _p(keys), C.c_uint32(keys.size), _p(loc))
        return loc

    def match_prefix(self, hashes, hash_off):
        hashes, hash_off = _arr(hashes, np.uint64), _arr(hash_off, np.uint64)
        R = hash_off.size - 1
        k_total, n_gpu = np.empty(R, np.uint32), np.empty(R, np.uint32)
        hit_loc = np.empty(hashes.size, np.uint32)
        lib().cwo_match_prefix(self._h, _p(hashes), _p(hash_off), C.c_uint32(R), _p(k_total), _p(n_gpu),
                               _p(hit_loc))
        return k_total, n_gpu, hit_loc


def schedule(need_d, n_gpu, arrival_seq, req_id, policy, free_blocks, evictable, max_admit):
    need_d, n_gpu = _arr(need_d, np.uint32), _arr(n_gpu, np.uint32)
    arrival_seq, req_id = _arr(arrival_seq, np.uint64), _arr(req_id, np.uint32)
    R = need_d.size
    order = np.empty(R, np.uint32)
    na, de = C.c_uint32(0), C.c_uint32(0)
    st = lib().cwo_schedule(C.c_uint32(R), _p(need_d), _p(n_gpu), _p(arrival_seq), _p(req_id), C.c_uint32(policy),
                            C.c_uint32(free_blocks), C.c_uint32(evictable), C.c_uint32(max_admit), _p(order),
                            C.byref(na), C.byref(de))
    if st:
        raise ValueError(f"cwo_schedule status {st}")
    return order, na.value, de.value


def admit_chunked(order, need_d, n_gpu, new_tokens, free_blocks, evictable, max_admit, token_budget):
    """PAPER.md L271 chunked prefill (R8).  Returns (chunk_tokens[R] by input index, num_admit, deficit)."""
    order, need_d, n_gpu = _arr(order, np.uint32), _arr(need_d, np.uint32), _arr(n_gpu, np.uint32)
    new_tokens = _arr(new_tokens, np.uint32)
    R = need_d.size
    chunk = np.zeros(R, np.uint32)
    na, de = C.c_uint32(0), C.c_uint32(0)
    st = lib().cwo_admit_chunked(C.c_uint32(R), _p(order), _p(need_d), _p(n_gpu), _p(new_tokens),
                                 C.c_uint32(free_blocks), C.c_uint32(evictable), C.c_uint32(max_admit),
                                 C.c_uint64(token_budget), _p(chunk), C.byref(na), C.byref(de))
    if st:
        raise ValueError(f"cwo_admit_chunked status {st}")
    return chunk, na.value, de.value


def session_tau(features, weights, bias, session_state, tau_override=None):
    features = _arr(features, np.uint8)
    S, F = features.shape
    weights, session_state = _arr(weights, np.int16), _arr(session_state, np.uint8)
    tau_override = _arr(tau_override, np.uint32)
    tau = np.empty(S, np.uint32)
    st = lib().cwo_session_tau(C.c_uint32(S), C.c_uint32(F), _p(features), _p(weights), C.c_int32(bias),
                               _p(session_state), _p(tau_override), _p(tau))
    if st:
        raise ValueError(f"cwo_session_tau status {st}")
    return tau


def block_score(tau, tick_now, last_access, depth) -> int:
    return int(lib().cwo_block_score(C.c_uint32(tau), C.c_uint32(tick_now), C.c_uint32(last_access),
                                     C.c_uint32(depth)))


def score_evict(tick_now, features, weights, bias, session_state, tau_override, deficit, blk_session,
                blk_last_access, blk_depth, blk_ref_flags, cap=None):
    """Returns (victims u32[n], victim_scores u64[n], status)."""
    features = _arr(features, np.uint8)
    S, F = features.shape
    weights, session_state = _arr(weights, np.int16), _arr(session_state, np.uint8)
    tau_override = _arr(tau_override, np.uint32)
    bs, bl = _arr(blk_session, np.uint32), _arr(blk_last_access, np.uint32)
    bd, br = _arr(blk_depth, np.uint32), _arr(blk_ref_flags, np.uint32)
    M = bs.size
    cap = M if cap is None else cap
    victims, scores = np.empty(max(cap, 1), np.uint32), np.empty(max(cap, 1), np.uint64)
    nv = C.c_uint32(0)
    st = lib().cwo_score_evict(C.c_uint32(tick_now), C.c_uint32(S), C.c_uint32(F), _p(features), _p(weights),
                               C.c_int32(bias), _p(session_state), _p(tau_override), C.c_uint32(deficit),
                               C.c_uint32(M), _p(bs), _p(bl), _p(bd), _p(br), _p(victims), _p(scores),
                               C.byref(nv), C.c_uint32(cap))
    if st == -1:
        raise ValueError("cwo_score_evict invalid argument")
    return victims[: nv.value].copy(), scores[: nv.value].copy(), st


def swap_out(pool, n_chunks, chunk_bytes, chunk_stride, block_stride, victims, dst, slots=None):
    pool, dst = _arr(pool, np.uint8), dst
    assert dst.dtype == np.uint8 and dst.flags.c_contiguous
    victims, slots = _arr(victims, np.uint32), _arr(slots, np.uint32)
    lib().cwo_swap_out(_p(pool), C.c_uint32(n_chunks), C.c_uint64(chunk_bytes), C.c_uint64(chunk_stride),
                       C.c_uint64(block_stride), _p(victims), C.c_uint32(victims.size), _p(slots), _p(dst))
    return dst


def swap_in(pool, n_chunks, chunk_bytes, chunk_stride, block_stride, src, dst_blocks, slots=None):
    assert pool.dtype == np.uint8 and pool.flags.c_contiguous
    src = _arr(src, np.uint8)
    dst_blocks, slots = _arr(dst_blocks, np.uint32), _arr(slots, np.uint32)
    lib().cwo_swap_in(_p(pool), C.c_uint32(n_chunks), C.c_uint64(chunk_bytes), C.c_uint64(chunk_stride),
                      C.c_uint64(block_stride), _p(slots), _p(src), _p(dst_blocks), C.c_uint32(dst_blocks.size))
    return pool


def predict_tau(cluster, elapsed_ms, sample_off, samples):
    """Paper predictor (R7).  Returns (tau u32[S], status)."""
    cluster, elapsed_ms = _arr(cluster, np.uint32), _arr(elapsed_ms, np.uint32)
    sample_off, samples = _arr(sample_off, np.uint64), _arr(samples, np.uint32)
    tau = np.empty(cluster.size, np.uint32)
    st = lib().cwo_predict_tau(C.c_uint32(cluster.size), _p(cluster), _p(elapsed_ms), C.c_uint32(sample_off.size - 1),
                               _p(sample_off), _p(samples), _p(tau))
    return tau, st
