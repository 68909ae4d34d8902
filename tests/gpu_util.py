"""Helpers for the `-m gpu` parity tests: numpy <-> device buffers (torch is used for device memory only)."""
import numpy as np
import torch

import paper_2606_16824_b200 as cw

_SIGNED = {np.dtype(np.uint64): np.int64, np.dtype(np.uint32): np.int32, np.dtype(np.uint16): np.int16}


def dev(a, dtype=None):
    """numpy array -> device tensor holding the same bytes (unsigned dtypes travel as their signed twins)."""
    a = np.ascontiguousarray(a, dtype=dtype)
    if a.dtype in _SIGNED:
        a = a.view(_SIGNED[a.dtype])
    return torch.from_numpy(a.copy()).cuda()


def host(t, dtype):
    """device tensor -> numpy array reinterpreted as `dtype`."""
    return t.cpu().numpy().view(dtype)


def zeros(n, dtype):
    dt = {np.uint64: torch.int64, np.uint32: torch.int32, np.uint8: torch.uint8, np.int32: torch.int32}[dtype]
    return torch.zeros(max(int(n), 1), dtype=dt, device="cuda")


def hash_off_of(tok_off):
    tok_off = np.asarray(tok_off, np.uint64)
    n = (tok_off[1:] - tok_off[:-1]) // np.uint64(16)
    ho = np.zeros(tok_off.size, np.uint64)
    np.cumsum(n, out=ho[1:])
    return ho


def gpu_hash(ctx, tokens, tok_off, salt=None, start_block=None, start_state=None, hashes=None, pad_front=0):
    """Runs cw_hash_blocks; returns (hashes u64[], hash_off).  pad_front shifts the token base by whole
    16-byte units only (the ABI wants a 16-byte aligned base; request starts may be any 4-byte offset)."""
    tok_off = np.asarray(tok_off, np.uint64)
    ho = hash_off_of(tok_off)
    R = tok_off.size - 1
    d_tok = dev(np.concatenate([np.asarray(tokens, np.int32), np.zeros(4, np.int32)]))
    d_hashes = zeros(int(ho[-1]), np.uint64) if hashes is None else dev(hashes)
    ctx.hash_blocks(d_tok, dev(tok_off), dev(ho), R, d_hashes,
                    start_block=None if start_block is None else dev(start_block, np.uint32),
                    start_state=None if start_state is None else dev(start_state, np.uint64),
                    salt=None if salt is None else dev(salt, np.uint64))
    st = ctx.sync(check=False)
    return host(d_hashes, np.uint64)[: int(ho[-1])], ho, st


def small_ctx(**kw):
    args = dict(num_blocks=1024, table_log2_slots=12, max_requests=4096, max_hashed_blocks=1 << 20, max_sessions=64,
                max_features=16)
    args.update(kw)
    return cw.Context(**args)
