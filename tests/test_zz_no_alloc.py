"""GPU parity — cw_hash_blocks_static (stage 1 with no ctx and no allocation: the scratch is a fixed static device
array) against the existing path cw_hash_blocks, bit-exact (integer work), and against the oracle.

Collected last on purpose (file name): the suite runs with pytest -x.  The test passes alone in a fresh process and
after the other tests: the entry point keeps no state a ctx shares, and it clears what must start at zero itself.
"""
import numpy as np
import pytest

import oracle
from harness import gen

pytestmark = pytest.mark.gpu


def _queue(g, R, long_len):
    lens = g.integers(0, 900, size=R)
    if long_len:
        lens[g.integers(0, R)] = long_len               # one request over many units / CTA ranges
    tok_off = np.concatenate([[0], np.cumsum(lens)]).astype(np.uint64)
    tokens = g.integers(0, gen.VOCAB, size=int(tok_off[-1]), dtype=np.int32)
    salt = g.integers(0, 1 << 63, size=R, dtype=np.uint64)
    return tokens, tok_off, salt


def test_static_scratch_hash_equals_the_ctx_path_on_two_calls_in_a_row():
    import torch

    import paper_2606_16824_b200 as cw
    from gpu_util import dev, gpu_hash, hash_off_of, host, small_ctx, zeros

    g = gen.rng(97, 0)
    # a large call (long request spanning many ranges), then at once a small one (few ranges, most of the grid idle;
    # the scratch still holds the first call's records and epoch), then a mid-sized one
    cases = [_queue(g, 3000, 300_000), _queue(g, 37, 70_000), _queue(g, 600, 0)]
    bufs = []
    for tokens, tok_off, salt in cases:                  # every caller-side buffer exists before the first call
        ho = hash_off_of(tok_off)
        bufs.append((dev(np.concatenate([tokens, np.zeros(4, np.int32)])), dev(tok_off), dev(ho), dev(salt),
                     zeros(int(ho[-1]), np.uint64), zeros(1, np.uint32), ho))
    torch.cuda.synchronize()
    before = torch.cuda.memory_allocated()
    for (d_tok, d_to, d_ho, d_salt, d_out, d_st, ho) in bufs:   # back to back on one stream, no sync in between
        cw.hash_blocks_static(d_tok, d_to, d_ho, d_to.numel() - 1, d_out, int(ho[-1]), salt=d_salt, status=d_st)
    torch.cuda.synchronize()
    assert torch.cuda.memory_allocated() == before
    ctx = small_ctx(max_hashed_blocks=1 << 21)
    for (tokens, tok_off, salt), (_, _, _, _, d_out, d_st, ho) in zip(cases, bufs):
        got = host(d_out, np.uint64)[: int(ho[-1])]
        ref, rho, st = gpu_hash(ctx, tokens, tok_off, salt=salt)          # the existing path
        exp, _ = oracle.hash_blocks(tokens, tok_off, salt=salt)
        assert st == 0 and int(host(d_st, np.uint32)[0]) == 0 and (rho == ho).all()
        assert (got == ref).all() and (got == exp).all()
    ctx.close()


def test_static_scratch_hash_resume_limits_and_status():
    import paper_2606_16824_b200 as cw
    from gpu_util import dev, hash_off_of, host, zeros
    import torch

    g = gen.rng(98, 0)
    tokens, tok_off, salt = _queue(g, 9, 20_000)
    ho = hash_off_of(tok_off)
    exp, _ = oracle.hash_blocks(tokens, tok_off, salt=salt)
    d_tok = dev(np.concatenate([tokens, np.zeros(4, np.int32)]))
    # resume: the first start_block hashes of every request are given, the rest is computed from start_state
    n = (ho[1:] - ho[:-1]).astype(np.int64)
    sb = (n // 2).astype(np.uint32)
    state = np.array([exp[int(ho[r]) + int(sb[r]) - 1] if sb[r] else 0 for r in range(n.size)], np.uint64)
    given = exp.copy()
    for r in range(n.size):
        given[int(ho[r]) + int(sb[r]): int(ho[r + 1])] = 0
    d_out = dev(given)
    cw.hash_blocks_static(d_tok, dev(tok_off), dev(ho), n.size, d_out, int(ho[-1]), start_block=dev(sb),
                          start_state=dev(state), salt=dev(salt))
    torch.cuda.synchronize()
    assert (host(d_out, np.uint64)[: int(ho[-1])] == exp).all()
    # beyond the static maximum: rejected on the host, nothing launched
    with pytest.raises(cw.CwError) as e:
        cw.hash_blocks_static(d_tok, dev(tok_off), dev(ho), cw.HASH_STATIC_MAX_REQUESTS + 1, d_out, int(ho[-1]))
    assert e.value.code == cw.CW_E_INVAL
    # device-detected: hash_off inconsistent with tok_off -> non-zero status word, then a clean call still works
    bad = ho.copy()
    bad[3:] += np.uint64(1)
    d_st, d_out2 = zeros(1, np.uint32), zeros(int(ho[-1]) + 1, np.uint64)
    cw.hash_blocks_static(d_tok, dev(tok_off), dev(bad), n.size, d_out2, int(ho[-1]) + 1, salt=dev(salt), status=d_st)
    torch.cuda.synchronize()
    assert int(host(d_st, np.uint32)[0]) != 0
    d_st.zero_()
    d_out3 = zeros(int(ho[-1]), np.uint64)
    cw.hash_blocks_static(d_tok, dev(tok_off), dev(ho), n.size, d_out3, int(ho[-1]), salt=dev(salt), status=d_st)
    torch.cuda.synchronize()
    assert int(host(d_st, np.uint32)[0]) == 0 and (host(d_out3, np.uint64)[: int(ho[-1])] == exp).all()
