"""GPU parity — stage 1 (cw_hash_blocks) against the oracle, bit-exact, through the C ABI."""
import json
import os

import numpy as np
import pytest

import oracle
from harness import gen

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx():
    from gpu_util import small_ctx
    c = small_ctx(max_hashed_blocks=1 << 21)
    yield c
    c.close()


def _check(ctx, tokens, tok_off, **kw):
    from gpu_util import gpu_hash
    got, ho, st = gpu_hash(ctx, tokens, tok_off, **kw)
    okw = {k: v for k, v in kw.items() if k in ("salt", "start_block", "start_state")}
    if "hashes" in kw:
        okw["hashes"] = np.array(kw["hashes"], np.uint64)
    exp, eho = oracle.hash_blocks(tokens, tok_off, **okw)
    assert st == 0
    assert (ho == eho).all()
    bad = np.nonzero(got != exp)[0]
    assert bad.size == 0, f"{bad.size} mismatches, first at {bad[:5]}"
    return got


def test_known_answer_vectors(ctx):
    kat = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "hash_kat.json")))
    from gpu_util import gpu_hash
    for c in kat["cases"]:
        tok = np.array(c["tokens"], np.int32)
        got, _, st = gpu_hash(ctx, tok, [0, tok.size], salt=[int(c["salt"], 16)])
        assert st == 0 and [f"{int(x):016x}" for x in got] == c["hashes"], c["name"]


def test_ragged_requests_all_alignments_and_tails(ctx):
    g = gen.rng(11, 0)
    # empty, sub-block, exact blocks, one unit (256 blocks) -1/0/+1, several units with ragged tail; the
    # cumulative offsets visit all four 4-byte alignments
    lens = [0, 5, 16, 17, 31, 32, 16 * 255 + 1, 16 * 256 + 2, 16 * 257 + 3, 16 * 1000 + 7, 1, 16 * 31 + 15,
            16 * 32, 16 * 33 + 9, 0, 16 * 513 + 6, 3]
    tok_off = np.concatenate([[0], np.cumsum(lens)]).astype(np.uint64)
    assert {int(o) % 4 for o in tok_off[:-1]} == {0, 1, 2, 3}
    tokens = g.integers(0, gen.VOCAB, size=int(tok_off[-1]), dtype=np.int32)
    salt = g.integers(0, 1 << 63, size=len(lens), dtype=np.uint64)
    _check(ctx, tokens, tok_off, salt=salt)
    _check(ctx, tokens, tok_off)  # NULL salt


def test_extreme_token_values_and_reserved_seeds(ctx):
    tok = np.array([0x7FFFFFFF, -1, -2147483648, 0] * 64, np.int32)
    _check(ctx, tok, [0, 100, tok.size], salt=[0, 0xFFFFFFFFFFFFFFFF])


def test_long_request_crosses_more_than_32_units(ctx):
    g = gen.rng(12, 0)
    n_blocks = 256 * 41 + 77  # 42 units: the look-back needs two 32-wide batches
    lens = [3, 16 * n_blocks + 5, 16 * 300]
    tok_off = np.concatenate([[0], np.cumsum(lens)]).astype(np.uint64)
    tokens = g.integers(0, gen.VOCAB, size=int(tok_off[-1]), dtype=np.int32)
    _check(ctx, tokens, tok_off, salt=[7, 8, 9])


def test_resume_from_start_block(ctx):
    g = gen.rng(13, 0)
    lens = [16 * 9 + 3, 16 * 600, 7, 16 * 1300 + 15, 16 * 256]
    tok_off = np.concatenate([[0], np.cumsum(lens)]).astype(np.uint64)
    tokens = g.integers(0, gen.VOCAB, size=int(tok_off[-1]), dtype=np.int32)
    salt = np.arange(1, 6, dtype=np.uint64)
    cold, ho = oracle.hash_blocks(tokens, tok_off, salt=salt)
    for sb in ([0, 0, 0, 0, 0], [9, 600, 0, 1300, 256], [3, 255, 0, 257, 1], [1, 512, 0, 1299, 255]):
        state = np.array([cold[int(ho[r]) + sb[r] - 1] if sb[r] else 0 for r in range(5)], np.uint64)
        init = np.full(cold.size, 0x1111111111111111, np.uint64)
        got = _check(ctx, tokens, tok_off, salt=salt, start_block=sb, start_state=state, hashes=init)
        for r in range(5):
            lo = int(ho[r])
            assert (got[lo:lo + sb[r]] == 0x1111111111111111).all()
            assert (got[lo + sb[r]:int(ho[r + 1])] == cold[lo + sb[r]:int(ho[r + 1])]).all()


def test_token_space_ranges_with_stretches_that_hold_no_work():
    """The ranges are cut in TOKEN space and moved to unit boundaries: long stretches of tokens without any unit
    (thousands of requests shorter than a block, requests resumed close to their end) leave ranges empty in the middle
    of the grid, a range start may hop over many requests, and a long request behind them still spans many ranges."""
    from gpu_util import small_ctx
    ctx = small_ctx(max_requests=12000, max_hashed_blocks=1 << 21)
    g = gen.rng(57, 0)
    lens = np.concatenate([g.integers(0, 16, size=4000),                 # no full block at all
                           [16 * 70_000 + 5],                            # one request over hundreds of ranges
                           g.integers(0, 16, size=3000),
                           g.integers(16 * 200, 16 * 3000, size=40),     # resumed close to their end below
                           g.integers(0, 40, size=2000),
                           [16 * 256 * 3, 16 * 256 * 3 + 1, 15, 16]]).astype(np.int64)
    R = lens.size
    tok_off = np.concatenate([[0], np.cumsum(lens)]).astype(np.uint64)
    tokens = g.integers(0, gen.VOCAB, size=int(tok_off[-1]), dtype=np.int32)
    salt = g.integers(0, 1 << 63, size=R, dtype=np.uint64)
    cold, ho = oracle.hash_blocks(tokens, tok_off, salt=salt)
    _check(ctx, tokens, tok_off, salt=salt)
    n = (ho[1:] - ho[:-1]).astype(np.int64)
    sb = np.zeros(R, np.int64)
    sb[7001:7041] = np.maximum(n[7001:7041] - g.integers(0, 3, size=40), 0)     # 0..2 blocks left to hash
    sb[4000] = 69_000
    state = np.array([cold[int(ho[r]) + int(sb[r]) - 1] if sb[r] else 0 for r in range(R)], np.uint64)
    init = np.full(cold.size, 0x2222222222222222, np.uint64)
    got = _check(ctx, tokens, tok_off, salt=salt, start_block=sb.astype(np.uint32), start_state=state, hashes=init)
    for r in (4000, 7001, 7020, 7040):
        lo = int(ho[r])
        assert (got[lo:lo + int(sb[r])] == 0x2222222222222222).all()
        assert (got[lo + int(sb[r]):int(ho[r + 1])] == cold[lo + int(sb[r]):int(ho[r + 1])]).all()
    ctx.close()


def test_scaled_stress_queue_and_repeatability(ctx):
    snap = gen.stress_snapshot(seed=5, S=8, L=32768, RB=1024, req_per_session=16, len_median=4096, len_min=64,
                               len_max=32768)
    a = _check(ctx, snap.tokens, snap.tok_off)
    b = _check(ctx, snap.tokens, snap.tok_off)  # the self-cleaning control block: second call identical
    assert (a == b).all()


def test_inconsistent_offsets_are_reported_not_crashing(ctx):
    from gpu_util import dev, zeros
    tok = dev(np.zeros(64, np.int32))
    tok_off = dev(np.array([0, 64], np.uint64))
    bad_hash_off = dev(np.array([0, 3], np.uint64))  # should be 4
    out = zeros(8, np.uint64)
    ctx.hash_blocks(tok, tok_off, bad_hash_off, 1, out)
    assert ctx.sync(check=False) == -1
    assert ctx.sync(check=False) == 0  # status is reported once


def test_host_side_argument_checks(ctx):
    import paper_2606_16824_b200 as cw
    from gpu_util import dev, zeros
    tok = dev(np.zeros(64, np.int32))
    off = dev(np.array([0, 64], np.uint64))
    ho = dev(np.array([0, 4], np.uint64))
    out = zeros(8, np.uint64)
    for args in [(None, off, ho, 1, out), (tok, None, ho, 1, out), (tok, off, ho, 1, None),
                 (tok.data_ptr() + 4, off, ho, 1, out), (tok, off, ho, 1 << 30, out)]:
        with pytest.raises(cw.CwError) as e:
            ctx.hash_blocks(*args)
        assert e.value.code == cw.CW_E_INVAL
    ctx.hash_blocks(tok, off, ho, 0, out)  # R = 0 is a no-op
    assert ctx.sync(check=False) == 0


def test_small_and_large_calls_interleaved_on_one_context():
    """Every call cuts its own token space into ranges (no plan pass) and its last CTA re-arms the range ticket and
    advances the epoch.  Small and large calls in any order on one context, including long requests that span many
    ranges (look-back over dependent ranges), must stay bit-exact."""
    from gpu_util import small_ctx
    ctx = small_ctx(max_requests=4096, max_hashed_blocks=1 << 21)
    g = gen.rng(41, 0)
    for rnd, R in enumerate([3, 700, 1, 512, 513, 2, 2, 900, 511, 40]):
        lens = g.integers(0, 600, size=R)
        lens[g.integers(0, R)] = int(g.integers(100_000, 400_000))     # one request over hundreds of units
        tok_off = np.concatenate([[0], np.cumsum(lens)]).astype(np.uint64)
        tokens = g.integers(0, gen.VOCAB, size=int(tok_off[-1]), dtype=np.int32)
        salt = g.integers(0, 2**63, size=R, dtype=np.uint64) if rnd % 2 else None
        _check(ctx, tokens, tok_off, **({"salt": salt} if salt is not None else {}))
    ctx.close()
