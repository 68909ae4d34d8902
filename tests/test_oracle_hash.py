"""Pins for the oracle's stage-1 hash (R1; SURVEY.md 8c stage 1).  CPU only.

The paper prints no hash value (it never describes hashing), so the pins are: constants re-derived from
their nothing-up-my-sleeve definitions with integer square roots, an independently derived INVERSE of fin,
zero/one special cases of the NH-style digest, the closed form of the affine chain evaluated with modular
exponentiation, resume == cold, prefix properties by brute force, and committed known-answer vectors.
"""
import json
import math
import os

import numpy as np
import pytest

import oracle

M64 = (1 << 64) - 1


def frac_sqrt(p):  # floor(2^64 * frac(sqrt p)) | 1
    return (math.isqrt(p << 128) & M64) | 1


A = (math.isqrt(5 << 128) - (1 << 64)) // 2          # floor(2^64 * (sqrt5 - 1)/2)
K2, K3, K5, K7, K11 = (frac_sqrt(p) for p in (2, 3, 5, 7, 11))


def unxorshift(x, s):
    y = x
    for _ in range(64 // s + 1):
        y = x ^ (y >> s)
    return y


def fin_inv(y):
    y = unxorshift(y, 32)
    y = (y * pow(K3, -1, 1 << 64)) & M64
    y = unxorshift(y, 29)
    y = (y * pow(K2, -1, 1 << 64)) & M64
    return unxorshift(y, 32)


def keys():
    out = []
    for m in range(8):
        x = oracle.fin((K11 * (m + 1)) & M64)
        out.append(((x >> 32) | 0x80000000, (x & 0xFFFFFFFF) | 0x80000000))
    return out


def as_i32(u):
    u &= 0xFFFFFFFF
    return u - (1 << 32) if u >= (1 << 31) else u


def test_constants_are_the_documented_irrationals():
    assert A == 0x9E3779B97F4A7C15 and A % 8 == 5
    assert (K2, K3, K5, K7, K11) == (0x6A09E667F3BCC909, 0xBB67AE8584CAA73B, 0x3C6EF372FE94F82B,
                                     0xA54FF53A5F1D36F1, 0x510E527FADE682D1)


def test_fin_is_the_bijection_with_the_derived_inverse():
    g = np.random.default_rng(1)
    for x in [0, 1, M64, 1 << 63] + [int(v) for v in g.integers(0, 1 << 63, size=200, dtype=np.uint64)]:
        assert fin_inv(oracle.fin(x)) == x
    assert oracle.fin(0) == 0


def test_digest_special_cases_zero_and_unit_multiplicands():
    k = keys()
    # every left multiplicand 0  ->  s = 0  ->  c = fin(K5)
    tok = []
    for ka, kb in k:
        tok += [as_i32(-ka), 12345]
    assert oracle.block_digest(tok) == oracle.fin(K5)
    # every left multiplicand 1  ->  s = sum (t_odd + kb_m)
    tok, s = [], 0
    for m, (ka, kb) in enumerate(k):
        t_odd = 1000 + 7 * m
        tok += [as_i32(1 - ka), t_odd]
        s += (t_odd + kb) & 0xFFFFFFFF
    assert oracle.block_digest(tok) == oracle.fin((s & M64) ^ K5)
    # one pair (a, b) only: s = a*b with the other left multiplicands zeroed
    tok = []
    for m, (ka, kb) in enumerate(k):
        tok += [as_i32((3 if m == 5 else 0) - ka), as_i32((0xFFFFFFF0 if m == 5 else 9) - kb)]
    assert fin_inv(oracle.block_digest(tok)) ^ K5 == 3 * 0xFFFFFFF0


def test_digest_depends_on_position_and_every_token():
    g = np.random.default_rng(2)
    tok = g.integers(0, 32000, size=16, dtype=np.int32)
    base = oracle.block_digest(tok)
    for i in range(16):
        t2 = tok.copy()
        t2[i] = (t2[i] + 1) % 32000
        assert oracle.block_digest(t2) != base
    for i in range(0, 16, 2):  # swapping two pairs / within a pair changes the digest
        t2 = tok.copy()
        t2[i], t2[i + 1] = tok[i + 1], tok[i]
        if tok[i] != tok[i + 1]:
            assert oracle.block_digest(t2) != base
    t2 = tok.copy()
    t2[0:2], t2[2:4] = tok[2:4].copy(), tok[0:2].copy()
    assert oracle.block_digest(t2) != base


@pytest.mark.parametrize("salt", [0, 0xDEADBEEFCAFEF00D])
def test_chain_closed_form(salt):
    g = np.random.default_rng(3)
    n = 37
    tok = g.integers(0, 32000, size=16 * n + 5, dtype=np.int32)  # +5: partial tail is never hashed
    h, off = oracle.hash_blocks(tok, [0, tok.size], salt=[salt])
    assert off.tolist() == [0, n] and h.size == n
    c = [oracle.block_digest(tok[16 * j:16 * j + 16]) for j in range(n)]
    h_init = oracle.fin(salt ^ K7)
    for j in range(n):
        closed = pow(A, j + 1, 1 << 64) * h_init + sum(pow(A, j - i, 1 << 64) * c[i] for i in range(j + 1))
        assert int(h[j]) == closed & M64


def test_resume_from_any_block_equals_cold_hash():
    g = np.random.default_rng(4)
    lens = [16 * 9 + 3, 16 * 4, 7, 16 * 13 + 15]
    tok = g.integers(0, 32000, size=sum(lens), dtype=np.int32)
    off = np.concatenate([[0], np.cumsum(lens)]).astype(np.uint64)
    salt = np.array([1, 2, 3, 4], np.uint64)
    cold, hoff = oracle.hash_blocks(tok, off, salt=salt)
    for sb in ([0, 0, 0, 0], [9, 4, 0, 13], [3, 1, 0, 7], [1, 4, 0, 12]):
        state = np.array([cold[int(hoff[r]) + sb[r] - 1] if sb[r] else 0 for r in range(4)], np.uint64)
        out = np.full(cold.size, 0x1111111111111111, np.uint64)
        oracle.hash_blocks(tok, off, start_block=sb, start_state=state, salt=salt, hashes=out)
        for r in range(4):
            lo, hi = int(hoff[r]), int(hoff[r + 1])
            assert (out[lo:lo + sb[r]] == 0x1111111111111111).all()      # untouched below start_block
            assert (out[lo + sb[r]:hi] == cold[lo + sb[r]:hi]).all()


def test_prefix_property_brute_force():
    g = np.random.default_rng(5)
    base = g.integers(0, 32000, size=16 * 12, dtype=np.int32)
    hb, _ = oracle.hash_blocks(base, [0, base.size])
    for pos in [0, 1, 15, 16, 17, 100, 16 * 12 - 1]:
        t2 = base.copy()
        t2[pos] = (t2[pos] + 1) % 32000
        h2, _ = oracle.hash_blocks(t2, [0, t2.size])
        first = pos // 16
        assert (h2[:first] == hb[:first]).all()
        assert (h2[first:] != hb[first:]).all()
    # different salts never share hashes; same salt + same tokens always do
    h3, _ = oracle.hash_blocks(base, [0, base.size], salt=[7])
    assert (h3 != hb).all()


def test_known_answer_vectors_match_committed_golden():
    path = os.path.join(os.path.dirname(__file__), "golden", "hash_kat.json")
    kat = json.load(open(path))
    for case in kat["cases"]:
        tok = np.array(case["tokens"], np.int32)
        h, _ = oracle.hash_blocks(tok, [0, tok.size], salt=[int(case["salt"], 16)])
        assert [f"{int(x):016x}" for x in h] == case["hashes"], case["name"]


def test_million_hashes_are_distinct_and_spread():
    g = np.random.default_rng(6)
    S, n = 64, 1024
    tok = g.integers(0, 32000, size=S * n * 16, dtype=np.int32)
    off = (np.arange(S + 1) * n * 16).astype(np.uint64)
    h, _ = oracle.hash_blocks(tok, off)
    assert np.unique(h).size == h.size
    slots = 1 << 17
    occ = np.bincount((h & np.uint64(slots - 1)).astype(np.int64), minlength=slots)
    assert abs((occ == 0).mean() - math.exp(-0.5)) < 0.01 and occ.max() <= 9
