"""Writes tests/golden/hash_kat.json — known-answer vectors for the stage-1 hash.

Calls ONLY the oracle (never the CUDA path).  PAPER.md prints no hash value (it does not describe
hashing at all; reading R1 defines it), so these are regression vectors of the pinned oracle:
the all-zero block, tokens 0..15, a 3-block chain and a non-zero salt (SURVEY.md 8c stage 1, pin iv).
Run:  python tests/golden/make_golden.py
"""
import json
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__)))))
import oracle  # noqa: E402


def case(name, tokens, salt):
    tok = np.array(tokens, np.int32)
    h, _ = oracle.hash_blocks(tok, [0, tok.size], salt=[salt])
    return dict(name=name, salt=f"{salt:016x}", tokens=[int(t) for t in tok], hashes=[f"{int(x):016x}" for x in h])


if __name__ == "__main__":
    g = np.random.Generator(np.random.Philox(key=[2606, 16824]))
    cases = [
        case("all_zero_block", [0] * 16, 0),
        case("tokens_0_to_15", list(range(16)), 0),
        case("three_block_chain", g.integers(0, 32000, size=48).tolist(), 0),
        case("nonzero_salt_with_tail", g.integers(0, 32000, size=16 * 5 + 9).tolist(), 0x0123456789ABCDEF),
        case("max_token_ids", [0x7FFFFFFF] * 32, 0xFFFFFFFFFFFFFFFF),
    ]
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "hash_kat.json")
    json.dump(dict(source="oracle/cw_oracle.cpp via tests/golden/make_golden.py", cases=cases), open(out, "w"), indent=1)
    print("wrote", out)
