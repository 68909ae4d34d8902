"""Instruction-mix summary of libcachewise.so, kernel by kernel (cuobjdump -sass), as Markdown on stdout.

    python -m paper_2606_16824_b200.sass_summary > profiles/r2_sass_summary.md

What to look for (B200_PROFILING.md "What proves a Blackwell-native kernel"): UBLKCP = TMA bulk copies
(cp.async.bulk), SYNCS = mbarrier operations, REDUX / MATCH = warp reductions and match.any, ATOMG / RED = global
atomics, LDG.E.128 = 16-byte slot loads.  No UTC*MMA / HMMA is expected: nothing on this path is a dense contraction.
"""
from __future__ import annotations

import collections
import re
import subprocess
import sys

from . import build

FAMILIES = ["UBLKCP", "UTMALDG", "UTMASTG", "SYNCS", "LDGSTS", "LDG", "STG", "LDS", "STS", "ATOMG", "ATOMS", "REDUX",
            "RED", "MATCH", "SHFL", "VOTE", "BAR", "MEMBAR", "IMAD", "LOP3", "ISETP", "BRA", "UTC", "HMMA", "CCTL"]


def summarise(lib: str):
    out = subprocess.check_output(["cuobjdump", "-sass", lib], text=True)
    kernels, cur = collections.OrderedDict(), None
    for line in out.splitlines():
        m = re.match(r"\s*Function : (\S+)", line)
        if m:
            cur = subprocess.check_output(["c++filt", m.group(1)], text=True).strip()
            cur = re.sub(r"\(anonymous namespace\)::", "", cur).split("(")[0]
            kernels[cur] = collections.Counter()
            continue
        m = re.match(r"\s*/\*[0-9a-f]{4,}\*/\s+(?:@!?U?P\d+\s+)?([A-Z0-9_.]+)", line)
        if m and cur:
            op = m.group(1)
            kernels[cur]["total"] += 1
            if op.startswith("CREDUX"):
                op = op[1:]  # uniform-register flavour of REDUX
            for fam in FAMILIES:
                if op.startswith(fam):
                    kernels[cur][fam] += 1
                    break
            if op.startswith("LDG.E.128") or op.startswith("LDG.E.ENL2.256"):
                kernels[cur]["LDG>=128b"] += 1
    return kernels


def main():
    lib = build.build()
    ks = summarise(lib)
    cols = ["total", "UBLKCP", "SYNCS", "LDG", "LDG>=128b", "STG", "LDS", "STS", "ATOMG", "RED", "ATOMS", "REDUX", "MATCH",
            "SHFL", "BAR", "MEMBAR", "UTC", "HMMA"]
    print("# SASS instruction mix per kernel (libcachewise.so, sm_100a)\n")
    print("Command: `python -m paper_2606_16824_b200.sass_summary` (cuobjdump -sass on the built library; static counts of")
    print("instructions in the binary, not executed counts).\n")
    print("| kernel | " + " | ".join(cols) + " |")
    print("|---|" + "---|" * len(cols))
    for name, c in ks.items():
        print(f"| `{name}` | " + " | ".join(str(c.get(k, 0)) for k in cols) + " |")
    tma = [k for k, c in ks.items() if c.get("UBLKCP")]
    print(f"\nTMA bulk copies (UBLKCP) in: {', '.join('`' + k + '`' for k in tma)}.")
    print("Tensor-core instructions (UTC*MMA / HMMA): " +
          ("none, as intended." if not any(c.get("UTC") or c.get("HMMA") for c in ks.values()) else "PRESENT."))


if __name__ == "__main__":
    sys.exit(main())
