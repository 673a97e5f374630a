"""SASS opcode histogram of the built libcomb.so, one row per kernel (markdown on stdout).

    python paper_2602_01519_b200/sass_histogram.py [path/to/libcomb.so]

Build check for the Blackwell-only instructions: UTCHMMA (tcgen05.mma kind::f16), UTCQMMA (kind::f8f6f4), UTCBAR (tcgen05.commit), LDTM / STTM
(tcgen05.ld / st), UTMALDG (TMA tensor load), UBLKCP (1-D bulk copy), SYNCS (mbarrier), plus the arithmetic that
dominates the CUDA-core paths. Needs cuobjdump and c++filt on PATH (CUDA toolkit, binutils); no GPU.
"""
from __future__ import annotations

import collections
import os
import re
import subprocess
import sys

COLS = ["UTCHMMA", "UTCQMMA", "UTCBAR", "LDTM", "STTM", "UTMALDG", "UBLKCP", "SYNCS", "MUFU", "REDUX", "FFMA2", "FFMA", "F2FP",
        "LDS", "STS", "LDG", "STG", "ATOMG", "SHFL", "BAR"]


def kernel_name(mangled: str) -> str:
    full = subprocess.run(["c++filt", mangled], capture_output=True, text=True).stdout.strip()
    m = re.search(r"(\w+<[^>]*>|\w+)\(", full.replace("comb::(anonymous namespace)::", ""))
    return m.group(1) if m else full


def histogram(lib: str):
    sass = subprocess.run(["cuobjdump", "-sass", lib], capture_output=True, text=True, check=True).stdout
    rows, cur = [], None
    for line in sass.splitlines():
        if "Function :" in line:
            cur = {"name": kernel_name(line.split("Function :")[1].strip()), "n": 0, "ops": collections.Counter()}
            rows.append(cur)
            continue
        m = re.match(r"\s+/\*[0-9a-f]{4,}\*/\s+(?:@!?U?P\d+\s+)?([A-Z][A-Z0-9_]*)", line)
        if m and cur is not None:
            cur["n"] += 1
            op = m.group(1)
            cur["ops"]["REDUX" if op in ("REDUX", "CREDUX") else op] += 1
    return rows


def main():
    here = os.path.dirname(os.path.abspath(__file__))
    lib = sys.argv[1] if len(sys.argv) > 1 else os.path.join(here, "libcomb.so")
    rows = histogram(lib)
    print("| kernel | instructions | " + " | ".join(COLS) + " |")
    print("|---|---|" + "---|" * len(COLS))
    for r in sorted(rows, key=lambda r: r["name"]):
        print("| `%s` | %d | %s |" % (r["name"], r["n"], " | ".join(str(r["ops"][c]) for c in COLS)))
    tot = collections.Counter()
    for r in rows:
        tot.update(r["ops"])
    print("| **all %d kernels** | %d | %s |" % (len(rows), sum(r["n"] for r in rows),
                                             " | ".join(str(tot[c]) for c in COLS)))


if __name__ == "__main__":
    main()
