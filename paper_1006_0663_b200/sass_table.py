"""`python -m paper_1006_0663_b200.sass_table` — per-kernel SASS instruction counts of the built libteuk.so.

Disassembles the library with cuobjdump and prints, for every kernel, how many TMA loads (UTMALDG), mbarrier operations
(SYNCS), asynchronous copies (LDGSTS = cp.async), FP64 arithmetic instructions, local-memory (spill) accesses, shared-memory
accesses and block barriers it contains: the evidence that the Blackwell data-movement paths are really in the binary and
that the multiprecision kernels do not spill.  Static counts (one per SASS instruction, not per execution)."""
from __future__ import annotations

import collections
import os
import re
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
COLS = ["UTMALDG", "SYNCS", "LDGSTS", "DADD", "DMUL", "DFMA", "LDL", "STL", "LDS", "STS", "BAR"]


def table(so: str) -> str:
    txt = subprocess.run(["cuobjdump", "-sass", so], capture_output=True, text=True, check=True).stdout
    rows = []
    for part in re.split(r"\n\s*Function : ", txt)[1:]:
        name = part.split("\n", 1)[0].strip()
        dem = subprocess.run(["cu++filt", name], capture_output=True, text=True).stdout.strip() or name
        dem = re.split(r"\((?!int\)|bool\))", dem)[0]
        for junk in ("void ", "tk::", "(int)", "(bool)"):
            dem = dem.replace(junk, "")
        c = collections.Counter(re.findall(r"^\s+/\*[0-9a-f]{4,6}\*/\s+(?:@!?U?P\d\s+)?([A-Z0-9_]+)", part, flags=re.M))
        rows.append((dem, sum(c.values()), *[c[k] for k in COLS]))
    out = ["| kernel | SASS instr | UTMALDG (TMA) | SYNCS (mbarrier) | LDGSTS (cp.async) | DADD | DMUL | DFMA | LDL | STL | LDS | STS | BAR |",
           "|" + "---|" * 13]
    for r in sorted(rows):
        out.append("| `" + r[0] + "` | " + " | ".join(str(x) for x in r[1:]) + " |")
    return "\n".join(out)


if __name__ == "__main__":
    print(table(sys.argv[1] if len(sys.argv) > 1 else os.path.join(HERE, "libteuk.so")))
