"""Per-kernel SASS opcode histogram of the built library (what proves which hardware path a kernel takes: UTC*MMA / LDTM =
tcgen05 + TMEM, UBLKCP / UTMALDG = TMA, IMMA / HMMA = legacy mma.sync, LDGSTS = cp.async).

    python -m paper_2606_31519_b200.sass_histogram [path/to/librbq_b200.so] > profiles/r02_sass_histogram.md

Needs only cuobjdump (no GPU).
"""
from __future__ import annotations

import collections
import re
import subprocess
import sys
from pathlib import Path

INTEREST = ("UTCHMMA", "UTCIMMA", "UTCQMMA", "UTCBAR", "UTCATOMSWS", "LDTM", "STTM", "UBLKCP", "UTMALDG", "UTMASTG", "SYNCS",
            "IMMA", "HMMA", "QMMA", "LDGSTS", "LDSM", "LDG", "STG", "LDS", "STS", "ATOMS", "ATOMG", "RED", "REDG", "LOP3", "POPC",
            "MUFU", "SHFL", "FFMA", "DADD", "DFMA", "BAR", "UCGABAR_ARV", "UCGABAR_WAIT", "CCTL", "MEMBAR", "ACQBULK")


def histogram(lib: Path):
    out = subprocess.run(["cuobjdump", "-sass", str(lib)], capture_output=True, text=True, check=True).stdout
    kernels, name = collections.OrderedDict(), None
    for line in out.splitlines():
        m = re.search(r"Function : (\S+)", line)
        if m:
            name = subprocess.run(["c++filt", m.group(1)], capture_output=True, text=True).stdout.strip()
            name = re.sub(r"\(anonymous namespace\)::", "", name)
            name = re.sub(r"\(.*", "", name).replace("void ", "")
            kernels[name] = collections.Counter()
            continue
        m = re.match(r"\s+/\*[0-9a-f]{4,}\*/\s+(?:@!?U?P\w+\s+)?([A-Z0-9_]+)", line)
        if m and name:
            kernels[name][m.group(1)] += 1
    return kernels


def main():
    lib = Path(sys.argv[1]) if len(sys.argv) > 1 else Path(__file__).resolve().parent / "librbq_b200.so"
    ks = histogram(lib)
    print(f"# SASS opcode histogram per kernel of `{lib.name}` (sm_100a)\n")
    print("Command: `python -m paper_2606_31519_b200.sass_histogram` (cuobjdump -sass on the built library; base mnemonics, "
          "modifiers dropped).  Only the mnemonics that identify a hardware path are listed, then the instruction total.\n")
    print("| kernel | instructions | path-defining mnemonics |")
    print("|---|---|---|")
    for name, c in ks.items():
        sel = ", ".join(f"{k} {c[k]}" for k in INTEREST if c.get(k))
        print(f"| `{name}` | {sum(c.values())} | {sel} |")


if __name__ == "__main__":
    main()
