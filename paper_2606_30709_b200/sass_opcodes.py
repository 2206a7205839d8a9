"""Per-kernel SASS opcode counts of libhga.so (evidence that the kernels are Blackwell-native; the profiling guide's
table: tcgen05.mma -> UTC*MMA, tcgen05.ld/st -> LDTM/STTM, TMA -> UTMALDG/UTMASTG/UBLKCP, commit -> UTCBAR).

    python -m paper_2606_30709_b200.sass_opcodes            # markdown table on stdout
"""
from __future__ import annotations

import collections
import re
import subprocess
import sys

from .binding import lib_path

OPS = ["UTCHMMA", "UTCBAR", "LDTM", "STTM", "UTMALDG", "UTMASTG", "UBLKCP", "SYNCS", "MUFU.EX2", "DFMA", "DMMA", "CREDUX", "HMMA"]


def kernel_opcodes(so: str):
    out = subprocess.run(["cuobjdump", "-sass", so], capture_output=True, text=True, check=True).stdout
    counts, name = collections.OrderedDict(), None
    for line in out.splitlines():
        m = re.search(r"Function : (\S+)", line)
        if m:
            name = subprocess.run(["c++filt", m.group(1)], capture_output=True, text=True).stdout.strip() or m.group(1)
            name = re.sub(r"\(anonymous namespace\)::|hga::|<unnamed>::", "", name)
            name = re.sub(r"\(.*", "", name)
            counts[name] = collections.Counter()
            continue
        m = re.match(r"\s+/\*[0-9a-f]{4,}\*/\s+(?:@!?U?P\d+\s+)?([A-Z0-9_.]+)", line)
        if m and name:
            op = m.group(1)
            for o in OPS:
                if op == o or op.startswith(o + "."):
                    counts[name][o] += 1
    return counts


def main():
    c = kernel_opcodes(lib_path())
    print("| kernel | " + " | ".join(OPS) + " |")
    print("|---|" + "---|" * len(OPS))
    for k, v in c.items():
        print(f"| `{k}` | " + " | ".join(str(v.get(o, 0)) for o in OPS) + " |")


if __name__ == "__main__":
    sys.exit(main())
