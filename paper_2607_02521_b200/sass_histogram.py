"""Opcode histogram of the built library: which Blackwell tensor / TMA / TMEM instructions each
kernel contains (`python -m paper_2607_02521_b200.sass_histogram [--md]`).

Evidence that the kernels are sm_100a-native (B200_PROFILING.md "What proves a Blackwell-native
kernel"): tcgen05.mma shows up in SASS as UTCHMMA (bf16) / UTCQMMA (fp8), tcgen05.ld as LDTM,
TMA loads / stores / prefetches as UTMALDG / UTMASTG / UTMAPF, tcgen05.commit as UTCBAR, and the
legacy mma.sync path would show up as HMMA (there is none).  Needs cuobjdump (CUDA toolkit)."""
from __future__ import annotations

import collections
import re
import subprocess
import sys

from .build import LIB, build

OPS = ("UTCHMMA", "UTCQMMA", "UTCHMMA.2CTA", "UTCQMMA.2CTA", "LDTM", "UTMALDG", "UTMASTG", "UTMAPF",
       "UTCBAR", "UTCBAR.2CTA", "HMMA", "MUFU.EX2", "MUFU.RCP")


def histogram():
    build()
    sass = subprocess.run(["cuobjdump", "-sass", LIB], check=True, capture_output=True, text=True).stdout
    counts = collections.OrderedDict()
    fn = None
    for line in sass.splitlines():
        m = re.search(r"Function : (\S+)", line)
        if m:
            fn = m.group(1)
            counts[fn] = collections.Counter()
            continue
        if fn is None:
            continue
        m = re.search(r"^\s*/\*[0-9a-f]+\*/\s+(?:@!?U?P\d+\s+)?([A-Z][A-Z0-9_.]*)", line)
        if not m:
            continue
        op = m.group(1)
        base = op.split(".")[0]
        if base in ("UTCHMMA", "UTCQMMA", "UTCBAR"):
            counts[fn][base + (".2CTA" if ".2CTA" in op else "")] += 1
        elif base in ("LDTM", "UTMALDG", "UTMASTG", "UTMAPF", "HMMA"):
            counts[fn][base] += 1
        elif op.startswith("MUFU.EX2") or op.startswith("MUFU.RCP"):
            counts[fn][op[:8]] += 1
    names = list(counts)
    dem = subprocess.run(["c++filt"], input="\n".join(names), capture_output=True, text=True).stdout.splitlines()
    short = [re.sub(r"\(.*", "", d).replace("void swiglu::", "") for d in dem]
    return [(s, counts[n]) for s, n in zip(short, names)]


def main():
    rows = histogram()
    print("| kernel | " + " | ".join(OPS) + " |")
    print("|---|" + "---|" * len(OPS))
    total = collections.Counter()
    for name, c in rows:
        total.update(c)
        print(f"| `{name}` | " + " | ".join(str(c.get(o, 0)) for o in OPS) + " |")
    print(f"| **all {len(rows)} kernels** | " + " | ".join(str(total.get(o, 0)) for o in OPS) + " |")


if __name__ == "__main__":
    sys.exit(main())
