"""SASS opcode histogram of the kernels in libtq.so (evidence for profiles/: UTCHMMA / LDTM = tcgen05, HMMA = mma.sync,
UBLKCP = cp.async.bulk, SYNCS = mbarrier).  `python -m paper_2603_26110_b200.sass_histogram` prints a markdown table."""
from __future__ import annotations

import collections
import re
import subprocess
import sys

from .build import LIB, build

WANT = ["UTCHMMA", "LDTM", "STTM", "HMMA", "UBLKCP", "UBLKPF", "SYNCS", "UTMALDG", "LDGSTS", "LDS", "STS", "LDG", "STG", "LOP3", "SHF",
        "IMAD", "FFMA", "FFMA2", "MUFU", "CREDUX", "BAR", "LDL", "STL"]
KERNELS = ("decode_main", "prep_kernel", "quantize_pack", "finish_kernel")


def main() -> int:
    build()
    sass = subprocess.run(["cuobjdump", "-sass", LIB], capture_output=True, text=True, check=True).stdout
    hist: dict[str, collections.Counter] = collections.defaultdict(collections.Counter)
    fn = None
    for line in sass.splitlines():
        m = re.match(r"\s*Function : (\S+)", line)
        if m:
            fn = m.group(1)
            continue
        m = re.match(r"\s*/\*[0-9a-f]{4,}\*/\s+(?:@!?U?P\d+\s+)?([A-Z][A-Z0-9_]*)", line)
        if m and fn:
            hist[fn][m.group(1)] += 1
    names = subprocess.run(["c++filt"] + list(hist), capture_output=True, text=True).stdout.split("\n")
    print("| kernel | instructions | " + " | ".join(WANT) + " |")
    print("|---|---:|" + "---:|" * len(WANT))
    for fn, nm in sorted(zip(hist, names), key=lambda x: x[1]):
        if not any(k in nm for k in KERNELS):
            continue
        short = nm.replace("tq::", "").replace("(anonymous namespace)::", "").replace("void ", "").split("(")[0]
        print(f"| `{short}` | {sum(hist[fn].values())} | " + " | ".join(str(hist[fn].get(w, 0)) for w in WANT) + " |")
    return 0


if __name__ == "__main__":
    sys.exit(main())
