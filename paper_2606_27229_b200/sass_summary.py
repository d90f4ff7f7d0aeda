"""Per-kernel histogram of the SASS mnemonics that show how a kernel of csrc/libcarve.so talks to the hardware:
tcgen05.mma (UTCHMMA), TMEM loads/stores (LDTM/STTM), TMA loads/stores/prefetches (UTMALDG/UTMASTG/UTMAPF), bulk copies
(UBLKCP), legacy tensor-core mma.sync (HMMA), ldmatrix/stmatrix (LDSM/STSM), mbarrier ops (SYNCS), shared loads (LDS)
generic loads (LD; should be 0: shared memory is addressed as shared) and packed fp32 pairs (FFMA2/FMUL2/FADD2).

    python -m paper_2606_27229_b200.sass_summary > profiles/r2_sass_summary.txt
"""
from __future__ import annotations

import collections
import re
import subprocess

from paper_2606_27229_b200 import build

COLS = ("UTCHMMA", "LDTM", "STTM", "UTMALDG", "UTMASTG", "UTMAPF", "UBLKCP", "HMMA.1688.F32.TF32", "HMMA.16816.F32.BF16",
        "LDSM", "STSM", "SYNCS", "LDS", "STS", "LD", "ST", "LDG", "STG", "MUFU", "FFMA2", "FMUL2", "FADD2", "BAR")


def main():
    lib = build.build()
    sass = subprocess.run(["cuobjdump", "-sass", lib], capture_output=True, text=True, check=True).stdout
    hist, size, name = collections.defaultdict(collections.Counter), collections.Counter(), None
    for ln in sass.splitlines():
        m = re.search(r"Function : (\S+)", ln)
        if m:
            name = subprocess.run(["c++filt", m.group(1)], capture_output=True, text=True).stdout.strip()
            name = re.sub(r"\(anonymous namespace\)::|carve::|void |\(.*", "", name)
            continue
        m = re.match(r"\s+/\*[0-9a-f]{4,6}\*/\s+(?:@!?U?P\d\s+)?([A-Z0-9_.]+)", ln)
        if m and name:
            op = m.group(1)
            size[name] += 1
            for c in COLS:
                if op == c or op.startswith(c + "."):
                    hist[name][c] += 1
    print("command: python -m paper_2606_27229_b200.sass_summary   (cuobjdump -sass paper_2606_27229_b200/csrc/libcarve.so, "
          "built with nvcc -gencode arch=compute_100a,code=sm_100a -lineinfo -O3)")
    print(f"{'kernel':58s} {'instrs':>6s} {'KB':>6s} " + " ".join(f"{c.split('.')[0] + ('.' + c.split('.')[-1] if '.' in c else ''):>9s}" for c in COLS))
    for k in sorted(size):
        print(f"{k[:58]:58s} {size[k]:6d} {size[k] * 16 / 1024:6.1f} " + " ".join(f"{hist[k][c]:9d}" for c in COLS))


if __name__ == "__main__":
    main()
