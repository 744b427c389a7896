"""Per-kernel SASS evidence of libawr.so as a markdown table (runs without a GPU):

    python -m paper_2606_05597_b200.sass_summary > profiles/r2_sass_summary.md

For every kernel of the library: registers, spill bytes, shared memory (cuobjdump -res-usage) and
the counts of the SASS mnemonics that show which Blackwell units it uses
(/opt/skills/guides/B200_PROFILING.md "What proves a Blackwell-native kernel"):
UTC*MMA = tcgen05.mma, UTCBAR = tcgen05.commit, LDTM = tcgen05.ld, UTMALDG = cp.async.bulk.tensor,
UBLKCP = 1-D cp.async.bulk, SYNCS = mbarrier, MUFU.EX2 = ex2.approx, HMMA = the legacy tensor path
(must be 0).  Template instantiations of one kernel are folded into one row (counts of the largest
instantiation, the number of instantiations in brackets)."""
from __future__ import annotations

import re
import subprocess
import sys
from collections import Counter, defaultdict

from . import build as _build

COLS = [("UTC*MMA", r"^UTC\w*MMA"), ("UTCBAR", r"^UTCBAR"), ("LDTM", r"^LDTM"), ("UTMALDG", r"^UTMALDG"),
        ("UBLKCP", r"^UBLKCP"), ("UTMASTG", r"^UTMASTG"), ("SYNCS", r"^SYNCS"), ("MUFU.EX2", r"^MUFU\.EX2"),
        ("HMMA", r"^HMMA"), ("LDG", r"^LDG"), ("STG", r"^STG"), ("LDS", r"^LDS"), ("LDL/STL", r"^(LDL|STL)")]


def demangle(names):
    out = subprocess.run(["c++filt"], input="\n".join(names), capture_output=True, text=True).stdout
    return dict(zip(names, out.splitlines()))


def family(d):
    """`awr::rows_rf_kernel<19, 2, false>(...)` -> (`rows_rf_kernel`, `<19, 2, false>`)."""
    m = re.match(r"(?:void )?(?:awr::)?(?:head::)?(\w+)(<[^(]*>)?\(", d)
    return (m.group(1), m.group(2) or "") if m else (d, "")


def main():
    lib = _build.build()
    sass = subprocess.run(["cuobjdump", "-sass", lib], capture_output=True, text=True, check=True).stdout
    res = subprocess.run(["cuobjdump", "-res-usage", lib], capture_output=True, text=True, check=True).stdout
    counts = defaultdict(Counter)
    size = Counter()
    cur = None
    for line in sass.splitlines():
        m = re.match(r"\s*Function : (\S+)", line)
        if m:
            cur = m.group(1)
            continue
        m = re.match(r"\s+/\*[0-9a-f]{4,}\*/\s+(?:@!?U?P\d+\s+)?([A-Z][A-Z0-9_.]*)", line)
        if m and cur:
            size[cur] += 1
            for name, pat in COLS:
                if re.match(pat, m.group(1)):
                    counts[cur][name] += 1
    usage = {}
    fn = None
    for line in res.splitlines():
        m = re.match(r"\s*Function (\S+):", line)
        if m:
            fn = m.group(1)
            continue
        m = re.search(r"REG:(\d+) STACK:(\d+) SHARED:(\d+) LOCAL:(\d+)", line)
        if m and fn:
            usage[fn] = tuple(int(x) for x in m.groups())
    names = sorted(size)
    dem = demangle(names)
    fam = defaultdict(list)
    for n in names:
        fam[family(dem[n])[0]].append(n)
    print("# SASS summary of libawr.so (sm_100a), per kernel\n")
    print("Made by `python -m paper_2606_05597_b200.sass_summary` (cuobjdump -sass / -res-usage of the "
          "in-tree build; no GPU needed).  One row per kernel; template instantiations are folded: "
          "the row shows the instantiation with the most instructions, `[n]` = instantiations.  "
          "STACK = bytes of local memory (spills).\n")
    hdr = ["kernel", "instr", "REG", "STACK"] + [c for c, _ in COLS]
    print("| " + " | ".join(hdr) + " |")
    print("|" + "---|" * len(hdr))
    for f in sorted(fam):
        big = max(fam[f], key=lambda n: size[n])
        reg, stack, _, _ = usage.get(big, (0, 0, 0, 0))
        label = "`%s%s` [%d]" % (f, family(dem[big])[1], len(fam[f]))
        row = [label, str(size[big]), str(reg), str(stack)] + [str(counts[big][c]) for c, _ in COLS]
        print("| " + " | ".join(row) + " |")
    tot = Counter()
    for n in names:
        tot.update(counts[n])
    print("\nWhole library (%d kernels): " % len(names) +
          ", ".join("%s %d" % (c, tot[c]) for c, _ in COLS) + ".")
    worst = sorted(((usage.get(n, (0, 0, 0, 0))[1], dem[n]) for n in names), reverse=True)[:5]
    print("\nLargest local-memory frames: " + "; ".join("%d B `%s`" % (s, family(d)[0] + family(d)[1])
                                                         for s, d in worst if s) + ".")


if __name__ == "__main__":
    sys.exit(main())
