"""Opcode histogram of the built kernels (cuobjdump -sass), the evidence that the Newton-Schulz kernels are
Blackwell-native: tcgen05.mma -> UTCHMMA, tcgen05.ld -> LDTM, TMA -> UTMALDG / UTMASTG, mbarrier -> SYNCS,
tcgen05.commit -> UTCBAR (B200_PROFILING.md "What proves a Blackwell-native kernel").

    python -m paper_2607_05895_b200.sass_histogram > profiles/r02_sass_ns.txt

Runs on the build box (no GPU needed); reads paper_2607_05895_b200/build/*.o.
"""
import collections
import os
import re
import subprocess
import sys

PKG = os.path.dirname(os.path.abspath(__file__))
KEEP = re.compile(r"^(UTC\w*|LDTM|STTM|UTMA\w*|UBLKCP|SYNCS|HMMA|HGMMA|QGMMA|IGMMA|ELECT|UCGABAR\w*|FFMA|DFMA|LDG|STG|LDS|STS|LDSM|"
                  r"ATOMG|REDG|RED|ATOM|MEMBAR|FENCE|NANOSLEEP|BAR|CCTL|F2FP|LDGSTS)$")


def histogram(obj):
    out = subprocess.run(["cuobjdump", "-sass", obj], stdout=subprocess.PIPE, text=True, check=True).stdout
    fn, hist = None, collections.OrderedDict()
    for line in out.splitlines():
        m = re.search(r"Function : (\S+)", line)
        if m:
            fn = m.group(1)
            hist[fn] = collections.Counter()
            continue
        m = re.match(r"\s+/\*[0-9a-f]{4,}\*/\s+(?:@!?U?P\d+\s+)?([A-Za-z0-9_.]+)", line)
        if m and fn:
            op = m.group(1)
            if KEEP.match(op.split(".")[0]):
                hist[fn][op] += 1
            hist[fn]["(all instructions)"] += 1
    return hist


def demangle(name):
    try:
        return subprocess.run(["c++filt", name], stdout=subprocess.PIPE, text=True).stdout.strip() or name
    except OSError:
        return name


def main():
    objs = sys.argv[1:] or [os.path.join(PKG, "build", f) for f in ("ns_tc.o", "ns_fused.o", "ns_fused2.o", "shampoo.o", "elementwise.o")]
    for obj in objs:
        print("== %s (sm_100a)" % os.path.relpath(obj, os.path.dirname(PKG)))
        for fn, h in histogram(obj).items():
            short = re.sub(r"\(anonymous namespace\)::|mfsdp::", "", demangle(fn))
            print("  %s" % short[:150])
            groups = collections.defaultdict(list)
            for op, n in sorted(h.items()):
                groups[op.split(".")[0]].append("%s x%d" % (op, n))
            for base in sorted(groups):
                print("      " + ", ".join(groups[base]))
        print()


if __name__ == "__main__":
    main()
