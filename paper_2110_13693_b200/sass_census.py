"""Opcode census of the built libwhp.so: for every kernel, the number of SASS instructions and how
many of them are the Blackwell / Hopper-class operations the design relies on (TMA tile loads and
stores, bulk copies, mbarrier operations, cp.async, the fused add-min of the next-fit chain, fp64
arithmetic, warp reductions). Evidence only — nothing at run time depends on it.

    python -m paper_2110_13693_b200.sass_census            # markdown table on stdout
"""
import collections
import re
import subprocess
import sys

from . import build

CLASSES = [("UTMALDG", r"^UTMALDG"), ("UTMASTG", r"^UTMASTG"), ("UBLKCP", r"^UBLKCP"),
           ("SYNCS", r"^SYNCS"), ("LDGSTS", r"^LDGSTS"), ("VIADDMNMX", r"^VIADDMNMX"),
           ("DADD/DMUL", r"^(DADD|DMUL)"), ("DFMA", r"^DFMA"), ("REDUX", r"^REDUX"),
           ("SHFL", r"^SHFL"), ("VOTE/MATCH", r"^(VOTE|MATCH)"), ("LDS", r"^LDS"), ("STS", r"^STS"),
           ("LDG", r"^LDG(?!STS)"), ("ATOM/RED", r"^(ATOM|RED)"), ("tensor (UTC*/HMMA)", r"^(UTC|HMMA)")]


def demangle(names):
    try:
        out = subprocess.run(["c++filt"], input="\n".join(names), capture_output=True, text=True).stdout
        return out.splitlines()
    except OSError:
        return names


def kernel_name(demangled):
    """`void (anonymous namespace)::k<(bool)1, 7>(args...)` -> `k<1, 7>`"""
    n = demangled.replace("(anonymous namespace)::", "").replace("void ", "")
    depth = 0
    for i, ch in enumerate(n):
        depth += ch == "<"
        depth -= ch == ">"
        if ch == "(" and depth == 0 and not n[:i].endswith("<"):
            n = n[:i]
            break
    return re.sub(r"\((bool|int)\)", "", n)


def census(so_path):
    sass = subprocess.run(["cuobjdump", "-sass", so_path], capture_output=True, text=True).stdout
    counts, fn = collections.OrderedDict(), None
    for line in sass.splitlines():
        m = re.search(r"Function : (\S+)", line)
        if m:
            fn = m.group(1)
            counts[fn] = collections.Counter()
            continue
        m = re.match(r"\s+/\*[0-9a-f]{4,}\*/\s+(@!?U?P\d+\s+)?([A-Z0-9_.]+)", line)
        if m and fn:
            op = m.group(2)
            counts[fn]["total"] += 1
            for name, pat in CLASSES:
                if re.match(pat, op):
                    counts[fn][name] += 1
    return counts


def main():
    so = build.build()
    counts = census(so)
    names = demangle(list(counts))
    short = [kernel_name(n) for n in names]
    print("| kernel | SASS instructions | " + " | ".join(n for n, _ in CLASSES) + " |")
    print("|---|---|" + "---|" * len(CLASSES))
    for (fn, c), s in sorted(zip(counts.items(), short), key=lambda x: x[1]):
        print(f"| `{s}` | {c['total']} | " + " | ".join(str(c[n]) for n, _ in CLASSES) + " |")
    return 0


if __name__ == "__main__":
    sys.exit(main())
