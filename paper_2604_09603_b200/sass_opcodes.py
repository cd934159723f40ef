"""Per-kernel count of the SASS opcodes that prove the Blackwell-native paths (B200_PROFILING.md):
tcgen05.mma -> UTC*MMA, tcgen05.ld / st -> LDTM / STTM, TMA -> UTMALDG / UBLKCP, tcgen05.commit -> UTCBAR,
packed fp32 -> FFMA2 / FADD2; HMMA would be the legacy mma.sync path.

    python -m paper_2604_09603_b200.sass_opcodes            # markdown table on stdout (profiles/r02_sass_opcodes.md)
"""
import collections
import os
import re
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
OPS = ["UTCHMMA", "UTCBAR", "LDTM", "STTM", "UTMALDG", "UTMAPF", "UBLKCP", "SYNCS", "USETMAXREG", "MUFU.EX2", "FFMA2", "FADD2",
       "F2FP", "HMMA", "LDG", "STG", "ATOMS", "SHFL"]


def main():
    lib = os.path.join(HERE, "libecho.so")
    sass = subprocess.run(["cuobjdump", "-sass", lib], capture_output=True, text=True, check=True).stdout
    counts, kernel = collections.OrderedDict(), None
    for ln in sass.splitlines():
        m = re.search(r"Function : (\S+)", ln)
        if m:
            name = subprocess.run(["cu++filt", m.group(1)], capture_output=True, text=True).stdout.strip() or m.group(1)
            kernel = re.sub(r"\(.*", "", name).replace("(anonymous namespace)::", "")
            counts[kernel] = collections.Counter()
            continue
        m = re.match(r"\s+/\*[0-9a-f]+\*/\s+(?:@!?U?P\d+\s+)?([A-Z0-9_.]+)", ln)
        if m and kernel:
            op = m.group(1)
            for o in OPS:
                if op == o or op.startswith(o + ".") or (o == "MUFU.EX2" and op.startswith("MUFU.EX2")):
                    counts[kernel][o] += 1
    print("| kernel | " + " | ".join(OPS) + " |")
    print("|---|" + "---|" * len(OPS))
    for k, c in counts.items():
        print(f"| `{k}` | " + " | ".join(str(c[o]) if c[o] else "" for o in OPS) + " |")


if __name__ == "__main__":
    sys.exit(main())
