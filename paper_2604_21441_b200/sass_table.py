"""Instruction-mix table of the built library, per kernel: `python -m paper_2604_21441_b200.sass_table > profiles/rNN_sass_table.md`.

Disassembles libnnp_b200.so with `cuobjdump -sass` and counts the SASS mnemonics that show what each kernel is made of
(B200_PROFILING.md "What proves a Blackwell-native kernel": tcgen05.mma -> UTC*MMA, tcgen05.ld/st -> LDTM/STTM,
cp.async.bulk -> UBLKCP, packed fp32 -> FFMA2/FMUL2/FADD2; HMMA would be the legacy mma.sync path).  Static counts of the
binary, not executed instructions.  Runs on the CPU box (no GPU needed)."""
import collections
import os
import re
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(HERE, "libnnp_b200.so")
COLS = ["UTCHMMA", "UTCBAR", "LDTM", "STTM", "UBLKCP", "SYNCS", "HMMA", "FFMA2", "FMUL2", "FADD2", "FFMA", "MUFU", "DFMA",
        "LDG", "STG", "LDS", "STS", "RED", "ATOM", "SHFL", "VOTE", "BAR"]


def demangle(names):
    try:
        out = subprocess.run(["c++filt"], input="\n".join(names), capture_output=True, text=True, check=True).stdout.splitlines()
        return dict(zip(names, out))
    except Exception:
        return {n: n for n in names}


def main():
    cuobjdump = os.environ.get("CUOBJDUMP", "/usr/local/cuda/bin/cuobjdump")
    sass = subprocess.run([cuobjdump, "-sass", LIB], capture_output=True, text=True, check=True).stdout
    counts, total, cur = collections.OrderedDict(), {}, None
    for line in sass.splitlines():
        m = re.match(r"\s*Function : (\S+)", line)
        if m:
            cur = m.group(1)
            counts[cur] = collections.Counter()
            total[cur] = 0
            continue
        m = re.match(r"\s*/\*[0-9a-f]{4,}\*/\s+(?:@!?U?P\d+\s+)?([A-Z0-9_]+)", line)
        if m and cur:
            op = m.group(1)
            total[cur] += 1
            for c in COLS:
                if op == c or (c in ("LDG", "STG", "LDS", "STS", "RED", "ATOM", "BAR", "MUFU", "SHFL", "VOTE", "SYNCS") and op.startswith(c)):
                    counts[cur][c] += 1
                    break
    names = demangle(list(counts))
    print("# SASS instruction mix per kernel (static counts, `cuobjdump -sass libnnp_b200.so`)\n")
    print("Command: `python -m paper_2604_21441_b200.build && python -m paper_2604_21441_b200.sass_table` (CPU box; sm_100a).\n")
    print("| kernel | instructions | " + " | ".join(COLS) + " |")
    print("|---|---|" + "---|" * len(COLS))
    for f in counts:
        short = re.sub(r"\(.*", "", names[f]).replace("void ", "").replace("nnp::", "")
        print(f"| `{short}` | {total[f]} | " + " | ".join(str(counts[f][c]) if counts[f][c] else "" for c in COLS) + " |")
    tot = collections.Counter()
    for f in counts:
        tot.update(counts[f])
    print("\nWhole library: " + ", ".join(f"{c} {tot[c]}" for c in COLS if tot[c]) + ".")
    if tot["HMMA"]:
        print("\nWARNING: legacy HMMA (mma.sync) instructions present.")


if __name__ == "__main__":
    sys.exit(main())
