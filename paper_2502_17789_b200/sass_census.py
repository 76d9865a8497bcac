"""Counts of the Blackwell-specific SASS mnemonics per kernel instantiation of the in-tree library.

    python -m paper_2502_17789_b200.sass_census > profiles/sass_census_r03.md

Runs `cuobjdump -sass` on libidg_b200.so (no GPU needed) and tabulates, per kernel, the instructions that show
what the build rests on: UTCHMMA (tcgen05.mma), STTM / LDTM (tensor-memory stores and loads), UTCBAR (tcgen05
commit), UTMALDG (TMA tensor loads), MUFU.SIN / MUFU.COS, FHFMA (mixed-precision FMA), FFMA2 (packed fp32)."""
import collections
import os
import re
import subprocess

from paper_2502_17789_b200.build import LIB

MNEMONICS = ("UTCHMMA", "UTCQMMA", "STTM", "LDTM", "UTCBAR", "UTMALDG", "MUFU.SIN", "MUFU.COS", "FHFMA", "FFMA2", "DFMA")


def census(lib=LIB):
    sass = subprocess.run(["cuobjdump", "-sass", lib], capture_output=True, text=True, check=True).stdout
    names = subprocess.run(["cu++filt"], input="\n".join(re.findall(r"Function : (\S+)", sass)), capture_output=True,
                           text=True).stdout.split("\n")
    out, cur, k = collections.OrderedDict(), None, 0
    for line in sass.split("\n"):
        m = re.search(r"Function : (\S+)", line)
        if m:
            cur = names[k] if k < len(names) and names[k] else m.group(1)
            k += 1
            out[cur] = collections.Counter()
            continue
        if cur is None:
            continue
        m = re.search(r"^\s+/\*[0-9a-f]+\*/\s+(?:@!?U?P\d+\s+)?([A-Z0-9_.]+)", line)
        if m:
            op = m.group(1)
            out[cur]["total"] += 1
            for mn in MNEMONICS:
                if op == mn or op.startswith(mn + "."):
                    out[cur][mn] += 1
    return out


def main():
    c = census()
    print("# SASS census of libidg_b200.so (round 3)\n")
    print("Command: `python -m paper_2502_17789_b200.sass_census` (= `cuobjdump -sass paper_2502_17789_b200/libidg_b200.so`,")
    print("mnemonics counted per kernel; built by `python -m paper_2502_17789_b200.build`, nvcc 12.9, sm_100a).\n")
    print("| kernel | SASS instructions | " + " | ".join(MNEMONICS) + " |")
    print("|---|---|" + "---|" * len(MNEMONICS))
    tot = collections.Counter()
    for name, cnt in c.items():
        short = re.sub(r"\((?:int|bool)\)", "", name)
        short = re.sub(r"^void idg::(?:\(anonymous namespace\)|<unnamed>)::", "", short)
        short = re.sub(r"\(.*$", "", short)
        print(f"| `{short}` | {cnt['total']} | " + " | ".join(str(cnt[m]) if cnt[m] else "" for m in MNEMONICS) + " |")
        tot.update(cnt)
    print(f"| **all {len(c)} kernels** | {tot['total']} | " + " | ".join(str(tot[m]) for m in MNEMONICS) + " |")
    print("\nUTCHMMA = `tcgen05.mma` (kind::f16 / kind::tf32), STTM / LDTM = `tcgen05.st` / `tcgen05.ld` (tensor memory),")
    print("UTCBAR = `tcgen05.commit`, UTMALDG = `cp.async.bulk.tensor` (TMA, the adder's patch boxes).  The rotating gridder")
    print("instantiations (last template argument 1) carry one `__sincosf` per 8 channels, the per-pair ones (0) one per pair.")


if __name__ == "__main__":
    main()
