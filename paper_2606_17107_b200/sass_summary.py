"""Per-kernel SASS / resource summary of the in-tree libkvr.so (what `profiles/*_sass_summary.md` is made with).

    python -m paper_2606_17107_b200.sass_summary            # markdown table on stdout

Counts, per kernel instantiation in the cubin: instructions, the mnemonics that prove the data path (UBLKCP = 1-D bulk
TMA, UTMALDG / UTMASTG = tensor-map TMA, SYNCS = mbarrier, UTC*MMA / LDTM / STTM = tcgen05 tensor cores and TMEM,
STG.E.128 / LDS.128 = 16-byte vector accesses, F2FP..E4M3 = fp8 conversions, DFMA = the fp64 angle table), and from
`cuobjdump -res-usage`: registers per thread, static shared memory, local-memory stack (spills).
"""
import os
import re
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(HERE, "libkvr.so")
PATTERNS = [("UBLKCP", r"\bUBLKCP"), ("UTMALDG", r"\bUTMALDG"), ("UTMASTG", r"\bUTMASTG"), ("UTMAPF", r"\bUTMAPF"),
            ("SYNCS", r"\bSYNCS"), ("UTCHMMA", r"\bUTC\w*MMA"), ("LDTM", r"\bLDTM"), ("STTM", r"\bSTTM"),
            ("UTCBAR", r"\bUTCBAR"), ("STG.128", r"\bSTG\.E(?:\.\w+)*\.128"), ("LDS.128", r"\bLDS(?:\.\w+)*\.128"),
            ("F2FP.E4M3", r"\bF2FP\S*E4M3"), ("DFMA", r"\bDFMA"), ("FFMA", r"\bFFMA"), ("MUFU", r"\bMUFU")]


def demangle(names):
    out = subprocess.run(["c++filt"], input="\n".join(names), capture_output=True, text=True, check=True).stdout
    return [re.sub(r"\(.*", "", d).replace("void ", "") for d in out.splitlines()]


def main():
    cuobjdump = os.environ.get("CUOBJDUMP", "/usr/local/cuda/bin/cuobjdump")
    sass = subprocess.run([cuobjdump, "-sass", LIB], capture_output=True, text=True, check=True).stdout
    res = subprocess.run([cuobjdump, "-res-usage", LIB], capture_output=True, text=True, check=True).stdout
    usage = {}
    for m in re.finditer(r"Function (\S+):\s*\n\s*(.*)", res):
        usage[m.group(1)] = {k: int(v) for k, v in re.findall(r"(REG|STACK|SHARED|LOCAL):(\d+)", m.group(2))}
    parts = re.split(r"\n\s*Function : ", sass)[1:]
    names = [p.split("\n", 1)[0].strip() for p in parts]
    rows = []
    for name, dem, body in zip(names, demangle(names), parts):
        n = len(re.findall(r"^\s+/\*[0-9a-f]{4,}\*/", body, flags=re.M))
        u = usage.get(name, {})
        rows.append([dem, n, u.get("REG"), u.get("STACK"), u.get("SHARED")] + [len(re.findall(p, body)) for _, p in PATTERNS])
    head = ["kernel", "instr", "regs", "stack B", "static smem B"] + [k for k, _ in PATTERNS]
    print("| " + " | ".join(head) + " |")
    print("|" + "---|" * len(head))
    for r in sorted(rows, key=lambda r: r[0]):
        print("| `" + str(r[0]) + "` | " + " | ".join(str(x) for x in r[1:]) + " |")
    return 0


if __name__ == "__main__":
    sys.exit(main())
