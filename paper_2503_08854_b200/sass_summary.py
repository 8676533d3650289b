"""SASS summary of the built kernels: `python -m paper_2503_08854_b200.sass_summary > profiles/<round>_sass.md`.

For every kernel of the object files under csrc/ (built by _build.py with -lineinfo): registers, shared memory and
spills from ptxas (csrc/ptxas.log), and a static instruction histogram from `cuobjdump -sass`: FP64-pipe
instructions (DFMA, DADD, DMUL, DSETP, ...), MUFU (the reciprocal / rsqrt seeds), warp votes and shuffles, global
and shared memory accesses, the TMA bulk copies (UBLKCP) and mbarrier operations (SYNCS) that prove the
Blackwell-native staging of kernel 1.  Static counts: how often an instruction EXECUTES is ncu's business
(k1_counts.py); this file shows what the binary contains.
"""
from __future__ import annotations

import collections
import os
import re
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
CLASSES = [
    ("fp64", re.compile(r"^(DFMA|DADD|DMUL|DSETP|DMNMX|F2F\.F64|I2F\.F64|F2I.*F64|D2|MUFU\.R(CP|SQ)64H)")),
    ("mufu", re.compile(r"^MUFU")),
    ("vote/shfl", re.compile(r"^(VOTE|SHFL|REDUX|MATCH)")),
    ("ldg/stg", re.compile(r"^(LDG|STG|LD\.|ST\.|RED|ATOMG|ATOM)")),
    ("lds/sts", re.compile(r"^(LDS|STS|ATOMS)")),
    ("tma bulk (UBLKCP)", re.compile(r"^UBLKCP")),
    ("mbarrier (SYNCS)", re.compile(r"^SYNCS")),
    ("branch", re.compile(r"^(BRA|BSSY|BSYNC|EXIT|CALL|RET|WARPSYNC|BAR)")),
]


def demangle(name: str) -> str:
    try:
        return subprocess.run(["cu++filt", name], capture_output=True, text=True).stdout.strip() or name
    except Exception:
        return name


def kernels_of(obj: str):
    out = subprocess.run(["cuobjdump", "-sass", obj], capture_output=True, text=True).stdout
    cur, res = None, collections.OrderedDict()
    for line in out.splitlines():
        m = re.search(r"Function : (\S+)", line)
        if m:
            cur = m.group(1)
            res[cur] = []
            continue
        m = re.match(r"\s+/\*[0-9a-f]{4}\*/\s+(.*?);", line)
        if m and cur:
            ins = m.group(1).strip()
            ins = re.sub(r"^@!?U?P\d+\s+", "", ins)
            res[cur].append(ins.split()[0])
    return res


def ptxas_info():
    info, cur = {}, None
    try:
        lines = open(os.path.join(CSRC, "ptxas.log")).read().splitlines()
    except Exception:
        return info
    for ln in lines:
        m = re.search(r"Compiling entry function '(\S+)'", ln)
        if m:
            cur = m.group(1)
            info[cur] = {"spill": "0/0"}
        m = re.search(r"(\d+) bytes spill stores, (\d+) bytes spill loads", ln)
        if m and cur:
            info[cur]["spill"] = "%s/%s" % (m.group(1), m.group(2))
        m = re.search(r"Used (\d+) registers", ln)
        if m and cur:
            info[cur]["regs"] = m.group(1)
            sm = re.search(r"(\d+) bytes smem", ln)
            info[cur]["smem"] = sm.group(1) if sm else "0 (+dynamic)"
    return info


def main():
    px = ptxas_info()
    print("| kernel | regs | static smem B | spill st/ld B | SASS instr. | " + " | ".join(c for c, _ in CLASSES) + " |")
    print("|---|---|---|---|---|" + "---|" * len(CLASSES))
    for obj in sorted(f for f in os.listdir(CSRC) if f.endswith(".o") and not f.endswith(".bounds.o")):
        for name, ins in kernels_of(os.path.join(CSRC, obj)).items():
            counts = []
            for _c, rx in CLASSES:
                counts.append(sum(1 for i in ins if rx.match(i)))
            p = px.get(name, {})
            full = demangle(name).replace("void ", "").replace("dt::", "").replace("(anonymous namespace)::", "").replace("<unnamed>::", "")
            head = full.split("(GatherParams")[0].split("(PropagateParams")[0]
            short = head[:head.rfind(">") + 1] if "<" in head else head.split("(")[0]
            print("| `%s` | %s | %s | %s | %d | %s |" % (short, p.get("regs", "?"), p.get("smem", "?"), p.get("spill", "?"),
                                                       len(ins), " | ".join(str(c) for c in counts)))


if __name__ == "__main__":
    sys.exit(main())
