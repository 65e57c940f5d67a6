"""SASS / resource digest of librqr.so: per kernel, the instruction counts that show which hardware paths execute.

  python -m paper_2309_05868_b200.sass_digest > profiles/r2_sass_digest.md

Runs `cuobjdump -sass` on the built library (no GPU needed) and reads the registers / spills from the build's ptxas log
(paper_2309_05868_b200/build/ptxas.log, written by build.py with -Xptxas -v).  Counts are STATIC instruction counts
of the kernel's SASS (unrolled loop bodies count once each), not executed instructions.
"""
from __future__ import annotations

import collections
import os
import re
import subprocess
import sys

from . import build

HERE = os.path.dirname(os.path.abspath(__file__))


def main():
    lib = build.build_lib()
    txt = subprocess.run(["cuobjdump", "-sass", lib], capture_output=True, text=True, check=True).stdout
    funcs = re.split(r"\n\s*Function : ", txt)[1:]
    log = open(os.path.join(HERE, "build", "ptxas.log")).read()
    regs = {}
    for m in re.finditer(r"Compiling entry function '([^']+)' for 'sm_100a'\n.*?\n\s*(\d+) bytes stack frame, (\d+) bytes spill "
                         r"stores, (\d+) bytes spill loads\n.*?Used (\d+) registers", log):
        regs[m.group(1)] = (int(m.group(5)), int(m.group(3)) + int(m.group(4)))
    names = [f.split("\n")[0].strip() for f in funcs]
    dem = subprocess.run(["c++filt"] + names, capture_output=True, text=True).stdout.strip().split("\n")
    rows = []
    absent = collections.Counter()
    for f, nm, d in zip(funcs, names, dem):
        ops = collections.Counter()
        for line in f.split("\n"):
            m = re.match(r"\s+/\*[0-9a-f]{4,}\*/\s+(?:@!?U?P\d+\s+)?([A-Z0-9_]+)", line)
            if m:
                ops[m.group(1)] += 1
        for op in ("UTCMMA", "UTCHMMA", "UTCQMMA", "UTCIMMA", "LDTM", "STTM", "UTMALDG", "UTMASTG", "HMMA", "IMMA", "QMMA"):
            absent[op] += ops[op]
        d = re.sub(r"\(.*", "", d).replace("void ", "")
        r = regs.get(nm, (0, 0))
        rows.append((d, sum(ops.values()), ops["DMMA"], ops["UBLKCP"], ops["UBLKRED"], ops["DFMA"] + ops["DMUL"] + ops["DADD"],
                     ops["LDS"] + ops["STS"], ops["RED"] + ops["ATOM"] + ops["ATOMG"] + ops["ATOMS"], ops["SYNCS"],
                     ops["MATCH"], r[0], r[1]))
    rows.sort()
    out = sys.stdout
    out.write("# SASS / resource digest of librqr.so (sm_100a), round 2\n\n")
    out.write("Command (no GPU needed; counts are static SASS instructions per kernel, registers and spill bytes from "
              "`-Xptxas -v`):\n\n```\npython -m paper_2309_05868_b200.sass_digest > profiles/r2_sass_digest.md\n```\n\n")
    out.write("What the columns show.  `DMMA` = `mma.sync.m8n8k4.f64` (the FP64 tensor path: `DMMA.8x8x4`); `UBLKCP` = "
              "`cp.async.bulk` global -> shared (the bulk-copy engine, TMA without a tensor map); `UBLKRED` = "
              "`cp.reduce.async.bulk ... add.f64` shared -> global (bulk reduction in the L2, the streaming CountSketch); "
              "`SYNCS` = mbarrier operations; `MATCH` = `match.any` (stable ranking of the A0 radix sort).\n\n")
    out.write("**Absent on purpose** (counts over the whole library): " + ", ".join("%s %d" % kv for kv in sorted(absent.items()))
              + ".  `tcgen05.mma` (SASS `UTC*MMA`) has no FP64 kind and the accumulators of an FP64 path cannot live in "
              "tensor memory (`LDTM` / `STTM`), so the Blackwell tensor path for this FP64 method is the warp-level DMMA "
              "with register accumulators.  `UTMALDG` (tensor-map TMA) is not used: V is a row-major matrix with a "
              "caller-chosen leading dimension, a row block is one contiguous range when ld = n, and the plain bulk copy "
              "needs no per-call descriptor (DESIGN.md section 8).\n\n")
    out.write("| kernel | SASS instr | DMMA | UBLKCP | UBLKRED | DFMA+DMUL+DADD | LDS+STS | RED/ATOM | SYNCS | MATCH | regs | spill B |\n")
    out.write("|---|---|---|---|---|---|---|---|---|---|---|---|\n")
    for r in rows:
        out.write("| `%s` | %d | %d | %d | %d | %d | %d | %d | %d | %d | %d | %d |\n" % r)


if __name__ == "__main__":
    main()
