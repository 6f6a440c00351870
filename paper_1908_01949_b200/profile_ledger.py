#!/usr/bin/env python3
"""Issue-slot ledger of a kernel: executed warp instructions per source line and per opcode.

Joins the per-instruction execution counts of an Nsight Compute report (`ncu -i REPORT --page source --csv`, SASS view)
with the source-line information of the very object the report was taken from (`nvdisasm --print-line-info-inline`,
needs -lineinfo at compile time), instruction by instruction, and prints
  * executed warp instructions per source line of the kernel file (inlined code is charged to the line of the kernel
    that called it), with the average number of active lanes,
  * the same per named region (line ranges given on the command line),
  * the opcode histogram, and the fp32 flops the executed instructions carry (thread level, packed forms included).
Divide by the number of loop iterations (the count of a line that executes once per iteration) to get instructions per
warp-step.  Used for profiles/r2_scan_ledger_*.md.

    python -m paper_1908_01949_b200.profile_ledger REPORT.ncu-rep OBJECT.o KERNEL_SUBSTRING [--per N] [--region NAME:FIRST-LAST ...]
                                                   [--listing OUT.txt]
--listing writes the SASS itself, one line per instruction that executes at least 0.02 times per unit: offset, executions
per unit, average active lanes, the instruction, and the source line it comes from.
"""
import collections
import csv
import os
import re
import subprocess
import sys
import tempfile


# fp32 flops per THREAD instruction (ncu's sass_thread_inst_executed_op_f* metrics do not count the packed forms)
FP32_FLOPS = {"FFMA": 2, "FMUL": 1, "FADD": 1, "FFMA2": 4, "FMUL2": 2, "FADD2": 2}


def disassemble(obj, kernel):
    d = tempfile.mkdtemp()
    subprocess.check_call(f"cd {d} && cuobjdump -xelf all {os.path.abspath(obj)} > /dev/null", shell=True)
    cub = [f for f in os.listdir(d) if f.endswith(".cubin")][0]
    dis = subprocess.check_output(["nvdisasm", "--print-line-info-inline", "-c", os.path.join(d, cub)], text=True).splitlines()
    start = next(i for i, l in enumerate(dis) if l.startswith(".text.") and kernel in l)
    insts, cur, pend = [], [], []
    for l in dis[start + 1:]:
        if l.startswith(".text.") and insts:
            break
        m = re.match(r'\s*//## File "([^"]+)", line (\d+)(?: inlined at "([^"]+)", line (\d+))?', l)
        if m:
            pend.append((os.path.basename(m.group(1)), int(m.group(2)), m.group(3) and os.path.basename(m.group(3)),
                         m.group(4) and int(m.group(4))))
            continue
        m = re.match(r"\s*/\*([0-9a-f]{4,})\*/\s+(.*?);", l)
        if m:
            if pend:
                cur, pend = pend, []
            insts.append((m.group(2).strip(), cur))
    return insts


def main(argv):
    rep, obj, kernel = argv[:3]
    per = float(argv[argv.index("--per") + 1]) if "--per" in argv else None
    regions = []
    for i, a in enumerate(argv):
        if a == "--region":
            name, rng = argv[i + 1].rsplit(":", 1)
            lo, hi = rng.split("-")
            regions.append((name, int(lo), int(hi)))
    insts = disassemble(obj, kernel)
    rows = list(csv.reader(subprocess.check_output(["ncu", "-i", rep, "--page", "source", "--csv"], text=True,
                                                   stderr=subprocess.DEVNULL).splitlines()))
    blk = next(j for j, r in enumerate(rows) if r and r[0] == "Kernel Name")
    hdr = rows[blk + 1]
    ci, ct = hdr.index("Instructions Executed"), hdr.index("Thread Instructions Executed")
    data = []
    for r in rows[blk + 2:]:
        if not r or r[0] == "Kernel Name":
            break
        data.append(r)
    assert len(data) == len(insts), f"{len(insts)} SASS instructions in the object, {len(data)} in the report: not the same build"
    by_line, thr_line, by_op = collections.Counter(), collections.Counter(), collections.Counter()
    total = 0
    flops = 0
    listing = open(argv[argv.index("--listing") + 1], "w") if "--listing" in argv else None
    listed = 0
    for k, ((text, chain), r) in enumerate(zip(insts, data)):
        cnt, thr = int(r[ci]), int(r[ct])
        total += cnt
        outer = None
        if chain:
            last = chain[-1]
            outer = (last[2], last[3]) if last[2] else (last[0], last[1])
        if listing and per and cnt >= 0.02 * per:
            inner = (chain[0][0], chain[0][1]) if chain else None
            where = "" if outer is None else f"{outer[0]}:{outer[1]}" + (f" <- {inner[0]}:{inner[1]}" if inner != outer else "")
            listing.write(f"/*{k * 16:05x}*/ {cnt / per:7.3f} {thr / max(cnt, 1):5.1f}  {text:72s} // {where}\n")
            listed += cnt
        by_line[outer] += cnt; thr_line[outer] += thr
        op = text.split()[1] if text.startswith("@") else text.split()[0]
        by_op[op.split(".")[0]] += cnt
        flops += thr * FP32_FLOPS.get(op.split(".")[0], 0)
    if listing:
        listing.write(f"# listed instructions: {listed / per:.1f} of {total / per:.1f} executed warp instructions per unit\n")
        listing.close()
    unit = (lambda c: f"{c / per:8.2f}") if per else (lambda c: f"{c:14d}")
    print(f"kernel {kernel}: {len(insts)} SASS instructions, {total} executed warp instructions" +
          (f", {total / per:.1f} per unit ({per:.0f} units)" if per else ""))
    print(f"fp32 flops executed (thread level; FFMA 2, FMUL / FADD 1, FFMA2 4, FMUL2 / FADD2 2): {flops}" +
          (f", {flops / per:.1f} per unit" if per else ""))
    if regions:
        print("\nper region" + (" (instructions per unit)" if per else ""))
        for name, lo, hi in regions:
            c = sum(v for k, v in by_line.items() if k and lo <= k[1] <= hi)
            print(f"  {name:34s} {unit(c)} {100 * c / total:6.2f} %")
    print("\nper source line (>= 0.3 % of the total)" + (" (instructions per unit)" if per else ""))
    for k in sorted(by_line, key=lambda x: (x or ("", 0))):
        c = by_line[k]
        if c * 1000 >= 3 * total:
            print(f"  {str(k):30s} {unit(c)} {100 * c / total:6.2f} %  lanes {thr_line[k] / max(c, 1):5.1f}")
    print("\nper opcode" + (" (instructions per unit)" if per else ""))
    for o, c in by_op.most_common(28):
        print(f"  {o:10s} {unit(c)} {100 * c / total:6.2f} %")


if __name__ == "__main__":
    main(sys.argv[1:])
