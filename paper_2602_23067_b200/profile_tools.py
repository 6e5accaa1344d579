"""Turns ncu reports and the built library into the text summaries kept under profiles/ (no GPU needed).

    python -m paper_2602_23067_b200.profile_tools summary <report.ncu-rep> <out.txt> "<command that made the report>"
    python -m paper_2602_23067_b200.profile_tools mix     <report.ncu-rep> <out.json> [<key>] "<command>"
    python -m paper_2602_23067_b200.profile_tools static  <kernel name regex> <out.txt>
    python -m paper_2602_23067_b200.profile_tools launches <ncu launch log.csv> <out.csv> "<command>"

summary  the counters DESIGN.md section 6 quotes, from `ncu -i <report> --page raw --csv`.
mix      the EXECUTED instruction mix of the row loop per warp-row (32 blocks), from the per-instruction counts of
         `ncu -i <report> --page source --csv` (needs a capture made with --import-source on / -lineinfo):
         shared-memory reads by width, global loads and stores, and thread-instructions per pipe.  bench.py builds
         the shared-memory-pipe roofline from this file instead of from a typed-in formula (SURVEY.md 8(d):
         "N_x = per-block thread-instruction counts ... of the shipped kernel, cross-checked with ncu").
static   per-opcode counts of the kernel's hot loop (the backward branch that encloses the most LDS) from
         `cuobjdump -sass` of the library: what the binary contains, all paths of the loop together.
"""
from __future__ import annotations

import collections
import csv
import json
import os
import re
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(HERE, "libb200gcm.so")

RAW_METRICS = (
    r"gpu__time_duration.sum$|sm__cycles_elapsed.avg$|sm__cycles_elapsed.avg.per_second|launch__registers_per_thread$|"
    r"launch__shared_mem_per_block_dynamic|launch__occupancy_limit_shared_mem|dram__bytes_read.sum$|dram__bytes_write.sum$|"
    r"gpu__dram_throughput.avg.pct|sm__throughput.avg.pct|smsp__inst_executed.sum$|smsp__issue_active.avg.pct|"
    r"sm__inst_executed_pipe_(alu|lsu|fma|uniform).avg.pct_of_peak_sustained_active|l1tex__data_pipe_lsu_wavefronts.avg.pct|"
    r"l1tex__data_pipe_lsu_wavefronts_mem_shared.sum$|l1tex__data_pipe_lsu_wavefronts_mem_shared_op_(ld|st).sum$|"
    r"l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum$|lts__t_bytes.sum$|"
    r"stalled_(short_scoreboard|mio_throttle|long_scoreboard|math_pipe_throttle|not_selected|wait|barrier)_per_issue_active.ratio|"
    r"sm__warps_active.avg.pct|sm__pipe_tensor_cycles_active.avg.pct_of_peak_sustained_(elapsed|active)$|"
    r"sm__inst_executed_pipe_tensor|smsp__inst_executed_pipe_(uniform|tmem)")

ALU = {"LOP3", "PRMT", "SHF", "IADD3", "IADD", "ISETP", "SEL", "LEA", "VIADD", "PLOP3", "MOV", "IABS", "IMNMX", "VIMNMX",
       "POPC", "FLO", "BREV", "SGXT", "BMSK", "LOP", "R2P", "P2R", "CS2R", "I2FP", "FSETP", "FMNMX", "VABSDIFF"}
FMA = {"IMAD", "FFMA", "FMUL", "FADD", "HFMA2", "IDP", "IMUL"}
LSU = {"LDS", "STS", "LDG", "STG", "LD", "ST", "LDL", "STL", "ATOM", "ATOMG", "ATOMS", "RED", "LDSM", "SHFL", "MEMBAR",
       "CCTL", "FENCE", "ERRBAR", "LDGSTS", "UBLKCP", "SYNCS"}


def opcode(sass: str) -> str:
    t = re.sub(r"^\s*@!?U?P\d+\s+", "", sass.strip())
    return t.split()[0].rstrip(";") if t else ""


def pipe_of(op: str) -> str:
    base = op.split(".")[0]
    if base.startswith("U") and base not in ("UBLKCP",):
        return "uniform"
    if base in LSU:
        return "lsu"
    if base in FMA:
        return "fma"
    if base in ALU:
        return "alu"
    if base in ("BRA", "BSSY", "BSYNC", "CALL", "RET", "EXIT", "BAR", "WARPSYNC", "BREAK", "NANOSLEEP", "YIELD", "JMP", "BRX"):
        return "control"
    return "other"


def _ncu_page(report: str, page: str) -> str:
    return subprocess.run(["ncu", "-i", report, "--page", page, "--csv"], capture_output=True, text=True, check=True).stdout


def summary(report: str, out: str, command: str) -> None:
    rows = list(csv.reader(_ncu_page(report, "raw").splitlines()))
    hdr, units = rows[0], rows[1]
    pat = re.compile(RAW_METRICS)
    with open(out, "w") as f:
        f.write("# ncu --set full summary (values of the profiled launches)\n# command: %s\n"
                "# report read with: ncu -i <report>.ncu-rep --page raw --csv  (python -m paper_2602_23067_b200.profile_tools summary)\n\n" % command)
        for vals in rows[2:]:
            for h, u, v in zip(hdr, units, vals):
                if h in ("Kernel Name", "Block Size", "Grid Size") or pat.search(h):
                    f.write("%-90s %-16s %s\n" % (h, u, v))
            f.write("\n")


def _library_fingerprint() -> dict:
    """Size and SHA-256 of the built libb200gcm.so next to this file: the binary the report was captured from (the
    capture and this step run on the same build).  bench.py compares it with the library it has loaded."""
    import hashlib
    lib = os.path.join(os.path.dirname(os.path.abspath(__file__)), "libb200gcm.so")
    data = open(lib, "rb").read()
    return {"bytes": len(data), "sha256": hashlib.sha256(data).hexdigest()}


def mix(report: str, out: str, key: str, command: str) -> None:
    """Per-warp-row executed instruction mix of the FIRST kernel in the report."""
    text = _ncu_page(report, "source")
    lines = text.splitlines()
    kernel = ""
    start = 0
    for i, l in enumerate(lines):
        if l.startswith('"Kernel Name"'):
            kernel = next(csv.reader([l]))[1]
        if l.startswith('"Address"'):
            start = i
            break
    rows = []
    hdr = next(csv.reader([lines[start]]))
    for l in lines[start + 1:]:
        if l.startswith('"Kernel Name"'):
            break                                             # next launch of the report
        r = next(csv.reader([l]))
        if len(r) == len(hdr):
            rows.append(dict(zip(hdr, r)))
    def num(r, k):
        try:
            return float(r.get(k, "0") or 0)
        except ValueError:
            return 0.0
    by_op = collections.Counter()
    by_pipe = collections.Counter()
    thread_by_pipe = collections.Counter()
    wf_shared = wf_shared_ideal = 0.0
    total = 0.0
    issued = 0.0
    for r in rows:
        op = opcode(r["Source"])
        # predicated-on thread instructions / 32: a warp instruction whose threads are all predicated off (the unused
        # one of two alternative loads, say) is issued but moves nothing; per block = per thread
        n = num(r, "Predicated-On Thread Instructions Executed") / 32.0
        issued += num(r, "Instructions Executed")
        if not op or n == 0:
            continue
        by_op[op] += n
        p = pipe_of(op)
        by_pipe[p] += n
        thread_by_pipe[p] += num(r, "Thread Instructions Executed")
        total += n
        wf_shared += num(r, "L1 Wavefronts Shared")
        wf_shared_ideal += num(r, "L1 Wavefronts Shared Ideal")
    lds128 = sum(v for k, v in by_op.items() if k.startswith("LDS") and ".128" in k)
    lds64 = sum(v for k, v in by_op.items() if k.startswith("LDS") and ".64" in k)
    lds32 = sum(v for k, v in by_op.items() if k.startswith("LDS")) - lds128 - lds64
    ldg128 = sum(v for k, v in by_op.items() if k.startswith("LDG") and ".128" in k)
    stg128 = sum(v for k, v in by_op.items() if k.startswith("STG") and ".128" in k)
    sts128 = sum(v for k, v in by_op.items() if k.startswith("STS") and ".128" in k)
    # every shared-memory wavefront of the launch, whoever caused it: the instructions above, bank conflicts, and the
    # tensor core's reads of its B operand (gcm_tc2 / gcm_tc: they show up in ncu as "bank conflict" wavefronts)
    wf_total = 0.0
    raw = list(csv.reader(_ncu_page(report, "raw").splitlines()))
    if len(raw) > 2 and "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum" in raw[0]:
        try:
            wf_total = float(raw[2][raw[0].index("l1tex__data_pipe_lsu_wavefronts_mem_shared.sum")])
        except ValueError:
            wf_total = 0.0
    # the launch's executed warp instructions from the hardware counter (the source page's per-line counts of the helper
    # warps' polling loops are sampled differently and do not add up to it: use this one for issue-rate arithmetic)
    inst_executed = 0.0
    if len(raw) > 2 and "smsp__inst_executed.sum" in raw[0]:
        try:
            inst_executed = float(raw[2][raw[0].index("smsp__inst_executed.sum")])
        except ValueError:
            inst_executed = 0.0
    # one STG.E.EF.128 (streaming store of a full row) per fast warp-row; the slow rows are a rounding error at the
    # sizes this is captured on.  GHASH-only launches store nothing: there a row is one streaming LDG.128.
    stream_st = sum(v for k, v in by_op.items() if k.startswith("STG") and ".EF" in k and ".128" in k)
    stream_ld = sum(v for k, v in by_op.items() if k.startswith("LDG") and ".EF" in k and ".128" in k)
    warp_rows = stream_st if stream_st else stream_ld
    if warp_rows <= 0:
        raise SystemExit("no streaming 128-bit store / load found: not a row-loop kernel?")
    per_row = lambda x: x / warp_rows
    entry = {
        "kernel": kernel, "command": command, "warp_rows": warp_rows, "library": _library_fingerprint(),
        "per_warp_row": {
            "lds32": per_row(lds32), "lds64": per_row(lds64), "lds128": per_row(lds128),
            "ldg128": per_row(ldg128), "stg128": per_row(stg128), "sts128": per_row(sts128),
            "shared_wavefronts_total": per_row(wf_total),
            "warp_instructions": per_row(total), "warp_instructions_issued": per_row(issued),
            "warp_instructions_executed_counter": per_row(inst_executed),
            "by_pipe_warp_instructions": {k: per_row(v) for k, v in sorted(by_pipe.items())},
            "shared_wavefronts": per_row(wf_shared), "shared_wavefronts_ideal": per_row(wf_shared_ideal),
            "top_opcodes": {k: round(per_row(v), 2) for k, v in by_op.most_common(24)},
        },
        # one warp-row = 32 blocks, one block per lane: warp-level counts per row = thread-level counts per block
        "note": "whole-kernel counts (predicated-on thread instructions / 32) divided by the number of warp-rows, prologue and "
                "epilogue included; warp_instructions_issued counts every issued warp instruction; "
                "a conflict-free LDS.32 is 1 shared-memory wavefront, an LDS.128 is 4",
    }
    data = {}
    if os.path.exists(out):
        data = json.load(open(out))
    data[key] = entry
    json.dump(data, open(out, "w"), indent=1, sort_keys=True)
    print(json.dumps({key: entry["per_warp_row"]}, indent=1))


def static(kernel_regex: str, out: str) -> None:
    names = subprocess.run(["cuobjdump", "-sass", LIB], capture_output=True, text=True, check=True).stdout
    funs = re.findall(r"Function : (\S+)", names)
    pick = [f for f in funs if re.search(kernel_regex, f)]
    with open(out, "w") as fo:
        fo.write("# static SASS of the hot loop: cuobjdump -sass -fun <kernel> %s\n"
                 "# made by: python -m paper_2602_23067_b200.profile_tools static '%s' <out>\n"
                 "# loop = the backward branch that encloses the most LDS; ALL paths of the loop body are counted (fast path, the\n"
                 "# byte-granular slow path and the every-8th-row counter refresh together); executed counts: sass_mix_*.json\n\n"
                 % (os.path.basename(LIB), kernel_regex))
        for fun in pick:
            txt = subprocess.run(["cuobjdump", "-sass", "-fun", fun, LIB], capture_output=True, text=True, check=True).stdout
            ins = []
            for l in txt.splitlines():
                m = re.match(r"\s+/\*([0-9a-f]{4,6})\*/\s+(.*?);", l)
                if m:
                    ins.append((int(m.group(1), 16), m.group(2)))
            loops = []
            for a, t in ins:
                m = re.search(r"\bBRA\b.*?0x([0-9a-f]+)", t)
                if m and int(m.group(1), 16) < a:
                    tgt = int(m.group(1), 16)
                    body = [x for (y, x) in ins if tgt <= y <= a]
                    nlds = sum(1 for x in body if opcode(x).startswith("LDS"))
                    loops.append((nlds, tgt, a, body))
            # the row loop: the smallest loop that still holds close to half of the kernel's table reads (the rest of
            # them sit in the one-off E_K(J0) / counter-cache code outside it)
            most = max((l[0] for l in loops), default=0)
            cand = [l for l in loops if l[0] >= 16 and l[0] >= 0.45 * most]
            best = min(cand, key=lambda l: len(l[3])) if cand else None
            if best is None:
                continue
            nlds, tgt, a, body = best
            ops = collections.Counter(opcode(x) for x in body)
            pipes = collections.Counter(pipe_of(opcode(x)) for x in body)
            fo.write("%s\n  whole kernel: %d instructions; hot loop 0x%x..0x%x: %d instructions\n" % (fun, len(ins), tgt, a, len(body)))
            fo.write("  by pipe: %s\n" % ", ".join("%s %d" % kv for kv in sorted(pipes.items())))
            fo.write("  table reads: LDS (32-bit) %d, LDS.128 %d; global: %s\n" % (
                sum(v for k, v in ops.items() if k == "LDS" or k.startswith("LDS.U") or k == "LDS.32"),
                sum(v for k, v in ops.items() if k.startswith("LDS") and ".128" in k),
                ", ".join("%s %d" % (k, v) for k, v in sorted(ops.items()) if k.startswith(("LDG", "STG")))))
            fo.write("  opcodes: %s\n\n" % ", ".join("%s %d" % kv for kv in ops.most_common(30)))


def launches(log: str, out_csv: str, command: str) -> None:
    """Compact copy of an `ncu --metrics gpu__time_duration.sum --csv` log (kernel names shortened) and the share of
    device time per kernel, printed as a markdown table."""
    rows = list(csv.reader(l for l in open(log) if l.startswith('"')))
    hdr = rows[0]
    ki, vi, gi, bi = hdr.index("Kernel Name"), hdr.index("Metric Value"), hdr.index("Grid Size"), hdr.index("Block Size")
    tot, cnt = collections.Counter(), collections.Counter()
    with open(out_csv, "w") as f:
        f.write("# %s\n" % command)
        f.write("id,kernel,grid,block,gpu__time_duration.sum [ns]\n")
        for r in rows[1:]:
            try:
                v = float(r[vi].replace(",", ""))
            except (ValueError, IndexError):
                continue
            name = re.sub(r"^void\s+", "", r[ki])
            name = re.sub(r"\(.*", "", name)
            name = re.sub(r"at::<unnamed>::|at::native::|at::", "torch ", name)[:64].strip()
            f.write("%s,%s,%s,%s,%.0f\n" % (r[0], name.replace(",", ";"), r[gi].replace(",", "x"), r[bi].replace(",", "x"), v))
            tot[name] += v
            cnt[name] += 1
    total = sum(tot.values())
    print("| kernel | launches | total ns | share |\n|---|---|---|---|")
    for k, v in tot.most_common():
        print("| `%s` | %d | %.0f | %.2f %% |" % (k, cnt[k], v, 100 * v / total))


def main(argv):
    if len(argv) >= 5 and argv[1] == "summary":
        summary(argv[2], argv[3], argv[4])
    elif len(argv) >= 6 and argv[1] == "mix":
        mix(argv[2], argv[3], argv[4], argv[5])
    elif len(argv) >= 5 and argv[1] == "launches":
        launches(argv[2], argv[3], argv[4])
    elif len(argv) >= 4 and argv[1] == "static":
        static(argv[2], argv[3])
    else:
        raise SystemExit(__doc__)


if __name__ == "__main__":
    main(sys.argv)
