"""Per-event instruction counts and DRAM traffic of the iterate kernel, read from an ncu report.

    python -m paper_2010_09341_b200.ncu_counts <report.ncu-rep> <workload> <n_events> [--md | --summary] [--launch K]

Reads the report with `ncu -i <report> --page raw --csv` (whole-launch counters) and `--page source --csv` (executed
count of every SASS instruction; needs --import-source at capture time and -lineinfo at compile time) and prints ONE
csv row: what one launch executed, divided by the events it processed --

    workload, kernel, n_events, kernel_us, dram_bytes, inst, fp64, fp32, imad_wide, imad, lop3, lds, atoms,
    smem_wavefronts, src_sha

`inst` .. `atoms` are warp instructions x 32 / n_events = thread instructions per event (retries of lost histogram races
included, predicated-off lanes counted: these are issue slots and pipe cycles, which is what bounds the kernel).
`smem_wavefronts` = l1tex__data_pipe_lsu_wavefronts_mem_shared.sum / n_events: shared-memory data-pipe wavefronts per
event (the pipe serves one per clock per SM); `src_sha` = build.kernel_source_sha() of the tree the report is parsed in
(parse right after the capture, from the same tree).
bench.py reads the committed table (profiles/r03_kernel_counts.csv) for the co-bounds of its roofline block and for
`roofline.traffic`; `--md` prints the opcode histogram as a markdown table instead (profiles/r03_sass_hist_*.md);
`--summary` prints the whole-launch counters the design discussion quotes (pipes, issue slots, shared-memory
wavefronts and bank conflicts, DRAM bytes, stall reasons per issued instruction) as a markdown table
(profiles/r03_ncu_full_*.md).  No GPU needed: ncu only parses the report.
"""
from __future__ import annotations

import collections
import csv
import re
import subprocess
import sys

from . import build as _build

FP64 = ("DADD", "DFMA", "DMUL", "DSETP")
FP32 = ("FADD", "FFMA", "FMUL", "FSETP", "FSEL", "FMNMX", "FCHK", "MUFU")
HEADER = "workload,kernel,n_events,kernel_us,dram_bytes,inst,fp64,fp32,imad_wide,imad,lop3,lds,atoms,smem_wavefronts,src_sha"
SUMMARY = """Kernel Name
gpu__time_duration.sum
launch__registers_per_thread
launch__shared_mem_per_block_dynamic
launch__block_size
launch__grid_size
smsp__inst_executed.sum
smsp__issue_active.avg.pct_of_peak_sustained_active
sm__inst_executed_pipe_fp64.avg.pct_of_peak_sustained_active
sm__pipe_fmaheavy_cycles_active.avg.pct_of_peak_sustained_elapsed
sm__pipe_fma_cycles_active.avg.pct_of_peak_sustained_active
sm__pipe_alu_cycles_active.avg.pct_of_peak_sustained_active
sm__inst_executed_pipe_lsu.avg.pct_of_peak_sustained_active
sm__inst_executed_pipe_xu.avg.pct_of_peak_sustained_active
sm__inst_executed_pipe_fma.avg.pct_of_peak_sustained_active
sm__inst_executed_pipe_alu.avg.pct_of_peak_sustained_active
sm__inst_executed_pipe_cbu.avg.pct_of_peak_sustained_active
sm__inst_executed_pipe_adu.avg.pct_of_peak_sustained_active
l1tex__data_pipe_lsu_wavefronts_mem_shared.sum
l1tex__data_pipe_lsu_wavefronts_mem_shared.sum.pct_of_peak_sustained_elapsed
l1tex__data_pipe_lsu_wavefronts_mem_shared_op_atom.sum
l1tex__data_pipe_lsu_wavefronts_mem_shared_op_ld.sum
l1tex__data_pipe_lsu_wavefronts_mem_shared_op_st.sum
l1tex__data_bank_conflicts_pipe_lsu_mem_shared_op_ld.sum
l1tex__data_bank_conflicts_pipe_lsu_mem_shared_op_atom.sum
smsp__inst_executed_op_shared_atom.sum
smsp__sass_inst_executed_op_shared_ld.sum
smsp__sass_inst_executed_op_shared_st.sum
dram__bytes_read.sum
dram__bytes_write.sum
sm__warps_active.avg.pct_of_peak_sustained_active
sm__throughput.avg.pct_of_peak_sustained_elapsed
sm__cycles_elapsed.avg
sm__cycles_elapsed.avg.per_second
smsp__thread_inst_executed_per_inst_executed.ratio
smsp__thread_inst_executed_pred_on_per_inst_executed.ratio""".splitlines()
STALL = "smsp__average_warps_issue_stalled_%s_per_issue_active.ratio"
STALLS = ("barrier", "branch_resolving", "dispatch_stall", "drain", "lg_throttle", "long_scoreboard", "math_pipe_throttle",
          "membar", "mio_throttle", "misc", "no_instruction", "not_selected", "selected", "short_scoreboard", "sleeping",
          "tex_throttle", "wait")


def _page(report, page):
    out = subprocess.run(["ncu", "-i", report, "--page", page, "--csv"], capture_output=True, text=True, check=True).stdout
    return list(csv.reader(out.splitlines()))


def raw_counters(report, launch=0):
    r = _page(report, "raw")
    hdr, row = r[0], r[2 + launch]
    return dict(zip(hdr, row))


def opcode_counts(report):
    """{opcode: warp instructions executed} over the first kernel of the report's source page."""
    rows = _page(report, "source")
    hdr = rows[1]
    i_src, i_exec = hdr.index("Source"), hdr.index("Instructions Executed")
    cnt = collections.Counter()
    for r in rows[2:]:
        if len(r) <= max(i_src, i_exec) or not r[i_src].strip():
            continue
        if r[0] == "Kernel Name":                        # a second kernel's block starts
            break
        op = re.sub(r"^@!?U?P\d+\s+", "", r[i_src].strip()).split()[0].rstrip(";")
        try:
            cnt[op] += int(r[i_exec] or 0)
        except ValueError:
            pass
    return cnt


def family(cnt, names):
    return sum(v for k, v in cnt.items() if k.split(".")[0] in names)


def main(argv):
    if len(argv) < 4:
        print(__doc__)
        return 2
    report, workload, n = argv[1], argv[2], float(argv[3])
    launch = int(argv[argv.index("--launch") + 1]) if "--launch" in argv else 0
    raw = raw_counters(report, launch)
    cnt = opcode_counts(report)
    per = 32.0 / n
    if "--summary" in argv:
        units = dict(zip(_page(report, "raw")[0], _page(report, "raw")[1]))
        print("`stall_*` = smsp__average_warps_issue_stalled_*_per_issue_active.ratio.\n\n| metric | unit | value |\n|---|---|---|")
        for m in SUMMARY:
            if m in raw:
                v = raw[m]
                if m == "Kernel Name":
                    v = re.sub(r"\(int\)|\(bool\)|vegas::", "", v)
                print("| %s | %s | %s |" % (m, units.get(m, ""), v))
        for st in STALLS:
            if STALL % st in raw:
                print("| stall_%s | %s | %s |" % (st, units.get(STALL % st, ""), raw[STALL % st]))
        return 0
    if "--md" in argv:
        total = sum(cnt.values())
        print("| opcode | warp instructions executed | thread instructions per event | share |\n|---|---|---|---|")
        for op, v in cnt.most_common():
            if v * per >= 0.05:
                print("| %s | %d | %.2f | %.1f %% |" % (op, v, v * per, 100.0 * v / total))
        print("| **total** | %d | %.2f | 100 %% |" % (total, total * per))
        return 0
    dram = float(raw.get("dram__bytes_read.sum", 0) or 0) + float(raw.get("dram__bytes_write.sum", 0) or 0)
    units = dict(zip(_page(report, "raw")[0], _page(report, "raw")[1]))
    scale = {"Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "byte": 1.0}
    dram = (float(raw.get("dram__bytes_read.sum", 0) or 0) * scale.get(units.get("dram__bytes_read.sum", "byte"), 1.0)
            + float(raw.get("dram__bytes_write.sum", 0) or 0) * scale.get(units.get("dram__bytes_write.sum", "byte"), 1.0))
    t = float(raw.get("gpu__time_duration.sum", 0) or 0) * {"ms": 1e3, "us": 1.0, "ns": 1e-3, "s": 1e6}.get(units.get("gpu__time_duration.sum", "us"), 1.0)
    kernel = re.sub(r"\(.*$", "", raw.get("Kernel Name", "")).replace("void ", "").replace("vegas::", "").replace("(int)", "").replace("(bool)", "")
    wide = sum(v for k, v in cnt.items() if k.startswith("IMAD.WIDE") or k.startswith("IMAD.HI"))
    imad = sum(v for k, v in cnt.items() if k.startswith("IMAD")) - wide
    lds = sum(v for k, v in cnt.items() if k.startswith("LDS"))
    atoms = sum(v for k, v in cnt.items() if k.startswith("ATOMS"))
    row = [workload, '"%s"' % kernel, "%d" % n, "%.2f" % t, "%.0f" % dram, "%.2f" % (sum(cnt.values()) * per),
           "%.2f" % (family(cnt, FP64) * per), "%.2f" % (family(cnt, FP32) * per), "%.2f" % (wide * per), "%.2f" % (imad * per),
           "%.2f" % (family(cnt, ("LOP3",)) * per), "%.2f" % (lds * per), "%.2f" % (atoms * per),
           "%.3f" % (float(raw.get("l1tex__data_pipe_lsu_wavefronts_mem_shared.sum", 0) or 0) / n), _build.kernel_source_sha()]
    print(",".join(row))
    return 0


if __name__ == "__main__":
    sys.exit(main(sys.argv))
