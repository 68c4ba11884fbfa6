"""Per-event instruction counts and DRAM traffic of the iterate kernel, read from an ncu report.

    python -m paper_2010_09341_b200.ncu_counts <report.ncu-rep> <workload> <n_events> [--md] [--launch K]

Reads the report with `ncu -i <report> --page raw --csv` (whole-launch counters) and `--page source --csv` (executed
count of every SASS instruction; needs --import-source at capture time and -lineinfo at compile time) and prints ONE
csv row: what one launch executed, divided by the events it processed --

    workload, kernel, n_events, kernel_us, dram_bytes, inst, fp64, fp32, imad_wide, imad, lop3, lds, atoms

`inst` .. `atoms` are warp instructions x 32 / n_events = thread instructions per event (retries of lost histogram races
included, predicated-off lanes counted: these are issue slots and pipe cycles, which is what bounds the kernel).
bench.py reads the committed table (profiles/r02_kernel_counts.csv) for the co-bounds of its roofline block and for
`roofline.traffic`; `--md` prints the opcode histogram as a markdown table instead (profiles/r02_sass_hist_*.md).
No GPU needed: ncu only parses the report.
"""
from __future__ import annotations

import collections
import csv
import re
import subprocess
import sys

FP64 = ("DADD", "DFMA", "DMUL", "DSETP")
FP32 = ("FADD", "FFMA", "FMUL", "FSETP", "FSEL", "FMNMX", "FCHK", "MUFU")
HEADER = "workload,kernel,n_events,kernel_us,dram_bytes,inst,fp64,fp32,imad_wide,imad,lop3,lds,atoms"


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
           "%.2f" % (family(cnt, ("LOP3",)) * per), "%.2f" % (lds * per), "%.2f" % (atoms * per)]
    print(",".join(row))
    return 0


if __name__ == "__main__":
    sys.exit(main(sys.argv))
