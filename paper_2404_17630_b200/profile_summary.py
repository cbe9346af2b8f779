"""Reduces an `ncu --set full` report to the tables kept under profiles/ (markdown on stdout).

    python -m paper_2404_17630_b200.profile_summary REPORT.ncu-rep [--sass KERNEL_REGEX ...] [--traffic WORKLOAD]

Reads the report with `ncu -i REPORT --page raw --csv` (one column per launch: duration, occupancy,
DRAM bytes, shared-memory wavefronts, stall reasons) and, for every --sass pattern, with
`ncu -i REPORT --page source --csv --kernel-name regex:PATTERN` (warp instructions and stall samples
summed by opcode, first matching launch).  --traffic prints the rows of profiles/traffic.csv
(workload,kernel,dram bytes per launch) that bench.py reports as `roofline.traffic`: launches of one
kernel name are summed when they are the size classes of one pass (k_flux, k_grad), chemistry
passes are summed per subcycle.  No GPU needed; only `ncu` on PATH.
"""
import collections
import csv
import hashlib
import io
import os
import subprocess
import sys

WANT = [("duration [ms]", "gpu__time_duration.sum"), ("grid", "launch__grid_size"), ("block", "launch__block_size"),
        ("registers / thread", "launch__registers_per_thread"),
        ("blocks / SM by registers", "launch__occupancy_limit_registers"),
        ("blocks / SM by shared memory", "launch__occupancy_limit_shared_mem"),
        ("achieved occupancy [%]", "sm__warps_active.avg.pct_of_peak_sustained_active"),
        ("DRAM read [Gbyte]", "dram__bytes_read.sum"), ("DRAM written [Gbyte]", "dram__bytes_write.sum"),
        ("DRAM throughput (% of peak)", "gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed"),
        ("L2 hit rate [%]", "lts__t_sector_hit_rate.pct"),
        ("L1/shared throughput (% of peak)", "l1tex__throughput.avg.pct_of_peak_sustained_active"),
        ("issue slots busy [%]", "sm__inst_issued.avg.pct_of_peak_sustained_active"),
        ("fp64 pipe (% of peak)", "sm__inst_executed_pipe_fp64.avg.pct_of_peak_sustained_active"),
        ("warp instructions", "smsp__inst_executed.sum"),
        ("active threads / warp instruction", "smsp__thread_inst_executed_per_inst_executed.ratio"),
        ("shared-memory wavefronts", "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum"),
        ("  of which bank conflicts", "l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum")]
BYTES = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}


def kernel_source_sha():
    """sha-256 (16 hex digits) of the kernel sources: profiles/traffic.csv rows carry it, so that bench.py
    never reports a capture of other kernels as its run's traffic."""
    h = hashlib.sha256()
    d = os.path.join(os.path.dirname(os.path.abspath(__file__)), "csrc")
    for f in ("rt_transport.cu", "rt_chem.cu", "rt_internal.cuh", "rt_kernels.cuh"):
        h.update(open(os.path.join(d, f), "rb").read())
    return h.hexdigest()[:16]


def _ncu(args):
    return subprocess.run(["ncu"] + args, capture_output=True, text=True, check=True).stdout


def raw_table(rep):
    rows = list(csv.reader(io.StringIO(_ncu(["-i", rep, "--page", "raw", "--csv"]))))
    hdr, units, data = rows[0], rows[1], rows[2:]
    col = {h: i for i, h in enumerate(hdr)}

    def num(r, m):
        return float(r[col[m]].replace(",", ""))

    def val(r, m):
        if m not in col:
            return "n/a"
        u = units[col[m]]
        try:
            x = num(r, m)
        except ValueError:
            return r[col[m]]
        if m == "gpu__time_duration.sum":
            return "%.3f" % (x / {"ns": 1e6, "us": 1e3, "ms": 1.0, "s": 1e-3}.get(u, 1.0))
        if "dram__bytes" in m:
            return "%.3f" % (x * BYTES.get(u, 1.0) / 1e9)
        return ("%.0f" % x) if abs(x) >= 1000 or x == int(x) else "%.2f" % x

    names = ["%s (id %s)" % (r[col["Kernel Name"]].split("(")[0], r[col["ID"]]) for r in data]
    out = ["| metric | " + " | ".join("`%s`" % n for n in names) + " |", "|---|" + "---|" * len(names)]
    for label, m in WANT:
        out.append("| %s | " % label + " | ".join(val(r, m) for r in data) + " |")
    stalls = sorted(h for h in hdr if h.startswith("smsp__average_warp") and "issue_stalled" in h and h.endswith(".ratio")
                    and "not_issued" not in h)
    out += ["", "| stall (cycles per issued instruction) | " + " | ".join("`%s`" % n for n in names) + " |",
            "|---|" + "---|" * len(names)]
    for h in stalls:
        out.append("| %s | " % h.split("issue_stalled_")[1].split("_per_warp")[0] + " | ".join(val(r, h) for r in data) + " |")
    traffic = collections.OrderedDict()
    for r in data:
        name = r[col["Kernel Name"]].split("<")[0].split("(")[0]
        b = sum(num(r, m) * BYTES.get(units[col[m]], 1.0) for m in ("dram__bytes_read.sum", "dram__bytes_write.sum"))
        traffic.setdefault(name, []).append((int(num(r, "launch__grid_size")), b))
    return "\n".join(out), traffic


def sass_table(rep, pattern):
    lines = _ncu(["-i", rep, "--page", "source", "--csv", "--kernel-name", "regex:" + pattern]).splitlines()
    starts = [i for i, l in enumerate(lines) if l.startswith('"Kernel Name"')]
    if not starts:
        return "(no launch matches %s)" % pattern
    rows = list(csv.DictReader(lines[starts[0] + 1:(starts[1] if len(starts) > 1 else len(lines))]))
    tot_s = sum(int(r["# Samples"]) for r in rows) or 1
    tot_i = sum(int(r["Instructions Executed"]) for r in rows) or 1
    agg = collections.defaultdict(lambda: [0, 0])
    for r in rows:
        op = [t for t in r["Source"].split() if not t.startswith("@")][0].rstrip(";")
        base = op.split(".")[0]
        if base in ("LDS", "STS", "LDG", "STG", "LDGSTS", "ST", "LD"):
            base = op if op.count(".") <= 2 else ".".join(op.split(".")[:3])
        agg[base][0] += int(r["# Samples"])
        agg[base][1] += int(r["Instructions Executed"])
    out = ["### `%s`: %d SASS instructions, %d warp instructions executed, %d stall samples" % (pattern, len(rows), tot_i, tot_s), "",
           "| opcode | warp instructions | share | stall samples | share |", "|---|---|---|---|---|"]
    for op, (s, i) in sorted(agg.items(), key=lambda kv: -kv[1][1])[:16]:
        out.append("| `%s` | %d | %.1f %% | %d | %.1f %% |" % (op, i, 100 * i / tot_i, s, 100 * s / tot_s))
    st = {c: sum(int(r[c] or 0) for r in rows) for c in rows[0] if c.startswith("stall_")}
    tt = sum(st.values()) or 1
    out += ["", "stall samples by reason: " + ", ".join("%s %.0f %%" % (c[6:], 100 * v / tt)
                                                        for c, v in sorted(st.items(), key=lambda kv: -kv[1])[:8]), ""]
    top = sorted(rows, key=lambda r: -int(r["# Samples"]))[:8]
    out.append("hottest instructions (stall samples): " + "; ".join("`%s` %d" % (" ".join(r["Source"].split()), int(r["# Samples"]))
                                                                    for r in top))
    return "\n".join(out)


def main(argv):
    if len(argv) < 2:
        print(__doc__)
        return 2
    rep, sass, workload = argv[1], [], None
    i = 2
    while i < len(argv):
        if argv[i] == "--sass":
            sass.append(argv[i + 1])
        elif argv[i] == "--traffic":
            workload = argv[i + 1]
        i += 2
    table, traffic = raw_table(rep)
    print(table)
    for pat in sass:
        print()
        print(sass_table(rep, pat))
    if workload:
        print()
        print("traffic.csv rows: workload,kernel,dram bytes read + written per launch (size classes of one pass summed, "
              "first pass of each kernel),sha of the kernel sources at the time of this reduction")
        for name, launches in traffic.items():
            # the size classes of one pass are consecutive launches with different grids
            grids, tot = [], 0.0
            for g, b in launches:
                if g in grids and not name.strip().endswith("k_chem"):   # (the chemistry passes of a subcycle are all summed)
                    break
                grids.append(g)
                tot += b
            print("%s,%s,%.0f,%s" % (workload, name.replace("void ", "").strip(), tot, kernel_source_sha()))
    return 0


if __name__ == "__main__":
    sys.exit(main(sys.argv))
