"""Turn ncu captures of the library's kernels into the text summaries kept under profiles/.

  python -m paper_2410_05985_b200.ncu_summary traffic  REP:WORKLOAD:OPTIMIZER[:KERNEL_REGEX[:SUMMARY]] [...]  > profiles/traffic.csv
  python -m paper_2410_05985_b200.ncu_summary summary  REP [KERNEL_REGEX]            > profiles/<name>.txt

`traffic` writes one csv row per capture: dram__bytes_read.sum + dram__bytes_write.sum of the
(last) matching kernel launch in REP, i.e. the number bench.py reports as roofline.traffic
(SUMMARY: the committed text summary of the same capture, written to the `source` column).
`summary` prints the counters DESIGN.md quotes (duration, DRAM bytes and throughput, occupancy,
registers, issue utilisation, top stall reasons) for every matching launch.
Both read the report with `ncu -i REP --page raw --csv`; nothing here runs on a GPU.
"""
import csv
import os
import io
import re
import subprocess
import sys

_UNIT = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12,
         "ns": 1e-6, "us": 1e-3, "usecond": 1e-3, "ms": 1.0, "msecond": 1.0, "s": 1e3, "second": 1e3}


def read_raw(rep):
    """-> (list of {metric: (value str, unit str)} per launch)."""
    out = subprocess.run(["ncu", "-i", rep, "--page", "raw", "--csv"], capture_output=True, text=True, check=True).stdout
    rows = list(csv.reader(io.StringIO(out)))
    head, units = rows[0], rows[1]
    return [{h: (v, u) for h, u, v in zip(head, units, r)} for r in rows[2:]]


def scaled(launch, metric):
    v, u = launch[metric]
    return float(v.replace(",", "")) * _UNIT.get(u, 1.0)


def pick(launches, pattern):
    sel = [l for l in launches if re.search(pattern, l["Kernel Name"][0])]
    if not sel:
        raise SystemExit("no kernel matching %r among %s" % (pattern, sorted({l["Kernel Name"][0] for l in launches})))
    return sel


def kernel_short(name):
    m = re.search(r"(layup_\w+(?:<[^>]*>)?)", name)
    return m.group(1).replace(" ", "") if m else name


def traffic(specs):
    """Rows carry the capture date and the git hash of the kernels captured (--git HASH first: the GPU
    box has no .git), so that bench.py can say how old the committed figure is (roofline.traffic_from)."""
    import datetime
    git = "?"
    if specs and specs[0] == "--git":
        git, specs = specs[1], specs[2:]
    captured = datetime.date.today().isoformat()
    w = csv.writer(sys.stdout, lineterminator="\n")
    w.writerow(["workload", "optimizer", "dram_bytes_per_launch", "kernel", "source", "captured", "git"])
    for spec in specs:
        parts = spec.split(":")
        rep, workload, optimizer = parts[:3]
        pattern = parts[3] if len(parts) > 3 and parts[3] else r"layup_update"
        source = parts[4] if len(parts) > 4 else rep
        l = pick(read_raw(rep), pattern)[-1]
        total = scaled(l, "dram__bytes_read.sum") + scaled(l, "dram__bytes_write.sum")
        w.writerow([workload, optimizer, int(round(total)), kernel_short(l["Kernel Name"][0]), source, captured, git])


_SASS = r"UTMALDG[.A-Z0-9_]*|UTMASTG[.A-Z0-9_]*|UBLKCP[.A-Z0-9_]*|SYNCS[.A-Z0-9_]*|LDG\.E[.A-Z0-9_]*|STG\.E[.A-Z0-9_]*|" \
        r"LDS[.A-Z0-9_]*|STS[.A-Z0-9_]*|DFMA|DADD|DMUL|FFMA|ATOMG[.A-Z0-9_]*|RED[.A-Z0-9_]*|ACQBULK|UTCBAR|TCGEN05[.A-Z0-9_]*|HMMA[.A-Z0-9_]*"


def sass(lib):
    """Counts, per kernel of the built library, the SASS mnemonics that show HOW it moves data (TMA tile
    loads UTMALDG, bulk copies UBLKCP, mbarrier ops SYNCS, plain LDG/STG, shared-memory and fp64 ops):
    `cuobjdump -sass` read as text, no GPU needed."""
    import subprocess
    txt = subprocess.run(["cuobjdump", "-sass", lib], check=True, capture_output=True, text=True).stdout
    print("# SASS instruction summary of %s (sm_100a), per kernel: static instruction counts" % os.path.basename(lib))
    print("# command: python -m paper_2410_05985_b200.ncu_summary sass > profiles/sass_summary.txt")
    print("# UTMALDG = TMA tensor-map tile load (.GATHER4 = tile::gather4), UBLKCP = 1-D bulk copy (cp.async.bulk),")
    print("# SYNCS = mbarrier arrive / try_wait / expect_tx, ATOMG/RED = global atomics, DFMA/DADD = fp64 pipe")
    name, counts, total = None, {}, 0

    def flush():
        if name is not None:
            short = subprocess.run(["c++filt", name], capture_output=True, text=True).stdout.strip() or name
            short = kernel_short(short)
            body = "  ".join("%s x%d" % kv for kv in sorted(counts.items(), key=lambda kv: (-kv[1], kv[0])))
            print("%-62s %6d instr | %s" % (short, total, body))

    for line in txt.splitlines():
        m = re.match(r"\s*Function : (\S+)", line)
        if m:
            flush()
            name, counts, total = m.group(1), {}, 0
            continue
        m = re.match(r"\s*/\*[0-9a-f]{4,}\*/\s+(?:@!?U?P\d+\s+)?([A-Z][A-Z0-9_.]*)", line)
        if m:
            total += 1
            op = m.group(1)
            if re.fullmatch(_SASS, op):
                counts[op] = counts.get(op, 0) + 1
    flush()


_SUMMARY = ["gpu__time_duration.sum", "dram__bytes_read.sum", "dram__bytes_write.sum",
            "gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed", "dram__throughput.avg.pct_of_peak_sustained_elapsed",
            "lts__throughput.avg.pct_of_peak_sustained_elapsed", "l1tex__throughput.avg.pct_of_peak_sustained_elapsed",
            "sm__throughput.avg.pct_of_peak_sustained_elapsed", "sm__inst_issued.avg.pct_of_peak_sustained_active",
            "sm__warps_active.avg.pct_of_peak_sustained_active", "sm__maximum_warps_per_active_cycle_pct",
            "launch__grid_size", "launch__block_size", "launch__registers_per_thread", "launch__shared_mem_per_block_dynamic",
            "launch__occupancy_limit_shared_mem", "launch__occupancy_limit_registers", "launch__waves_per_multiprocessor",
            "sm__cycles_elapsed.avg.per_second", "dram__cycles_elapsed.avg.per_second",
            "sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_active", "sm__inst_executed_pipe_fp64.sum",
            "sm__pipe_alu_cycles_active.avg.pct_of_peak_sustained_active", "sm__pipe_fma_cycles_active.avg.pct_of_peak_sustained_active",
            "sm__inst_executed_pipe_xu.sum", "smsp__inst_executed.sum"]


def summary(rep, pattern):
    launches = pick(read_raw(rep), pattern)
    for l in launches:
        print("kernel: %s" % l["Kernel Name"][0])
        for m in _SUMMARY:
            if m in l and l[m][0] != "":
                print("  %-62s %s %s" % (m, l[m][0], l[m][1]))
        if "dram__bytes_read.sum" in l and "gpu__time_duration.sum" in l:
            tot = scaled(l, "dram__bytes_read.sum") + scaled(l, "dram__bytes_write.sum")
            ms = scaled(l, "gpu__time_duration.sum")
            print("  %-62s %.3f GB in %.4f ms = %.0f GB/s (under ncu: cold caches, serialised)" % (
                "dram read+write", tot / 1e9, ms, tot / 1e9 / (ms * 1e-3)))
        stalls = sorted(((float(v[0].replace(",", "")), k) for k, v in l.items()
                         if k.startswith("smsp__average_warps_issue_stalled") and k.endswith("_per_issue_active.ratio")
                         and v[0] not in ("", "n/a")), reverse=True)
        if not stalls:
            stalls = sorted(((float(v[0].replace(",", "")), k) for k, v in l.items()
                             if k.startswith("smsp__average_warp_latency_issue_stalled") and v[0] not in ("", "n/a")), reverse=True)
        for val, k in stalls[:8]:
            print("  stall %-56s %.3f" % (k.replace("smsp__average_warps_issue_stalled_", "").replace("smsp__average_warp_latency_issue_stalled_", "")
                                          .replace("_per_issue_active.ratio", "").replace(".ratio", ""), val))
        print()


def main(argv):
    if argv and argv[0] == "sass":
        sass(argv[1] if len(argv) > 1 else os.path.join(os.path.dirname(os.path.abspath(__file__)), "csrc", "liblayup.so"))
        return 0
    if len(argv) >= 2 and argv[0] == "traffic":
        traffic(argv[1:])
    elif len(argv) >= 2 and argv[0] == "summary":
        summary(argv[1], argv[2] if len(argv) > 2 else r"layup_")
    else:
        raise SystemExit(__doc__)


if __name__ == "__main__":
    main(sys.argv[1:])
