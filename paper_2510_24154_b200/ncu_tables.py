"""Text tables from an ncu report of the transport kernel (profiling aid; how the files under profiles/ are made).

    python -m paper_2510_24154_b200.ncu_tables functions REPORT.ncu-rep            > profiles/..._per_function.txt
    python -m paper_2510_24154_b200.ncu_tables summary   REPORT.ncu-rep KEY HISTORIES   (row KEY of profiles/ncu_transport_summary.csv)

functions: `ncu -i REPORT --page source --csv --print-source cuda,sass`; every row with a "Line No" is a CUDA source line carrying
the sums over the SASS attributed to it (inlined code counts for the line of the innermost inlined function); a row of
transport.cu goes to the function whose body textually contains the line, rows of other files are listed under [file name].
summary: `ncu -i REPORT --page raw --csv`; the metrics named in profiles/r02_README.md.  Needs ncu, no GPU."""
import csv
import io
import os
import re
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "csrc", "transport.cu")


def ncu_csv(report, *page):
    out = subprocess.run(["ncu", "-i", report, "--csv"] + list(page), capture_output=True, text=True).stdout
    return list(csv.reader(io.StringIO(out)))


def function_of_line():
    pat = re.compile(r"^(?:template\s*<[^>]*>\s*)?(?:static\s+)?(?:__device__|__global__|inline|static|int|void|size_t)[^;{]*?\b([A-Za-z_][A-Za-z0-9_]*)\s*\([^;]*$")
    fn, cur, depth = {}, "file scope", 0
    for i, l in enumerate(open(SRC).read().split("\n"), 1):
        if depth <= 1:                                    # namespace scope
            m = pat.match(l)
            if m and not l.startswith("#") and not l.strip().startswith("//"):
                name = m.group(1)
                if name not in ("__launch_bounds__", "__align__"):
                    cur = name
                elif "transport_kernel" in l:
                    cur = "transport_kernel"
                elif "sample_source_kernel" in l:
                    cur = "sample_source_kernel"
        fn[i] = cur
        code = l.split("//")[0]
        depth += code.count("{") - code.count("}")
    return fn


def functions(report):
    rows = ncu_csv(report, "--page", "source", "--print-source", "cuda,sass")
    hdr = next(r for r in rows if r and r[0] == "Line No")
    col = {n: i for i, n in reversed(list(enumerate(hdr)))}
    stall = [n for n in hdr if n.startswith("stall_") and "Not Issued" not in n]
    fn_at, agg, cur_file = function_of_line(), {}, ""
    for r in rows:
        if r and r[0] == "File Path":
            cur_file = r[1]
            continue
        if not r or not r[0].isdigit() or len(r) < len(hdr):
            continue
        try:
            w, t, s = (float(r[col[k]] or 0) for k in ("Instructions Executed", "Thread Instructions Executed", "# Samples"))
            st = [float(r[col[k]] or 0) for k in stall]
        except ValueError:                                 # a header line whose quotes break the CSV
            continue
        f = fn_at.get(int(r[0]), "?") if cur_file.endswith("transport.cu") else "[" + cur_file.split("/")[-1] + "]"
        a = agg.setdefault(f, [0.0, 0.0, 0.0] + [0.0] * len(stall))
        a[0] += w; a[1] += t; a[2] += s
        for k, v in enumerate(st):
            a[3 + k] += v
    W, T, S = (sum(a[k] for a in agg.values()) for k in range(3))
    show = ["stall_no_inst", "stall_long_sb", "stall_short_sb", "stall_wait", "stall_barrier", "stall_math", "stall_branch_resolving", "stall_not_selected"]
    print("total warp instr %.3e thread instr %.3e samples %d avg lanes %.2f" % (W, T, S, T / W))
    print("%-26s %7s %6s %7s | %s  (%% of the samples of the function)" % ("function", "winstr%", "lanes", "sampl%", " ".join(s[6:14] for s in show)))
    for f, a in sorted(agg.items(), key=lambda kv: -kv[1][2]):
        if a[0] == 0:
            continue
        print("%-26s %6.1f%% %6.1f %6.1f%% | %s" % (f, 100 * a[0] / W, a[1] / a[0], 100 * a[2] / S,
              " ".join("%8.1f" % (100 * a[3 + stall.index(k)] / max(a[2], 1)) for k in show)))


def summary(report, key, n):
    rows = ncu_csv(report, "--page", "raw")
    m = {h: (v, u) for h, u, v in zip(rows[0], rows[1], rows[2])}

    def f(name):
        v, u = m[name]
        return float(v.replace(",", "")) * {"Gbyte": 1e9, "Mbyte": 1e6, "Kbyte": 1e3, "ms": 1e-3, "us": 1e-6, "ns": 1e-9}.get(u, 1.0)
    row = {"key": key, "histories": int(n), "report": os.path.basename(report), "duration_ms": round(f("gpu__time_duration.sum") * 1e3, 4),
           "dram_bytes_per_history": round((f("dram__bytes_read.sum") + f("dram__bytes_write.sum")) / n, 2),
           "warp_instr_per_history": round(f("smsp__inst_executed.sum") / n, 2),
           "lanes_per_warp_instr": round(f("smsp__thread_inst_executed_per_inst_executed.ratio"), 3),
           "lanes_pred_on": round(f("smsp__thread_inst_executed_pred_on_per_inst_executed.ratio"), 3),
           "issue_slot_pct": round(f("smsp__issue_active.avg.pct_of_peak_sustained_active"), 2),
           "ipc": round(f("sm__inst_executed.avg.per_cycle_active"), 3), "l2_hit_pct": round(f("lts__t_sector_hit_rate.pct"), 2),
           "registers": int(f("launch__registers_per_thread"))}
    path = os.path.join(os.path.dirname(HERE), "profiles", "ncu_transport_summary.csv")
    old = [r for r in csv.DictReader(open(path)) if r["key"] != key] if os.path.exists(path) else []
    with open(path, "w", newline="") as fh:
        w = csv.DictWriter(fh, fieldnames=list(row.keys()))
        w.writeheader()
        for r in old + [row]:
            w.writerow(r)
    print(row)


if __name__ == "__main__":
    if len(sys.argv) >= 3 and sys.argv[1] == "functions":
        functions(sys.argv[2])
    elif len(sys.argv) >= 5 and sys.argv[1] == "summary":
        summary(sys.argv[2], sys.argv[3], float(sys.argv[4]))
    else:
        sys.exit(__doc__)
