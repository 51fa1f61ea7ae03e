"""Text summary of an Nsight Compute report of the library's kernels.

    python -m paper_2008_02478_b200.ncu_summary REPORT.ncu-rep --config C5 [--traffic profiles/ncu_traffic.csv]

Reads the report through `ncu -i REPORT --page raw --csv` and `--page source --csv` (ncu is on the
CPU box too; no GPU needed), prints
  * one column per profiled launch with the counters DESIGN.md argues from, and
  * per kernel the share of warp-stall samples of every barrier-separated phase (the kernels are
    sequences of phases, csrc/launcher.cuh) with its top stall reasons and instruction mix.
With --traffic it also appends `config,kernel,dram_bytes_read,dram_bytes_write,csrc_sha` rows to the
CSV that bench.py quotes as `roofline.traffic` (only for the kernel sources the capture was taken from).
Measurement tooling: it runs none of the method's arithmetic.
"""
import argparse
import csv
import hashlib
import io
import os
import re
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))

METRICS = [
    "gpu__time_duration.sum", "dram__bytes_read.sum", "dram__bytes_write.sum", "lts__t_sector_hit_rate.pct",
    "lts__t_sectors_srcunit_tex_op_read.sum", "sm__warps_active.avg.pct_of_peak_sustained_active",
    "launch__registers_per_thread", "launch__occupancy_limit_registers", "launch__occupancy_limit_shared_mem",
    "launch__waves_per_multiprocessor", "sm__pipe_fma_cycles_active.avg.pct_of_peak_sustained_active",
    "sm__inst_executed_pipe_lsu.avg.pct_of_peak_sustained_active", "smsp__issue_active.avg.pct_of_peak_sustained_active",
    "smsp__inst_executed.sum", "l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum",
    "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum", "l1tex__data_pipe_lsu_wavefronts.avg.pct_of_peak_sustained_elapsed",
    "l1tex__t_sectors_pipe_lsu_mem_global_op_ld.sum", "l1tex__t_requests_pipe_lsu_mem_global_op_ld.sum",
    "l1tex__t_sectors_pipe_lsu_mem_global_op_st.sum", "l1tex__t_requests_pipe_lsu_mem_global_op_st.sum",
    "smsp__average_warps_issue_stalled_barrier_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_long_scoreboard_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_short_scoreboard_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_mio_throttle_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_lg_throttle_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_wait_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_math_pipe_throttle_per_issue_active.ratio",
    "launch__shared_mem_config_size",
]


def csrc_sha():
    h = hashlib.sha256()
    d = os.path.join(HERE, "csrc")
    for name in sorted(os.listdir(d)):
        # the hot path: kernel headers, the launcher, the translation units that instantiate them and the C ABI
        if name.endswith((".h", ".cuh")) or name.startswith("tu_") or name == "boris_demag.cu":
            h.update(name.encode())
            h.update(open(os.path.join(d, name), "rb").read())
    return h.hexdigest()[:16]


def ncu_page(report, page):
    out = subprocess.run(["ncu", "-i", report, "--page", page, "--csv"], capture_output=True, text=True)
    if out.returncode != 0:
        raise SystemExit("ncu failed: " + out.stderr[-2000:])
    return list(csv.reader(io.StringIO(out.stdout)))


def short_kernel(name):
    m = re.search(r"phase_kernel<(?:bd::)?(\w+)<([^>]*)>", name)
    if m:
        return m.group(1), f"{m.group(1)}<{m.group(2).replace('(int)', '')}>"
    m = re.search(r"(k_\w+)", name)
    return (m.group(1), m.group(1)) if m else (name[:24], name[:40])


def raw_table(report):
    rows = ncu_page(report, "raw")
    hdr, units, data = rows[0], rows[1], rows[2:]
    col = {h: i for i, h in enumerate(hdr)}
    names = [short_kernel(r[col["Kernel Name"]]) for r in data]
    lines = ["%-76s %-9s %s" % ("kernel", "", " | ".join(n[1] for n in names)),
             "%-76s %-9s %s" % ("grid", "", " | ".join(r[col["Grid Size"]] for r in data))]
    for m in METRICS:
        if m in col:
            lines.append("%-76s %-9s %s" % (m[:76], units[col[m]][:9], " | ".join(r[col[m]] for r in data)))
    traffic = [(names[i][0], int(float(r[col["dram__bytes_read.sum"]].replace(",", "")) * unit_scale(units[col["dram__bytes_read.sum"]])),
                int(float(r[col["dram__bytes_write.sum"]].replace(",", "")) * unit_scale(units[col["dram__bytes_write.sum"]])))
               for i, r in enumerate(data)] if "dram__bytes_read.sum" in col else []
    return lines, traffic


def unit_scale(u):
    return {"byte": 1, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}.get(u, 1)


def phase_table(report):
    rows = ncu_page(report, "source")
    lines, seen = [], set()
    i = 0
    while i < len(rows):
        r = rows[i]
        if not (r and r[0] == "Kernel Name"):
            i += 1
            continue
        name, hdr = r[1], rows[i + 1]
        j = i + 2
        body = []
        while j < len(rows) and not (rows[j] and rows[j][0] == "Kernel Name"):
            body.append(rows[j])
            j += 1
        i = j
        ci = {h: k for k, h in enumerate(hdr)}
        if "# Samples" not in ci or name in seen:
            continue
        seen.add(name)
        stall_cols = [h for h in hdr if h.startswith("stall_") and "Not Issued" not in h]
        ph, acc = 0, {}
        for b in body:
            if len(b) < len(hdr):
                continue
            d = acc.setdefault(ph, {"samples": 0, "inst": 0})
            d["samples"] += int(b[ci["# Samples"]] or 0)
            d["inst"] += int(b[ci["Instructions Executed"]] or 0)
            for h in stall_cols:
                d[h] = d.get(h, 0) + int(b[ci[h]] or 0)
            op = b[ci["Source"]]
            for key in ("LDG", "STG", "LDS", "STS", "SHFL", "FFMA2", "FADD2", "FMUL2", "MOV", "LDL", "STL"):
                if key in op:
                    d["n_" + key] = d.get("n_" + key, 0) + int(b[ci["Instructions Executed"]] or 0)
            if "BAR.SYNC" in op:
                ph += 1
        tot = max(sum(d["samples"] for d in acc.values()), 1)
        lines.append(f"{short_kernel(name)[1]}: {len(body)} SASS instructions, {tot} stall samples")
        for p, d in acc.items():
            top = sorted(((d[h], h[6:]) for h in stall_cols), reverse=True)[:4]
            mix = ", ".join(f"{k[2:]} {v / 1e6:.1f}M" for k, v in sorted(d.items()) if k.startswith("n_"))
            lines.append(f"  phase {p}: {100 * d['samples'] / tot:5.1f} % of samples, {d['inst'] / 1e6:6.1f} M warp instructions | "
                         + ", ".join(f"{h} {100 * v / max(d['samples'], 1):.0f}%" for v, h in top) + f" | {mix}")
    return lines


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("report")
    ap.add_argument("--config", required=True, help="workload the report was captured on (C1..C5 or a mesh)")
    ap.add_argument("--traffic", default=None, help="CSV to append the DRAM byte counts to (profiles/ncu_traffic.csv)")
    ap.add_argument("--no-phases", action="store_true")
    args = ap.parse_args()
    lines, traffic = raw_table(args.report)
    print("\n".join(lines))
    if not args.no_phases:
        print()
        print("\n".join(phase_table(args.report)))
    if args.traffic:
        new = not os.path.exists(args.traffic)
        with open(args.traffic, "a") as f:
            if new:
                f.write("config,kernel,dram_bytes_read,dram_bytes_write,csrc_sha\n")
            sha = csrc_sha()
            for k, rd, wr in traffic:
                f.write(f"{args.config},{k},{rd},{wr},{sha}\n")
        print(f"\n[appended {len(traffic)} rows to {args.traffic}, csrc_sha {csrc_sha()}]", file=sys.stderr)


if __name__ == "__main__":
    main()
