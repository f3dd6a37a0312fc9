"""Summarise an `ncu --set full` report of this library's kernels into profiles/ (text only; nothing here runs a GPU).

    python -m paper_2602_03857_b200.ncu_summary REPORT.ncu-rep --config C [--tag NAME] [--command "..."]

reads the report with `ncu -i REPORT --page raw --csv` (ncu is on the CPU box too) and
  * updates profiles/kernel_metrics.csv: one row per (kernel, config) with the figures bench.py quotes instead of
    hard-coding them - FP64-pipe thread-instructions executed per node evaluation (or per pair for the per-pair
    kernel), DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum), duration, pipe utilisation;
  * writes profiles/NAME.md with the same figures, the stall breakdown and the command that produced the report.
The evaluations (pairs) one launch processes come from the workload generator's sizes for `--config`.
"""
import argparse
import csv
import io
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
CSV_PATH = os.path.join(ROOT, "profiles", "kernel_metrics.csv")
COLUMNS = ["kernel", "config", "log2d", "launch", "duration_ms", "units_per_launch", "unit", "fp64_inst_per_eval",
           "fp64_pipe_pct", "issue_active_pct", "dram_bytes_per_launch", "lds_wavefront_pct", "registers", "block",
           "grid", "sm_mhz", "report"]

# kernel-name fragment -> (short name, unit of work)
KERNELS = [("forward_nodes", "forward_nodes", "eval"), ("adjoint_nodes", "adjoint_nodes", "eval"),
           ("pair_tile_kernel<0", "tabulate_f64", "pair"), ("pair_tile_kernel<1", "tabulate_f32", "pair"),
           ("pair_tile_kernel<2", "gram_diag", "pair"), ("gemvt_kernel", "gemvt", "byte"), ("gemv_kernel", "gemv", "byte")]


def _num(s):
    try:
        return float(str(s).replace(",", ""))
    except ValueError:
        return float("nan")


def read_report(path):
    out = subprocess.run(["ncu", "-i", path, "--page", "raw", "--csv"], capture_output=True, text=True, check=True).stdout
    rows = list(csv.reader(io.StringIO(out)))
    hdr, units = rows[0], rows[1]
    return [dict(zip(hdr, r)) for r in rows[2:]], dict(zip(hdr, units))


def to_base(value, unit):
    """ncu prints byte and time metrics with a scaled unit (Kbyte, Mbyte, ms, us ...)."""
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12, "ns": 1e-6, "us": 1e-3, "ms": 1.0,
             "s": 1e3, "second": 1e3, "msecond": 1.0, "usecond": 1e-3, "nsecond": 1e-6}
    return value * scale.get(unit.strip(), 1.0)


def summarise(path, config, sizes):
    rows, units = read_report(path)
    N, M, Nn, elem = sizes
    out = []
    for r in rows:
        name = r.get("Kernel Name", "")
        hit = next(((short, unit) for frag, short, unit in KERNELS if frag in name), None)
        if hit is None:
            continue
        short, unit = hit
        g = lambda k: _num(r.get(k, "nan"))
        if g("sm__throughput.avg.pct_of_peak_sustained_elapsed") != g("sm__throughput.avg.pct_of_peak_sustained_elapsed"):
            continue                                        # a launch ncu did not finish collecting (NaN metrics)
        dur = to_base(g("gpu__time_duration.sum"), units.get("gpu__time_duration.sum", "ms"))
        # --set full carries the FP64 op counts as per-cycle rates summed over the SM sub-partitions: x elapsed cycles
        mhz = to_base(g("sm__cycles_elapsed.avg.per_second"), "") * {"Ghz": 1e3, "Mhz": 1.0, "hz": 1e-6}.get(
            units.get("sm__cycles_elapsed.avg.per_second", "Ghz").strip(), 1e3)
        cycles = g("sm__cycles_elapsed.avg") if "sm__cycles_elapsed.avg" in r else dur * 1e-3 * mhz * 1e6
        fp64 = sum(g(f"smsp__sass_thread_inst_executed_op_{op}_pred_on.sum.per_cycle_elapsed")
                   for op in ("dfma", "dmul", "dadd")) * cycles
        n_units = {"eval": float(N) * Nn, "pair": float(N) * M, "byte": float(N) * M * elem}[unit]
        dram = to_base(g("dram__bytes_read.sum"), units.get("dram__bytes_read.sum", "byte")) + \
            to_base(g("dram__bytes_write.sum"), units.get("dram__bytes_write.sum", "byte"))
        stalls = {k.replace("smsp__average_warps_issue_stalled_", "").replace("_per_issue_active.ratio", ""): _num(v)
                  for k, v in r.items() if k.startswith("smsp__average_warps_issue_stalled_")
                  and k.endswith("_per_issue_active.ratio")}
        out.append(dict(kernel=short, config=config, log2d=int(", 1>" in name or "<2, 2>" in name or ", 2>" in name),
                        launch=name.split("(")[0].strip(), duration_ms=dur, units_per_launch=n_units, unit=unit,
                        fp64_inst_per_eval=fp64 / n_units if unit != "byte" else float("nan"),
                        fp64_pipe_pct=g("sm__inst_executed_pipe_fp64.avg.pct_of_peak_sustained_active"),
                        issue_active_pct=g("smsp__issue_active.avg.pct_of_peak_sustained_active"),
                        dram_bytes_per_launch=dram,
                        lds_wavefront_pct=g("l1tex__data_pipe_lsu_wavefronts_mem_shared.sum.pct_of_peak_sustained_elapsed"),
                        registers=g("launch__registers_per_thread"), block=r.get("Block Size", ""),
                        grid=r.get("Grid Size", ""), sm_mhz=mhz,
                        report=os.path.basename(path), _stalls=stalls))
    return out


def update_csv(new_rows):
    old = []
    if os.path.exists(CSV_PATH):
        with open(CSV_PATH) as f:
            old = list(csv.DictReader(f))
    key = lambda r: (r["kernel"], str(int(float(r["config"]))))
    keep = {key(r): r for r in old}
    for r in new_rows:
        keep[key(r)] = {c: (f"{r[c]:.6g}" if isinstance(r[c], float) else r[c]) for c in COLUMNS}
    os.makedirs(os.path.dirname(CSV_PATH), exist_ok=True)
    with open(CSV_PATH, "w", newline="") as f:
        w = csv.DictWriter(f, fieldnames=COLUMNS)
        w.writeheader()
        for k in sorted(keep):
            w.writerow({c: keep[k].get(c, "") for c in COLUMNS})


def write_md(tag, new_rows, command, config):
    path = os.path.join(ROOT, "profiles", f"{tag}.md")
    with open(path, "w") as f:
        f.write(f"# {tag}: ncu --set full summary, config {config}\n\n")
        f.write("Command (run under gpurun on one B200; the plain run of the same command exited 0 first):\n\n")
        f.write(f"    {command}\n\n")
        f.write("Read on the CPU box with `python -m paper_2602_03857_b200.ncu_summary` (`ncu -i ... --page raw --csv`).  "
                "Durations are under the profiler (serialised, cold cache): bench.py's CUDA-event times are the ones "
                "quoted as results.\n\n")
        for r in new_rows:
            f.write(f"## {r['kernel']}  (`{r['launch']}`)\n\n")
            f.write(f"| metric | value |\n|---|---|\n")
            f.write(f"| grid / block / registers | {r['grid']} / {r['block']} / {r['registers']:.0f} |\n")
            f.write(f"| duration | {r['duration_ms']:.3f} ms at {r['sm_mhz']:.0f} MHz |\n")
            f.write(f"| work per launch | {r['units_per_launch']:.4g} {r['unit']}s |\n")
            if r["unit"] != "byte":
                f.write(f"| FP64-pipe thread-instructions per {r['unit']} (DFMA + DMUL + DADD, executed) | "
                        f"{r['fp64_inst_per_eval']:.2f} |\n")
            f.write(f"| sm__inst_executed_pipe_fp64 (% of peak, active) | {r['fp64_pipe_pct']:.1f} |\n")
            f.write(f"| smsp__issue_active (%) | {r['issue_active_pct']:.1f} |\n")
            f.write(f"| shared-memory wavefronts (% of peak) | {r['lds_wavefront_pct']:.1f} |\n")
            f.write(f"| DRAM bytes per launch (read + write) | {r['dram_bytes_per_launch']:.4g} |\n")
            st = sorted(((v, k) for k, v in r["_stalls"].items() if v == v and v >= 0.05), reverse=True)
            f.write("| warp stalls per issue (>= 0.05) | " + ", ".join(f"{k} {v:.2f}" for v, k in st) + " |\n\n")
    return path


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("report")
    ap.add_argument("--config", type=int, required=True)
    ap.add_argument("--tag", default=None)
    ap.add_argument("--command", default="(not recorded)")
    a = ap.parse_args()
    sys.path.insert(0, ROOT)
    from paper_2602_03857_b200 import workloads
    wl = workloads.make(a.config)
    elem = 4 if wl.N * wl.M * 8 > 100e9 else 8
    rows = summarise(a.report, a.config, (wl.N, wl.M, wl.n_nodes, elem))
    if not rows:
        sys.exit("no kernel of this library in the report")
    update_csv(rows)
    tag = a.tag or os.path.splitext(os.path.basename(a.report))[0]
    print(write_md(tag, rows, a.command, a.config))
    for r in rows:
        print(f"{r['kernel']}: {r['duration_ms']:.3f} ms, fp64/unit {r['fp64_inst_per_eval']:.2f}, "
              f"pipe {r['fp64_pipe_pct']:.1f} %, DRAM {r['dram_bytes_per_launch']:.3g} B")


if __name__ == "__main__":
    main()
