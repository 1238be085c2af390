"""Turns an Nsight Compute report of the step kernels into the text summaries kept under profiles/.

    python -m paper_2401_03008_b200.ncu_summary gpurun_out/prof_r2.ncu-rep --tag r2 --n 256 [--scheme uct-ho]

reads the report with `ncu -i <rep> --page raw --csv` (no GPU needed) and writes
    profiles/<tag>_ncu_full.md    per-kernel table of the metrics DESIGN.md quotes, with the capture command
    profiles/<tag>_traffic.json   dram__bytes_read.sum + dram__bytes_write.sum per cell and kernel class, stamped with
                                  the sha256 of the CUDA sources it was captured on; bench.py reports roofline.traffic
                                  from it and reports null when the sources have changed since.
The capture command itself (run under gpurun, after the same command exited 0 without ncu) is printed by --help-capture.
Post-processing of profiler output only: nothing here is on the numerical path.
"""
import argparse
import csv
import hashlib
import io
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
CSRC = os.path.join(ROOT, "paper_2401_03008_b200", "csrc")

CAPTURE = ('ncu --set full --clock-control none --import-source on -k regex:"k_prim|k_flux|k_uct|k_bupd" -s 24 -c 6 '
           '-o gpurun_out/prof_{tag} python bench.py --steps 2 --warmup 3 --no-cpu --e2e-steps 1 --kernel-steps 1')

METRICS = [
    ("time (`gpu__time_duration.sum`)", "gpu__time_duration.sum"),
    ("DRAM read (`dram__bytes_read.sum`)", "dram__bytes_read.sum"),
    ("DRAM write (`dram__bytes_write.sum`)", "dram__bytes_write.sum"),
    ("FP64 pipe active % (`sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_active`)",
     "sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_active"),
    ("issue slots busy % (`smsp__issue_active.avg.pct_of_peak_sustained_active`)", "smsp__issue_active.avg.pct_of_peak_sustained_active"),
    ("achieved occupancy % (`sm__warps_active.avg.pct_of_peak_sustained_active`)", "sm__warps_active.avg.pct_of_peak_sustained_active"),
    ("registers/thread (`launch__registers_per_thread`)", "launch__registers_per_thread"),
    ("static smem/block (`launch__shared_mem_per_block_static`)", "launch__shared_mem_per_block_static"),
    ("dynamic smem/block (`launch__shared_mem_per_block_dynamic`)", "launch__shared_mem_per_block_dynamic"),
    ("warp instructions (`smsp__inst_executed.sum`)", "smsp__inst_executed.sum"),
    ("LDGSTS warp instructions (`smsp__inst_executed_op_ldgsts.sum`)", "smsp__inst_executed_op_ldgsts.sum"),
    ("shared-memory wavefronts (`l1tex__data_pipe_lsu_wavefronts_mem_shared.sum`)", "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum"),
    ("L2 hit % (`lts__t_sector_hit_rate.pct`)", "lts__t_sector_hit_rate.pct"),
    ("avg active threads/instr (`smsp__thread_inst_executed_per_inst_executed.ratio`)", "smsp__thread_inst_executed_per_inst_executed.ratio"),
    ("smem bank conflicts (`l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum`)", "l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum"),
    ("grid size (`launch__grid_size`)", "launch__grid_size"),
    ("block size (`launch__block_size`)", "launch__block_size"),
    ("elapsed cycles (`sm__cycles_elapsed.max`)", "sm__cycles_elapsed.max"),
]
STALLS = "smsp__average_warps_issue_stalled_%s_per_issue_active.ratio"
UNIT_SCALE = {"Gbyte": 1e9, "Mbyte": 1e6, "Kbyte": 1e3, "byte": 1.0, "ms": 1.0, "us": 1e-3, "ns": 1e-6, "s": 1e3,
              "msecond": 1.0, "usecond": 1e-3, "nsecond": 1e-6, "second": 1e3}


def kernel_source_hash():
    """sha256 over the CUDA sources the library is built from: ties an ncu capture to the kernels it measured."""
    h = hashlib.sha256()
    for f in sorted(os.listdir(CSRC)):
        if f.endswith((".cu", ".cuh")):
            h.update(f.encode())
            with open(os.path.join(CSRC, f), "rb") as fh:
                h.update(fh.read())
    return h.hexdigest()


def kernel_class(name):
    if "k_prim" in name:
        return "k_prim"
    if "k_flux" in name:
        for d, c in (("<0", "k_flux_x"), ("<1", "k_flux_y"), ("<2", "k_flux_z"), ("<(int)0", "k_flux_x"),
                     ("<(int)1", "k_flux_y"), ("<(int)2", "k_flux_z")):
            if "k_flux" + d in name or "k_flux_flat" + d in name:
                return c
        return "k_flux"
    if "k_uct" in name:
        return "k_uct"
    if "k_bupd" in name or "k_update" in name:
        return "k_update"
    return None


def read_report(path):
    out = subprocess.run(["ncu", "-i", path, "--page", "raw", "--csv"], capture_output=True, text=True, check=True).stdout
    rows = list(csv.reader(io.StringIO(out)))
    hdr, units = rows[0], rows[1]
    recs = []
    for r in rows[2:]:
        if len(r) != len(hdr):
            continue
        d = {}
        for k, u, v in zip(hdr, units, r):
            try:
                d[k] = float(v.replace(",", "")) * UNIT_SCALE.get(u, 1.0) if u in UNIT_SCALE else float(v.replace(",", ""))
            except ValueError:
                d[k] = v
        recs.append(d)
    return recs


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("report", nargs="?")
    ap.add_argument("--tag", default="r2")
    ap.add_argument("--n", type=int, default=256)
    ap.add_argument("--scheme", default="uct-ho")
    ap.add_argument("--help-capture", action="store_true")
    args = ap.parse_args()
    if args.help_capture or not args.report:
        print(CAPTURE.format(tag=args.tag))
        return
    cells = float(args.n) ** 3
    recs = read_report(args.report)
    md = ["# %s_ncu_full.md — `ncu --set full` of one RK stage (stage 2 of a step) at %d^3" % (args.tag, args.n), "",
          "Command (under `gpurun`, one B200, after the identical command had exited 0 without ncu in the same call):", "",
          "```", CAPTURE.format(tag=args.tag), "```", "",
          "Summarised with `python -m paper_2401_03008_b200.ncu_summary %s --tag %s --n %d` (reads the report with "
          "`ncu -i ... --page raw --csv`).  N = %d cells; flop = DADD + DMUL + 2 DFMA (thread level, predicated on). "
          "Times under ncu are cold-cache and serialised; the CUDA-event averages are in the bench lines." %
          (os.path.basename(args.report), args.tag, args.n, int(cells)), "",
          "kernel sources sha256 at capture: `%s`" % kernel_source_hash(), ""]
    traffic = {"source_sha256": kernel_source_hash(), "scheme": args.scheme, "n": args.n,
               "report": os.path.basename(args.report), "md": "profiles/%s_ncu_full.md" % args.tag, "kernels": {}}
    for d in recs:
        name = str(d.get("Kernel Name", ""))
        cls = kernel_class(name)
        md += ["## `%s`" % name, "", "| metric | value |", "|---|---|"]
        for label, key in METRICS:
            if key in d:
                v = d[key]
                md.append("| %s | %s |" % (label, ("%.6g" % v) if isinstance(v, float) else v))
        get = lambda k: float(d.get(k, 0.0) or 0.0)
        # --set full holds the FP64 thread-instruction counts per elapsed cycle of an SM sub-partition
        pre = "smsp__sass_thread_inst_executed_op_%s_pred_on.sum.per_cycle_elapsed"
        cyc = get("smsp__cycles_elapsed.max") or get("sm__cycles_elapsed.max")
        flop = (get(pre % "dadd") + get(pre % "dmul") + 2.0 * get(pre % "dfma")) * cyc
        t_ms = get("gpu__time_duration.sum")
        dram = get("dram__bytes_read.sum") + get("dram__bytes_write.sum")
        if t_ms > 0:
            md.append("| **derived** flop/cell, TFLOP/s | %.0f, %.2f |" % (flop / cells, flop / (t_ms * 1e-3) * 1e-12))
            md.append("| **derived** DRAM bytes/launch, bytes/cell, GB/s | %.4g, %.1f, %.0f |" %
                      (dram, dram / cells, dram / (t_ms * 1e-3) * 1e-9))
            md.append("| **derived** warp instructions per warp of 32 cells | %.0f |" % (get("smsp__inst_executed.sum") / (cells / 32.0)))
        stalls = []
        for k, v in d.items():
            if k.startswith("smsp__average_warps_issue_stalled_") and k.endswith("_per_issue_active.ratio") and isinstance(v, float):
                stalls.append((v, k[len("smsp__average_warps_issue_stalled_"):-len("_per_issue_active.ratio")]))
        stalls.sort(reverse=True)
        md.append("| top stall reasons (warps per issue) | %s |" % ", ".join("%s %.2f" % (n, v) for v, n in stalls[:6]))
        md.append("")
        if cls and cls not in traffic["kernels"] and dram > 0:
            traffic["kernels"][cls] = {"kernel": name, "dram_bytes_per_cell": dram / cells, "time_ms_under_ncu": t_ms}
    out_md = os.path.join(ROOT, "profiles", "%s_ncu_full.md" % args.tag)
    with open(out_md, "w") as f:
        f.write("\n".join(md) + "\n")
    with open(os.path.join(ROOT, "profiles", "%s_traffic.json" % args.tag), "w") as f:
        json.dump(traffic, f, indent=1)
        f.write("\n")
    print("wrote", out_md, "and profiles/%s_traffic.json" % args.tag, "(classes: %s)" % ", ".join(sorted(traffic["kernels"])))


if __name__ == "__main__":
    main()
