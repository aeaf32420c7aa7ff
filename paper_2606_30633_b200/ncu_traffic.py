"""Turn `ncu --set full` captures of the hot-path kernels into the two things the repo keeps of them:

    python -m paper_2606_30633_b200.ncu_traffic --key cfg5_f64 --source profiles/r2_cfg5_f64.md gpurun_out/r2_prof_cfg5.ncu-rep

  * a text summary per kernel (the counters DESIGN.md argues with: duration, registers, occupancy limits, pipe
    utilisation, issue slots, DRAM bytes, hit rates, top stall reasons), printed to stdout for the profiles/*.md file;
  * `profiles/ncu_traffic.json`: DRAM bytes (dram__bytes_read.sum + dram__bytes_write.sum) of ONE launch of each
    kernel, keyed by "<key>" (cfg<k>_<precision>) and by the stage name bench.py uses, which bench.py reads for
    `roofline.traffic` (it cannot run a profiler itself).  Existing keys of the file are kept.

The capture is read with `ncu -i <rep> --page raw --csv` (works without a GPU).  Holds no arithmetic of the method.
"""
import argparse
import csv
import io
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
STAGE_OF = (("gl_ray_fwd_kernel", "ray_fwd"), ("gl_ray_comp_kernel", "ray_fwd"), ("gl_conv_fwd", "conv_chi2"),
            ("gl_conv_bwd", "conv_transpose"), ("gl_ray_adj_kernel", "ray_adjoint"), ("gl_unpack_kernel", "unpack_prior"),
            ("gl_finalize_kernel", "finalize"), ("gl_prep_kernel", "prep"), ("gl_amp_solve_kernel", "amplitude_solve"),
            ("gl_shp_coef_kernel", "ray_adjoint_coef"), ("gl_bin_planes_kernel", "bin_planes"))
SHOW = ["gpu__time_duration.sum", "launch__registers_per_thread", "launch__block_size", "launch__grid_size",
        "launch__occupancy_limit_registers", "launch__occupancy_limit_shared_mem", "launch__occupancy_limit_warps",
        "sm__warps_active.avg.pct_of_peak_sustained_active", "sm__inst_executed_pipe_fp64.avg.pct_of_peak_sustained_active",
        "sm__inst_executed_pipe_fma.avg.pct_of_peak_sustained_active", "sm__inst_executed_pipe_xu.avg.pct_of_peak_sustained_active",
        "sm__inst_executed_pipe_alu.avg.pct_of_peak_sustained_active", "sm__inst_executed_pipe_lsu.avg.pct_of_peak_sustained_active",
        "sm__pipe_tensor_cycles_active.avg.pct_of_peak_sustained_active",
        "smsp__issue_active.avg.pct_of_peak_sustained_active", "smsp__inst_executed.sum", "dram__bytes_read.sum",
        "dram__bytes_write.sum", "l1tex__t_sector_hit_rate.pct", "lts__t_sector_hit_rate.pct",
        "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum", "l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum",
        "gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed"]
STALL_PREFIX = "smsp__average_warps_issue_stalled_"
STALL_SUFFIX = "_per_issue_active.ratio"
UNIT_SCALE = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}


def read_raw(rep):
    txt = subprocess.run(["ncu", "-i", rep, "--page", "raw", "--csv"], check=True, capture_output=True, text=True).stdout
    rows = list(csv.reader(io.StringIO(txt)))
    hdr = next(i for i, r in enumerate(rows) if "Kernel Name" in r)
    names, units = rows[hdr], rows[hdr + 1]
    return names, units, rows[hdr + 2:]


def num(x):
    try:
        return float(x.replace(",", ""))
    except ValueError:
        return None


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("reports", nargs="+")
    ap.add_argument("--key", required=True, help="cfg<k>_<f64|f32>")
    ap.add_argument("--source", required=True, help="the profiles/*.md file that documents the capture")
    ap.add_argument("--json", default=os.path.join(ROOT, "profiles", "ncu_traffic.json"))
    a = ap.parse_args()
    per_stage = {}
    for rep in a.reports:
        names, units, rows = read_raw(rep)
        col = {n: i for i, n in enumerate(names)}
        kcol = col["Kernel Name"]
        for r in rows:
            if len(r) <= kcol:
                continue
            kname = r[kcol]
            stage = next((s for pat, s in STAGE_OF if pat in kname), None)
            print("== %s" % kname[:110])
            for mname in SHOW:
                if mname in col and r[col[mname]] != "":
                    print("   %-70s %s %s" % (mname, r[col[mname]], units[col[mname]]))
            stalls = []
            for n, i in col.items():
                if n.startswith(STALL_PREFIX) and n.endswith(STALL_SUFFIX) and num(r[i]) is not None:
                    stalls.append((num(r[i]), n[len(STALL_PREFIX):-len(STALL_SUFFIX)]))
            stalls.sort(reverse=True)
            print("   stalls (warps per issue): " + ", ".join("%s %.2f" % (n, v) for v, n in stalls[:7]))
            if stage is None:
                continue
            tot = 0.0
            for mname in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
                v = num(r[col[mname]]) if mname in col else None
                if v is None:
                    tot = None
                    break
                tot += v * UNIT_SCALE.get(units[col[mname]], 1.0)
            if tot is not None:
                per_stage.setdefault(stage, {"kernel": kname.split("(")[0][:100], "launches": []})["launches"].append(tot)
    tab = {}
    if os.path.exists(a.json):
        with open(a.json) as f:
            tab = json.load(f)
    tab[a.key] = {s: {"kernel": d["kernel"], "dram_bytes_per_launch": sum(d["launches"]) / len(d["launches"]),
                      "launches_captured": len(d["launches"]), "source": a.source} for s, d in sorted(per_stage.items())}
    with open(a.json, "w") as f:
        json.dump(tab, f, indent=1, sort_keys=True)
    print("wrote %s [%s]: %s" % (a.json, a.key, {s: "%.4g GB" % (d["dram_bytes_per_launch"] / 1e9) for s, d in tab[a.key].items()}),
          file=sys.stderr)


if __name__ == "__main__":
    main()
