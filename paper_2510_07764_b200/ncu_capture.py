"""Record the counters of one `ncu --set full` capture of a cell kernel in ncu_captured.json (read by bench.py).

    ncu -i gpurun_out/<name>.ncu-rep --page raw --csv > raw.csv
    python -m paper_2510_07764_b200.ncu_capture raw.csv --key C5:8:p0 --profile profiles/<summary>.md [--kernel k_cells_tab]

bench.py's roofline object reports executed FP64 flop and DRAM traffic only from a capture whose workload key
(workload:batch:precision[:tmapDEX]) and kernel-source hash match the run; this script writes that record.  The
first launch in the csv whose name contains --kernel is used.  Prints a markdown table row set for profiles/.
"""
import argparse
import csv
import hashlib
import json
import os

HERE = os.path.dirname(os.path.abspath(__file__))
JSON_PATH = os.path.join(HERE, "ncu_captured.json")
def hashed_files(key):
    """the sources that define the cell kernel of a capture key (same rule as bench.kernel_source_files)"""
    files = ["ppm_common.cuh", "ppm_cells.cuh"]
    if ":d1" in key:
        files.append("ppm_cells_lin.cuh")
    if ":tmap" in key:
        files.append("ppm_cells_map.cuh")
    if ":p1" in key:
        files.append("ppm_cells32.cuh")
        if ":tmap" in key:
            files.append("ppm_cells_map32.cuh")
    return files


UNIT = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12,
        "ns": 1e-9, "us": 1e-6, "ms": 1e-3, "s": 1.0, "usecond": 1e-6, "nsecond": 1e-9, "msecond": 1e-3, "second": 1.0}

WANT = {
    # thread-level instruction counts: `--set full` reports them per elapsed cycle; parse() multiplies by smsp_cycles
    "dfma_per_cycle": "smsp__sass_thread_inst_executed_op_dfma_pred_on.sum.per_cycle_elapsed",
    "dadd_per_cycle": "smsp__sass_thread_inst_executed_op_dadd_pred_on.sum.per_cycle_elapsed",
    "dmul_per_cycle": "smsp__sass_thread_inst_executed_op_dmul_pred_on.sum.per_cycle_elapsed",
    "ffma_per_cycle": "smsp__sass_thread_inst_executed_op_ffma_pred_on.sum.per_cycle_elapsed",
    "fadd_per_cycle": "smsp__sass_thread_inst_executed_op_fadd_pred_on.sum.per_cycle_elapsed",
    "fmul_per_cycle": "smsp__sass_thread_inst_executed_op_fmul_pred_on.sum.per_cycle_elapsed",
    "smsp_cycles": "smsp__cycles_elapsed.avg",
    "l2_sectors": "lts__t_sectors.sum",
    "dram_read_bytes": "dram__bytes_read.sum",
    "dram_write_bytes": "dram__bytes_write.sum",
    "time_s": "gpu__time_duration.sum",
    "cycles": "sm__cycles_elapsed.max",
    "inst_executed": "smsp__inst_executed.sum",
    "fp64_pipe_pct": "sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_active",
    "issue_active_pct": "smsp__issue_active.avg.pct_of_peak_sustained_active",
    "xu_pipe_pct": "sm__inst_executed_pipe_xu.avg.pct_of_peak_sustained_active",
    "fma_pipe_pct": "sm__inst_executed_pipe_fma.avg.pct_of_peak_sustained_active",
    "alu_pipe_pct": "sm__inst_executed_pipe_alu.avg.pct_of_peak_sustained_active",
    "lsu_pipe_pct": "sm__inst_executed_pipe_lsu.avg.pct_of_peak_sustained_active",
    "smem_wavefronts": "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum",
    "smem_wavefronts_pct": "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum.pct_of_peak_sustained_elapsed",
    "smem_bank_conflicts": "l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum",
    "registers": "launch__registers_per_thread",
    "warps_active_pct": "sm__warps_active.avg.pct_of_peak_sustained_active",
    "occupancy_pct": "sm__warps_active.avg.pct_of_peak_sustained_active",
}


def _code_only(text):
    """the source without comments and with white space collapsed (same rule as bench.py)"""
    import re
    text = re.sub(r"/\*.*?\*/", " ", text, flags=re.S)
    text = re.sub(r"//[^\n]*", " ", text)
    return " ".join(text.split())


def source_hash(key):
    h = hashlib.sha256()
    for f in hashed_files(key):
        with open(os.path.join(HERE, "csrc", f), "r") as fh:
            h.update(_code_only(fh.read()).encode())
    return h.hexdigest()[:16]


def parse(path, kernel):
    rows = [r for r in csv.reader(open(path)) if r]
    start = next(i for i, r in enumerate(rows) if "Kernel Name" in r)
    hdr, units = rows[start], rows[start + 1]
    kn = hdr.index("Kernel Name")
    for r in rows[start + 2:]:
        if kernel in r[kn]:
            out = {"kernel": r[kn].split("(")[0]}
            for k, m in WANT.items():
                if m in hdr:
                    j = hdr.index(m)
                    try:
                        v = float(r[j].replace(",", ""))
                    except ValueError:
                        continue
                    out[k] = v * UNIT.get(units[j], 1.0)
            for op in ("dfma", "dadd", "dmul", "ffma", "fadd", "fmul"):
                if op + "_per_cycle" in out and "smsp_cycles" in out:
                    out[op] = out.pop(op + "_per_cycle") * out["smsp_cycles"]
            if "l2_sectors" in out:
                out["l2_bytes"] = 32.0 * out["l2_sectors"]
            return out
    raise SystemExit("no launch of %s in %s" % (kernel, path))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("raw_csv")
    ap.add_argument("--key", required=True)
    ap.add_argument("--profile", required=True, help="the profiles/ summary that documents this capture")
    ap.add_argument("--kernel", default="k_cells")
    ap.add_argument("--no-write", action="store_true")
    a = ap.parse_args()
    c = parse(a.raw_csv, a.kernel)
    c["dram_bytes"] = c.get("dram_read_bytes", 0.0) + c.get("dram_write_bytes", 0.0)
    c["source_hash"] = source_hash(a.key)
    c["hashed_sources"] = hashed_files(a.key)
    c["profile"] = a.profile
    if not a.no_write:
        try:
            data = json.load(open(JSON_PATH))
        except (OSError, ValueError):
            data = {"captures": {}}
        data["captures"][a.key] = c
        with open(JSON_PATH, "w") as f:
            json.dump(data, f, indent=1, sort_keys=True)
            f.write("\n")
    print("| metric | %s |\n|---|---|" % a.key)
    for k in sorted(c):
        print("| %s | %s |" % (k, c[k]))


if __name__ == "__main__":
    main()
