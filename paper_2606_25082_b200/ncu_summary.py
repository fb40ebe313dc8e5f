"""Turns `ncu -i <capture>.ncu-rep --page raw --csv` into the per-kernel summary that bench.py reads for `roofline.traffic`.

    ncu --set full --clock-control none --import-source on -k regex:sim_thread -s 7 -c 1 -f -o gpurun_out/prof python bench.py ...
    ncu -i gpurun_out/prof.ncu-rep --page raw --csv > gpurun_out/prof_raw.csv
    python -m paper_2606_25082_b200.ncu_summary gpurun_out/prof_raw.csv --workload C5 --n-envs 65536 --out profiles/ncu_summary.json

One entry per kernel name (as the library reports it: mig_sim_kernel_name), carrying the hash of csrc/ at capture time, so
that bench.py can tell a capture of the present kernels from a stale one (it then prints traffic = null).  No arithmetic of
the simulated method lives here; this is measurement bookkeeping.
"""
from __future__ import annotations

import argparse
import csv
import glob
import hashlib
import json
import os
import re

HERE = os.path.dirname(os.path.abspath(__file__))

WANTED = {
    "dram__bytes_read.sum": "dram_bytes_read",
    "dram__bytes_write.sum": "dram_bytes_write",
    "gpu__time_duration.sum": "duration_ms",
    "sm__inst_executed.sum": "warp_inst_executed",
    "smsp__inst_executed.sum": "warp_inst_executed",
    "smsp__thread_inst_executed.sum": "thread_inst_executed",
    "sass__thread_inst_executed_true_per_opcode": "thread_inst_executed_true",
    "sm__inst_executed.sum.pct_of_peak_sustained_elapsed": "issue_pct_of_peak_elapsed",
    "smsp__thread_inst_executed_per_inst_executed.ratio": "active_threads_per_inst",
    "sm__cycles_elapsed.avg.per_second": "sm_ghz",
    "sm__warps_active.avg.per_cycle_active": "warps_active_per_sm",
    "launch__registers_per_thread": "registers",
    "l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum": "smem_bank_conflicts",
    "l1tex__t_sectors_pipe_lsu_mem_global_op_ld.sum": "global_ld_sectors",
    "l1tex__t_requests_pipe_lsu_mem_global_op_ld.sum": "global_ld_requests",
    "smsp__sass_average_data_bytes_per_sector_mem_global_op_ld.ratio": "global_ld_bytes_per_sector",
    "smsp__sass_average_data_bytes_per_sector_mem_global_op_st.ratio": "global_st_bytes_per_sector",
}
SCALE = {"Gbyte": 1e9, "Mbyte": 1e6, "Kbyte": 1e3, "byte": 1.0, "ms": 1.0, "us": 1e-3, "s": 1e3, "ns": 1e-6, "Ghz": 1.0, "Mhz": 1e-3}


def csrc_sha16() -> str:
    h = hashlib.sha256()
    for f in sorted(glob.glob(os.path.join(HERE, "csrc", "*")) + glob.glob(os.path.join(HERE, "..", "include", "*.h"))):
        with open(f, "rb") as fh:
            h.update(os.path.basename(f).encode() + b"\0" + fh.read())
    return h.hexdigest()[:16]


def canonical(name: str) -> str:
    """'void migsim::sim_thread_kernel<64, 0, 0>(SimArgs)' -> 'sim_thread_kernel<64,false,false>' (the library's spelling)."""
    m = re.search(r"(\w+)(<[^>]*>)?\s*\(", name)
    if not m:
        return name
    base, targs = m.group(1), m.group(2) or ""
    if targs:
        parts = [p.strip() for p in targs[1:-1].split(",")]
        parts = [parts[0]] + [{"0": "false", "1": "true"}.get(p, p) for p in parts[1:]]
        targs = "<" + ",".join(parts) + ">"
    return base + targs


def parse(path: str) -> list[dict]:
    with open(path, newline="") as f:
        rows = [r for r in csv.reader(f) if r]
    start = next(i for i, r in enumerate(rows) if "Kernel Name" in r)
    hdr, units = rows[start], rows[start + 1]
    out = []
    for vals in rows[start + 2:]:
        rec = {}
        for h, u, v in zip(hdr, units, vals):
            if h == "Kernel Name":
                rec["kernel_raw"] = v
                rec["kernel"] = canonical(v)
            elif h in WANTED:
                try:
                    rec[WANTED[h]] = float(v.replace(",", "")) * SCALE.get(u, 1.0)
                except ValueError:
                    pass
        out.append(rec)
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("raw_csv")
    ap.add_argument("--workload", required=True)
    ap.add_argument("--n-envs", type=int, required=True)
    ap.add_argument("--out", required=True)
    ap.add_argument("--command", default="", help="the ncu command line that made the capture (recorded verbatim)")
    ap.add_argument("--sum-first", type=int, default=0, help="instead of one entry per kernel: ONE entry, the sums over the first N launches of the capture")
    ap.add_argument("--sum-key", default="", help="kernel field of that entry")
    a = ap.parse_args()
    try:
        with open(a.out) as f:
            doc = json.load(f)
    except Exception:
        doc = {}
    recs = parse(a.raw_csv)
    if a.sum_first:                                          # e.g. the eleven products of ONE training step
        part = recs[:a.sum_first]
        assert len(part) == a.sum_first and a.sum_key, "capture shorter than --sum-first, or no --sum-key"
        tot = {"kernel": a.sum_key, "launches": a.sum_first, "kernels": [r["kernel"] for r in part]}
        for k in ("dram_bytes_read", "dram_bytes_write", "duration_ms", "warp_inst_executed"):
            tot[k] = sum(r.get(k, 0.0) for r in part)
        recs = [tot]
    for rec in recs:
        rec.update(workload=a.workload, n_envs=a.n_envs, csrc_sha16=csrc_sha16(), command=a.command)
        if "dram_bytes_read" in rec and "dram_bytes_write" in rec:
            rec["dram_bytes"] = rec["dram_bytes_read"] + rec["dram_bytes_write"]
        doc["%s|%s|%d" % (rec["kernel"], a.workload, a.n_envs)] = rec
    with open(a.out, "w") as f:
        json.dump(doc, f, indent=1, sort_keys=True)
    print("wrote", a.out, "entries:", sorted(doc))


if __name__ == "__main__":
    main()
