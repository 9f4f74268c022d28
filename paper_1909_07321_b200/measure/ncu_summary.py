"""Text summary of one kernel launch of an Nsight Compute report -- the tool that writes profiles/rNN_full_*.txt.

    ncu --set full --clock-control none --import-source on -k regex:<kernel> -s <skip> -c 1 -o rep <command>
    python -m paper_1909_07321_b200.measure.ncu_summary rep.ncu-rep --title "..." --command "<the ncu line>" > profiles/rNN_full_x.txt

It calls `ncu -i rep --page raw --csv` and `ncu -i rep --page source --csv` (ncu must be on PATH; no GPU needed to
read a report) and prints: the counters the roofline argument rests on, DRAM bytes per launch, L2 -> SM bytes per launch
and per SM clock, the spread of the per-SM active cycles, warp samples and executed instructions by SASS opcode, and
the stall reasons.  Nothing here is on the product path; it only reads reports.
"""
from __future__ import annotations

import argparse
import csv
import io
import re
import subprocess
import sys
from collections import defaultdict

RAW_METRICS = [
    "gpu__time_duration.sum", "sm__cycles_elapsed.max", "sm__cycles_active.min", "sm__cycles_active.avg", "sm__cycles_active.max",
    "launch__grid_size", "launch__block_size", "launch__registers_per_thread", "launch__shared_mem_per_block_dynamic",
    "launch__cluster_size",
    "sm__inst_executed_pipe_tensor_subpipe_dmma.avg.pct_of_peak_sustained_active",
    "sm__ops_path_tensor_src_fp64.sum", "sm__ops_path_tensor_src_fp64.avg.pct_of_peak_sustained_elapsed",
    "sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_active",
    "sm__inst_executed_pipe_tensor_subpipe_imma.avg.pct_of_peak_sustained_active",
    "sm__throughput.avg.pct_of_peak_sustained_elapsed",
    "dram__bytes_read.sum", "dram__bytes_write.sum", "dram__throughput.avg.pct_of_peak_sustained_elapsed",
    "lts__t_sector_hit_rate.pct", "lts__throughput.avg.pct_of_peak_sustained_elapsed", "lts__t_bytes.sum", "lts__t_sectors.sum",
    "lts__t_sectors_srcunit_tex_op_read.sum", "lts__t_sectors_srcunit_tex_op_write.sum",
    "l1tex__m_xbar2l1tex_read_bytes.sum", "l1tex__m_xbar2l1tex_read_bytes.sum.per_second",
    "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum", "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum.pct_of_peak_sustained_elapsed",
    "l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum",
    "smsp__inst_executed.sum", "sm__warps_active.avg.pct_of_peak_sustained_active",
]
TO_BYTES = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}
TO_SECONDS = {"ns": 1e-9, "us": 1e-6, "ms": 1e-3, "s": 1.0, "second": 1.0}


def _ncu_csv(report: str, page: str) -> list[list[str]]:
    out = subprocess.run(["ncu", "-i", report, "--page", page, "--csv"], check=True, capture_output=True, text=True).stdout
    start = out.find('"')                                    # ncu may print notices ahead of the table
    return list(csv.reader(io.StringIO(out[start:])))


def raw_metrics(report: str, launch: int = 0) -> dict[str, tuple[str, str]]:
    """{metric: (value, unit)} of launch number `launch` of the report."""
    rows = _ncu_csv(report, "raw")
    names, units, vals = rows[0], rows[1], rows[2 + launch]
    return {n: (v, u) for n, u, v in zip(names, units, vals)}


def _num(m: dict, key: str):
    if key not in m or m[key][0] in ("", "n/a"):
        return None
    return float(m[key][0].replace(",", ""))


def _bytes(m: dict, key: str):
    v = _num(m, key)
    return None if v is None else v * TO_BYTES.get(m[key][1], 1.0)


def opcode_table(report: str):
    """[(opcode, samples, warp instructions executed)] summed over the SASS lines of the source page, and the stall
    reasons' sample totals."""
    rows = _ncu_csv(report, "source")
    hi = next(i for i, r in enumerate(rows) if r and r[0] == "Address")
    hdr = rows[hi]
    col = {h: i for i, h in enumerate(hdr)}
    i_src, i_smp, i_exe = col["Source"], col["# Samples"], col["Instructions Executed"]
    stall_cols = [(h, i) for h, i in col.items() if h.startswith("stall_") and "Not Issued" not in h]
    ops = defaultdict(lambda: [0, 0])
    stalls = defaultdict(int)
    for r in rows[hi + 1:]:
        if len(r) <= max(i_src, i_smp, i_exe):
            continue
        text = re.sub(r"^\s*(@!?U?P\d+\s+)?", "", r[i_src])
        op = text.split()[0].split(".")[0] if text.split() else "?"
        ops[op][0] += int(r[i_smp] or 0)
        ops[op][1] += int(r[i_exe] or 0)
        for h, i in stall_cols:
            if i < len(r) and r[i].isdigit():
                stalls[h] += int(r[i])
    return sorted(((o, s, e) for o, (s, e) in ops.items()), key=lambda x: -x[1]), sorted(stalls.items(), key=lambda x: -x[1])


def summarise(report: str, title: str, command: str, launch: int = 0, top: int = 14) -> str:
    m = raw_metrics(report, launch)
    out = [f"# {title}", f"# kernel: {m.get('Kernel Name', ('?', ''))[0]}",
           f"# command (after the same command exited 0 without ncu): {command}",
           f"# summary written by `python -m paper_1909_07321_b200.measure.ncu_summary {report.split('/')[-1]}` from `ncu -i ... --page raw --csv` and `--page source --csv`",
           "", "## raw metrics"]
    for k in RAW_METRICS:
        if k in m and m[k][0] not in ("", "n/a"):
            out.append(f"{k:<100} {m[k][0]:>20} {m[k][1]}")
    out += ["", "## derived"]
    rd, wr = _bytes(m, "dram__bytes_read.sum"), _bytes(m, "dram__bytes_write.sum")
    if rd is not None and wr is not None:
        out.append(f"DRAM bytes per launch: read {rd / 1e6:.1f} MB + write {wr / 1e6:.1f} MB = {(rd + wr) / 1e6:.1f} MB")
    t = _num(m, "gpu__time_duration.sum")
    t_s = t * TO_SECONDS.get(m["gpu__time_duration.sum"][1], 1.0) if t is not None else None
    cyc, grid = _num(m, "sm__cycles_elapsed.max"), _num(m, "launch__grid_size")
    sect = _num(m, "lts__t_sectors_srcunit_tex_op_read.sum")
    if sect is not None and t_s and cyc:
        b = 32.0 * sect
        out.append(f"L2 -> SM (lts__t_sectors_srcunit_tex_op_read x 32 B): {b / 1e6:.1f} MB per launch = {b / t_s / 1e12:.2f} TB/s"
                   f" = {b / cyc / max(grid or 1, 1):.1f} B/clk per CTA of the grid ({int(grid or 0)} CTAs)")
    lo, av, hi = (_num(m, f"sm__cycles_active.{s}") for s in ("min", "avg", "max"))
    if None not in (lo, av, hi, cyc):
        out.append(f"SM active cycles min / avg / max over the SMs: {lo:.0f} / {av:.0f} / {hi:.0f} of {cyc:.0f} elapsed "
                   f"(avg/elapsed {av / cyc:.3f}, min/max {lo / hi:.3f})")
    try:
        ops, stalls = opcode_table(report)
    except (StopIteration, KeyError, subprocess.CalledProcessError):
        ops, stalls = [], []
    if ops:
        total = sum(s for _, s, _ in ops) or 1
        out += ["", f"## warp samples by SASS opcode (total {total}) and warp-level instructions executed"]
        for o, s, e in ops[:top]:
            out.append(f"{o:<12} samples {s:>8} ({100.0 * s / total:5.1f} %)   executed {e:>12}")
    if stalls:
        total = sum(v for _, v in stalls) or 1
        out += ["", "## stall reasons (samples)"]
        for h, v in stalls[:10]:
            out.append(f"{h:<40} {v:>8} ({100.0 * v / total:5.1f} %)")
    return "\n".join(out) + "\n"


def main() -> int:
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("report")
    ap.add_argument("--title", default="ncu --set full capture")
    ap.add_argument("--command", default="(not given)")
    ap.add_argument("--launch", type=int, default=0, help="which launch of the report (default: the first)")
    a = ap.parse_args()
    sys.stdout.write(summarise(a.report, a.title, a.command, a.launch))
    return 0


if __name__ == "__main__":
    sys.exit(main())
