"""Summarise an ncu raw-page CSV as a markdown table, and record the DRAM traffic per launch.

    ncu -i capture.ncu-rep --page raw --csv > capture.csv
    python -m paper_1211_0126_b200.ncu_summary capture.csv --out profiles/r02_dslash_r12.md \
        --title "..." --command "ncu --set full ..." \
        [--traffic profiles/r02_traffic.json --key cfg5_32x32x32x64/f32/nrhs12 --commit <hash>]

With --launch-list the input is the log of `ncu --metrics gpu__time_duration.sum --csv --log-file ...` and the output a
per-kernel table of launches / time / share.  Otherwise the markdown lists, per captured launch, the counters DESIGN.md section 6 argues with (duration, DRAM bytes and
throughput, L2 sectors and L2 throughput, L1 hit rate, LSU wavefronts, issue slots, stalls, occupancy).  With
--traffic, the mean over the captured launches of dram__bytes_read.sum + dram__bytes_write.sum is stored under
--key together with the commit of the kernels; bench.py reports that number as `roofline.traffic`.
No arithmetic of the method lives here; this is a measurement aid for users of the library.
"""
from __future__ import annotations

import argparse
import csv
import json
import os

WANT = [
    ("Kernel Name", "kernel"), ("gpu__time_duration.sum", "duration"), ("launch__grid_size", "grid"), ("launch__block_size", "block"),
    ("launch__registers_per_thread", "regs/thread"), ("launch__shared_mem_per_block_dynamic", "dyn smem/block"),
    ("dram__bytes_read.sum", "DRAM read"), ("dram__bytes_write.sum", "DRAM write"),
    ("gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed", "DRAM throughput % of peak"),
    ("lts__t_sectors_srcunit_tex.sum", "L2 sectors from SMs"),
    ("lts__t_sectors.sum", "L2 sectors, all sources"),
    ("lts__throughput.avg.pct_of_peak_sustained_elapsed", "L2 (lts) throughput % of peak"),
    ("lts__t_sectors.avg.pct_of_peak_sustained_elapsed", "L2 sector throughput % of peak"),
    ("lts__t_sector_hit_rate.pct", "L2 hit rate %"),
    ("l1tex__t_sector_hit_rate.pct", "L1 hit rate %"),
    ("l1tex__throughput.avg.pct_of_peak_sustained_active", "L1/TEX throughput % of peak"),
    ("l1tex__data_pipe_lsu_wavefronts.sum.pct_of_peak_sustained_elapsed", "LSU data-pipe wavefronts % of peak"),
    ("l1tex__data_pipe_lsu_wavefronts_mem_shared.sum", "shared-memory wavefronts"),
    ("l1tex__data_pipe_lsu_wavefronts.sum", "LSU data-pipe wavefronts"),
    ("l1tex__m_xbar2l1tex_read_bytes.sum", "L2 -> SM bytes over the crossbar (reads)"),
    ("l1tex__m_l1tex2xbar_write_bytes.sum", "SM -> L2 bytes over the crossbar (writes)"),
    ("smsp__inst_executed.sum", "warp instructions"), ("smsp__issue_active.avg.pct_of_peak_sustained_active", "issue slots busy %"),
    ("sm__warps_active.avg.pct_of_peak_sustained_active", "achieved occupancy %"),
    ("smsp__warps_eligible.avg.per_cycle_active", "eligible warps per scheduler cycle"),
    ("sm__inst_executed_pipe_fma.sum.pct_of_peak_sustained_active", "FMA pipe %"),
    ("sm__inst_executed_pipe_fp64.sum.pct_of_peak_sustained_active", "FP64 pipe %"),
    ("sm__inst_executed_pipe_tensor.sum.pct_of_peak_sustained_active", "tensor pipe %"),
    ("smsp__average_warps_issue_stalled_long_scoreboard_per_issue_active.ratio", "stall long_scoreboard (warps/issue)"),
    ("smsp__average_warps_issue_stalled_barrier_per_issue_active.ratio", "stall barrier"),
    ("smsp__average_warps_issue_stalled_short_scoreboard_per_issue_active.ratio", "stall short_scoreboard"),
    ("smsp__average_warps_issue_stalled_lg_throttle_per_issue_active.ratio", "stall lg_throttle"),
    ("smsp__average_warps_issue_stalled_mio_throttle_per_issue_active.ratio", "stall mio_throttle"),
    ("smsp__average_warps_issue_stalled_math_pipe_throttle_per_issue_active.ratio", "stall math_pipe_throttle"),
    ("smsp__average_warps_issue_stalled_wait_per_issue_active.ratio", "stall wait"),
    ("smsp__average_warps_issue_stalled_not_selected_per_issue_active.ratio", "stall not_selected"),
    ("sm__cycles_elapsed.avg.per_second", "SM clock"),
]


def read_rows(path):
    rows = list(csv.reader(open(path)))
    while rows and (not rows[0] or rows[0][0] != "ID"):      # ncu prints "==PROF==" lines before the table
        rows.pop(0)
    if len(rows) < 3:
        raise SystemExit(f"{path}: no ncu raw table found")
    return rows[0], rows[1], rows[2:]


def to_float(v):
    try:
        return float(v.replace(",", ""))
    except ValueError:
        return None


def table(hdr, units, rows):
    idx = {h: i for i, h in enumerate(hdr)}
    n = len(rows)
    out = ["| metric | " + " | ".join(f"launch {k + 1}" for k in range(n)) + " |", "|---|" + "---|" * n]
    for key, name in WANT:
        if key not in idx:
            continue
        vals = []
        for r in rows:
            v = r[idx[key]]
            if key == "Kernel Name":
                v = v.replace("void <unnamed>::", "").split("(")[0]
            else:
                f = to_float(v)
                v = f"{f:.4g}" if f is not None else v
            vals.append(v)
        u = units[idx[key]]
        out.append(f"| {name}{' [' + u + ']' if u else ''} | " + " | ".join(vals) + " |")
    return "\n".join(out)


def dram_bytes(hdr, units, rows):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch, in bytes (ncu prints them in scaled units)."""
    idx = {h: i for i, h in enumerate(hdr)}
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}
    tot = []
    for r in rows:
        b = 0.0
        for key in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
            b += to_float(r[idx[key]]) * scale[units[idx[key]]]
        tot.append(b)
    return tot


def launch_list(path, out_md, out_csv, title, command, note):
    """`ncu --metrics gpu__time_duration.sum --csv --log-file x.csv ...` -> a table of launches, total time and share per
    kernel (markdown) and the log reduced to (id, kernel, duration_us) (csv)."""
    rows = list(csv.reader(open(path)))
    while rows and (not rows[0] or rows[0][0] != "ID"):
        rows.pop(0)
    if len(rows) < 2:
        raise SystemExit(f"{path}: no ncu table found")
    hdr = rows[0]
    ki, vi, ui, mi = hdr.index("Kernel Name"), hdr.index("Metric Value"), hdr.index("Metric Unit"), hdr.index("Metric Name")
    scale = {"ns": 1e-3, "us": 1.0, "ms": 1e3, "s": 1e6}
    recs = []
    for r in rows[1:]:
        if len(r) <= vi or r[mi] != "gpu__time_duration.sum":
            continue
        name = r[ki].replace("void <unnamed>::", "").replace("<unnamed>::", "").split("(")[0]
        recs.append((name, to_float(r[vi]) * scale[r[ui]]))
    tot, cnt = {}, {}
    for name, us in recs:
        tot[name] = tot.get(name, 0.0) + us
        cnt[name] = cnt.get(name, 0) + 1
    T = sum(tot.values())
    text = f"# {title}\n\n"
    if command:
        text += f"Command (B200 box; the same command had just exited 0 without ncu):\n\n    {command}\n\n"
    text += (f"`{os.path.basename(out_csv)}` beside this file is that log reduced to (id, kernel, duration). {len(recs)} launches, "
             f"{T / 1e3:.2f} ms of kernel time; per-launch times under ncu are cold-cache and serialised, so compare SHARES with "
             "bench.py's `roofline.share_of_step`, not absolutes.\n\n")
    text += "| launches | total ms | share | avg us | kernel |\n|---|---|---|---|---|\n"
    for name in sorted(tot, key=lambda k: -tot[k]):
        text += f"| {cnt[name]} | {tot[name] / 1e3:.2f} | {100 * tot[name] / T:.1f} % | {tot[name] / cnt[name]:.1f} | `{name}` |\n"
    if note:
        text += "\n" + note + "\n"
    with open(out_md, "w") as f:
        f.write(text)
    with open(out_csv, "w") as f:
        f.write("id,kernel,duration_us\n")
        for k, (name, us) in enumerate(recs):
            f.write(f'{k},"{name}",{us:.2f}\n')


def sass_histogram(path, out_md, title, command, note, units, inst_executed=0.0):
    """`ncu -i x.ncu-rep --page source --csv [--kernel-name ... --launch-skip k --launch-count 1]` -> executed warp
    instructions per opcode and per `units` / 32 warp-units, the share of stall samples per opcode, and for the memory
    opcodes the L1 tag requests (global) or wavefronts (shared) per executed instruction."""
    import re
    rows = list(csv.reader(open(path)))
    kernel = rows[0][1] if rows and len(rows[0]) > 1 else ""
    hdr = next(r for r in rows if r and r[0] == "Address")
    ix = {n: i for i, n in enumerate(hdr)}
    data = [r for r in rows[rows.index(hdr) + 1:] if len(r) >= len(hdr) and to_float(r[ix["Instructions Executed"]]) is not None]
    ex, samp, tags, wav = {}, {}, {}, {}
    for r in data:
        m = re.match(r"\s*(@!?U?P\d+\s+)?([A-Z0-9_.]+)", r[ix["Source"]])
        op = (m.group(2) if m else "?").split(".")[0]
        n = to_float(r[ix["Instructions Executed"]])
        ex[op] = ex.get(op, 0.0) + n
        samp[op] = samp.get(op, 0.0) + (to_float(r[ix["# Samples"]]) or 0.0)
        tags[op] = tags.get(op, 0.0) + (to_float(r[ix["L1 Tag Requests Global"]]) or 0.0)
        wav[op] = wav.get(op, 0.0) + (to_float(r[ix["L1 Wavefronts Shared"]]) or 0.0)
    tot, ns, wu = sum(ex.values()), sum(samp.values()) or 1.0, units / 32.0
    # the source page can count a launch's instructions more than once (it did, twice, for the persistent tile kernel):
    # normalise to smsp__inst_executed.sum of the same launch when given
    if inst_executed > 0:
        f = inst_executed / tot
        ex = {k: v * f for k, v in ex.items()}
        tags = {k: v * f for k, v in tags.items()}
        wav = {k: v * f for k, v in wav.items()}
        tot = inst_executed
    text = f"# {title}\n\n"
    if command:
        text += f"Command:\n\n    {command}\n\n"
    text += f"Kernel: `{kernel.replace('void <unnamed>::', '').split('(Geom')[0]}`; {tot:.4g} warp instructions = {tot / wu:.1f} per 32 units ({units} units).\n\n"
    text += "| opcode | per 32 units | share of instructions | share of stall samples | L1 tag requests / shared wavefronts per instruction |\n|---|---|---|---|---|\n"
    for op in sorted(ex, key=lambda k: -ex[k]):
        if ex[op] / tot < 0.002:
            continue
        mem = f"{tags[op] / ex[op]:.2f} tags" if tags[op] else (f"{wav[op] / ex[op]:.2f} wavefronts" if wav[op] else "")
        text += f"| {op} | {ex[op] / wu:.1f} | {100 * ex[op] / tot:.1f} % | {100 * samp[op] / ns:.1f} % | {mem} |\n"
    if note:
        text += "\n" + note + "\n"
    with open(out_md, "w") as f:
        f.write(text)


def main():
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("csv")
    ap.add_argument("--sass-histogram", type=int, metavar="UNITS", help="treat `csv` as an ncu source-page csv of ONE launch that processed UNITS (site, source) units; markdown to --out")
    ap.add_argument("--inst-executed", type=float, default=0.0, help="smsp__inst_executed.sum of that launch (raw page): the histogram is normalised to it")
    ap.add_argument("--launch-list", help="treat `csv` as an ncu gpu__time_duration log; write the reduced csv here (markdown to --out)")
    ap.add_argument("--out", help="markdown file to write (default: stdout)")
    ap.add_argument("--title", default="ncu summary")
    ap.add_argument("--command", default="", help="the full command that made the capture (named in the file)")
    ap.add_argument("--note", default="")
    ap.add_argument("--traffic", help="JSON file to update with the mean DRAM bytes per launch")
    ap.add_argument("--key", help="entry of the JSON file: workload/prec/nrhsN")
    ap.add_argument("--commit", default="", help="commit of the kernels the capture was taken at")
    a = ap.parse_args()
    if a.sass_histogram:
        if not a.out:
            raise SystemExit("--sass-histogram needs --out")
        sass_histogram(a.csv, a.out, a.title, a.command, a.note, a.sass_histogram, a.inst_executed)
        return
    if a.launch_list:
        if not a.out:
            raise SystemExit("--launch-list needs --out")
        launch_list(a.csv, a.out, a.launch_list, a.title, a.command, a.note)
        return
    hdr, units, rows = read_rows(a.csv)
    per = dram_bytes(hdr, units, rows)
    text = f"# {a.title}\n\n"
    if a.command:
        text += f"Command (B200 box; the same command had just exited 0 without ncu):\n\n    {a.command}\n\n"
    text += f"read with `ncu -i <report>.ncu-rep --page raw --csv`, summarised by `python -m paper_1211_0126_b200.ncu_summary`.\n\n"
    text += table(hdr, units, rows) + "\n\n"
    text += "DRAM bytes per launch (read + write): " + ", ".join(f"{b / 1e9:.3f} GB" for b in per) + f"; mean {sum(per) / len(per) / 1e9:.3f} GB.\n"
    if a.note:
        text += "\n" + a.note + "\n"
    if a.out:
        with open(a.out, "w") as f:
            f.write(text)
    else:
        print(text)
    if a.traffic:
        if not a.key:
            raise SystemExit("--traffic needs --key")
        d = json.load(open(a.traffic)) if os.path.exists(a.traffic) else {}
        idx = {h: i for i, h in enumerate(hdr)}
        d[a.key] = {"bytes_per_launch": sum(per) / len(per), "per_launch": per, "commit": a.commit,
                    "summary": a.out or "", "kernels": sorted({r[idx["Kernel Name"]].replace("void <unnamed>::", "").split("(")[0] for r in rows})}
        with open(a.traffic, "w") as f:
            json.dump(d, f, indent=1, sort_keys=True)
            f.write("\n")


if __name__ == "__main__":
    main()
