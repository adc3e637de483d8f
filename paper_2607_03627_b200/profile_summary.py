"""Turn an Nsight Compute report of bench.py into the tracked artefacts under profiles/.

    python -m paper_2607_03627_b200.profile_summary gpurun_out/r02c_full.ncu-rep --tag r02c --config 3 \
        --command "ncu --set full ... python bench.py ..."

writes
    profiles/<tag>_summary.md     one table row per captured launch of the attempt kernels (duration, DRAM bytes, L2 sectors,
                                  issue utilisation, stall reasons), the command that made the report
    profiles/r02_traffic.json     {"uc_config<N>": {"k_primal": bytes, "k_dual": bytes, "source": ...}}: DRAM read + write
                                  bytes per launch (mean over the captured launches), which bench.py reports as
                                  roofline.traffic -- so that number is tied to a tracked capture, not typed in by hand.
Needs the `ncu` command line tool (it only READS the report; nothing is profiled here)."""
from __future__ import annotations

import argparse
import csv
import io
import json
import os
import subprocess

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

METRICS = [
    ("gpu__time_duration.sum", "us"),
    ("dram__bytes_read.sum", "DRAM read"),
    ("dram__bytes_write.sum", "DRAM write"),
    ("gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed", "DRAM % of peak"),
    ("lts__t_sectors_srcunit_tex.sum", "L2 sectors from SMs"),
    ("lts__t_sector_hit_rate.pct", "L2 hit %"),
    ("l1tex__t_sector_hit_rate.pct", "L1 hit %"),
    ("smsp__inst_executed.sum", "warp instructions"),
    ("smsp__issue_active.avg.pct_of_peak_sustained_active", "issue active %"),
    ("smsp__cycles_active.avg", "SMSP cycles active (avg)"),
    ("sm__cycles_elapsed.max", "SM cycles elapsed"),
    ("launch__registers_per_thread", "registers"),
    ("launch__shared_mem_per_block_dynamic", "dynamic smem"),
]


def read_raw(report: str):
    out = subprocess.run(["ncu", "-i", report, "--page", "raw", "--csv"], capture_output=True, text=True, check=True).stdout
    rows = list(csv.reader(io.StringIO(out)))
    return rows[0], rows[1], rows[2:]


def sass_mix(report: str, kernel: str):
    """Executed warp instructions by opcode for the first captured launch of `kernel` (ncu source page, SASS view) and
    the number of pipeline steps it ran (= executed LDGDEPBAR, one cp.async.commit_group per step)."""
    out = subprocess.run(["ncu", "-i", report, "--page", "source", "--csv", "--kernel-name", f"regex:{kernel}"],
                         capture_output=True, text=True, check=True).stdout
    rows = list(csv.reader(io.StringIO(out)))
    heads = [i for i, r in enumerate(rows) if r and r[0] == "Address"]
    if not heads:
        return None
    hdr = rows[heads[0]]
    body = [r for r in rows[heads[0] + 1:(heads[1] - 1 if len(heads) > 1 else None)] if r and r[0].startswith("0x")]
    ie, isrc = hdr.index("Instructions Executed"), hdr.index("Source")
    mix, total = {}, 0
    for r in body:
        try:
            e = int(r[ie])
        except ValueError:
            continue
        w = r[isrc].split()
        op = (w[1] if w[0].startswith("@") else w[0]).split(".")[0]
        mix[op] = mix.get(op, 0) + e
        total += e
    return total, mix, len(body)


def aggregate_launches(raw_csv: str, out_csv: str):
    """Per-kernel aggregation of an `ncu --metrics gpu__time_duration.sum --csv` launch list: launches, mean and total
    duration, share of the total (cold-cache, serialised launches: compare shares, not absolute times)."""
    rows = [r for r in csv.reader(open(raw_csv)) if len(r) > 10]
    hdr = rows[0]
    ik, iv, iu, im = hdr.index("Kernel Name"), hdr.index("Metric Value"), hdr.index("Metric Unit"), hdr.index("Metric Name")
    agg = {}
    for r in rows[1:]:
        if r[im] != "gpu__time_duration.sum":
            continue
        us = float(r[iv].replace(",", "")) * {"ns": 1e-3, "us": 1.0, "ms": 1e3}.get(r[iu], 1e-3)
        a = agg.setdefault(r[ik].split("(")[0], [0, 0.0])
        a[0] += 1; a[1] += us
    total = sum(v[1] for v in agg.values()) or 1.0
    with open(out_csv, "w") as f:
        f.write("kernel,launches,mean_us,total_us,share_pct\n")
        for k, (n, t) in sorted(agg.items(), key=lambda kv: -kv[1][1]):
            f.write(f"{k},{n},{t / n:.2f},{t:.1f},{100 * t / total:.2f}\n")
    return agg


def to_bytes(value: str, unit: str) -> float:
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
    return float(value) * scale.get(unit, 1.0)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("report")
    ap.add_argument("--tag", required=True)
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--command", default="", help="the full command that produced the report (recorded in the summary)")
    ap.add_argument("--launches", default="", help="raw `ncu --metrics gpu__time_duration.sum --csv` launch list to aggregate into profiles/<tag>_launches.csv")
    ap.add_argument("--launches-command", default="")
    args = ap.parse_args()
    hdr, units, data = read_raw(args.report)
    col = {h: i for i, h in enumerate(hdr)}
    lines = [f"# {args.tag}: Nsight Compute capture of the attempt kernels (UC config {args.config})", ""]
    if args.command:
        lines += ["Command (one B200 under gpurun, after the same command exited 0 without ncu):", "", "```", args.command, "```", ""]
    lines += ["Report read here with `python -m paper_2607_03627_b200.profile_summary` (`ncu -i <report> --page raw --csv`).", ""]
    names = [m for m, _ in METRICS if m in col]
    lines += ["| launch | kernel | " + " | ".join(dict(METRICS)[m] for m in names) + " | top stall reasons (share of samples) |",
              "|---|---|" + "---|" * (len(names) + 1)]
    traffic = {}
    for k, d in enumerate(data):
        kern = d[col["Kernel Name"]].split("(")[0]
        cells = []
        for m in names:
            v, u = d[col[m]], units[col[m]]
            try:
                cells.append(f"{float(v):,.2f} {u}".strip() if "." in v and float(v) < 1e6 else f"{float(v):,.0f} {u}".strip())
            except ValueError:
                cells.append(v)
        stalls = []
        for h in hdr:
            if "pcsamp_warps_issue_stalled" in h and "_not_issued" not in h:
                try:
                    stalls.append((float(d[col[h]]), h.replace("smsp__pcsamp_warps_issue_stalled_", "")))
                except ValueError:
                    pass
        tot = sum(v for v, _ in stalls) or 1.0
        top = ", ".join(f"{n} {100 * v / tot:.0f}%" for v, n in sorted(stalls, reverse=True)[:6])
        lines.append(f"| {k} | {kern} | " + " | ".join(cells) + f" | {top} |")
        if "dram__bytes_read.sum" in col:
            b = to_bytes(d[col["dram__bytes_read.sum"]], units[col["dram__bytes_read.sum"]]) + \
                to_bytes(d[col["dram__bytes_write.sum"]], units[col["dram__bytes_write.sum"]])
            traffic.setdefault(kern, []).append(b)
    lines += ["", "## Executed SASS of the first captured launch of each kernel (ncu source page, `--import-source on`)", "",
              "A pipeline step = 32 rows x up to 4 entries (one `cp.async.commit_group`, SASS `LDGDEPBAR`, per step).", "",
              "| kernel | static SASS instructions | warp instructions executed | steps | per step | asynchronous copies `LDGSTS` | plain loads `LDG` | stores `STG` | "
              "TMA (`UBLKCP` / `UTMALDG`) | most executed opcodes per step |", "|---|---|---|---|---|---|---|---|---|---|"]
    for kern in ("k_primal", "k_dual"):
        m = sass_mix(args.report, kern)
        if not m:
            continue
        total, mix, nstatic = m
        steps = max(mix.get("LDGDEPBAR", 0), 1)
        top = ", ".join(f"{op} {c / steps:.1f}" for op, c in sorted(mix.items(), key=lambda kv: -kv[1])[:12])
        lines.append(f"| {kern} | {nstatic:,} | {total:,} | {steps:,} | {total / steps:.0f} | {mix.get('LDGSTS', 0):,} | {mix.get('LDG', 0):,} | "
                     f"{mix.get('STG', 0):,} | {mix.get('UBLKCP', 0) + mix.get('UTMALDG', 0)} | {top} |")
    os.makedirs(os.path.join(ROOT, "profiles"), exist_ok=True)
    if args.launches:
        agg = aggregate_launches(args.launches, os.path.join(ROOT, "profiles", f"{args.tag}_launches.csv"))
        total = sum(v[1] for v in agg.values()) or 1.0
        lines += ["", f"## Launch list (`profiles/{args.tag}_launches.csv`)", ""]
        if args.launches_command:
            lines += ["```", args.launches_command, "```", ""]
        lines += ["Cold-cache, serialised launches: the SHARE of a kernel is what compares with the un-profiled run, not its absolute time.", "",
                  "| kernel | launches | mean us | share of the kernel time |", "|---|---|---|---|"]
        for k, (n, t) in sorted(agg.items(), key=lambda kv: -kv[1][1]):
            lines.append(f"| {k} | {n} | {t / n:.2f} | {100 * t / total:.2f} % |")
    with open(os.path.join(ROOT, "profiles", f"{args.tag}_summary.md"), "w") as f:
        f.write("\n".join(lines) + "\n")
    tpath = os.path.join(ROOT, "profiles", "r02_traffic.json")
    try:
        allt = json.load(open(tpath))
    except Exception:
        allt = {}
    allt[f"uc_config{args.config}"] = {k: int(sum(v) / len(v)) for k, v in traffic.items()}
    allt[f"uc_config{args.config}"]["source"] = f"profiles/{args.tag}_summary.md (dram__bytes_read.sum + dram__bytes_write.sum, mean over {len(data)} captured launches, cold L2 per replay)"
    with open(tpath, "w") as f:
        json.dump(allt, f, indent=1)
        f.write("\n")
    print(f"wrote profiles/{args.tag}_summary.md and profiles/r02_traffic.json")


if __name__ == "__main__":
    main()
