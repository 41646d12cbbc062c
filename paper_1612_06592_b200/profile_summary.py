"""Post-processing of an `ncu --set full` capture into the text/JSON summaries kept under profiles/.

    python -m paper_1612_06592_b200.profile_summary <capture.ncu-rep> --bench <bench line .json> --tag r2_x
        [--json profiles/ncu_summary.json] [--md profiles/r2_x_ncu_full.md]

Reads the raw page of the capture (ncu -i ... --page raw --csv), takes per kernel the DRAM bytes, the busiest
units and the instruction count, joins them with the algorithmic bytes per launch that bench.py printed for the same
build and workload, and (a) updates profiles/ncu_summary.json, the file bench.py reads `roofline.traffic` and
`roofline.limiter` from, (b) writes a markdown table.  Nothing here runs on the GPU."""
from __future__ import annotations

import argparse
import csv
import io
import json
import os
import re
import subprocess

METRICS = [
    "gpu__time_duration.sum", "launch__grid_size", "launch__registers_per_thread", "dram__bytes_read.sum",
    "dram__bytes_write.sum", "gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed",
    "smsp__issue_active.avg.pct_of_peak_sustained_active", "sm__pipe_fma_cycles_active.avg.pct_of_peak_sustained_active",
    "sm__inst_executed_pipe_alu.avg.pct_of_peak_sustained_active", "sm__inst_executed_pipe_lsu.avg.pct_of_peak_sustained_active",
    "sm__pipe_tensor_cycles_active.avg.pct_of_peak_sustained_active", "smsp__inst_executed.sum",
    "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum", "l1tex__throughput.avg.pct_of_peak_sustained_elapsed",
    "lts__throughput.avg.pct_of_peak_sustained_elapsed", "lts__t_sector_hit_rate.pct",
]
LIMITERS = {"gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed": "dram",
            "smsp__issue_active.avg.pct_of_peak_sustained_active": "issue slots",
            "sm__pipe_fma_cycles_active.avg.pct_of_peak_sustained_active": "fp32 (FMA) pipe",
            "l1tex__throughput.avg.pct_of_peak_sustained_elapsed": "l1tex / shared-memory data path",
            "lts__throughput.avg.pct_of_peak_sustained_elapsed": "L2",
            "sm__pipe_tensor_cycles_active.avg.pct_of_peak_sustained_active": "tensor pipe"}


def short(name: str) -> str:
    m = re.search(r"(\w+_kernel)", name)
    return m.group(1) if m else name


def read_raw(rep: str):
    out = subprocess.run(["ncu", "-i", rep, "--page", "raw", "--csv"], capture_output=True, text=True, check=True).stdout
    rows = list(csv.reader(io.StringIO(out)))
    hdr, units = rows[0], rows[1]
    res = []
    for r in rows[2:]:
        d = {"name": short(r[hdr.index("Kernel Name")])}
        for m in METRICS:
            if m in hdr:
                v = r[hdr.index(m)].replace(",", "")
                try:
                    d[m] = float(v)
                except ValueError:
                    d[m] = None
                d[m + "#unit"] = units[hdr.index(m)]
        res.append(d)
    return res


def phases(rep: str, kernel: str, min_share: float = 0.01):
    """Warp-stall samples of `kernel` from the source page of the capture (ncu -i ... --page source --csv), summed over
    the stretches of SASS between barriers (BAR / SYNCS / EXIT): one row per stretch with its share of the samples, the
    warp instructions executed, the most frequent opcodes and the most frequent stall reasons."""
    out = subprocess.run(["ncu", "-i", rep, "--page", "source", "--csv", "--kernel-name", f"regex:{kernel}"],
                         capture_output=True, text=True).stdout
    rows = list(csv.reader(io.StringIO(out)))
    start = next((i for i, r in enumerate(rows) if r and r[0] == "Address"), None)
    if start is None:
        return []
    hdr = rows[start]
    ix = {h: i for i, h in enumerate(hdr)}
    stalls = [h for h in hdr if h.startswith("stall_") and "Not Issued" not in h]
    data = []
    for r in rows[start + 1:]:
        if len(r) != len(hdr) or r[0] == "Address":
            break                                   # the next launch of the same kernel
        data.append(r)
    total = sum(int(r[ix["# Samples"]] or 0) for r in data) or 1
    segs, cur = [], None

    def new(i):
        return {"first": i, "samples": 0, "exec": 0, "ops": {}, "stalls": {}}
    cur = new(0)
    for i, r in enumerate(data):
        words = r[ix["Source"]].split()
        op = words[1] if words and words[0].startswith("@") and len(words) > 1 else (words[0] if words else "")
        cur["samples"] += int(r[ix["# Samples"]] or 0)
        e = int(r[ix["Instructions Executed"]] or 0)
        cur["exec"] += e
        cur["ops"][op.split(".")[0]] = cur["ops"].get(op.split(".")[0], 0) + e
        for st in stalls:
            cur["stalls"][st[6:]] = cur["stalls"].get(st[6:], 0) + int(r[ix[st]] or 0)
        if op.startswith(("BAR", "SYNCS", "EXIT")):
            cur["last"] = i
            segs.append(cur)
            cur = new(i + 1)
    cur["last"] = len(data) - 1
    segs.append(cur)
    res = []
    for sg in segs:
        if sg["samples"] / total < min_share:
            continue
        top = sorted(sg["ops"].items(), key=lambda x: -x[1])[:5]
        st = sorted(sg["stalls"].items(), key=lambda x: -x[1])[:4]
        res.append({"sass": f"{sg['first']}-{sg['last']}", "share": sg["samples"] / total, "warp_instr": sg["exec"],
                    "top_ops": ", ".join(f"{k} {v / 1e6:.0f}M" for k, v in top if v),
                    "top_stalls": ", ".join(f"{k} {v / max(1, sg['samples']):.0%}" for k, v in st if v)})
    return res


def to_bytes(v, unit):
    mult = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}.get(unit, 1.0)
    return None if v is None else v * mult


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("rep")
    ap.add_argument("--bench", required=True, help="JSON line printed by bench.py for the same build and workload")
    ap.add_argument("--tag", required=True)
    ap.add_argument("--json", default=os.path.join("profiles", "ncu_summary.json"))
    ap.add_argument("--md", default=None)
    ap.add_argument("--command", default="", help="the command line that made the capture (recorded in the summary)")
    ap.add_argument("--phases", default="", help="kernel name (regex) whose warp-stall samples are split at its barriers")
    args = ap.parse_args()
    bench = json.loads(open(args.bench).read().strip().splitlines()[-1])
    cfg = re.match(r"(configs\[\d\])", bench["config"]["workload"]).group(1)
    alg = {k["kernel"]: k["algorithmic_GB_per_launch"] for k in bench["kernels"]}
    kernels = read_raw(args.rep)
    summary = json.load(open(args.json)) if os.path.exists(args.json) else {}
    entry = summary.setdefault(cfg, {})
    lines = [f"# {args.tag}: ncu --set full, {bench['config']['workload']}", ""]
    if args.command:
        lines += ["Command (under gpurun on one B200, directly after the same command exited 0 without ncu):", "",
                  "```", args.command, "```", ""]
    lines += ["| metric | " + " | ".join(k["name"] for k in kernels) + " |", "|---|" + "---|" * len(kernels)]
    for m in METRICS:
        lines.append(f"| {m} [{kernels[0].get(m + '#unit', '')}] | " +
                     " | ".join("" if k.get(m) is None else f"{k[m]:.6g}" for k in kernels) + " |")
    for k in kernels:
        rd = to_bytes(k.get("dram__bytes_read.sum"), k.get("dram__bytes_read.sum#unit"))
        wr = to_bytes(k.get("dram__bytes_write.sum"), k.get("dram__bytes_write.sum#unit"))
        pct = {n: k.get(m) or 0.0 for m, n in LIMITERS.items()}
        lim = max(pct, key=pct.get)
        e = {"dram_GB_per_launch": (rd + wr) / 1e9 if rd is not None and wr is not None else None,
             "algorithmic_GB_per_launch": alg.get(k["name"]),
             "limiter": f"{lim} ({pct[lim]:.0f} % busy; " + ", ".join(f"{n} {v:.0f} %" for n, v in pct.items() if n != lim) + ")",
             "fma_pipe_frac": pct["fp32 (FMA) pipe"] / 100.0, "issue_frac": pct["issue slots"] / 100.0,
             "warp_instructions": k.get("smsp__inst_executed.sum"), "source": args.tag}
        entry[k["name"]] = e
        if e["dram_GB_per_launch"] and e["algorithmic_GB_per_launch"]:
            lines.append("")
            lines.append(f"{k['name']}: DRAM traffic {e['dram_GB_per_launch']:.3f} GB per launch vs "
                         f"{e['algorithmic_GB_per_launch']:.3f} GB algorithmic (ratio "
                         f"{e['dram_GB_per_launch'] / e['algorithmic_GB_per_launch']:.3f}); busiest unit: {e['limiter']}.")
    if args.phases:
        ph = phases(args.rep, args.phases)
        if ph:
            lines += ["", f"{args.phases}: warp-stall samples between barriers (source page of the same capture, first "
                          "launch; SASS line ranges of this build):", "",
                      "| SASS lines | share of samples | warp instructions | most executed opcodes | top stall reasons |",
                      "|---|---|---|---|---|"]
            lines += [f"| {p['sass']} | {p['share']:.1%} | {p['warp_instr'] / 1e6:.1f} M | {p['top_ops']} | {p['top_stalls']} |"
                      for p in ph]
    os.makedirs(os.path.dirname(args.json) or ".", exist_ok=True)
    json.dump(summary, open(args.json, "w"), indent=1, sort_keys=True)
    md = args.md or os.path.join("profiles", f"{args.tag}_ncu_full.md")
    open(md, "w").write("\n".join(lines) + "\n")
    print(md, args.json)


if __name__ == "__main__":
    main()
