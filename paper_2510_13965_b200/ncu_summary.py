"""Turns `ncu -i <report>.ncu-rep --page raw --csv` (a `--set full` capture of one RK stage of bench.py) into the per-kernel JSON that
bench.py reads for `roofline.traffic` and the executed-FP64 figures, and into the markdown table kept under profiles/.

    ncu -i gpurun_out/prof.ncu-rep --page raw --csv > raw.csv
    python -m paper_2510_13965_b200.ncu_summary raw.csv --zones 2097152 --points 2406104 --commit <hash> --command "<the ncu command>" \
        --json profiles/r2_ncu_c4_128.json --md profiles/r2_ncu_c4_128.md

Per kernel class (the classes of mhd_patch_profile_read): duration, DRAM bytes per zone (dram__bytes_read.sum + dram__bytes_write.sum),
FP64-pipe utilisation (sm__inst_executed_pipe_fp64), executed thread-level FP64 flops per zone (DADD + DMUL + 2 DFMA, predicated-on), registers,
top stall reasons. Nothing here runs on the hot path."""
import argparse
import csv
import json

CLASS_OF = [("k_fill_ghosts", "fill_ghosts"), ("k_con2prim", "con2prim"), ("k_ccz4_algebra", "ccz4_algebra"), ("k_recon_x", "recon_x"),
            ("k_recon_march<1", "recon_y"), ("k_recon_march<2", "recon_z"), ("k_rk_combine", "rk_combine"), ("k_copy", "rk_combine"),
            ("k_point_flux", "point_flux"), ("k_adv_ko", "adv_ko"), ("k_les", "les"), ("k_m1_point", "m1_point"), ("k_m1_div", "m1_div"),
            ("k_m1_march", "m1_div"), ("k_m1_implicit", "m1_implicit"), ("k_m1_backreact", "m1_implicit"), ("k_m1_gravity", "m1_implicit")]


def kernel_class(name):
    for key, cls in CLASS_OF:
        if key in name:
            return cls
    return None


def _num(x):
    try:
        return float(x.replace(",", ""))
    except ValueError:
        return None


def summarise(path, zones, points):
    rows = list(csv.reader(open(path)))
    hdr, units, body = rows[0], rows[1], rows[2:]
    col = {h: i for i, h in enumerate(hdr)}

    def get(r, name, scale_units=True):
        if name not in col:
            return None
        v = _num(r[col[name]])
        if v is None or not scale_units:
            return v
        u = units[col[name]].lower()
        mult = {"gbyte": 1e9, "mbyte": 1e6, "kbyte": 1e3, "byte": 1.0, "us": 1.0, "ms": 1e3, "ns": 1e-3, "s": 1e6}.get(u, 1.0)
        return v * mult

    stall_cols = [h for h in hdr if h.startswith("smsp__average_warps_issue_stalled") and h.endswith("per_issue_active.ratio")]
    out = {}
    for r in body:
        name = r[col["Kernel Name"]]
        cls = kernel_class(name)
        if cls is None:
            continue
        cyc = get(r, "smsp__cycles_elapsed.avg") or get(r, "sm__cycles_elapsed.max")
        flops = None
        parts = [get(r, "smsp__sass_thread_inst_executed_op_%s_pred_on.sum.per_cycle_elapsed" % k) for k in ("dadd", "dmul", "dfma")]
        if cyc and all(p is not None for p in parts):
            flops = (parts[0] + parts[1] + 2.0 * parts[2]) * cyc
        per = points if cls in ("fill_ghosts",) else zones
        stalls = sorted(((_num(r[col[h]]) or 0.0, h.split("stalled_")[1].split("_per")[0]) for h in stall_cols), reverse=True)[:4]
        e = {"kernel": name[:80], "time_us": get(r, "gpu__time_duration.sum"), "registers": get(r, "launch__registers_per_thread", False),
             "dram_bytes": (get(r, "dram__bytes_read.sum") or 0.0) + (get(r, "dram__bytes_write.sum") or 0.0),
             "fp64_pipe_pct": get(r, "sm__inst_executed_pipe_fp64.avg.pct_of_peak_sustained_active", False),
             "dram_pct": get(r, "gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed", False),
             "warps_active_pct": get(r, "sm__warps_active.avg.pct_of_peak_sustained_active", False),
             "issue_active_pct": get(r, "smsp__issue_active.avg.pct_of_peak_sustained_active", False),
             "executed_fp64_flops": flops, "top_stalls": ["%s=%.2f" % (n, v) for v, n in stalls]}
        e["dram_bytes_per_zone"] = e["dram_bytes"] / per
        e["executed_fp64_flops_per_zone"] = flops / zones if flops is not None else None
        if cls in out:                               # several launches of a class in the capture: keep the sum
            o = out[cls]
            for k in ("time_us", "dram_bytes", "dram_bytes_per_zone", "executed_fp64_flops", "executed_fp64_flops_per_zone"):
                if o[k] is not None and e[k] is not None:
                    o[k] += e[k]
            o["launches"] += 1
        else:
            e["launches"] = 1
            out[cls] = e
    return out


def markdown(kern, meta):
    lines = ["# ncu --set full summary: %s" % meta.get("title", ""), "", "Command (on a B200 via gpurun, after the same command exited 0 without ncu):", "",
             "    " + meta.get("command", ""), "", "commit %s, %d zones, %d grid points per launch" % (meta.get("commit"), meta["zones"], meta["points"]), "",
             "| class | kernel | launches | time us | regs | DRAM B/zone | DRAM % | FP64 pipe % | executed FP64 flop/zone | warps active % | issue active % | top stalls |",
             "|---|---|---|---|---|---|---|---|---|---|---|---|"]
    for cls, e in kern.items():
        lines.append("| %s | `%s` | %d | %.1f | %s | %.1f | %s | %s | %s | %s | %s | %s |" % (
            cls, e["kernel"].replace("|", "/")[:48], e["launches"], e["time_us"], e["registers"], e["dram_bytes_per_zone"], e["dram_pct"], e["fp64_pipe_pct"],
            "%.0f" % e["executed_fp64_flops_per_zone"] if e["executed_fp64_flops_per_zone"] is not None else "-", e["warps_active_pct"],
            e["issue_active_pct"], " ".join(e["top_stalls"])))
    tot = sum(e["dram_bytes_per_zone"] for c, e in kern.items())
    lines += ["", "Sum of DRAM bytes per zone over the captured launches: %.0f B (algorithmic 1280 B per zone-stage)." % tot]
    return "\n".join(lines) + "\n"


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("raw_csv")
    ap.add_argument("--zones", type=int, required=True)
    ap.add_argument("--points", type=int, required=True)
    ap.add_argument("--commit", default="unknown")
    ap.add_argument("--command", default="")
    ap.add_argument("--title", default="")
    ap.add_argument("--json")
    ap.add_argument("--md")
    a = ap.parse_args()
    kern = summarise(a.raw_csv, a.zones, a.points)
    meta = {"commit": a.commit, "command": a.command, "zones": a.zones, "points": a.points, "title": a.title}
    if a.json:
        json.dump({"meta": meta, "kernels": kern}, open(a.json, "w"), indent=1)
    if a.md:
        open(a.md, "w").write(markdown(kern, meta))
    if not a.json and not a.md:
        print(json.dumps({"meta": meta, "kernels": kern}, indent=1))


if __name__ == "__main__":
    main()
