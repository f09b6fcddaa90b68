"""ORACLE (test infrastructure) — algorithmic operation count of the hot path (F_alg of SURVEY.md 8(d)).

    python -m oracle.count_ops            # writes tests/golden/op_counts.json

Runs the operation-counting build of the oracle (orc_count.cpp: the same sources, `double` replaced by a counting
wrapper; no FMA can form) on a 16^3 instance of each workload and records, per interior zone and per step of the path,
how many add/sub, mul, div, sqrt, compare/min/max and transcendental operations the algorithm performs when it is
written out term by term as in the paper. Every operation counts as one flop. The oracle does not share
subexpressions between steps (e.g. it recomputes derivatives for the fluid sources and 1/(12 h) per stencil), so this
is an upper estimate of the work a fused implementation needs; bench.py reports it beside the FP64 instruction
counts measured by ncu (profiles/).
"""
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from paper_2510_13965_b200 import synth  # noqa: E402


def count(cfg):
    oracle.use_counting(True)
    try:
        n = cfg["n"]
        zones = n[0] * n[1] * n[2]
        o = oracle.Oracle(cfg["params"], n[0], n[1], n[2], cfg["ng"], cfg["dx"], table=cfg.get("table"))
        U, P = cfg["U"].copy(), cfg["P"].copy()
        o.prim2con(U, P)
        o.fill_ghosts(U, cfg["bc"])

        def run(fn, per):
            oracle.count_reset()
            r = fn()
            c = oracle.count_get()
            c = {k: v / per for k, v in c.items()}
            c["flops"] = sum(c.values())
            return r, c

        out = {"zones": zones, "points": o.npts}
        (Pp, _), out["con2prim_per_point"] = run(lambda: o.con2prim(U), o.npts)
        _, out["ccz4_per_zone"] = run(lambda: o.rhs(U, Pp, "ccz4"), zones)
        _, out["grmhd_flux_per_zone"] = run(lambda: o.rhs(U, Pp, "grmhd_flux"), zones)
        _, out["grmhd_src_per_zone"] = run(lambda: o.rhs(U, Pp, "grmhd_src"), zones)
        # advective + KO part of the CCZ4 RHS: 22 fields x 3 axes x (beta * dadv + add) and (dko + add)
        u = np.linspace(0.0, 1.0, 7) ** 2
        _, adv = run(lambda: oracle.stencil("dadv", u, 1, 0.1, 0.3), 1)
        _, ko = run(lambda: oracle.stencil("dko", u, 1, 0.1, 0.1), 1)
        out["adv_ko_per_zone"] = {"flops": 22 * 3 * (adv["flops"] + 2 + ko["flops"] + 1)}
        K = [np.zeros_like(U)]
        _, out["rk_combine_per_zone_per_term"] = run(lambda: o.rk_combine(U, K, [0.5], 0.1), zones)
        if "V" in cfg:                   # grey M1, 3 species: implicit solve per point, explicit part per zone
            V = cfg["V"].copy()
            o.fill_ghosts(V, cfg["bc"])
            (_, _), out["m1_implicit_per_point"] = run(lambda: o.m1_implicit(U, Pp, V, 0.25 * 0.25 * cfg["dx"]), o.npts)
            _, out["m1_rhs_per_zone"] = run(lambda: o.m1_rhs(U, Pp, V), zones)
        ratio = o.npts / zones
        out["per_zone_stage_flops"] = (out["con2prim_per_point"]["flops"] * ratio + out["ccz4_per_zone"]["flops"]
                                       + out["grmhd_flux_per_zone"]["flops"] + out["grmhd_src_per_zone"]["flops"]
                                       + 2.5 * out["rk_combine_per_zone_per_term"]["flops"])
        if "V" in cfg:
            out["per_zone_stage_flops"] += out["m1_implicit_per_point"]["flops"] * ratio + out["m1_rhs_per_zone"]["flops"]
        return out
    finally:
        oracle.use_counting(False)


def main():
    res = {"c1": count(synth.config1(n=16)), "c3": count(synth.config3(n=16)), "c4": count(synth.config4(n=16)),
           "c5": count(synth.config5(n=16, crop_on_star=True))}
    path = os.path.join(ROOT, "tests", "golden", "op_counts.json")
    with open(path, "w") as f:
        json.dump(res, f, indent=1, sort_keys=True)
    for k, v in res.items():
        print(k, "flops per zone-stage: %.0f" % v["per_zone_stage_flops"],
              {a: round(b["flops"]) for a, b in v.items() if isinstance(b, dict)})


if __name__ == "__main__":
    main()
