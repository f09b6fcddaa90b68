#!/usr/bin/env python
"""bench.py — zone-stage updates/s of the MHDuet per-stage hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c1|c3|c4] [--n SIZE] [--impl ours|reference]

A "step" is one full explicit RK4 time step of one patch = 4 passes of the whole hot path
(fill_ghosts -> con2prim -> rhs -> rk_stage), so one step performs 4 * n^3 zone-stage updates.
N > 1 (torchrun): the path does not shard (north_star: no multi-GPU decomposition) -> N independent replicas,
weak scaling, value = sum over ranks / max-over-ranks time.

One JSON line is printed by rank 0; see DESIGN.md "Measurement" for the roofline arithmetic.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "zone-stage updates/s"
STAGES = 4


def workload_inputs(name, n, les_cm=0.0, les_other=0.0):
    """Seeded synthetic inputs (paper_2510_13965_b200.synth); returns cfg dict with U (metric, Bbar), P (rho, Ye, eps, v)."""
    from paper_2510_13965_b200 import synth
    if name == "c1" and les_cm != 0.0:      # LES sub-grid-scale term on (App. A, C_M): ghost width 5, ideal gas
        cfg = synth.config1_tiled(n, ng=5)
        cfg["params"].update(les_C_M=les_cm, les_C_N=les_other, les_C_Y=les_other, les_C_T=les_other)
        return cfg
    if name == "c4" and les_cm != 0.0:      # the paper's production setting: tabulated EoS + C_M = 8
        cfg = synth.config4(n=n, ng=5)
        cfg["params"].update(les_C_M=les_cm, les_C_N=les_other, les_C_Y=les_other, les_C_T=les_other)
        return cfg
    if les_cm != 0.0:
        raise ValueError("--les-cm is available for the workloads c1 and c4")
    if name == "c1":
        return synth.config1_tiled(n)
    if name == "c3":
        return synth.config3(n=n)
    if name == "c4":
        return synth.config4(n=n)
    if name == "c5":                    # two stars + M1 on the full half-width-60 patch (0.3 % star)
        return synth.config5(n=n)
    if name == "c5crop":                # the same state on a patch centred on one star (40 % star): exercises the stiff cores
        return synth.config5(n=n, crop_on_star=True)
    raise ValueError(name)


def max_over_ranks(value, device=None):
    """Replicas-only scaling: the only exchange of the N > 1 path is this reduction of the timed
    region over ranks (MAX), after which value = world * units / time. Works on any torch.distributed backend."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_throughput(world, zones, stages, steps, ms_max):
    """whole-job zone-stage updates per second of `world` independent replicas (weak scaling)"""
    return world * zones * stages * steps / (ms_max * 1e-3)


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms during the timed region."""
    Q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        sm = [float(r[0]) for r in self.rows if len(r) >= 7 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 7 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [nm for i, nm in enumerate(names) if any(len(r) >= 7 and r[3 + i].lower().startswith("active") for r in self.rows)]
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None, "reasons": reasons,
                "samples": len(sm)}


def cpu_info():
    model = "unknown"
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                model = line.split(":", 1)[1].strip()
                break
    except OSError:
        pass
    return {"nproc": os.cpu_count() or 1, "cpu_model": model}


def oracle_leg(cfg_name, n_sample, steps, threads=1, les_cm=0.0, les_other=0.0):
    """The oracle as it stands on a bounded sample of the workload: threads = 1 is the plain single-threaded build, threads > 1 the
    -fopenmp build of the same sources (outermost grid loops only, arithmetic unchanged); returns (value, seconds, zone_stages, threads)."""
    import oracle
    from paper_2510_13965_b200 import synth
    threads = oracle.use_threads(threads)
    cfg = workload_inputs(cfg_name, n_sample, les_cm, les_other)
    n = cfg["n"]
    o = oracle.Oracle(cfg["params"], n[0], n[1], n[2], cfg["ng"], cfg["dx"], table=cfg.get("table"))
    U, P = cfg["U"].copy(), cfg["P"].copy()
    o.prim2con(U, P)
    dt = 0.25 * cfg["dx"]
    t0 = time.perf_counter()
    if "V" in cfg:
        ae, we, ai, wi = synth.imex_tableau()
        o.evolve_imex(U, cfg["V"].copy(), cfg["bc"], ae, we, ai, wi, dt, steps)
        nst = len(we)
    else:
        a, w = synth.tableau("rk4")
        o.evolve(U, cfg["bc"], a, w, dt, steps)
        nst = len(w)
    sec = time.perf_counter() - t0
    zs = float(n[0] * n[1] * n[2] * nst * steps)
    oracle.use_threads(1)
    return zs / sec, sec, zs, threads


def falg_nonredundant(workload, eos_kind, nonatmo, pts_per_zone, nstages, m1):
    """Algorithmic FP64 flops per zone and LAUNCH of each kernel class, every quantity counted once (FMA = 2): the itemised count of
    SURVEY 8(d) (DESIGN.md section 6 lists the items). Nothing the kernels recompute for their own convenience is in here."""
    d_first, d_second, d_mixed, d_adv, d_ko = 4.0, 7.0, 20.0, 9.0, 8.0          # flops of one stencil application (Eqs. 60-62, l.454-460)
    deriv_centred = 48 * d_first + 33 * d_second + 33 * d_mixed                 # 16 fields x 3, 11 fields x (3 + 3)
    ccz4_pointwise = 2150.0                                                     # Eqs. (13)-(26): Christoffels, Ricci (the Gamma~ Gamma~ sum ~0.5 k with the contraction over m done once), D_i D_j alpha, RHS
    grmhd_sources = 300.0                                                       # right-hand sides of Eq. (32) from the same derivatives
    mp5 = 60.0 * 20.0                                                           # 60 reconstructions x Eq. (70) + the test of Eq. (72); the limiter (up to ~80 more) not claimed
    splitting = 600.0                                                           # Eqs. (65), (69), (64) for 10 fields x 3 directions, lambda maxima
    c2p = (2000.0 if eos_kind != 2 else 2000.0 + 10000.0) * nonatmo * pts_per_zone   # bracketed solve ~15 evaluations; table: + gathers / log10 / exp10 per evaluation
    out = {"fill_ghosts": 0.0, "con2prim": c2p, "ccz4_algebra": deriv_centred + ccz4_pointwise + grmhd_sources,
           "adv_ko": 66 * d_adv + 66 * d_ko, "point_flux": 500.0 * pts_per_zone,
           "recon_x": (mp5 + splitting) / 3, "recon_y": (mp5 + splitting) / 3, "recon_z": (mp5 + splitting) / 3,
           "rk_combine": 2.0 * 2.5 * 32,
           # M1: closure root + fluxes ~2 k per species, implicit 4x4 Newton ~1 k per species and iteration (SURVEY: +6-8 k per zone-stage in all)
           "les": (26 * 3 * 4 + 36 * 5 + 300 + 150) * pts_per_zone,              # 78 gradients, 36 contracted products, (A12)-(A16), auxiliary fields
           "m1_point": 3 * 1200.0 * pts_per_zone if m1 else 0.0, "m1_div": 3 * 500.0 if m1 else 0.0, "m1_implicit": 3 * 800.0 * pts_per_zone if m1 else 0.0}
    return out


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    n_s = args.ref_n
    vals = []
    nthr = max(1, args.ref_threads)
    for _ in range(args.warmup):
        oracle_leg(args.workload, 16, 1, args.ref_threads, args.les_cm, args.les_other)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        v, sec, zs, nthr = oracle_leg(args.workload, n_s, 1, args.ref_threads, args.les_cm, args.les_other)
        vals.append((zs, sec))
    total = time.perf_counter() - t0
    value = sum(z for z, _ in vals) / sum(s for _, s in vals)
    sample = "%d^3 instance of workload %s, 1 RK step per bench step, %d thread(s)" % (n_s, args.workload, nthr)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": "zone-stages/s", "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * total / max(args.steps, 1), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "%s_%d" % (args.workload, args.n), "bounded_sample": sample},
        "cpu_baseline": dict({"value": value, "unit": "zone-stages/s", "cores": nthr, "kind": "oracle", "sample": sample,
                              "pins": "oracle pinned except readings R1, R10, R17, R26 (unpinnable against the paper; DESIGN.md section 4)"}, **cpu_info()),
        "e2e": {"value": value, "unit": "zone-stages/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="c4", help="c4 (BASELINE configs[3], the 256^3 workload the metric is quoted on), c1, c3, c5, c5crop")
    ap.add_argument("--n", type=int, default=256)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--ref-n", type=int, default=40, help="sample size of the oracle legs")
    ap.add_argument("--ref-threads", type=int, default=1, help="--impl reference: threads of the oracle (1 = the plain build)")
    ap.add_argument("--decomp", default=None, help="e.g. 1x1x2: ONE patch split into bricks over the ranks, halo exchange fused with the ghost fill "
                                                   "(strong scaling; needs world = product, or world 1 for the self-neighbour check); default: replicas")
    ap.add_argument("--les-other", type=float, default=0.0, help="with --les-cm: the other three SGS coefficients C_N = C_Y = C_T of App. A (the paper's runs: 0)")
    ap.add_argument("--les-cm", type=float, default=0.0, help="workloads c1 / c4 with the LES sub-grid-scale term of the induction equation, C_M (paper: 8); ghost width 5")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist
    from paper_2510_13965_b200 import binding, synth
    from paper_2510_13965_b200 import build as _build
    if int(os.environ.get("LOCAL_RANK", "0")) == 0:
        _build.build()                  # refresh the in-tree library if a source is newer (seconds when up to date)

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the hot path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    cfg = workload_inputs(args.workload, args.n, args.les_cm, args.les_other)
    n, ng = cfg["n"], cfg["ng"]
    m1 = "V" in cfg
    nstages = 3 if m1 else STAGES
    grid = None
    if args.decomp:                       # ONE patch of the workload's size split over the ranks (strong scaling)
        from paper_2510_13965_b200 import decomp
        grid = decomp.brick_grid(world, [int(x) for x in args.decomp.lower().split("x")])
        box = decomp.local_box(rank, grid, n)
        n_glob, n = n, tuple(hi - lo for lo, hi in box)
        for key in ("U", "P", "V"):
            if key in cfg:
                cfg[key] = decomp.cut_local(cfg[key], rank, grid, n_glob, ng)
    zones = n[0] * n[1] * n[2]
    patch = binding.Patch(cfg["params"], n, ng, cfg["dx"], stages=nstages, table=cfg.get("table"), device="cuda:%d" % local, m1=m1)
    halo_imports = []
    if grid is not None:
        if world == 1:                    # one GPU: the brick is its own neighbour across z, with the epoch words of the multi-GPU protocol
            for d in ((0, 0, 1), (0, 0, -1)):
                for name, (slot, t) in decomp.state_slots(patch).items():
                    binding.mhd_patch_set_neighbor(patch.h, slot, d, t.data_ptr(), patch.npts)
                binding.mhd_patch_set_neighbor_word(patch.h, d, binding.mhd_patch_halo_words(patch.h))
            cfg["bc"] = list(cfg["bc"][:4]) + [2, 2] if cfg["bc"][4] == 0 and cfg["bc"][5] == 0 else cfg["bc"]
        else:
            cfg["bc"], halo_imports = decomp.connect_distributed(patch, rank, grid, cfg["bc"])
    if m1:                              # config 5: IMEX(3,3,2) pair (R1), 3 stages per step
        tab = binding.make_tableau(*synth.imex_tableau())
        patch.V.copy_(torch.as_tensor(cfg["V"]))
        advance = patch.advance_imex
    else:
        tab = binding.make_tableau(*synth.tableau("rk4"))
        advance = patch.advance
    dt = 0.25 * cfg["dx"]
    # initial data: metric + Bbar in U, (rho, Ye, eps, v) in P; conserved fields from the library's own prim2con kernel
    patch.upload(U=cfg["U"], P=cfg["P"])
    patch.prim2con()
    patch.fill_ghosts(cfg["bc"])
    U_init = patch.U.clone()
    V_init = patch.V.clone() if m1 else None
    torch.cuda.synchronize()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing -------------------------------------------------------------------------------
    for _ in range(args.warmup):
        advance(tab, cfg["bc"], dt, 1)
    torch.cuda.synchronize()
    patch.U.copy_(U_init)
    if m1:
        patch.V.copy_(V_init)
    patch.profile(True)
    patch.profile_read()
    sampler = ClockSampler(local)
    sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record()
    advance(tab, cfg["bc"], dt, args.steps)              # K full RK steps = 4K (IMEX: 3K) passes of the whole path, one C-ABI call
    ev1.record()
    barrier()
    ms = ev0.elapsed_time(ev1)
    clocks = sampler.stop()
    prof = patch.profile_read()
    patch.profile(False)
    status = patch.status()
    ms = max_over_ranks(ms, device="cuda")
    value = aggregate_throughput(world, zones, nstages, args.steps, ms)

    # ---- end to end through the host-buffer entry point (H2D of the state, advance, D2H of state + flags) ------
    e2e = None
    if not args.no_e2e:
        hostU = U_init.cpu().pin_memory()
        hostV = V_init.cpu().pin_memory() if m1 else None
        hostF = torch.zeros(patch.flags.shape[1:], dtype=torch.uint8).pin_memory()
        src, srcV = hostU.clone(), (hostV.clone() if m1 else None)
        e_steps = max(1, min(args.steps, 3))

        def host_step():
            if m1:
                patch.advance_imex_host(tab, cfg["bc"], dt, 1, hostU, hostV, hostF)
            else:
                patch.advance_host(tab, cfg["bc"], dt, 1, hostU, hostF)
        host_step()                                                  # warm-up
        hostU.copy_(src)
        if m1:
            hostV.copy_(srcV)
        barrier()
        t0 = time.perf_counter()
        for _ in range(e_steps):
            host_step()
        torch.cuda.synchronize()
        sec = time.perf_counter() - t0
        sec = max_over_ranks(sec, device="cuda")
        nbytes = hostU.numel() * 8 + (hostV.numel() * 8 if m1 else 0)
        e2e = {"value": world * zones * nstages * e_steps / sec, "unit": "zone-stages/s", "h2d_bytes_per_step": nbytes,
               "d2h_bytes_per_step": nbytes + hostF.numel(), "steps": e_steps,
               "entry_point": "mhd_advance_imex_host" if m1 else "mhd_advance_host"}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel -----------------------------------------------
    # The path is bound by the plain FP64 pipe ("alu"): ~11-13 kflop per zone-stage against 1.28 kB of algorithmic HBM traffic is ~9 flop/B,
    # the ridge of this GPU is 34 TFLOP/s / 6.5 TB/s = 5.2 flop/B. Peak = FP64 FMA throughput measured by the library's own register-resident
    # DFMA probe (nominal 148 SMs x 64 lanes x 2 flop x 1.965 GHz = 37.2 TFLOP/s).
    # Numerator = ALGORITHMIC flops, every derivative, flux and symmetric component counted once (falg_nonredundant below, the itemised count of
    # SURVEY 8(d) / DESIGN.md section 6), never more than what the kernel executed (ncu: DADD + DMUL + 2 DFMA thread instructions of the tracked
    # capture profiles/r2_ncu_c4_128.json). The oracle's operation count (tests/golden/op_counts.json) is NOT used: the oracle recomputes on purpose.
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    hbm_peak, hbm_src = (peaks["hbm_gbs"], "measured") if "hbm_gbs" in peaks else (6650.0, "fallback")
    fp64_peak = binding.mhd_probe_fp64_flops(patch.stream()) / 1e12
    pts_per_zone = patch.npts / zones
    nonatmo = 1.0 - status["n_atmo"] / status["n_points"]
    alg_flops = falg_nonredundant(args.workload, cfg["params"]["eos_kind"], nonatmo, pts_per_zone, nstages, m1)
    # algorithmic doubles moved per zone and launch (reads + writes at the minimum)
    alg_doubles = {"fill_ghosts": 0.0, "con2prim": 18 + 16, "ccz4_algebra": 22 + 10 + 5 + 32, "adv_ko": 22 * 3, "recon_x": 21 + 20,
                   "recon_y": 21 + 20, "recon_z": 21 + 20, "rk_combine": 3.75 * 32, "point_flux": 29 + 33,
                   "m1_point": 21 + 15 + 75, "m1_div": 15 + 75 + 22 + 15, "m1_implicit": 21 + 15 + 30, "les": 17 + 26 + 26 + 12}
    # ncu figures of the tracked capture (written by `python -m paper_2510_13965_b200.ncu_summary`; per-zone figures carry over to this size, the
    # tiles are the same); null when the capture is of another workload class
    cap, cap_meta = {}, None
    try:
        capj = json.load(open(os.path.join(ROOT, "profiles", "r2_ncu_c4_128.json")))
        cap_meta = capj["meta"]
        if not m1:
            cap = capj["kernels"]
    except Exception:
        pass
    total_kernel_ms = sum(v[0] for v in prof.values())
    dom = max(prof, key=lambda k: prof[k][0])
    dom_ms, dom_launches = prof[dom]
    sec_per_launch = dom_ms / max(dom_launches, 1) * 1e-3
    exe = {k: (cap[k]["executed_fp64_flops_per_zone"] if k in cap else None) for k in prof}
    if not args.workload.startswith("c4"):
        exe["con2prim"] = None               # the capture is of workload c4: its con2prim count (table EoS, 42 % star) does not carry over

    def claimed(k):                         # algorithmic flops of class k per zone, capped by what the kernel executed
        return min(alg_flops[k], exe[k]) if exe.get(k) is not None else alg_flops[k]
    achieved = claimed(dom) * zones / sec_per_launch / 1e12
    F_alg = sum(claimed(k) * (prof[k][1] / max(args.steps * nstages, 1)) for k in prof if prof[k][1] > 0)    # per zone-stage, launches per stage counted
    launched = [k for k in prof if prof[k][1] > 0]
    F_exe = (sum(exe[k] * (prof[k][1] / max(args.steps * nstages, 1)) for k in launched)
             if cap and all(exe.get(k) is not None for k in launched) else None)       # only when the capture covers every kernel of this workload
    step_tflops = F_alg * value / world / 1e12
    roofline = {"bound": "alu", "kernel": dom, "achieved": achieved, "peak": fp64_peak, "unit": "TFLOP/s", "frac": achieved / fp64_peak,
                "peak_source": "measured: FP64 DFMA probe of the library (mhd_probe_fp64_flops); nominal 37.2",
                "numerator": "algorithmic flops, each derivative / flux / symmetric component once (bench.falg_nonredundant), capped by the executed DADD+DMUL+2*DFMA of the ncu capture",
                "traffic": cap[dom]["dram_bytes_per_zone"] * zones if dom in cap else None,
                "traffic_source": ("dram__bytes_read.sum + dram__bytes_write.sum per zone of the ncu --set full capture profiles/r2_ncu_c4_128.json (commit %s) x zones of this run"
                                   % cap_meta["commit"]) if dom in cap else None,
                "alg_bytes": alg_doubles[dom] * 8.0 * zones,
                "fp64_pipe_busy_ncu": cap[dom]["fp64_pipe_pct"] / 100.0 if dom in cap and cap[dom]["fp64_pipe_pct"] is not None else None,
                "executed_flops_per_zone_ncu": exe.get(dom),
                "kernel_ms_per_launch": dom_ms / max(dom_launches, 1),
                "share_of_step": dom_ms / total_kernel_ms if total_kernel_ms else None,
                "alg_flops_per_zone": alg_flops[dom],
                "hbm": {"achieved_gbs": alg_doubles[dom] * 8.0 * zones / sec_per_launch / 1e9, "peak_gbs": hbm_peak, "peak_source": hbm_src},
                "kernel_ms_per_step": {k: v[0] / args.steps for k, v in prof.items()},
                "kernel_frac_of_fp64_peak": {k: (claimed(k) * zones / (v[0] / max(v[1], 1) * 1e-3) / 1e12 / fp64_peak if v[0] > 0 else None)
                                             for k, v in prof.items()},
                # whole step against the binding roof: T_bound = max(B_alg / BW, F_alg / P_fp64) per zone-stage
                "step": {"alg_flops_per_zone_stage": F_alg, "executed_flops_per_zone_stage_ncu": F_exe, "alg_bytes_per_zone_stage": 1280 if not m1 else 1880,
                         "achieved_tflops": step_tflops, "frac_of_fp64_peak": step_tflops / fp64_peak,
                         "frac_of_hbm_peak": (1280.0 if not m1 else 1880.0) * value / world / 1e9 / hbm_peak,
                         "dram_bytes_per_zone_stage_ncu": sum(cap[k]["dram_bytes_per_zone"] for k in cap) if cap else None,
                         "binding": "alu", "target": 0.5}}

    cpu = None
    if not args.no_cpu_baseline:
        v, sec, zs, _ = oracle_leg(args.workload, args.ref_n, 1, les_cm=args.les_cm, les_other=args.les_other)
        nall = os.cpu_count() or 1
        va, seca, _, nthr = oracle_leg(args.workload, args.ref_n, 1, threads=nall, les_cm=args.les_cm, les_other=args.les_other) if nall > 1 else (v, sec, zs, 1)
        cpu = dict({"value": v, "unit": "zone-stages/s", "cores": 1, "kind": "oracle",
                    "sample": "%d^3 instance of workload %s, 1 RK step (%.1f s), single thread" % (args.ref_n, args.workload, sec),
                    "all_cores": {"value": va, "cores": nthr, "seconds": seca, "build": "-fopenmp on the outermost grid loops, arithmetic unchanged"},
                    "pins": "oracle pinned except readings R1, R10, R17, R26 (unpinnable against the paper; DESIGN.md section 4)"}, **cpu_info())

    bad = []
    if status["n_fatal"] or status["n_noconv"]:
        bad.append("n_fatal=%d n_noconv=%d after the timed region: the state left the method's domain of validity" % (status["n_fatal"], status["n_noconv"]))
    if status.get("halo_timeout"):
        bad.append("a halo wait expired")
    out = {
        "metric": METRIC, "value": value, "unit": "zone-stages/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": "%s_%d%s" % (args.workload, args.n, ("_les%g" % args.les_cm + ("_nyt%g" % args.les_other if args.les_other else "")) if args.les_cm else ""), "grid": list(n), "ghosts": ng, "rk": "rk4", "eos_kind": cfg["params"]["eos_kind"],
                   "l2": "inputs (32 fields x %.0f MB) far larger than L2; no flush needed" % (patch.npts * 8 / 1e6),
                   "non_atmosphere_fraction": 1.0 - status["n_atmo"] / status["n_points"], "parallelism": "replicas" if world > 1 else "single"},
        "clocks": clocks, "e2e": e2e, "gpu_launches": int(sum(v[1] for v in prof.values())),
        "roofline": roofline, "cpu_baseline": cpu, "flags": {k: v for k, v in status.items() if k != "n_points"},
    }
    if grid is not None:
        out["scaling"] = "strong"
        out["config"]["parallelism"] = "bricks %s, halo exchange fused with the ghost fill%s" % (
            "x".join(str(g) for g in grid), " (one GPU: the brick is its own neighbour across z)" if world == 1 else "")
    if bad:
        out["invalid"] = "; ".join(bad)
    print(json.dumps(out))
    if bad:
        sys.stderr.write("bench.py: INVALID RUN: %s\n" % "; ".join(bad))
        sys.exit(1)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
