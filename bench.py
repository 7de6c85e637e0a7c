#!/usr/bin/env python
"""bench.py -- cell updates/s of the unsplit patch-group update on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--dtype f32|f64]

A "step" is one pass of the whole hot path over one batch of synthetic patch groups:
hydro_dt (CFL reduction) -> hydro_solve (steps (1)-(5)), the time-step
formed on the device from the reduction (no host sync inside the timed region).  The workload is
BASELINE.json configs[2] (the AMR-shaped batch the metric's CTU+PLM+Roe fp32 number is quoted on):
8192 patch groups of 16^3 cells with 3 ghost cells (22^3 input), 5 fp32 variables SoA, one
CTU + PLM (van Leer) + Roe step with the patch-boundary fluxes returned.  Inputs (1.7 GB) exceed L2.

Prints ONE JSON line (rank 0).  Keys beyond the base contract: roofline, cpu_baseline, e2e, clocks,
gpu_launches, and f64 (the same step in double precision, same kernels templated on double).
--impl reference times the CPU oracle (oracle/, plain C++ on the host cores) on the same config.
"""
import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "cell updates/sec (CTU+PLM+Roe, fp32/fp64) and % of HBM/FLOP roofline"
UNIT = "cell updates/s"
NG, GHOST, GAMMA, DH, CFL = 8192, 3, 5.0 / 3.0, 1.0, 0.5
CELLS = 16 ** 3
SCHEME, RIEMANN, LIMITER = 2, 3, 1  # CTU, Roe, van Leer (PLM on primitive variables: opts defaults)


def load_json(path, default=None):
    try:
        with open(path) as f:
            return json.load(f)
    except Exception:
        return default


def workload_name(dtype):
    return f"configs[2]: AMR batch, {NG} patch groups x 16^3 cells, g={GHOST} (22^3 in), {dtype}, CTU+PLM(vanLeer)+Roe, face fluxes on"


def algorithmic_flops_per_cell(dtype):
    """Counted on the oracle with a counting scalar (oracle/count_flops.py -> oracle/flops_per_cell.json);
    falls back to the hand estimate of SURVEY.md 8(d) until that file exists."""
    d = load_json(os.path.join(ROOT, "oracle", "flops_per_cell.json"), {})
    e = d.get("ctu_plm_roe_vanleer_g3", {})
    if "flops_per_cell" in e:
        return float(e["flops_per_cell"]), "counted (oracle/count_flops.py)"
    return 2300.0, "hand estimate (SURVEY.md 8(d))"


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""
    REASONS = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
               0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting", 0x10: "sync_boost"}

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.stop_flag, self.samples, self.mask, self.max_mhz, self.ok = index, False, [], 0, None, False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception:
            self.ok = False

    def run(self):
        if not self.ok:
            return
        while not self.stop_flag:
            try:
                self.samples.append(self.nv.nvmlDeviceGetClockInfo(self.h, self.nv.NVML_CLOCK_SM))
                self.mask |= int(self.nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
            except Exception:
                pass
            time.sleep(0.005)

    def summary(self):
        if not self.ok or not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["nvml unavailable"]}
        s = sorted(self.samples)
        return {"sm_mhz": s[len(s) // 2], "sm_max_mhz": self.max_mhz, "samples": len(s),
                "reasons": [n for b, n in self.REASONS.items() if self.mask & b]}


def physical_gpu_index(local):
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local])
        except Exception:
            return local
    return local


def time_oracle(G, dt, nthreads, target_s=12.0):
    """The oracle as it stands on a bounded sample: calibrate on 2*nthreads groups, then whole passes of
    hydro_dt + hydro_solve over the first n groups, repeated until ~target_s of CPU work has been done."""
    from oracle import oracle as O
    n0 = min(len(G), 2 * nthreads)
    t0 = time.perf_counter()
    O.hydro_dt(G[:n0], GAMMA, 0)
    O.hydro_solve(G[:n0], dt, DH, GAMMA, SCHEME, RIEMANN, LIMITER, nthreads=nthreads)
    per_group = (time.perf_counter() - t0) / n0
    n = int(max(n0, min(len(G), target_s / max(per_group, 1e-9))))
    passes, t0 = 0, time.perf_counter()
    while True:
        O.hydro_dt(G[:n], GAMMA, 0)
        O.hydro_solve(G[:n], dt, DH, GAMMA, SCHEME, RIEMANN, LIMITER, nthreads=nthreads)
        passes += 1
        el = time.perf_counter() - t0
        if el >= 0.8 * target_s or passes >= 64:
            break
    return passes * n * CELLS / el, n, el, passes


def ncu_counters(key):
    """Per-launch counters of the dominant kernel from the committed ncu --set full capture of this same workload
    (profiles/kernel_counters.json, written from the .ncu-rep by the command named in it): DRAM bytes, executed
    FP thread-instructions (fadd, fmul, ffma / dadd, dmul, dfma), FMA / FP64 pipe utilisation."""
    d = load_json(os.path.join(ROOT, "profiles", "kernel_counters.json"), {}) or {}
    return d.get(key)


def measured_peaks():
    """ALU peaks measured on this pool's B200 by `python bench.py --table peaks` (profiles/alu_peaks.json)."""
    return load_json(os.path.join(ROOT, "profiles", "alu_peaks.json"), {}) or {}


def alu_roofline(dtype, kernel_ms, flops_cell, ncells, sm_max, key):
    """The three fractions of the ALU roofline for one hydro_solve launch of `ncells` cell updates:
    frac          = oracle-counted (algorithmic) flops / time / MEASURED FMA peak      (the metric's fraction)
    frac_executed = flops the kernel actually executes (ncu: fadd + fmul + 2 ffma thread-instructions) / time / peak
    pipe_pct      = sm__inst_executed_pipe_fma (fp64: pipe_fp64) of the committed capture."""
    lanes = 128 if dtype == "f32" else 64
    nominal = 148 * lanes * 2 * sm_max * 1e6 / 1e12
    mp = measured_peaks()
    peak = mp.get("fp32_tflops_ffma" if dtype == "f32" else "fp64_tflops")
    src = "measured: register-resident %s loop, python bench.py --table peaks -> profiles/alu_peaks.json" % ("FFMA" if dtype == "f32" else "DFMA")
    if not peak:
        peak, src = nominal, f"nominal (profiles/alu_peaks.json missing): 148 SM x {lanes} lanes x 2 x {sm_max:.0f} MHz"
    achieved = flops_cell * ncells / (kernel_ms * 1e-3) / 1e12
    r = {"achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak, "peak_source": src,
         "peak_nominal": nominal, "frac_of_nominal": achieved / nominal}
    c = ncu_counters(key)
    if c:
        ex = c.get("flops_executed_per_launch")
        if ex and c.get("cells_per_launch"):
            ex_t = ex * (ncells / c["cells_per_launch"]) / (kernel_ms * 1e-3) / 1e12
            r.update({"executed_tflops": ex_t, "frac_executed": ex_t / peak, "flops_executed_per_cell": ex / c["cells_per_launch"]})
        r["pipe_pct"] = c.get("pipe_pct")
        r["issue_active_pct"] = c.get("issue_active_pct")
        r["traffic"] = c.get("dram_bytes_per_launch")
        r["counters_source"] = c.get("source")
    else:
        r.update({"frac_executed": None, "pipe_pct": None, "traffic": None})
    return r


def run_reference(args):
    """--impl reference: the CPU oracle on the host cores, same config/metric; rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    import numpy as np
    from oracle import oracle as O
    from paper_1103_3373_b200 import workloads as wl
    dtype = "float32" if args.dtype == "f32" else "float64"
    nthreads = min(O.max_threads(), len(os.sched_getaffinity(0)))
    nsample = int(os.environ.get("HYDRO_REF_GROUPS", 32 * nthreads))
    G = wl.amr_batch(nsample, g=GHOST, gamma=GAMMA, seed=0, dtype=dtype).numpy()
    smax = O.hydro_dt(G, GAMMA, 0)
    dt = float(G.dtype.type(CFL * DH / smax))
    for _ in range(max(0, min(args.warmup, 1))):
        O.hydro_solve(G[:nthreads], dt, DH, GAMMA, SCHEME, RIEMANN, LIMITER, nthreads=nthreads)
    steps = max(1, args.steps)
    budget = float(os.environ.get("HYDRO_REF_BUDGET_S", "120"))
    t0 = time.perf_counter()
    done = 0
    for _ in range(steps):
        O.hydro_dt(G, GAMMA, 0)
        O.hydro_solve(G, dt, DH, GAMMA, SCHEME, RIEMANN, LIMITER, nthreads=nthreads)
        done += 1
        if time.perf_counter() - t0 > budget:
            break
    el = time.perf_counter() - t0
    value = done * nsample * CELLS / el
    sample = f"{nsample} of {NG} patch groups per step, {done} steps, {nthreads} OpenMP threads over groups (PAPER.md:137)"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": done,
        "warmup": args.warmup, "ms_per_step": 1e3 * el / done, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": args.dtype, "data": "synthetic",
        "config": {"workload": workload_name(args.dtype), "note": "CPU oracle (oracle/hydro_oracle.cpp, g++ -O2 -ffp-contract=off) on a bounded sample"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": nthreads, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def run_table(args):
    """--table variants | grid: CUDA-event timings through the binding (2 warm-ups, 5 launches), inputs resident in HBM."""
    import numpy as np
    import torch
    from paper_1103_3373_b200 import binding as B, workloads as wl
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)

    def ev(f, reps=5):
        for _ in range(2):
            f()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(reps):
            f()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / reps

    rows = []
    if args.table == "peaks":
        return run_peaks(args, B, dev)
    if args.table == "variants":
        Ng = 4096
        names, rn = {0: "MHM", 1: "VL", 2: "CTU"}, {0: "exact", 1: "HLLE", 2: "HLLC", 3: "Roe"}
        # fraction of the MEASURED FMA roof by the oracle's operation count, where oracle/count_flops.py counted the variant
        fpc = load_json(os.path.join(ROOT, "oracle", "flops_per_cell.json"), {}) or {}
        mp = measured_peaks()

        def alu_frac(scheme, recon, rs, es, ms):
            key = [k for k in fpc if k.startswith("%s_%s_%s_" % (names[scheme].lower(), "ppm" if recon else "plm", rn[rs].lower()))]
            peak = mp.get("fp32_tflops_ffma" if es == 4 else "fp64_tflops")
            if not key or not peak:
                return {}
            fl = fpc[key[0]]["flops_per_cell"]
            return {"flops_per_cell": fl, "frac": fl * Ng * CELLS / (ms * 1e-3) / 1e12 / peak}
        for tdt in (torch.float32, torch.float64):
            for scheme in (2, 0, 1):
                for recon in (0, 1):
                    for rs in (3, 2, 1, 0):
                        if scheme != 2 and rs in (1, 0):
                            continue
                        if args.only and args.only.lower() != ",".join((names[scheme], "PPM" if recon else "PLM", rn[rs],
                                                                         "fp32" if tdt == torch.float32 else "fp64")).lower():
                            continue
                        g = B.hydro_min_ghost(scheme, recon)
                        u = wl.amr_batch(Ng, g=g, gamma=GAMMA, seed=0, dtype=str(tdt).replace("torch.", ""), device=dev)
                        out = torch.empty((Ng, 5, 16, 16, 16), dtype=tdt, device=dev)
                        ff = torch.empty((Ng, 9, 5, 16, 16), dtype=tdt, device=dev)
                        ms = ev(lambda: B.hydro_solve(u, 0.05, DH, GAMMA, scheme, rs, LIMITER, recon=recon, out=out, face_flux=ff))
                        rows.append({"precision": "fp32" if tdt == torch.float32 else "fp64", "scheme": names[scheme],
                                     "recon": "PPM" if recon else "PLM", "riemann": rn[rs], "ms": ms,
                                     "cell_updates_per_s": Ng * CELLS / (ms * 1e-3),
                                     "fused": bool(B.hydro_fused_fits(tdt, scheme, recon, g))})
                        rows[-1].update(alu_frac(scheme, recon, rs, 4 if tdt == torch.float32 else 8, ms))
                        del u, out, ff
        # the directionally split relaxing-TVD scheme (the low-arithmetic-intensity contrast).  By the oracle's count
        # (1 271 flops against 83 B per cell update: three sweeps, 5.9 cell-sweeps per interior cell) it is still above the B200's
        # machine balance of ~11 flop/B, so both fractions are reported: of the FMA roof (the binding one) and of the copy peak
        peaks = load_json(os.path.join(ROOT, "MEASURED_PEAKS.json"), {}) or {}
        hbm = float(peaks.get("hbm_gbs") or 6650.0)
        for split, tdt in ((sp, t) for sp in ("RTVD", "WAF") for t in (torch.float32, torch.float64)):
            es = 4 if tdt == torch.float32 else 8
            if args.only and args.only.lower() != split.lower() + ",-,-," + ("fp32" if es == 4 else "fp64"):
                continue
            u = wl.amr_batch(Ng, g=3, gamma=GAMMA, seed=0, dtype=str(tdt).replace("torch.", ""), device=dev)
            out = torch.empty((Ng, 5, 16, 16, 16), dtype=tdt, device=dev)
            ff = torch.empty((Ng, 9, 5, 16, 16), dtype=tdt, device=dev)
            ws = torch.empty(B.lib().hydro_rtvd_workspace_bytes(Ng, es), dtype=torch.uint8, device=dev)
            fn = B.hydro_rtvd_solve if split == "RTVD" else B.hydro_waf_solve
            ms = ev(lambda: fn(u, 0.05, DH, GAMMA, 0, out=out, face_flux=ff, workspace=ws))
            byt = es * Ng * (5 * 22 ** 3 + 5 * CELLS + 45 * 256)
            rows.append({"precision": "fp32" if es == 4 else "fp64", "scheme": split + " (split)", "recon": "-", "riemann": "-", "ms": ms,
                         "cell_updates_per_s": Ng * CELLS / (ms * 1e-3), "fused": True,
                         "hbm_gbs": byt / ms / 1e6, "hbm_frac": byt / ms / 1e6 / hbm})
            fl = (fpc.get("rtvd_g3" if split == "RTVD" else "waf_g3") or {}).get("flops_per_cell")
            peak = mp.get("fp32_tflops_ffma" if es == 4 else "fp64_tflops")
            if fl and peak:
                rows[-1].update({"flops_per_cell": fl, "frac": fl * Ng * CELLS / (ms * 1e-3) / 1e12 / peak, "bound": "alu"})
            del u, out, ff, ws
        print(json.dumps({"table": "variants", "groups": Ng, "limiter": "van Leer", "rows": rows}))
        return
    for N, tdt in ((512, torch.float32), (256, torch.float64)):
        es = 4 if tdt == torch.float32 else 8
        for g in (2, 3):
            U = torch.rand((5, N, N, N), dtype=tdt, device=dev) + 1.0
            Ng, S = (N // 16) ** 3, 16 + 2 * g
            G = B.hydro_gather(U, g)
            out = torch.empty((Ng, 5, 16, 16, 16), dtype=tdt, device=dev)
            tg = ev(lambda: B.hydro_gather(U, g, groups=G))
            ts = ev(lambda: B.hydro_scatter(out, (N, N, N), grid=U))
            rows.append({"kernel": "gather/scatter", "N": N, "precision": "fp32" if es == 4 else "fp64", "g": g, "gather_ms": tg,
                         "gather_gbs": es * 5 * (N ** 3 + Ng * S ** 3) / tg / 1e6, "scatter_ms": ts,
                         "scatter_gbs": es * 10 * N ** 3 / ts / 1e6})
            del U, G, out
        torch.cuda.empty_cache()
    for N in (256, 512):
        U = torch.from_numpy(wl.blast_grid(128, dtype=np.float32)).to(dev).repeat(1, N // 128, N // 128, N // 128).contiguous()
        for label, kw in (("hydro_solve_grid (one launch per step)", {}), ("gather -> hydro_solve -> scatter", {"nghost": 2})):
            ms = ev(lambda: B.hydro_advance(U, 10, 1.0, GAMMA, SCHEME, RIEMANN, LIMITER, cfl=0.4, **kw), 2) / 10
            rows.append({"kernel": "hydro_advance, CTU+PLM+Roe fp32, " + label, "N": N, "ms_per_step": ms,
                         "cell_updates_per_s": N ** 3 / (ms * 1e-3)})
    print(json.dumps({"table": "grid", "rows": rows}))


def run_counters(args):
    """--table counters --rep-f32 A.ncu-rep --rep-f64 B.ncu-rep: distil the committed `ncu --set full` captures of the dominant
    kernel (one launch of hydro_solve on the bench workload) into profiles/kernel_counters.json, which the bench line reads
    for frac_executed / pipe_pct / traffic.  Runs here (no GPU): `ncu -i <rep> --page raw --csv`."""
    import csv
    import subprocess
    out = {"_command": "python bench.py --table counters --rep-f32 %s --rep-f64 %s" % (args.rep_f32, args.rep_f64),
           "_capture": "ncu --set full --clock-control none --import-source on -k regex:ctu_lean_kernel -s 3 -c 1 -o <rep> "
                       "python bench.py --steps 3 --warmup 3 --no-extras [--dtype f64]"}
    for key, rep in (("solve_f32", args.rep_f32), ("solve_f64", args.rep_f64)):
        if not rep:
            continue
        txt = subprocess.run(["ncu", "-i", rep, "--page", "raw", "--csv"], capture_output=True, text=True, check=True).stdout
        rows = list(csv.reader(txt.splitlines()))
        hdr, vals = rows[0], rows[2]
        m = {h: v for h, v in zip(hdr, vals)}

        def f(name):
            return float(m[name].replace(",", ""))
        # executed FP thread-instructions by opcode from the source page (predicated-on threads of every SASS instruction)
        src = subprocess.run(["ncu", "-i", rep, "--page", "source", "--csv"], capture_output=True, text=True, check=True).stdout
        srows = list(csv.reader(src.splitlines()))
        sh = srows[1]
        i_src, i_thr = sh.index("Source"), sh.index("Predicated-On Thread Instructions Executed")
        ops = ("FADD", "FMUL", "FFMA") if key == "solve_f32" else ("DADD", "DMUL", "DFMA")
        fl = [0.0, 0.0, 0.0]
        for r in srows[2:]:
            if len(r) <= i_thr or not r[i_thr]:
                continue
            tok = r[i_src].split()
            op = (tok[1] if tok and tok[0].startswith("@") and len(tok) > 1 else (tok[0] if tok else "")).split(".")[0]
            if op in ops:
                fl[ops.index(op)] += float(r[i_thr])
        pipe = f("sm__inst_executed_pipe_fma.avg.pct_of_peak_sustained_active" if key == "solve_f32"
                 else "sm__inst_executed_pipe_fp64.avg.pct_of_peak_sustained_active")
        unit = {h: u for h, u in zip(hdr, rows[1])}

        def gb(name):  # ncu prints dram bytes in a scaled unit
            scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}[unit[name]]
            return f(name) * scale
        out[key] = {
            "kernel": m.get("Kernel Name", "")[:80], "cells_per_launch": NG * CELLS,
            "thread_inst_add_mul_fma": fl, "flops_executed_per_launch": fl[0] + fl[1] + 2 * fl[2],
            "pipe_pct": pipe, "issue_active_pct": f("smsp__issue_active.avg.pct_of_peak_sustained_active"),
            "warp_inst_per_launch": f("smsp__inst_executed.sum"),
            "registers": f("launch__registers_per_thread"),
            "local_ld": f("smsp__sass_inst_executed_op_local_ld.sum"), "local_st": f("smsp__sass_inst_executed_op_local_st.sum"),
            "dram_bytes_per_launch": gb("dram__bytes_read.sum") + gb("dram__bytes_write.sum"),
            "ncu_duration_ms": f("gpu__time_duration.sum") * {"ms": 1.0, "us": 1e-3, "s": 1e3}.get(unit["gpu__time_duration.sum"], 1.0),
            "source": os.path.basename(rep)}
    with open(os.path.join(ROOT, "profiles", "kernel_counters.json"), "w") as fo:
        json.dump(out, fo, indent=1)
    print(json.dumps(out))


def run_peaks(args, B, dev):
    """--table peaks: MEASURED ALU peaks.  Register-resident loops of hydro_alu_peak_launch on all SMs
    (4 CTAs x 512 threads per SM, 16 independent chains per thread), each kind run back to back for ~1 s under the
    clock sampler and timed with CUDA events; the best 0.25 s window counts as the burst figure, the whole second as
    the sustained one.  Writes profiles/alu_peaks.json (read by the bench line for roofline.peak)."""
    import torch
    sms = torch.cuda.get_device_properties(dev).multi_processor_count
    blocks, threads, iters = sms * 4, 512, 2048
    scratch = torch.empty(blocks * threads * 8, dtype=torch.uint8, device=dev)
    out = {"table": "peaks", "gpu": torch.cuda.get_device_name(dev), "sms": sms, "blocks": blocks, "threads": threads,
           "chains_per_thread": 16, "command": "python bench.py --table peaks", "kinds": {}}
    for kind in ("ffma", "ffma_const", "ffma2", "fmul_fadd", "ffma_fmnmx", "ffma2_fmnmx", "dfma", "mufu"):
        ops = B.hydro_alu_peak_launch(kind, blocks, threads, iters, scratch)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        B.hydro_alu_peak_launch(kind, blocks, threads, iters, scratch)
        e1.record()
        torch.cuda.synchronize()
        one = e0.elapsed_time(e1) * 1e-3
        n = max(8, int(1.0 / max(one, 1e-6)))
        evs = [torch.cuda.Event(enable_timing=True) for _ in range(n + 1)]
        sampler = ClockSampler(physical_gpu_index(dev.index or 0))
        sampler.start()
        evs[0].record()
        for k in range(n):
            B.hydro_alu_peak_launch(kind, blocks, threads, iters, scratch)
            evs[k + 1].record()
        torch.cuda.synchronize()
        sampler.stop_flag = True
        sampler.join()
        ts = [evs[k].elapsed_time(evs[k + 1]) * 1e-3 for k in range(n)]
        w = max(1, int(0.25 / max(one, 1e-6)))
        burst = max(ops * w / sum(ts[k:k + w]) for k in range(0, n - w + 1))
        out["kinds"][kind] = {"ops_per_launch": ops, "launches": n, "sustained_tops": ops * n / sum(ts) / 1e12,
                              "burst_tops": burst / 1e12, "clocks": sampler.summary()}
    # issue probes: the same arithmetic issued as scalar FFMA pairs or as packed FFMA2, inside the instruction mix of the kernels
    out["issue_probe"] = {"_what": "TFLOP/s of the FP32 part of each mix (higher = the mix issues faster); scalar vs packed side by side"}
    for sc, pk in (("2ffma_shf", "ffma2_shf"), ("6ffma_sel_shf", "3ffma2_sel_shf"), ("8ffma_sel_mufu_shf", "4ffma2_sel_mufu_shf")):
        row = {}
        for kind in (sc, pk):
            ops = B.hydro_alu_peak_launch(kind, blocks, threads, iters, scratch)
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(5):
                B.hydro_alu_peak_launch(kind, blocks, threads, iters, scratch)
            e1.record()
            torch.cuda.synchronize()
            row[kind] = ops * 5 / (e0.elapsed_time(e1) * 1e-3) / 1e12
        row["packed_over_scalar"] = row[pk] / row[sc]
        out["issue_probe"][sc + " vs " + pk] = row
    k = out["kinds"]
    out["fp32_tflops"] = max(k["ffma"]["sustained_tops"], k["ffma2"]["sustained_tops"], k["ffma_const"]["sustained_tops"])
    out["fp32_tflops_ffma"] = k["ffma"]["sustained_tops"]
    out["fp64_tflops"] = k["dfma"]["sustained_tops"]
    out["nominal"] = {"fp32_tflops": sms * 128 * 2 * 1.965e9 / 1e12, "fp64_tflops": sms * 64 * 2 * 1.965e9 / 1e12,
                      "rule": "SMs x 128 (64) FMA lanes x 2 x 1965 MHz"}
    for d in ("profiles", "gpurun_out"):  # gpurun_out/ is what comes back from a GPU box; profiles/ is the committed copy
        if os.path.isdir(os.path.join(ROOT, d)):
            with open(os.path.join(ROOT, d, "alu_peaks.json"), "w") as f:
                json.dump(out, f, indent=1)
    print(json.dumps(out))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=("ours", "reference"))
    ap.add_argument("--dtype", default="f32", choices=("f32", "f64"))
    ap.add_argument("--ng", type=int, default=NG, help="patch groups per GPU (default: the config's 8192)")
    ap.add_argument("--kernel", default="auto", choices=("auto", "staged", "fused"))
    ap.add_argument("--no-extras", action="store_true", help="skip the e2e / cpu_baseline / f64 legs (profiling runs)")
    ap.add_argument("--table", default=None, choices=("variants", "grid", "peaks", "counters"),
                    help="instead of the bench line: one JSON line with per-variant hydro_solve timings (4096 groups), or with the\n"
                         "uniform-grid kernels (gather / scatter bandwidth, whole-step rates); context for DESIGN.md, profiles/")
    ap.add_argument("--only", default=None, help="--table variants: run ONE row, e.g. CTU,PPM,exact,fp32 or RTVD,-,-,fp32 (the ncu\n"
                    "captures of the other kernels under profiles/ are taken with it)")
    ap.add_argument("--rep-f32", default=None, help="--table counters: ncu report of the fp32 dominant kernel")
    ap.add_argument("--rep-f64", default=None, help="--table counters: ncu report of the fp64 dominant kernel")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.table == "counters":
        return run_counters(args)
    if args.table:
        return run_table(args)

    import torch
    import torch.distributed as dist
    from paper_1103_3373_b200 import binding as B, shard, workloads as wl

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    B.lib()
    warmup = max(3, args.warmup)
    steps = max(1, args.steps)
    impl = {"auto": B.IMPL_AUTO, "staged": B.IMPL_STAGED, "fused": B.IMPL_FUSED}[args.kernel]
    Ng = args.ng

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def device_leg(tdtype, nsteps, nwarm, sample_clocks):
        """K steps of hydro_dt -> [max all-reduce over ranks] -> hydro_solve, inputs resident in HBM."""
        name = str(tdtype).replace("torch.", "")
        u = wl.amr_batch(Ng, g=GHOST, gamma=GAMMA, seed=1000 * rank, dtype=name, device=dev)
        out = torch.empty((Ng, 5, 16, 16, 16), dtype=tdtype, device=dev)
        ff = torch.empty((Ng, 9, 5, 16, 16), dtype=tdtype, device=dev)
        smax = torch.empty((), dtype=tdtype, device=dev)
        status = torch.zeros(3, dtype=torch.int64, device=dev)

        def step():
            B.hydro_dt(u, GAMMA, 0, max_speed=smax)
            shard.global_max(smax)  # the path's only exchange: one scalar max; no-op at N = 1
            B.hydro_solve(u, 0.0, DH, GAMMA, SCHEME, RIEMANN, LIMITER, out=out, face_flux=ff, status=status,
                          max_speed=smax, cfl=CFL, impl=impl)

        for _ in range(nwarm):
            step()
        ev = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(nsteps)]
        t_begin, t_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        sampler = ClockSampler(physical_gpu_index(local)) if sample_clocks else None
        barrier()
        if sampler:
            sampler.start()
        t_begin.record()
        for k in range(nsteps):
            ev[k][0].record()
            B.hydro_dt(u, GAMMA, 0, max_speed=smax)
            shard.global_max(smax)
            ev[k][1].record()
            B.hydro_solve(u, 0.0, DH, GAMMA, SCHEME, RIEMANN, LIMITER, out=out, face_flux=ff, status=status,
                          max_speed=smax, cfl=CFL, impl=impl)
            ev[k][2].record()
        t_end.record()
        barrier()
        if sampler:
            sampler.stop_flag = True
            sampler.join()
        total_ms = t_begin.elapsed_time(t_end)
        if world > 1:
            t = torch.tensor([total_ms], dtype=torch.float64, device=dev)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            total_ms = float(t.item())
        dt_ms = sum(e[0].elapsed_time(e[1]) for e in ev) / nsteps
        solve_ms = sum(e[1].elapsed_time(e[2]) for e in ev) / nsteps
        st = status.cpu().tolist()
        return {"total_ms": total_ms, "dt_ms": dt_ms, "solve_ms": solve_ms, "status": st, "u": u,
                "clocks": sampler.summary() if sampler else None, "smax": float(smax.item())}

    main_dtype = torch.float32 if args.dtype == "f32" else torch.float64
    leg = device_leg(main_dtype, steps, warmup, True)
    value = world * Ng * CELLS * steps / (leg["total_ms"] * 1e-3)
    es = 4 if args.dtype == "f32" else 8
    S = 16 + 2 * GHOST

    # ---- roofline of the dominant kernel (hydro_solve): plain-ALU bound ----
    peaks = load_json(os.path.join(ROOT, "MEASURED_PEAKS.json"), {}) or {}
    clocks = leg["clocks"] or {}
    sm_max = float(peaks.get("sm_max_mhz") or clocks.get("sm_max_mhz") or 1965.0)
    flops_cell, flops_src = algorithmic_flops_per_cell(args.dtype)
    bytes_cell = es * (5 * S ** 3 + 5 * CELLS + 45 * 256) / CELLS
    hbm = float(peaks.get("hbm_gbs") or 6650.0)
    hbm_src = "measured (MEASURED_PEAKS.json)" if peaks.get("hbm_gbs") else "fallback (B200_PROFILING.md)"
    if impl != B.IMPL_STAGED and B.hydro_fused_fits(main_dtype, SCHEME, B.PLM, GHOST):
        kernel_name = "hydro_solve (ctu_lean_kernel: fused z-marching CTU, phase-crossing state in shared memory)"
    else:
        kernel_name = "hydro_solve (staged_kernel)"
    roofline = {"bound": "alu", "kernel": kernel_name}
    roofline.update(alu_roofline(args.dtype, leg["solve_ms"], flops_cell, Ng * CELLS, sm_max, f"solve_{args.dtype}"))
    roofline.update({
        "flops_per_cell": flops_cell, "flops_source": flops_src,
        "kernel_ms": leg["solve_ms"], "share_of_step": leg["solve_ms"] / (leg["solve_ms"] + leg["dt_ms"]),
        "hbm": {"bytes_per_cell": bytes_cell, "achieved_gbs": bytes_cell * Ng * CELLS / (leg["solve_ms"] * 1e-3) / 1e9,
                "peak_gbs": hbm, "peak_source": hbm_src,
                "hydro_dt_gbs": 5 * es * Ng * CELLS / (leg["dt_ms"] * 1e-3) / 1e9,
                "hydro_dt_frac": 5 * es * Ng * CELLS / (leg["dt_ms"] * 1e-3) / 1e9 / hbm},
        "cells_per_s_at_alu_roof": roofline["peak"] * 1e12 / flops_cell,
        "cells_per_s_at_hbm_roof": hbm * 1e9 / bytes_cell,
    })

    result = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": steps, "warmup": warmup,
        "ms_per_step": leg["total_ms"] / steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": args.dtype, "data": "synthetic",
        "config": {"workload": workload_name(args.dtype), "groups_per_gpu": Ng, "l2": "inputs (1.7 GB fp32) larger than L2; no flush",
                   "step": "hydro_dt + hydro_solve, dt formed on device", "kernel": args.kernel,
                   "parallelism": f"{world} x independent patch-group shards (max all-reduce of one scalar)"},
        "roofline": roofline, "clocks": clocks, "gpu_launches": 2 * steps, "status": leg["status"],
    }

    def e2e_leg(tdtype, smax_val, nrep):
        """The same metric through hydro_pipeline_solve with HOST buffers: pinned in / out, H2D and D2H
        copies inside the timed region."""
        name = str(tdtype).replace("torch.", "")
        esz = 4 if tdtype == torch.float32 else 8
        hin = torch.empty((Ng, 5, S, S, S), dtype=tdtype, pin_memory=True)
        hin.copy_(wl.amr_batch(Ng, g=GHOST, gamma=GAMMA, seed=1000 * rank, dtype=name, device=dev))
        hout = torch.empty((Ng, 5, 16, 16, 16), dtype=tdtype, pin_memory=True)
        hff = torch.empty((Ng, 9, 5, 16, 16), dtype=tdtype, pin_memory=True)
        hs = torch.zeros((), dtype=tdtype)
        pipe = B.HydroPipeline(tdtype, GHOST, groups_per_chunk=512, nstreams=4, device=dev)
        dt0 = CFL * DH / smax_val
        pipe.solve(hin, hout, hff, dt0, DH, GAMMA, SCHEME, RIEMANN, LIMITER, max_speed=hs, impl=impl)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(nrep):
            pipe.solve(hin, hout, hff, dt0, DH, GAMMA, SCHEME, RIEMANN, LIMITER, max_speed=hs, impl=impl)
        torch.cuda.synchronize()
        e2e_s = (time.perf_counter() - t0) / nrep
        pipe.close()
        r = {"value": Ng * CELLS / e2e_s, "unit": UNIT, "h2d_bytes_per_step": hin.numel() * esz,
             "d2h_bytes_per_step": (hout.numel() + hff.numel()) * esz + esz, "ms_per_step": 1e3 * e2e_s,
             "pcie_gbs": (hin.numel() + hout.numel() + hff.numel()) * esz / e2e_s / 1e9,
             "api": "hydro_pipeline_solve (pinned host in/out, 4 streams x 512-group chunks; hydro_dt of the updated state fused per chunk)"}
        return r, hin, dt0

    if rank == 0 and world == 1 and not args.no_extras:
        del leg["u"]
        torch.cuda.empty_cache()
        # ---- e2e: HOST buffers through the C ABI pipeline, copies inside the timed region
        result["e2e"], hin, dt0 = e2e_leg(main_dtype, leg["smax"], max(2, min(5, steps)))
        # ---- cpu_baseline: the oracle as it stands, bounded sample: all host cores (OpenMP over groups)
        # and ONE thread (the paper quotes its speed-ups against one core and against four)
        from oracle import oracle as O
        nthreads = min(O.max_threads(), len(os.sched_getaffinity(0)))
        G = hin.numpy()
        cpu_v, cpu_n, cpu_s, cpu_p = time_oracle(G, float(G.dtype.type(dt0)), nthreads, target_s=10.0)
        one_v, one_n, one_s, one_p = time_oracle(G, float(G.dtype.type(dt0)), 1, target_s=8.0)
        result["cpu_baseline"] = {"value": cpu_v, "unit": UNIT, "cores": nthreads, "kind": "oracle",
                                  "sample": f"first {cpu_n} of {Ng} patch groups of the same batch, {cpu_p} passes of hydro_dt + one {args.dtype} CTU+PLM+Roe step, {cpu_s:.1f} s, OpenMP over groups",
                                  "one_thread": {"value": one_v, "unit": UNIT, "cores": 1,
                                                 "sample": f"first {one_n} groups, {one_p} passes, {one_s:.1f} s, single thread"}}
        del hin, G
        torch.cuda.empty_cache()
        # ---- the other precision: device-resident leg with the same roofline fractions, and its own e2e
        other = torch.float64 if args.dtype == "f32" else torch.float32
        oname = "f64" if args.dtype == "f32" else "f32"
        n2 = max(3, steps // 2)
        leg2 = device_leg(other, n2, 3, False)
        del leg2["u"]
        torch.cuda.empty_cache()
        v2 = Ng * CELLS * n2 / (leg2["total_ms"] * 1e-3)
        r2 = {"bound": "alu"}
        r2.update(alu_roofline(oname, leg2["solve_ms"], flops_cell, Ng * CELLS, sm_max, f"solve_{oname}"))
        r2["kernel_ms"] = leg2["solve_ms"]
        e2, hin2, _ = e2e_leg(other, leg2["smax"], 2)
        del hin2
        result[oname] = {"value": v2, "unit": UNIT, "ms_per_step": leg2["total_ms"] / n2, "roofline": r2, "e2e": e2}
    elif "u" in leg:
        del leg["u"]
    if "e2e" not in result:
        result["e2e"] = None
    if rank == 0:
        print(json.dumps(result))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
