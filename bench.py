#!/usr/bin/env python
"""bench.py -- cell-updates/s of the MHD step on B200 (one JSON line; contract in DESIGN.md "Measurement").

A "step" is one pass of the whole hot path over the resident state: one c_max reduction, dt = cfl/c_max on
the device, six L_i operators (fluid + B pair each), t += 2 dt.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c4|c5|c3|small] [--impl reference]

N > 1: one process per GPU under torchrun, each rank advances its own replica of the workload ("replicas
only": the paper's method is single-GPU); value = cells advanced by all ranks / max time.
"""
from __future__ import annotations

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

import numpy as np

WORKLOADS = {
    # name: (generator, n, precision, BASELINE.json config)
    "c4": ("turbulence", 512, "f32", "configs[3]: 3-D turbulence-like state, 512^3, fp32, periodic, cfl 0.8"),
    "c5": ("turbulence", 512, "f64", "configs[4]: same seeded state, 512^3, fp64, periodic, cfl 0.8"),
    "c3": ("blast3d", 256, "f32", "configs[2]: 3-D MHD blast wave, 256^3, fp32, periodic, cfl 0.8"),
    "small": ("turbulence", 128, "f32", "reduced 128^3 fp32 turbulence-like state (not a BASELINE config)"),
    # the paper's own 3-D blast wave (E6, B = (1,1,1)/sqrt 3) at its largest size; Table 3 has its ms/step
    "e6": ("blast3d_paper", 128, "f32", "paper E6: 3-D blast wave, 128^3, fp32, B=(1,1,1)/sqrt(3) (PAPER.md:539-559; not a BASELINE config)"),
}
# BASELINE.md section 1, the paper's own number for the same workload on another machine (context, not the target):
# 128^3 fp32 3-D blast on a GTX 480, 161.33 ms/step (Table 3) = 13.0 M cell-updates/s
PAPER_RATE = {"e6": 128 ** 3 / 161.33e-3}


def _gen(inputs, gen, n, **kw):
    if gen == "turbulence":
        return inputs.turbulence(n, **kw)
    return inputs.blast3d(n, paper_field=(gen == "blast3d_paper"), **kw)
ALGO_WORDS_STEP = 96          # ideal: each of the six L_i reads 8 fields and writes 8
CFL = 0.8
SPEC_PEAK_GBS = 8000.0        # the data-sheet HBM3e figure north_star words its target on (context; the roofline uses the measured copy rate)
# configs' own step counts (BASELINE.json): the headline line is timed at --steps, `long_run` repeats it at these
CONFIG_STEPS = {"c4": 100, "c5": 50, "c3": 200}


def ncu_traffic(workload, kernel):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel`, from the committed post-processing of the
    ncu --set full capture (profiles/r02_traffic.json names the capture it came from); None where no capture exists"""
    p = os.path.join(ROOT, "profiles", "r02_traffic.json")
    try:
        return json.load(open(p))["traffic_bytes_per_launch"][workload][kernel]
    except Exception:
        return None


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.12)
        self.proc.terminate()
        rows = [r for (t, r) in self.rows if t0 <= t <= t1 + 0.06] or [r for (_, r) in self.rows[-3:]]
        sm, smax, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            c = [x.strip() for x in r.split(",")]
            try:
                sm.append(float(c[0])); smax.append(float(c[1])); pw.append(float(c[2]))
            except Exception:
                continue
            for nm, v in zip(names, c[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def make_state(gen, n, prec, device):
    """seeded synthetic state of the workload, built on the device with torch (plumbing), in run precision"""
    import torch
    from paper_0908_4362_b200 import inputs
    kw = dict(xp=torch, xp_kw={"device": device})
    f, meta = _gen(inputs, gen, n, **kw)
    dt = torch.float32 if prec == "f32" else torch.float64
    out = [a.to(dt).contiguous() for a in f]
    del f
    torch.cuda.empty_cache()
    return out, meta


def l2_note(state_bytes):
    """how the timed state compares with the 126 MB L2 (timing rule: inputs larger than L2, or say so)"""
    gb = state_bytes / 1e9
    if state_bytes > 4 * 126e6:
        return f"state {gb:.2f} GB per copy >> 126 MB L2 (inputs larger than L2, no flush needed)"
    return f"state {gb:.3f} GB per copy is NOT large against the 126 MB L2: partly L2-resident, not an HBM data point"


def oracle_rate(gen, prec, budget_s=12.0, n=96, threads=None):
    """the oracle as it stands, timed on the host cores on a bounded sample of the workload"""
    import oracle
    from paper_0908_4362_b200 import inputs
    n_all = oracle.num_threads()
    if threads:
        oracle.set_num_threads(threads)
    try:
        return _oracle_rate(oracle, inputs, gen, prec, budget_s, n)
    finally:
        oracle.set_num_threads(n_all)


def _oracle_rate(oracle, inputs, gen, prec, budget_s, n):
    f, meta = _gen(inputs, gen, n)
    dt = np.float32 if prec == "f32" else np.float64
    st = [np.array(a, dtype=dt) for a in f]
    oracle.run(st, meta["gamma"], meta["bc"], 0, 1, CFL)            # page in / warm caches
    steps, t0 = 0, time.perf_counter()
    while True:
        oracle.run(st, meta["gamma"], meta["bc"], steps + 1, 1, CFL)
        steps += 1
        el = time.perf_counter() - t0
        if el > budget_s or steps >= 200:
            break
    return (n ** 3) * steps / el, oracle.num_threads(), f"{gen} {n}^3 {prec}, {steps} steps in {el:.1f} s"


def run_reference(args, rank, world):
    """--impl reference: the oracle (deliberately slow CPU program), same metric/config keys"""
    if rank != 0:
        return
    gen, n, prec, desc = WORKLOADS[args.workload]
    import oracle
    from paper_0908_4362_b200 import inputs
    ns = 96 if n >= 96 else n
    f, meta = _gen(inputs, gen, ns)
    dt = np.float32 if prec == "f32" else np.float64
    st = [np.array(a, dtype=dt) for a in f]
    k0 = 0
    for _ in range(args.warmup):
        oracle.run(st, meta["gamma"], meta["bc"], k0, 1, CFL); k0 += 1
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.run(st, meta["gamma"], meta["bc"], k0, 1, CFL); k0 += 1
    el = time.perf_counter() - t0
    val = ns ** 3 * args.steps / el
    sample = f"{gen} {ns}^3 {prec} sub-sample of the {n}^3 workload, {args.steps} steps"
    print(json.dumps({
        "impl": "reference", "metric": "MHD cell-updates/sec", "value": val, "unit": "cell-updates/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * el / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": prec, "data": "synthetic",
        "config": {"workload": f"{args.workload}: {desc}", "cfl": CFL, "sample": sample},
        "cpu_baseline": {"value": val, "unit": "cell-updates/s", "cores": oracle.num_threads(), "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": val, "unit": "cell-updates/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="c4", choices=sorted(WORKLOADS))
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-breakdown", action="store_true")
    ap.add_argument("--no-long-run", action="store_true", help="skip the second timed run at the config's own step count")
    ap.add_argument("--no-others", action="store_true", help="skip the short fp64 (c5) and 256^3 (c3) legs")
    ap.add_argument("--e2e-contexts", type=int, default=2, help="independent contexts pipelining the end-to-end jobs")
    ap.add_argument("--option", action="append", default=[], help="key=value passed to mhd_set_option")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3)

    from paper_0908_4362_b200.replicas import Replicas, env_rank
    rank, local_rank, world = env_rank()
    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    import torch
    from paper_0908_4362_b200 import binding as B      # raises if libmhd.so is missing: no fallback

    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local_rank)
    device = f"cuda:{local_rank}"
    rep = Replicas(backend="nccl", device=device)      # replicas only: barrier + max-over-ranks timing, no data-path collective
    barrier = rep.barrier

    gen, n, prec, desc = WORKLOADS[args.workload]
    N = n ** 3
    esize = 4 if prec == "f32" else 8
    state, meta = make_state(gen, n, prec, device)
    ws = torch.empty(B.mhd_workspace_bytes(n, n, n, B.MHD_F32 if prec == "f32" else B.MHD_F64), dtype=torch.uint8, device=device)
    stream = torch.cuda.Stream(device=device)
    sol = B.Solver(n, n, n, meta["gamma"], prec, meta["bc"], workspace=ws, stream=stream)
    for kv in args.option:
        k, v = kv.split("=")
        sol.set_option(k, int(v))
    torch.cuda.synchronize()
    sol.set_state(state)

    ev = lambda: torch.cuda.Event(enable_timing=True)

    # ---- device-resident throughput -----------------------------------------------------------
    def timed(sl, strm, steps):
        """steps of mhd_step between two CUDA events on the context's stream; clocks sampled during the region"""
        with torch.cuda.stream(strm):
            sampler = ClockSampler(local_rank)
            sampler.start()
            time.sleep(0.15)
            barrier()
            l0 = sl.launch_count()
            e0, e1 = ev(), ev()
            w0 = time.time()
            e0.record(strm)
            sl.step(steps, CFL, sync=False)
            e1.record(strm)
            barrier()
            w1 = time.time()
            l1 = sl.launch_count()
        return rep.max_over_ranks(e0.elapsed_time(e1)), sampler.stop(w0, w1), int(l1 - l0)

    with torch.cuda.stream(stream):
        sol.step(args.warmup, CFL, sync=True)
    ms, clocks, launches = timed(sol, stream, args.steps)
    t_now = sol.time()        # also surfaces a poisoned state
    value = N * world * args.steps / (ms * 1e-3)
    peak, peak_src = peaks()
    step_bytes = ALGO_WORDS_STEP * esize

    # the same at the config's own step count (BASELINE.json: c4 100 steps): long runs sit under the 1000 W power cap
    long_run = None
    ksteps = CONFIG_STEPS.get(args.workload)
    if ksteps and ksteps != args.steps and not args.no_long_run:
        lms, lclocks, _ = timed(sol, stream, ksteps)
        lval = N * world * ksteps / (lms * 1e-3)
        long_run = {"steps": ksteps, "ms_per_step": lms / ksteps, "value": lval, "clocks": lclocks,
                    "roofline_step_frac": step_bytes * (lval / world) / 1e9 / peak,
                    "roofline_step_frac_of_spec_peak": step_bytes * (lval / world) / 1e9 / SPEC_PEAK_GBS}

    # ---- per-kernel breakdown and roofline of the dominant kernel (rank 0) ---------------------
    roofline, breakdown = None, None
    if rank == 0 and not args.no_breakdown:
        dtv, _ = sol.cfl_dt(CFL)
        # algorithmic words per cell of each row follow the PATH THAT RAN, read off the kernel launches one apply makes
        # (ADVICE r2): a fluid kernel moves 13 words (8 in, 5 out), a B pair 8 (rho, m_d, 3 B in; 3 B out), a kernel that
        # fuses B pair + fluid 16, one that fuses two B pairs 8; mhd_apply adds one 1-thread launch that sets dt
        WORDS_BY_LAUNCHES = {"lrev": {1: (16, "one fused kernel"), 2: (8 + 13, "B pair kernel + fluid kernel")},
                             "mid": {2: (13 + 16, "fluid kernel + one kernel fusing B pair, B pair, fluid"),
                                     3: (13 + 8 + 13, "fluid + one kernel fusing the two B pairs + fluid"),
                                     4: (13 + 8 + 8 + 13, "fluid, B pair, B pair, fluid: four kernels")}}
        kinds = [("fluid_x", B.MHD_OP_FLUID, 0, 13), ("fluid_y", B.MHD_OP_FLUID, 1, 13), ("fluid_z", B.MHD_OP_FLUID, 2, 13),
                 ("bpair_x", B.MHD_OP_BPAIR, 0, 8), ("bpair_y", B.MHD_OP_BPAIR, 1, 8), ("bpair_z", B.MHD_OP_BPAIR, 2, 8),
                 ("lrev_x", B.MHD_OP_SWEEP_REVERSE, 0, "lrev"), ("lrev_y", B.MHD_OP_SWEEP_REVERSE, 1, "lrev"),
                 ("lrev_z", B.MHD_OP_SWEEP_REVERSE, 2, "lrev"),
                 ("mid_y", B.MHD_OP_MIDDLE_PAIR, 1, "mid"), ("mid_z", B.MHD_OP_MIDDLE_PAIR, 2, "mid")]
        breakdown = {}
        reps = 5
        with torch.cuda.stream(stream):
            for name, op, d, words in kinds:
                sol.set_state(state)                           # repeated single operators are not a stable scheme: start each kind
                dtv, _ = sol.cfl_dt(CFL)                       # from the workload's initial state, dt at its CFL limit
                l0 = sol.launch_count()
                sol.apply(op, d, 0, dtv)                       # warm
                nk = sol.launch_count() - l0 - 1               # kernels of one apply, without the 1-thread set_dt launch
                path = None
                if isinstance(words, str):
                    words, path = WORDS_BY_LAUNCHES[words].get(nk, (None, f"{nk} kernels"))
                a, b = ev(), ev()
                torch.cuda.synchronize()
                a.record(stream)
                for _ in range(reps):
                    sol.apply(op, d, 0, dtv)
                b.record(stream)
                torch.cuda.synchronize()
                kms = a.elapsed_time(b) / reps                 # includes the 1-thread set_dt launch (~2 us)
                breakdown[name] = {"ms": kms, "algo_GBps": (words * esize * N / (kms * 1e-3) / 1e9) if words else None,
                                   "words_per_cell": words, "kernels_per_apply": nk}
                if path:
                    breakdown[name]["path"] = path
            # the stand-alone c_max pass (first step / after mhd_apply only; steps fuse it into their last kernel):
            # cmax_reuse = 0 makes every mhd_cfl_dt run the reduction instead of returning the cached c_max
            sol.set_state(state)
            sol.set_option("cmax_reuse", 0)
            sol.cfl_dt(CFL)
            a, b = ev(), ev()
            torch.cuda.synchronize()
            a.record(stream)
            for _ in range(reps):
                sol.cfl_dt(CFL)
            b.record(stream)
            torch.cuda.synchronize()
            sol.set_option("cmax_reuse", 1)
            kms = a.elapsed_time(b) / reps             # includes the D2H read of dt and its synchronisation
            breakdown["cfl"] = {"ms": kms, "algo_GBps": 8 * esize * N / (kms * 1e-3) / 1e9, "words_per_cell": 8,
                                "includes": "per call: the reduction kernel, the 1-thread dt kernel, the D2H read of dt and the stream synchronisation mhd_cfl_dt does (a step pays none of this: its reduction is fused into its last kernel)"}
        # Dominant kernel = largest share of a step.  Launches per step, averaged over the three sweep orders:
        # fluid_y, fluid_z 2 each (one kernel template, fluid_yz_ring_kernel, 4 launches), B pair y/z 2 each
        # (bpair_ring_kernel, 4 launches), fluid_x 1 + bpair_x 1 (forward L_x) and the reverse L_x (1).
        share = {"fluid_yz": 2 * (breakdown["fluid_y"]["ms"] + breakdown["fluid_z"]["ms"]),
                 "bpair_yz": 2 * (breakdown["bpair_y"]["ms"] + breakdown["bpair_z"]["ms"]),
                 "fluid_x": breakdown["fluid_x"]["ms"], "bpair_x": breakdown["bpair_x"]["ms"],
                 "lrev_x": breakdown["lrev_x"]["ms"]}
        dom = max(share, key=share.get)
        if dom.endswith("_yz"):
            a_, b_ = breakdown[dom[:-2] + "y"], breakdown[dom[:-2] + "z"]
            kms, words = 0.5 * (a_["ms"] + b_["ms"]), a_["words_per_cell"]
        else:
            kms, words = breakdown[dom]["ms"], breakdown[dom]["words_per_cell"]
        ach = words * esize * N / (kms * 1e-3) / 1e9
        # DRAM bytes one step actually moves (ncu dram__bytes of every kernel x its launches per step, profiles/r02_traffic.json)
        # over the measured step time: the "achieved HBM GB/s" north_star's >= 60 % target is worded on
        lpstep = {"fluid_yz": 4, "bpair_yz": 4, "fluid_x": 1, "bpair_x": 1, "lrev_x": 1}
        tr = {k: ncu_traffic(args.workload, k) for k in lpstep}
        if all(v is not None for v in tr.values()) and sol.launch_count() > 0 and breakdown["lrev_x"]["kernels_per_apply"] == 1:
            dram_step = float(sum(tr[k] * lpstep[k] for k in lpstep))
        elif all(tr.get(k) is not None for k in ("fluid_yz", "bpair_yz", "fluid_x", "bpair_x")):
            dram_step = float(tr["fluid_yz"] * 4 + tr["bpair_yz"] * 4 + tr["fluid_x"] * 2 + tr["bpair_x"] * 2)   # reverse L_x as two kernels
        else:
            dram_step = None
        step_s = (ms / args.steps) * 1e-3
        roofline = {"bound": "hbm", "kernel": dom, "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                    "frac_is": f"the dominant kernel ({dom}) alone on its own {words} words per cell; the whole step is roofline.step",
                    "traffic": ncu_traffic(args.workload, dom), "peak_source": peak_src,
                    "frac_of_spec_peak": ach / SPEC_PEAK_GBS,
                    "algorithmic_bytes_per_launch": words * esize * N, "ms_per_launch": kms,
                    "share_of_step": share[dom] / sum(share.values()),
                    "step": {"algorithmic_bytes_per_cell_step": ALGO_WORDS_STEP * esize,
                             "achieved": ALGO_WORDS_STEP * esize * (value / world) / 1e9,
                             "frac": ALGO_WORDS_STEP * esize * (value / world) / 1e9 / peak,
                             "frac_of_spec_peak": ALGO_WORDS_STEP * esize * (value / world) / 1e9 / SPEC_PEAK_GBS,
                             "dram_bytes_per_step_ncu": dram_step,
                             "dram_gbs_achieved": (dram_step / step_s / 1e9) if dram_step else None,
                             "dram_frac_of_measured_peak": (dram_step / step_s / 1e9 / peak) if dram_step else None,
                             "dram_frac_of_spec_peak": (dram_step / step_s / 1e9 / SPEC_PEAK_GBS) if dram_step else None,
                             "dram_source": "profiles/r02_traffic.json (ncu --set full, dram__bytes_read.sum + dram__bytes_write.sum per launch) x launches per step / the step time measured here"}}

    # ---- end to end through the C ABI with HOST buffers ----------------------------------------
    e2e = None
    if not args.no_e2e:
        # Every job = H2D of its 8 input fields from pinned host memory, one mhd_step, D2H of the 8 result fields,
        # all through the C ABI with HOST pointers.  Jobs are independent, so two contexts (own workspace, own
        # stream) driven by two host threads keep both PCIe directions and the SMs busy at once; one context
        # alone alternates between them (--e2e-contexts 1 measures that).
        import threading
        nctx = max(1, args.e2e_contexts)
        k_e2e = 3
        sols, hosts = [sol], []
        for _ in range(1, nctx):
            ws2 = torch.empty(ws.numel(), dtype=torch.uint8, device=device)
            s2 = B.Solver(n, n, n, meta["gamma"], prec, meta["bc"], workspace=ws2, stream=torch.cuda.Stream(device=device))
            for kv in args.option:
                k, v = kv.split("=")
                s2.set_option(k, int(v))
            sols.append(s2)
        for _ in range(nctx):
            host = [torch.empty((n, n, n), dtype=state[0].dtype, pin_memory=True) for _ in range(8)]
            for h, s in zip(host, state):
                h.copy_(s)
            hosts.append(host)
        torch.cuda.synchronize()
        errs = []

        def worker(sl, host):
            try:
                torch.cuda.set_device(local_rank)      # the current device is per host thread
                for _ in range(k_e2e):
                    sl.set_state(host)                 # H2D of the job's inputs (pinned host memory)
                    sl.step(1, CFL, sync=True)
                    sl.get_state(host)                 # D2H of the job's result
            except Exception as ex:                    # surfaces in the main thread
                errs.append(ex)

        threads = [threading.Thread(target=worker, args=(sl, h)) for sl, h in zip(sols, hosts)]
        barrier()
        t0 = time.perf_counter()
        for t in threads:
            t.start()
        for t in threads:
            t.join()
        barrier()
        el = time.perf_counter() - t0
        if errs:
            raise errs[0]
        el = rep.max_over_ranks(el)
        jobs = k_e2e * nctx
        e2e = {"value": N * world * jobs / el, "unit": "cell-updates/s", "h2d_bytes_per_step": 8 * N * esize,
               "d2h_bytes_per_step": 8 * N * esize, "steps": jobs, "contexts": nctx}
        for s2 in sols[1:]:
            s2.close()
        del hosts

    # ---- the other bandwidth-bound configs, short legs: c5 (512^3 fp64) and c3 (256^3 fp32 blast) -------------
    # BASELINE.json's metric is "fp32 & fp64 at 256^3/512^3": the headline line is c4; these make the rest driver-measured
    others = None
    if world == 1 and args.workload == "c4" and not args.no_others:
        sol.close()
        sol = None
        del ws, state
        torch.cuda.empty_cache()
        others = {}
        for name, ksteps in (("c5", 10), ("c3", 50)):
            g2, n2, p2, d2 = WORKLOADS[name]
            st2, m2 = make_state(g2, n2, p2, device)
            ws2 = torch.empty(B.mhd_workspace_bytes(n2, n2, n2, B.MHD_F32 if p2 == "f32" else B.MHD_F64), dtype=torch.uint8, device=device)
            s2 = B.Solver(n2, n2, n2, m2["gamma"], p2, m2["bc"], workspace=ws2, stream=stream)
            torch.cuda.synchronize()
            s2.set_state(st2)
            with torch.cuda.stream(stream):
                s2.step(args.warmup, CFL, sync=True)
            oms, oclk, _ = timed(s2, stream, ksteps)
            s2.time()
            oval = n2 ** 3 * ksteps / (oms * 1e-3)
            es2 = 4 if p2 == "f32" else 8
            others[name] = {"workload": d2, "dtype": p2, "steps": ksteps, "ms_per_step": oms / ksteps, "value": oval,
                            "unit": "cell-updates/s", "clocks": oclk,
                            "roofline_step_frac": ALGO_WORDS_STEP * es2 * oval / 1e9 / peak,
                            "roofline_step_frac_of_spec_peak": ALGO_WORDS_STEP * es2 * oval / 1e9 / SPEC_PEAK_GBS,
                            "l2": l2_note(8 * n2 ** 3 * es2)}
            s2.close()
            del s2, ws2, st2
            torch.cuda.empty_cache()
        # c1 (1-D Brio-Wu 512, fp64, outflow) and c2 (2-D Orszag-Tang 256^2, fp32 and fp64): a few thousand cells, bound by
        # launch latency (a step is ten launches replayed as a CUDA graph), reported for completeness of "each config"
        from paper_0908_4362_b200 import inputs as _inp
        # ... and the largest sizes of the paper's own Tables 1 and 2 with the paper's GTX 480 ms per step beside them
        # (another machine: context)
        for name, (fgen, shape, p2, ksteps, d2, paper_ms) in {
                "c1": (_inp.brio_wu, (512, 1, 1), "f64", 100, "configs[0]: 1-D Brio-Wu, 512x1x1, fp64, outflow, cfl 0.8", 3.21),
                "c2_f32": (_inp.orszag_tang, (256, 256, 1), "f32", 500, "configs[1]: 2-D Orszag-Tang, 256x256x1, fp32, periodic, cfl 0.8", 12.48),
                "c2_f64": (_inp.orszag_tang, (256, 256, 1), "f64", 500, "configs[1]: 2-D Orszag-Tang, 256x256x1, fp64, periodic, cfl 0.8", 21.59),
                "t1_4096_f32": (_inp.brio_wu, (4096, 1, 1), "f32", 200, "paper Table 1: 1-D Brio-Wu, 4096x1x1, fp32", 4.31),
                "t2_1024_f32": (_inp.orszag_tang, (1024, 1024, 1), "f32", 200, "paper Table 2: 2-D Orszag-Tang, 1024x1024x1, fp32", 96.43),
                "t2_1024_f64": (_inp.orszag_tang, (1024, 1024, 1), "f64", 200, "paper Table 2: 2-D Orszag-Tang, 1024x1024x1, fp64", 144.48)}.items():
            f2_, m2 = fgen(shape[0])
            dt2 = np.float32 if p2 == "f32" else np.float64
            s2 = B.Solver(shape[0], shape[1], shape[2], m2["gamma"], p2, m2["bc"], stream=stream)
            s2.set_state([np.ascontiguousarray(a, dtype=dt2) for a in f2_])
            with torch.cuda.stream(stream):
                s2.step(args.warmup, CFL, sync=True)
            oms, oclk, _ = timed(s2, stream, ksteps)
            s2.time()
            ncell = shape[0] * shape[1] * shape[2]
            others[name] = {"workload": d2, "dtype": p2, "steps": ksteps, "ms_per_step": oms / ksteps,
                            "value": ncell * ksteps / (oms * 1e-3), "unit": "cell-updates/s", "clocks": oclk,
                            "l2": l2_note(8 * ncell * (4 if p2 == "f32" else 8)),
                            "paper_gtx480_ms_per_step": paper_ms, "vs_paper_gtx480": paper_ms / (oms / ksteps)}
            s2.close()

    cpu = None
    if rank == 0 and not args.no_cpu_baseline:
        v, cores, sample = oracle_rate(gen, prec)
        cpu = {"value": v, "unit": "cell-updates/s", "cores": cores, "kind": "oracle", "sample": sample}
        # the baseline of record (the paper's own CPU comparison is a serial code on one core)
        v1, c1, sample1 = oracle_rate(gen, prec, budget_s=6.0, threads=1)
        cpu["serial"] = {"value": v1, "unit": "cell-updates/s", "cores": c1, "kind": "oracle", "sample": sample1}

    if rank == 0:
        out = {
            "metric": "MHD cell-updates/sec", "value": value, "unit": "cell-updates/s", "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": (value / PAPER_RATE[args.workload] if args.workload in PAPER_RATE else None),
            "dtype": prec, "data": "synthetic",
            "config": {"workload": f"{args.workload}: {desc}", "grid": [n, n, n], "cfl": CFL, "gamma": meta["gamma"],
                       "parallelism": "replicas only" if world > 1 else "single GPU",
                       "l2": l2_note(8 * N * esize),
                       "t_grid_after": t_now},
            "clocks": clocks, "gpu_launches": launches, "kernels": breakdown, "others": others, "e2e": e2e,
            "roofline": roofline, "cpu_baseline": cpu, "long_run": long_run,
        }
        # LAST in the line, compact: the whole of BASELINE.json's metric ("fp32 & fp64 at 256^3/512^3") in one place, so
        # that a record which keeps only the tail of the line still carries it
        def brief(r):
            return None if not r else {"steps": r["steps"], "ms_per_step": round(r["ms_per_step"], 4), "value": round(r["value"]),
                                       "step_frac_of_measured_peak": round(r["roofline_step_frac"], 4),
                                       "step_frac_of_spec_peak": round(r["roofline_step_frac_of_spec_peak"], 4),
                                       "sm_mhz": (r.get("clocks") or {}).get("sm_mhz"), "reasons": (r.get("clocks") or {}).get("reasons")}
        out["summary"] = {
            "unit": "cell-updates/s; fractions are 96 words per cell-step (384 B fp32, 768 B fp64) x value over the HBM peak (measured copy rate / 8 TB/s data sheet)",
            f"{args.workload}_at_--steps": {"steps": args.steps, "ms_per_step": round(ms / args.steps, 4), "value": round(value),
                                           "step_frac_of_measured_peak": roofline and round(roofline["step"]["frac"], 4),
                                           "step_frac_of_spec_peak": roofline and round(roofline["step"]["frac_of_spec_peak"], 4),
                                           "dram_gbs_achieved": roofline and roofline["step"]["dram_gbs_achieved"] and round(roofline["step"]["dram_gbs_achieved"], 1),
                                           "dram_frac_of_spec_peak": roofline and roofline["step"]["dram_frac_of_spec_peak"] and round(roofline["step"]["dram_frac_of_spec_peak"], 4),
                                           "sm_mhz": clocks.get("sm_mhz") if clocks else None},
            f"{args.workload}_at_config_steps": brief(long_run),
            "c5_512^3_f64": brief((others or {}).get("c5")), "c3_256^3_f32": brief((others or {}).get("c3")),
            "dominant_kernel_frac": roofline and round(roofline["frac"], 4),
            "cpu_oracle_sample": cpu and cpu.get("sample"),
        }
        print(json.dumps(out))
    if sol is not None:
        sol.close()
    rep.close()


if __name__ == "__main__":
    main()
