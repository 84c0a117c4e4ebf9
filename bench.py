"""bench.py — radiation cell-updates/s of one full gray-M1 sub-step on B200 (BASELINE.json `metric`).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C4|C5|C3|CP] [--impl native|reference]

A "step" is one pass of the whole hot path over the resident fields, one rt_substep call: ghost fill ->
thick-limit pre-pass -> k_substep_fused (ONE kernel: reconstruction, f-fix, closure, wave speeds, Riemann fluxes of
the three directions, flux divergence + geometric sources, floor, opacities, implicit coupling, CFL rate of the
updated state) -> one-thread dt finalise; the time step stays on the device.  `--fused-seg -1` runs the same call
on the per-direction kernels (x1/x2/x3 sweeps + implicit), `--api split` times the three-call form rt_cfl_dt
(8-byte result to the host) -> rt_explicit_step -> rt_implicit_step.  Default workload: C4,
the 256^3 Cartesian config the north_star target is quoted on (C5 = the spherical one).
Prints ONE JSON line (see DESIGN.md "Measurement" for every key).  `--impl reference` times the CPU
oracle instead (the only other place oracle/ may be executed besides the cpu_baseline leg).
N > 1 (torchrun): the path does not shard (north_star: one GPU, no collectives) -> N independent
replicas, value = N x cells x K / max-over-ranks time, "scaling": "weak".
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

METRIC = "radiation cell-updates/sec (fp64, 1 B200)"
UNIT = "cell-updates/s"

FUSED_CFL = True
FUSED_KERNEL = True   # rt_substep runs k_substep_fused (2-D / 3-D grids, --fused-seg >= 0, --api fused)

# fp64-pipe roof by formula, kept beside the MEASURED one (rt_measure_fp64, same process): 148 SMs x 64 lanes/clk x 1.965 GHz
FP64_FORMULA_TINST = 148 * 64 * 1.965e9 / 1e12
N_SM = 148
REGIONS = 5           # timed regions of K steps each; the line reports the median (SURVEY 8(d) "Timing")


def method_bytes_per_cell(feedback):
    """compulsory HBM traffic of one sub-step: read E, F, rho, T (+ m) and write E, F, T (+ m)"""
    return 88.0 + (48.0 if feedback else 0.0)


# Algorithmic bytes per interior cell and launch: 8 B x (fields read + written)
def bytes_per_cell(kind, thick, feedback):
    return {
        "thick_limit": 24.0 if not FUSED_KERNEL else 32.0,     # read rho, T; write lim (+ rho kappa_P for the fused kernel)
        "sweep_x1": 64.0 + (8.0 if thick else 0.0),            # read U 4 (+ lim); write U_out 4
        "sweep_x2": 96.0 + (8.0 if thick else 0.0),            # read U 4 (+ lim) + U_out 4; write U_out 4
        "sweep_x3": 96.0 + (8.0 if thick else 0.0),
        "implicit": 88.0 + (48.0 if feedback else 0.0),        # read E,F,rho,T (+m); write E,F,T (+m)
        "cfl": 32.0 if not FUSED_CFL else 0.0,                 # split API: read E,F; fused: a one-thread finalise kernel
        "ghost_fill": 0.0,                                     # O(surface)
        # k_substep_fused: read U 4 (+ lim), rho, T (+ m 3); write E, F, T (+ m 3)
        "fused": 88.0 + (16.0 if thick else 0.0) + (48.0 if feedback else 0.0),   # thick: + lim + rho kappa_P
    }[kind]


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="C4")
    ap.add_argument("--impl", default="native", choices=["native", "reference"])
    ap.add_argument("--size", type=int, default=0, help="override the grid side (debug only; marks the line)")
    ap.add_argument("--api", default="fused", choices=["fused", "split"])
    ap.add_argument("--fused-seg", type=int, default=0, help="rt_set_tuning fused_seg: 0 auto, -1 per-direction kernels, >0 x3 segment")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-also", action="store_true", help="skip the second north_star config (C5 beside C4)")
    ap.add_argument("--graph", action="store_true", help="replay the sub-steps from a CUDA graph of two (latency-bound grids)")
    return ap.parse_args()


def make_workload(name, size=0):
    import rt_workloads as W
    if size:
        if name in ("C3", "C4", "CP"):
            return W.BY_NAME[name](nside=size)
        if name == "C5":
            return W.c5(n=(size, size // 2, size))
    return W.BY_NAME[name]()


def workload_config(w, args):
    n = w.n
    cfg = {"workload": "%s: %s %dx%dx%d, %s" % (w.name, ("cartesian", "cylindrical", "spherical")[w.geometry], n[0], n[1], n[2],
                                                w.notes),
           "cells": w.ncells, "substep": ("rt_substep (k_substep_fused, device-resident dt)" if args.fused_seg >= 0 else
                                       "rt_substep (per-direction kernels, device-resident dt)") if args.api == "fused" else
           "rt_cfl_dt + rt_explicit_step + rt_implicit_step",
           "solver": "HLL/GLF alternating" if w.solver_schedule else ("HLL" if w.params["solver"] == 0 else "GLF"),
           "thick_limit": int(w.params["thick_limit"]), "feedback_momentum": int(w.params["feedback_momentum"]),
           "l2": "inputs larger than L2 (%.2f GB resident fields vs 126 MB)" % (13 * 8 * float(__import__("numpy").prod(w.shape)) / 1e9),
           "parallelism": "replicas only" if args.gpus > 1 else "1 GPU"}
    if args.size:
        cfg["debug_size_override"] = args.size
    return cfg


class ClockSampler(threading.Thread):
    """samples SM clock and throttle reasons through NVML while the timed region runs"""

    def __init__(self, index, period=0.02):
        super().__init__(daemon=True)
        self.index, self.period = index, period
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop_evt = threading.Event()
        self.ok = False
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
        nv = self.nv
        names = {"hw_slowdown": nv.nvmlClocksThrottleReasonHwSlowdown,
                 "hw_thermal_slowdown": nv.nvmlClocksThrottleReasonHwThermalSlowdown,
                 "sw_thermal_slowdown": nv.nvmlClocksThrottleReasonSwThermalSlowdown,
                 "sw_power_cap": nv.nvmlClocksThrottleReasonSwPowerCap,
                 "hw_power_brake": nv.nvmlClocksThrottleReasonHwPowerBrakeSlowdown}
        while not self._stop_evt.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(self.period)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=2.0)
        s = sorted(self.samples)
        return {"sm_mhz": s[len(s) // 2] if s else None, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(s)}


def replicas_throughput(ms_local, cells, steps, world, device=None):
    """whole-job throughput of `world` independent replicas (DESIGN.md Sect. 9: the path does not shard): every rank
    runs `steps` sub-steps over `cells` cells in ms_local milliseconds; the job takes the slowest rank's time.
    Returns (cell-updates/s over all ranks, max-over-ranks ms).  Uses the initialised process group when world > 1."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms_local], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms_max = float(t.item())
    return world * cells * steps / (ms_max * 1e-3), ms_max


# ------------------------------------------------------------------------------------------ native arm
def one_substep(rt, g, w, st, step_index):
    """the whole hot path once"""
    if w.solver_schedule:
        g.set_params(rt.make_params(**dict(w.params, solver=w.solver_at(step_index))))
    if FUSED_CFL:
        g.substep(st.dt_dev, w.cfl, st.rho, st.T, st.mom, st.U, st.U2)
        st.U, st.U2 = st.U2, st.U
        return None
    dt = g.cfl_dt(st.U, w.cfl)
    g.explicit_step(dt, st.rho, st.T, st.U, st.U2)
    g.implicit_step(dt, st.rho, st.T, st.mom, st.U2)
    st.U, st.U2 = st.U2, st.U
    return dt


def csrc_hash():
    """sha256 over the CUDA sources k_substep_fused and its launch are built from (everything under csrc/ except the two
    files that hold only self-contained extras: the fp64 microbenchmark kernels and the no-alloc CFL entry point): ties
    the ncu-derived instruction counts under profiles/ to the code they were taken from"""
    import hashlib
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2606_26268_b200", "csrc")
    for f in sorted(os.listdir(d)):
        if f in ("rt_kernels_measure.cuh", "rt_noalloc.cu"):
            continue
        with open(os.path.join(d, f), "rb") as fh:
            h.update(f.encode() + b"\0" + fh.read())
    return h.hexdigest()[:16]


def load_fp64_counts(workload):
    """executed fp64-pipe thread instructions per cell-update and ncu's fp64-pipe-active % of k_substep_fused, from
    profiles/fp64_counts.txt (written by bench_ncu_counts.py from an `ncu --page source/raw --csv` export).  Returns
    None when the file is missing or was taken from other sources than the ones in the tree (stale)."""
    try:
        with open(os.path.join(ROOT, "profiles", "fp64_counts.txt")) as fh:
            d = json.load(fh)
    except Exception:
        return None
    if d.get("csrc_hash") != csrc_hash():
        return {"stale": True, "capture_csrc_hash": d.get("csrc_hash"), "tree_csrc_hash": csrc_hash()}
    return d.get("workloads", {}).get(workload)


def measure_fp64_peak(rt, dev):
    """DFMA microbenchmark in this process (rt_measure_fp64), 8 warps per SM sub-partition, ~10 ms per launch, best of 3,
    in 1e12 DFMA thread instructions per second:
      chains8      8 chains x = fma(x, a, b), a and b shared by the chains (the operand reuse cache serves them)
      two_reg      4 chains x = fma(x, y_c, const): two register operands, like DMUL / DADD  -> the pipe's own rate
      three_reg    4 chains x = fma(x, y_c, z_c): three different register pairs -> the register file's rate (3 cycles)
      *_plus_fmul  the same with 4 independent fp32 multiplies per 4 DFMAs: what an instruction of another pipe costs
                   while the fp64 pipe is busy (DESIGN.md Sect. 5)
    The roof bench.py divides by is the best of the first two."""
    out = {}
    for key, code in (("chains8", 8), ("two_reg", 204), ("three_reg", 304), ("two_reg_plus_fmul", 214), ("three_reg_plus_fmul", 314)):
        best = 0.0
        for _ in range(3):
            ms, n = rt.measure_fp64(148 * 4, 256, code, 20000 if code == 8 else 40000, device=dev)
            best = max(best, n / (ms * 1e-3))
        out[key] = best / 1e12
    out["peak"] = max(out["chains8"], out["two_reg"])
    return out


def measure_workload(args, rt, drv, w, dev, world, K, Wm, regions, barrier):
    """the device-resident timing of one workload: returns a dict with value, ms_per_step (median of `regions` timed regions
    of K sub-steps), per-kernel times, clocks, launches and the live state.  --graph: the sub-steps are replayed from a
    CUDA graph holding two of them (the ping-pong of the two state buffers; K is rounded up to an even number), which is
    how a launch-latency-bound grid (C1, C2) would be driven; everything then runs on a side stream."""
    import contextlib
    import torch
    side = torch.cuda.Stream(dev) if args.graph else None
    ctx = torch.cuda.stream(side) if side is not None else contextlib.nullcontext()
    with ctx:
        g = drv.grid_from_workload(w, device=dev)
        g.set_tuning(fused_seg=args.fused_seg)
        st = drv.DeviceState(g, w)
        st.dt_dev = torch.zeros(1, dtype=torch.float64, device=dev)
        g.cfl_dt_async(st.U, w.cfl, st.dt_dev)
        sampler = ClockSampler(dev.index if dev.index is not None else 0, period=0.002)
        sampler.start()
        step = 0
        for _ in range(Wm + (Wm & 1 if args.graph else 0)):   # an even count keeps the buffer roles of the captured pair
            one_substep(rt, g, w, st, step)
            step += 1
        graph = None
        if args.graph:
            K += K & 1
            torch.cuda.synchronize()
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(graph, stream=side):
                one_substep(rt, g, w, st, step)
                one_substep(rt, g, w, st, step + 1)

        def run(nsteps):
            nonlocal step
            if graph is not None:
                for _ in range(nsteps // 2):
                    graph.replay()
            else:
                for _ in range(nsteps):
                    one_substep(rt, g, w, st, step)
                    step += 1

        ms_regions, launches = [], 0
        per_step = None
        for _ in range(regions):
            barrier()
            l0 = g.launch_count()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            run(K)
            e1.record()
            barrier()
            launches = g.launch_count() - l0
            ms_regions.append(e0.elapsed_time(e1))
        clocks = sampler.stop()
        ms_med = sorted(ms_regions)[len(ms_regions) // 2]
        value, ms_max = replicas_throughput(ms_med, w.ncells, K, world, dev)

        # per-kernel device times over K more steps (instrumented pass, eager launches): CUDA events on the launching
        # stream, inside the library
        g.set_profiling(True)
        l0 = g.launch_count()
        for _ in range(K):
            one_substep(rt, g, w, st, step)
            step += 1
        eager_launches = g.launch_count() - l0
        kt = g.kernel_times()
        g.set_profiling(False)
        if graph is not None:
            launches = eager_launches      # kernels per K steps: a replay launches what the capture recorded
    return {"g": g, "st": st, "value": value, "ms_per_step": ms_max / K, "ms_regions": [round(m / K, 5) for m in ms_regions],
            "kt": kt, "clocks": clocks, "launches": int(launches), "step": step, "K": K}


def roofline_block(w, m, K, world, peaks, fp64_peak):
    """roofline of the dominant kernel (HBM, on the METHOD's compulsory bytes), every kernel's own figures, the whole
    sub-step, and the fp64-pipe side block"""
    thick, feedback = bool(w.params["thick_limit"]), bool(w.params["feedback_momentum"]) and w.mom is not None
    kt = m["kt"]
    kernels = {}
    tot_ms = sum(v[0] for v in kt.values())
    for name, (tot, cnt) in kt.items():
        if cnt == 0:
            continue
        avg = tot / cnt
        b = bytes_per_cell(name, thick, feedback) * w.ncells
        kernels[name] = {"launches_per_step": cnt / K, "avg_ms": round(avg, 5), "share": round(tot / tot_ms, 4),
                         "alg_bytes": b, "GBps": round(b / (avg * 1e-3) / 1e9, 1) if avg > 0 else None}
    dom = max(kernels, key=lambda k: kt[k][0])
    avg_ms = kernels[dom]["avg_ms"]
    # the method's bytes for the kernel that does the whole sub-step; a per-direction kernel keeps its own algorithmic bytes
    mb = method_bytes_per_cell(feedback) if dom == "fused" else bytes_per_cell(dom, thick, feedback)
    alg = mb * w.ncells
    achieved = alg / (avg_ms * 1e-3) / 1e9
    sub_bytes = sum(bytes_per_cell(k, thick, feedback) * kernels[k]["launches_per_step"] for k in kernels)
    sub_GBps = sub_bytes * m["value"] / world / 1e9
    method_GBps = method_bytes_per_cell(feedback) * m["value"] / world / 1e9
    roof = {"bound": "hbm", "kernel": dom, "achieved": round(achieved, 1), "peak": peaks["hbm_gbs"], "unit": "GB/s",
            "frac": round(achieved / peaks["hbm_gbs"], 4), "traffic": load_traffic(dom, w.name),
            "peak_source": peaks["source"],
            "bytes_per_cell": mb, "bytes_note": "compulsory bytes of the method for one sub-step (SURVEY 8(d)): read E, F, rho, T"
            " (+ m), write E, F, T (+ m); the kernel's own algorithmic bytes (adds the lim and rho kappa_P arrays of the"
            " pre-pass) are in kernels.%s.alg_bytes" % dom,
            "alg_bytes_per_launch": alg, "avg_launch_ms": avg_ms, "kernels": kernels,
            "kernel_ms_sum_per_step": round(tot_ms / K, 4),
            "substep": {"method_bytes_per_cell": method_bytes_per_cell(feedback), "method_GBps": round(method_GBps, 1),
                        "method_frac": round(method_GBps / peaks["hbm_gbs"], 4),
                        "alg_bytes_per_cell_all_kernels": sub_bytes, "alg_GBps": round(sub_GBps, 1),
                        "alg_frac": round(sub_GBps / peaks["hbm_gbs"], 4)}}
    # fp64 pipe: the roof that binds the fused kernel (DESIGN.md Sect. 5).  Peak MEASURED in this process; executed
    # instructions per cell from the committed ncu capture of the same sources (refused when stale)
    probes = fp64_peak
    fp64_peak = probes["peak"]
    alu = {"peak_measured_Tinst": round(fp64_peak, 3), "peak_formula_Tinst": round(FP64_FORMULA_TINST, 3),
           "peak_source": "rt_measure_fp64 in this run: the better of DFMA chains with shared operands (8 per thread) and"
                          " with two register operands (4 per thread), 8 warps per SM sub-partition",
           "probes_Tinst": {k: round(v, 3) for k, v in probes.items() if k != "peak"}}
    cnt = load_fp64_counts(w.name) if dom == "fused" else None
    if cnt and not cnt.get("stale"):
        inst = cnt["fp64_thread_inst_per_cell"]
        ach = inst * w.ncells / (avg_ms * 1e-3) / 1e12
        alu.update({"executed_fp64_thread_inst_per_cell": inst, "achieved_Tinst": round(ach, 3),
                    "frac_of_measured": round(ach / fp64_peak, 4), "ncu_pipe_fp64_active_pct": cnt.get("pipe_fp64_active_pct"),
                    "counts_source": "profiles/fp64_counts.txt (bench_ncu_counts.py; same csrc hash as the tree)"})
        # the issue slot: every executed warp instruction holds it for max(pipe, even source registers, odd source
        # registers) cycles (2 for the fp64 pipe, 3 for a DFMA with three register operands, 1 otherwise), one after the
        # other; the sum over the kernel's instruction stream is its own lower bound on this device
        ic = cnt.get("issue_cycles_per_warp_of_cells")
        sm_mhz = (m.get("clocks") or {}).get("sm_mhz")
        if ic and sm_mhz:
            bound_ms = ic * (w.ncells / 32.0) / (N_SM * 4) / (sm_mhz * 1e6) * 1e3
            alu["issue"] = {"cycles_per_warp_of_cells": ic, "bound_ms": round(bound_ms, 4), "frac": round(bound_ms / avg_ms, 4),
                            "sm_mhz": sm_mhz,
                            "note": "issue cycles of the executed instruction stream (ncu capture) / (148 SMs x 4 schedulers x"
                                    " the SM clock sampled during the timed region) over the measured launch time"}
    elif cnt:
        alu.update(cnt)
    roof["alu"] = alu
    return roof


def run_native(args):
    import numpy as np
    import torch
    import torch.distributed as dist
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py: no CUDA device; the product has no CPU path")
    from paper_2606_26268_b200 import rt
    from rt_workloads import drive_rt as drv

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    global FUSED_CFL, FUSED_KERNEL
    FUSED_CFL = args.api == "fused"
    FUSED_KERNEL = FUSED_CFL and args.fused_seg >= 0
    K, Wm = args.steps, max(args.warmup, 0)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    peaks = load_peaks()
    fp64_peak = measure_fp64_peak(rt, dev)
    w = make_workload(args.workload, args.size)
    m = measure_workload(args, rt, drv, w, dev, world, K, Wm, REGIONS, barrier)
    K = m["K"]
    out = {"metric": METRIC, "value": m["value"], "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
           "ms_per_step": m["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": "f64", "data": "synthetic", "config": workload_config(w, args), "clocks": m["clocks"],
           "gpu_launches": m["launches"], "timing": {"regions": REGIONS, "steps_per_region": K, "reported": "median", "cuda_graph": bool(args.graph),
                                                       "ms_per_step_regions": m["ms_regions"]},
           "roofline": roofline_block(w, m, K, world, peaks, fp64_peak)}

    # ---- end to end: host buffers, copies inside the timed region
    if not args.no_e2e:
        out["e2e"] = run_e2e(rt, m["g"], w, m["st"], K, world, dev, barrier)
    del m
    torch.cuda.empty_cache()

    # ---- the other north_star config in the same line (C5 beside C4 and vice versa), same protocol, 3 regions
    other = {"C4": "C5", "C5": "C4"}.get(args.workload)
    if other and not args.size and not args.no_also:
        w2 = make_workload(other)
        m2 = measure_workload(args, rt, drv, w2, dev, world, K, Wm, 3, barrier)
        r2 = roofline_block(w2, m2, K, world, peaks, fp64_peak)
        out["also"] = {other: {"value": m2["value"], "unit": UNIT, "ms_per_step": m2["ms_per_step"],
                               "ms_per_step_regions": m2["ms_regions"], "config": workload_config(w2, args),
                               "gpu_launches": m2["launches"], "roofline": r2}}
        del m2, w2
        torch.cuda.empty_cache()
        # the two launch-latency-bound configs ("report cell-updates/s and us per sub-step only"), replayed from
        # a CUDA graph of two sub-steps, 200 sub-steps per region
        import copy
        lat = {}
        for name in ("C1a", "C2"):
            a2 = copy.copy(args)
            a2.graph = True
            w3 = make_workload(name)
            m3 = measure_workload(a2, rt, drv, w3, dev, world, 200, 4, 3, barrier)
            lat[name] = {"us_per_substep": round(m3["ms_per_step"] * 1e3, 2), "value": m3["value"], "unit": UNIT,
                         "cells": w3.ncells, "cuda_graph": True, "launches_per_substep": m3["launches"] / m3["K"]}
            del m3, w3
        out["also"]["latency_bound"] = lat
        torch.cuda.empty_cache()
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        out["cpu_baseline"] = cpu_baseline(w)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps(out))


def load_peaks():
    """roofline denominator: the driver-measured copy bandwidth (MEASURED_PEAKS.json), else the guide's fallback"""
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as fh:
            d = json.load(fh)
        return {"hbm_gbs": float(d["hbm_gbs"]), "source": "of measured (MEASURED_PEAKS.json hbm_gbs, copy)"}
    except Exception:
        return {"hbm_gbs": 6650.0, "source": "of fallback (B200_PROFILING.md 6.65 TB/s)"}


def load_traffic(kernel, workload):
    """DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum) of the fused kernel from the committed ncu
    capture of the same sources (profiles/fp64_counts.txt), or None (another kernel, no capture, stale capture)"""
    if kernel != "fused":
        return None
    c = load_fp64_counts(workload)
    return c.get("dram_bytes_per_launch") if c and not c.get("stale") else None


def run_e2e(rt, g, w, st, K, world, dev, barrier):
    """same metric with HOST buffers: every step copies the sub-step's inputs (E, F, rho, T, m) from pinned
    host memory to the device, runs the sub-step through the C ABI, and copies the results (E, F, T, m) back.
    Software-pipelined over two device buffer sets and three streams: the copy-in of step i+1 overlaps the
    sub-step and the copy-out of step i (PCIe is full duplex); every step still moves all of its own bytes."""
    import torch
    import torch.distributed as dist

    class Set:
        def __init__(self, src):
            self.U = [t.clone() for t in src.U]
            self.U2 = [t.clone() for t in src.U2]
            self.rho, self.T = src.rho.clone(), src.T.clone()
            self.mom = [t.clone() for t in src.mom] if src.mom is not None else None
            self.ins = list(self.U) + [self.rho, self.T] + (list(self.mom) if self.mom is not None else [])
            self.outs = list(self.U2) + [self.T] + (list(self.mom) if self.mom is not None else [])

    sets = [Set(st), Set(st)]
    host_in = [t.cpu().pin_memory() for t in sets[0].ins]
    host_out = [torch.empty_like(host_in[0]).pin_memory() for _ in sets[0].outs]
    h2d = sum(t.numel() * 8 for t in host_in)
    d2h = sum(t.numel() * 8 for t in host_out)
    cs = torch.cuda.current_stream(dev)          # the stream the grid was created on
    s_in, s_out = torch.cuda.Stream(dev), torch.cuda.Stream(dev)
    ev_in = [torch.cuda.Event() for _ in range(2)]
    ev_comp = [torch.cuda.Event() for _ in range(2)]
    ev_out = [torch.cuda.Event() for _ in range(2)]

    def step(i):
        S = sets[i % 2]
        b = i % 2
        with torch.cuda.stream(s_in):
            s_in.wait_event(ev_out[b])           # the results of this set's previous step have left the device
            for d, h in zip(S.ins, host_in):
                d.copy_(h, non_blocking=True)
            ev_in[b].record(s_in)
        cs.wait_event(ev_in[b])
        if w.solver_schedule:
            g.set_params(rt.make_params(**dict(w.params, solver=w.solver_at(i))))
        if FUSED_CFL:   # the input state is new every step: its CFL first, then the whole sub-step, no host sync
            g.cfl_dt_async(S.U, w.cfl, st.dt_dev)
            g.substep(st.dt_dev, w.cfl, S.rho, S.T, S.mom, S.U, S.U2)
        else:
            dt = g.cfl_dt(S.U, w.cfl)
            g.explicit_step(dt, S.rho, S.T, S.U, S.U2)
            g.implicit_step(dt, S.rho, S.T, S.mom, S.U2)
        ev_comp[b].record(cs)
        with torch.cuda.stream(s_out):
            s_out.wait_event(ev_comp[b])
            for h, d in zip(host_out, S.outs):
                h.copy_(d, non_blocking=True)
            ev_out[b].record(s_out)

    def drain():
        cs.wait_event(ev_out[0])
        cs.wait_event(ev_out[1])

    Ke = max(4, min(K, 10))
    step(0)
    step(1)
    drain()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(cs)
    for i in range(Ke):
        step(i)
    drain()                                       # the timed region ends when the last result is in host memory
    e1.record(cs)
    barrier()
    value, ms = replicas_throughput(e0.elapsed_time(e1), w.ncells, Ke, world, dev)
    del sets
    return {"value": value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
            "steps": Ke, "ms_per_step": ms / Ke,
            "note": "pinned host buffers -> device -> C-ABI sub-step -> pinned host buffers; two device buffer sets, "
                    "copy-in / sub-step / copy-out of consecutive steps overlap on three streams"}


# ------------------------------------------------------------------------------------------ the oracle, timed
def time_oracle(w, nsteps, warm=0):
    """nsteps full sub-steps (CFL + explicit + implicit) of the CPU oracle as it stands, all host cores"""
    from oracle import ort
    og = ort.grid_from_workload(w)
    state = None
    if warm:
        U, T, mom, _ = ort.run_substeps(og, w, warm)
        state = (U, T, mom)
    t0 = time.perf_counter()
    ort.run_substeps(og, w, nsteps, state=state)
    dt = time.perf_counter() - t0
    return w.ncells * nsteps / dt, dt, ort.max_threads()


def cpu_baseline(w):
    """the oracle as it stands on the box's host cores: all threads (OpenMP), and one thread (SURVEY 8(d) "Timing")"""
    from oracle import ort
    n = 2 if w.ncells > 4_000_000 else 5
    v, secs, cores = time_oracle(w, n)
    ort.set_num_threads(1)
    try:
        v1, secs1, _ = time_oracle(w, 1)
    finally:
        ort.set_num_threads(cores)
    return {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": "%d full sub-steps of the same %s workload (%d cells), %.1f s, OpenMP on %d threads" % (n, w.name, w.ncells,
                                                                                                            secs, cores),
            "single_thread": {"value": v1, "unit": UNIT, "cores": 1,
                              "sample": "1 full sub-step of the same workload, %.1f s" % secs1}}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w = make_workload(args.workload, args.size)
    K, Wm = args.steps, max(args.warmup, 0)
    from oracle import ort
    og = ort.grid_from_workload(w)
    state = None
    if Wm:
        U, T, mom, _ = ort.run_substeps(og, w, Wm)
        state = (U, T, mom)
    t0 = time.perf_counter()
    ort.run_substeps(og, w, K, state=state)
    secs = time.perf_counter() - t0
    v = w.ncells * K / secs
    cores = ort.max_threads()
    sample = "each step = one full sub-step of the %s workload (%d cells) on %d host threads" % (w.name, w.ncells, cores)
    out = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": K, "warmup": Wm,
           "ms_per_step": secs * 1e3 / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
           "data": "synthetic", "config": workload_config(w, args),
           "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
           "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
    print(json.dumps(out))


if __name__ == "__main__":
    a = parse_args()
    if a.impl == "reference":
        run_reference(a)
    else:
        run_native(a)
