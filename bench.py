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
FUSED_KERNEL = True   # rt_substep runs k_substep_fused (3-D grids, --fused-seg >= 0, --api fused)

# fp64-pipe roof (DESIGN.md Sect. 5): 148 SMs x 64 fp64 lanes/clk x 1.965 GHz (B200_PROFILING.md unit counts and clock)
FP64_PEAK_TINST = 148 * 64 * 1.965e9 / 1e12
# Algorithmic fp64-pipe instructions (DFMA/DMUL/DADD/DSETP) per cell-update of k_substep_fused: ncu's executed count of
# the committed capture (profiles/r1_ncu_full_fused.md) x the useful-lane fraction of the launch (30 of 32 lanes along
# x1 and the ragged last tile, edge-row extras, segment ends) -- derivation in DESIGN.md Sect. 5.
FUSED_FP64_PER_CELL = {"C4": 0.5 * (692.0 + 588.0),   # HLL / GLF alternate
                       "C5": 741.0}                    # HLL, spherical (opacity tables are evaluated in the pre-pass)


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
    w = make_workload(args.workload, args.size)
    g = drv.grid_from_workload(w, device=dev)
    g.set_tuning(fused_seg=args.fused_seg)
    st = drv.DeviceState(g, w)
    st.dt_dev = torch.zeros(1, dtype=torch.float64, device=dev)
    g.cfl_dt_async(st.U, w.cfl, st.dt_dev)
    thick, feedback = bool(w.params["thick_limit"]), bool(w.params["feedback_momentum"]) and w.mom is not None
    K, Wm = args.steps, max(args.warmup, 0)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing (value)
    step = 0
    for _ in range(Wm):
        one_substep(rt, g, w, st, step)
        step += 1
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    l0 = g.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(K):
        one_substep(rt, g, w, st, step)
        step += 1
    e1.record()
    barrier()
    clocks = sampler.stop()
    launches = g.launch_count() - l0
    ms = e0.elapsed_time(e1)
    value, ms_max = replicas_throughput(ms, w.ncells, K, world, dev)

    # ---- per-kernel device times over the same K steps (second, instrumented pass): roofline
    g.set_profiling(True)
    for _ in range(K):
        one_substep(rt, g, w, st, step)
        step += 1
    kt = g.kernel_times()
    g.set_profiling(False)
    peaks = load_peaks()
    kernels = {}
    for name, (tot, cnt) in kt.items():
        if cnt == 0:
            continue
        avg = tot / cnt
        b = bytes_per_cell(name, thick, feedback) * w.ncells
        kernels[name] = {"launches_per_step": cnt / K, "avg_ms": round(avg, 5), "share": None,
                         "alg_bytes": b, "GBps": round(b / (avg * 1e-3) / 1e9, 1) if avg > 0 else None}
    tot_ms = sum(v[0] for v in kt.values())
    for name in kernels:
        kernels[name]["share"] = round(kt[name][0] / tot_ms, 4)
    dom = max(kernels, key=lambda k: kt[k][0])
    achieved = kernels[dom]["GBps"]
    roofline = {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                "frac": round(achieved / peaks["hbm_gbs"], 4), "traffic": load_traffic(dom, w.name),
                "peak_source": peaks["source"], "alg_bytes_per_launch": kernels[dom]["alg_bytes"],
                "avg_launch_ms": kernels[dom]["avg_ms"], "kernels": kernels,
                "substep_alg_bytes_per_cell": sum(bytes_per_cell(k, thick, feedback) * kernels[k]["launches_per_step"]
                                                  for k in kernels),
                "substep_GBps": None, "kernel_ms_sum_per_step": round(tot_ms / K, 4)}
    if dom == "fused" and w.name in FUSED_FP64_PER_CELL and not args.size:
        # the fused kernel is bound by the fp64 pipe, not by HBM (DESIGN.md Sect. 5): report it against that roof and
        # keep its HBM figure beside it
        inst = FUSED_FP64_PER_CELL[w.name] * w.ncells
        ach = inst / (kernels[dom]["avg_ms"] * 1e-3) / 1e12
        roofline.update({"bound": "alu", "achieved": round(ach, 3), "peak": round(FP64_PEAK_TINST, 3),
                         "unit": "Tinst/s (fp64 pipe: DFMA/DMUL/DADD/DSETP thread instructions)",
                         "frac": round(ach / FP64_PEAK_TINST, 4),
                         "peak_source": "148 SMs x 64 fp64 lanes/clk x 1.965 GHz (B200_PROFILING.md unit counts and clock)",
                         "alg_fp64_inst_per_cell": FUSED_FP64_PER_CELL[w.name],
                         "hbm": {"achieved": achieved, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                                 "frac": round(achieved / peaks["hbm_gbs"], 4), "peak_source": peaks["source"]}})
    roofline["substep_GBps"] = round(roofline["substep_alg_bytes_per_cell"] * value / world / 1e9, 1)
    roofline["substep_frac"] = round(roofline["substep_GBps"] / peaks["hbm_gbs"], 4)

    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
           "ms_per_step": ms_max / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": "f64", "data": "synthetic", "config": workload_config(w, args), "clocks": clocks,
           "gpu_launches": int(launches), "roofline": roofline}

    # ---- end to end: host buffers, copies inside the timed region
    if not args.no_e2e:
        out["e2e"] = run_e2e(rt, g, w, st, K, world, dev, barrier)
    del st
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
    """DRAM bytes per launch of `kernel` from the committed ncu --set full capture (profiles/ncu_traffic.csv,
    written by hand from the capture named in profiles/ncu_traffic.md), or None"""
    try:
        with open(os.path.join(ROOT, "profiles", "ncu_traffic.csv")) as fh:
            for line in fh.read().splitlines()[1:]:
                wl, k, b = line.split(",")
                if wl == workload and k == kernel:
                    return float(b)
    except Exception:
        pass
    return None


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
    n = 2 if w.ncells > 4_000_000 else 5
    v, secs, cores = time_oracle(w, n)
    return {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": "%d full sub-steps of the same %s workload (%d cells), %.1f s, OpenMP on %d threads" % (n, w.name, w.ncells,
                                                                                                            secs, cores)}


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
