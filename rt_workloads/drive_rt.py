"""Driving a described workload (rt_workloads.Workload) through the CUDA library: call sequencing only, used by the
GPU tests, bench.py and __graft_entry__.smoke().  No method arithmetic here and none in the binding it calls
(paper_2606_26268_b200.rt marshals arguments; every step of the path runs in the kernels behind the C ABI).
This module is NOT imported by `import rt_workloads`: the oracle side never pulls the CUDA package in."""
import torch

from paper_2606_26268_b200 import rt
from paper_2606_26268_b200.rt import make_params, opacity_from_spec, Grid


def grid_from_workload(w, device="cuda:0"):
    g = Grid(w.geometry, w.n, w.xf[0], w.xf[1], w.xf[2], w.bc, device=device)
    g.set_params(make_params(**w.params))
    for which, spec in w.opacities.items():
        g.set_opacity(which, opacity_from_spec(spec))
    return g


class DeviceState:
    """device-resident copy of a workload's fields: U (two buffers), rho, T, mom"""

    def __init__(self, g, w):
        self.U = [g.to_device(a) for a in w.U]
        self.U2 = [t.clone() for t in self.U]  # ghosts of FIXED boundaries must exist in both buffers
        self.rho = g.to_device(w.rho)
        self.T = g.to_device(w.T)
        self.mom = [g.to_device(a) for a in w.mom] if w.mom is not None else None


def substep(g, w, st, dt, step_index=0):
    """one sub-step = rt_explicit_step + rt_implicit_step on the device state (buffers swap)"""
    if w.solver_schedule:
        g.set_params(make_params(**dict(w.params, solver=w.solver_at(step_index))))
    g.explicit_step(dt, st.rho, st.T, st.U, st.U2)
    g.implicit_step(dt, st.rho, st.T, st.mom, st.U2)
    st.U, st.U2 = st.U2, st.U


def run_substeps(g, w, nsub, dts=None, st=None):
    """nsub sub-steps of workload w; dts = fixed time steps, else rt_cfl_dt each step.
    Returns (state, list of dt used)."""
    st = st if st is not None else DeviceState(g, w)
    used = []
    for s in range(nsub):
        if w.solver_schedule:
            g.set_params(make_params(**dict(w.params, solver=w.solver_at(s))))
        dt = float(dts[s]) if dts is not None else g.cfl_dt(st.U, w.cfl)
        used.append(dt)
        g.explicit_step(dt, st.rho, st.T, st.U, st.U2)
        g.implicit_step(dt, st.rho, st.T, st.mom, st.U2)
        st.U, st.U2 = st.U2, st.U
    return st, used


def run_substeps_fused(g, w, nsub, st=None):
    """nsub sub-steps through rt_substep: the time step never leaves the device (seeded by rt_cfl_dt_async,
    then produced by the CFL reduction fused behind each implicit half).  Returns (state, dt tensor of the
    NEXT sub-step, list of the dt used as a device tensor history)."""
    st = st if st is not None else DeviceState(g, w)
    dt_dev = torch.zeros(1, dtype=torch.float64, device=g.device)
    hist = torch.zeros(nsub, dtype=torch.float64, device=g.device)
    g.cfl_dt_async(st.U, w.cfl, dt_dev)
    for s in range(nsub):
        if w.solver_schedule:
            g.set_params(make_params(**dict(w.params, solver=w.solver_at(s))))
        hist[s:s + 1].copy_(dt_dev)
        g.substep(dt_dev, w.cfl, st.rho, st.T, st.mom, st.U, st.U2)
        st.U, st.U2 = st.U2, st.U
    return st, dt_dev, hist


def run_rk2(g, w, nsteps, st=None):
    """nsteps RK2 steps through rt_rk2_step (time step resident on the device).  Returns (state, dt history tensor)."""
    st = st if st is not None else DeviceState(g, w)
    W2 = [t.clone() for t in st.U]
    dt_dev = torch.zeros(1, dtype=torch.float64, device=g.device)
    hist = torch.zeros(nsteps, dtype=torch.float64, device=g.device)
    g.cfl_dt_async(st.U, w.cfl, dt_dev)
    for s in range(nsteps):
        hist[s:s + 1].copy_(dt_dev)
        g.rk2_step(dt_dev, w.cfl, st.rho, st.T, st.mom, st.U, st.U2, W2)
    return st, hist
