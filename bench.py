#!/usr/bin/env python
"""bench.py -- FP64 MEG6 RHS + SSP-RK3 throughput on B200 (BASELINE.json metric).

One "step" = one SSP-RK3 step = three passes of the whole hot path (ghosts, gradients, three flux sweeps, the last
one fused with residual assembly + RK3 update + primitive conversion) over the workload; the K timed steps are one
meg6_rk3_steps call (state resident on the device); the end-to-end number calls meg6_rk3_step per step between a
host -> device copy of the whole state and a device -> host copy of the result, E2E_STATES independent states in flight
on three streams (the one-state, strictly sequential form is reported beside it as e2e.serial).
value = N_cells * 3 * steps / seconds, in Mcell-updates/s per RK stage, summed over all ranks (independent replicas for --gpus > 1: the path is single-GPU).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c4|c3|c1|c2] [--impl reference]
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)
import workloads as W  # noqa: E402

METRIC = "FP64 MEG6 RHS Mcell-updates/s per RK stage"
UNIT = "Mcell-updates/s/stage"
E2E_STATES = 3        # independent states in flight in the end-to-end measurement (copy in / step / copy out overlap)
# Nominal FP64 (DFMA-pipe) thread-instruction rate: 148 SMs x 64 lanes/clk x clock; the roof bench.py
# reports is MEASURED by the library's DFMA micro-benchmark (meg6_fp64_peak), this is printed beside it
FP64_LANES_PER_SM_CLK = 64
N_SM = 148
# DRAM traffic per launch (dram__bytes_read.sum + dram__bytes_write.sum) and FP64-pipe activity of the sweeps from the
# committed `ncu --set full` captures (never measured by this script: a run under ncu is not a bench run).  `state` says
# which flow state and clock the capture saw; the timed region of this script is the mid-run, power-capped state.
NCU = {}
try:
    with open(os.path.join(ROOT, "profiles", "ncu_constants.json")) as _f:
        NCU = json.load(_f)
except Exception:
    pass


def make_workload(name):
    if name == "c4":
        return W.c4_jet()
    if name == "c4_small":
        return W.c4_jet(ni=160, nj=100, nk=100)
    if name == "c3":
        return W.c3_tgv(n=128)
    if name == "c1":
        return W.c1_vortex(n=32)
    if name == "c2":
        return W.c2_dynamic_freestream(n=64)
    if name.startswith("c2_"):                       # moving-mesh freestream at other sizes
        return W.c2_dynamic_freestream(n=int(name[3:]))
    if name == "c5":
        return W.c5_tgv_mig4(n=384)
    if name.startswith("c5_"):                       # large-grid sweep of config 5: c5_128 ... c5_384
        return W.c5_tgv_mig4(n=int(name[3:]))
    if name.startswith("c3_"):                       # same sweep with MEG6
        return W.c3_tgv(n=int(name[3:]))
    raise SystemExit("unknown workload " + name)


def peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            p = json.load(f)
        return p["hbm_gbs"], p.get("sm_max_mhz", 1965.0), "measured (MEASURED_PEAKS.json)"
    except Exception:
        return 6650.0, 1965.0, "fallback (B200_PROFILING.md)"


def bytes_per_cell_stage(prm, sponge_frac):
    """Compulsory HBM doubles per cell per RK stage of the shipped kernel set.
    sponge_frac: None without a sponge, else the fraction of cells with sigma != 0 (Q_ref is read only there)."""
    v, m, ig = prm["viscous"], prm["moving"], prm.get("scheme", 0) == 1
    k = {}
    nf = 6 if v else 5
    k["prim"] = 0.0                                # once per meg6_rk3_steps call (11 doubles / (3 K) per cell-stage)
    met = (10 if v else 3) + (1 if m else 0)
    if ig:
        # MIG4: 3 nf segmented line solves (read f, write the gradient); sweeps read P, P' and two 5-field gradient groups
        k["grad"] = 3 * nf * 2
        base = nf + nf + met + (10 if v else 0)
    else:
        k["grad"] = GRAD_DOUBLES if v else 0
        base = nf + met + (SWEEP_GRAD_DOUBLES if v else 0)   # primitive tile, interface metrics, stored gradients
    k["flux_eta"] = base + 5 + (ETA_GRAD_DOUBLES if (v and not ig) else 0)   # first sweep: writes the residual [+ its own gradients]
    k["flux_zeta"] = base + 5 + 5                   # reads and writes it
    # last sweep, fused with assembly + RK3 stage + primitives of the new state:
    # reads residual 5, U 5, U0 5 (stages 2-3), 1/J 1 [, (1/J)_t 1] [, sigma 1, Q_ref 5 where sigma != 0]; writes U 5,
    # U0 5 (stage 1), P_next 6 (every stage: inside meg6_rk3_steps the last sweep of a step writes the primitives of the
    # next step's first stage)
    sp = 0.0 if sponge_frac is None else 1.0 + 5.0 * sponge_frac
    k["flux_xi"] = base + 5 + 5 + 10.0 / 3 + 1 + (1 if m else 0) + sp + 5 + 5.0 / 3 + 6
    k["metrics"] = (6 + 3 + 9 + 9 + 1 + 6 + 3 * met + 1) if m else 0   # nodes+modes, xc, cd, met, rj, xt+mt, faces, rjt
    return {a: 8.0 * b for a, b in k.items()}


# stored tangential gradients of the viscous flux (MEG6): k_grad reads (u,v,w,T) and writes the 8 arrays of the xi and zeta
# gradients, the eta sweep (first) writes the 4 arrays of the eta gradients it has in its tiles; each sweep reads the 8
# arrays of its two tangential directions
GRAD_DOUBLES = 4 + 8
ETA_GRAD_DOUBLES = 4
SWEEP_GRAD_DOUBLES = 8


def default_develop(wl, wl_name, develop):
    """untimed steps that advance the flow before the timed ones: half of the config's step count for the jet"""
    return develop if develop is not None else (wl["steps"] // 2 if wl_name.startswith("c4_jet") else 0)


def make_config(wl, wl_name, prm, cells, dt, world, slabs, develop, warmup):
    """The `config` object of the JSON line: the workload BASELINE.json's metric is quoted on.  Both arms print the same
    object (the reference arm times a bounded sample of it and says so in `cpu_baseline.sample`)."""
    stage_bytes = sum(bytes_per_cell_stage(prm, sponge_fraction(wl)).values())
    return {"workload": wl_name, "cells": cells, "viscous": prm["viscous"], "moving": prm["moving"],
            "scheme": "MIG4" if prm.get("scheme", 0) == 1 else "MEG6", "dt": dt,
            "parallelism": ("zeta slabs x%d, 6-layer halo exchange per stage" if slabs else "replicas x%d") % world,
            "l2": "working set %.1f GB per stage >> 126 MB L2 (no flush needed)" % (stage_bytes * cells / max(world if slabs else 1, 1) / 1e9),
            "state": "timed after %d untimed steps of the config's %s-step run (warm-up included)" % (
                max(develop, warmup), wl.get("steps"))}


def sponge_fraction(wl):
    sg = wl.get("sigma")
    return None if sg is None else float(np.count_nonzero(sg)) / sg.size


def input_hashes(wl):
    """SHA-256 of the generated arrays (oracle and GPU provably see the same bits)"""
    h = {"nodes": W.sha256(wl["x"], wl["y"], wl["z"]), "U0": W.sha256(wl["U0"])}
    if wl.get("dx_mode") is not None:
        h["modes"] = W.sha256(wl["dx_mode"], wl["dy_mode"], wl["dz_mode"])
    if wl.get("sigma") is not None:
        h["sponge"] = W.sha256(wl["sigma"], wl["U_ref"])
    for f, pin in sorted(wl.get("inflow", {}).items()):
        h["inflow%d" % int(f)] = W.sha256(pin)
    return h


def cpu_model():
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except Exception:
        pass
    return "unknown"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu):
        self.rows, self.proc, self.gpu = [], None, gpu

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.gpu), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[1])); mx.append(float(r[2]))
                for n, v in zip(names, r[5:9]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                pass
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


SAMPLE = dict(ni=160, nj=100, nk=100)


def oracle_sample(threads=None, grid=None):
    """The CPU oracle as it stands, timed on a bounded sample of the C4 workload (1/8 of the cells): one RK3 step.
    Returns (record, seconds, (grid, workload)) -- the grid can be reused for another thread count (static mesh)."""
    from oracle import meg6_oracle as O
    nthr = threads or (os.cpu_count() or 1)
    if grid is None:
        O.set_threads(os.cpu_count() or 1)
        wl = W.c4_jet(**SAMPLE)
        g = O.Grid(wl)
        g.metrics_compute(0.0)
    else:
        g, wl = grid
    O.set_threads(nthr)
    U = wl["U0"].copy()
    t0 = time.perf_counter()
    g.rk3_step(U, 0.0, wl["dt"])
    dt = time.perf_counter() - t0
    n = U[0].size
    rec = {"value": n * 3 / dt / 1e6, "unit": UNIT, "cores": O.get_threads(), "kind": "oracle",
           "sample": "c4_jet %dx%dx%d (%.1f M cells, 1/8 of the workload), 1 RK3 step, %.1f s"
                     % (SAMPLE["ni"], SAMPLE["nj"], SAMPLE["nk"], n / 1e6, dt),
           "cpu_model": cpu_model(), "nproc": os.cpu_count()}
    return rec, dt, (g, wl)


def cpu_baseline():
    """(b) all host cores and (a) one thread -- the paper's like-for-like is one Xeon Gold 5115 core"""
    rec, _, grid = oracle_sample()
    one, dt1, _ = oracle_sample(threads=1, grid=grid)
    rec["single_thread"] = {"value": one["value"], "unit": UNIT, "cores": 1, "sample": one["sample"]}
    return rec


def ref_config(args):
    """our arm's `config` for the default workload (no GPU needed: the jet has a fixed dt)"""
    wl = W.c4_jet(ni=20, nj=20, nk=20)               # parameters and step count only; the sizes are set below
    full = dict(ni=320, nj=200, nk=200)
    prm = dict(wl["params"], **full)
    name = "c4_jet_%dx%dx%d" % (full["ni"], full["nj"], full["nk"])
    sg = W.c4_jet(**SAMPLE)                           # sponge fraction of the sample mesh (same relative layer widths)
    return make_config(dict(wl, sigma=sg["sigma"]), name, prm, full["ni"] * full["nj"] * full["nk"], wl["dt"], 1, False,
                       default_develop(wl, name, args.develop), max(args.warmup, 3))


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    vals = []
    base = None
    grid = None
    for s in range(args.warmup + args.steps):
        base, dt, grid = oracle_sample(grid=grid)
        if s >= args.warmup:
            vals.append((base["value"], dt))
    v = float(np.mean([a for a, _ in vals]))
    ms = float(np.mean([b for _, b in vals])) * 1e3
    base["value"] = v
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": ref_config(args),
            "cpu_baseline": base,
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def max_over_ranks(values, dist, device):
    """Device-side times of one rank -> the maximum over all ranks (the job ends when the slowest rank does)."""
    import torch
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t]


def whole_job_throughput(ncell_per_rank, steps, world, ms):
    """Mcell-updates/s per RK stage of the whole job: every rank advances its own replica of ncell cells by
    `steps` RK3 steps (3 stages each) in `ms` milliseconds (max over ranks).  Weak scaling, no data-path collective."""
    return ncell_per_rank * 3 * steps * world / (ms * 1e-3) / 1e6


def run_ours(args):
    import torch
    from paper_2303_10785_b200 import Grid
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    # everything on one stream of our own (the library captures CUDA graphs, which the legacy default stream cannot)
    torch.cuda.set_stream(torch.cuda.Stream(dev))
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    wl = make_workload(args.workload)
    wl_name = wl["name"]
    slabs = args.decomp == "slabs" and world > 1
    stepper = None
    if slabs:
        # strong scaling: the workload cut into `world` zeta slabs, one per rank, six-layer halo exchange of the
        # primitives per RK stage over NCCL point-to-point (paper_2303_10785_b200/slabs.py)
        from paper_2303_10785_b200.slabs import SlabStepper, slab_cuts
        p0 = wl["params"]
        blocks, links = W.split_blocks(wl, ((p0["ni"],), (p0["nj"],), slab_cuts(p0["nk"], world)))
        dt_fixed = wl["dt"]
        wl = blocks[rank]
        wl["dt"] = dt_fixed
        remote = {face: nb for home, face, nb in links if home == rank}
        del blocks
    prm = wl["params"]
    ncell = prm["ni"] * prm["nj"] * prm["nk"]
    ncell_job = ncell * world                      # replicas: every rank its own copy
    if slabs:                                      # slabs: the ranks share one copy; the slabs differ by up to a plane
        tn = torch.tensor([ncell], dtype=torch.int64, device=dev)
        dist.all_reduce(tn, op=dist.ReduceOp.SUM)
        ncell_job = int(tn.item())
    g = Grid(wl, device=dev)
    if args.metrics_only:
        return run_metrics_only(args, g, wl, dev)
    if slabs:   # ghost coordinates of the cut faces come from the neighbour slab: the stepper exchanges them
        stepper = SlabStepper(g, remote, moving=bool(prm["moving"]), offsets=wl["link_offset"])
        stepper.metrics_compute(wl["t0"])
    else:
        g.metrics_compute(wl["t0"])
    U = torch.as_tensor(wl["U0"], device=dev).contiguous()
    if wl["dt"] is not None:
        dt = wl["dt"]
    else:
        dt = g.cfl_dt(U, wl["cfl"])      # on-device Eq. B.2/B.3 (no oracle on the product path)
        if slabs:                        # one time step for the whole job: the minimum over the slabs
            tdt = torch.tensor([dt], dtype=torch.float64, device=dev)
            dist.all_reduce(tdt, op=dist.ReduceOp.MIN)
            dt = float(tdt.item())
    step = stepper.rk3_step if stepper else g.rk3_step
    stream = torch.cuda.current_stream(dev)

    def steps(U, t, n):
        """n RK3 steps of constant dt with U resident on the device: one meg6_rk3_steps call (single grid), else n calls"""
        if stepper:
            for q in range(n):
                stepper.rk3_step(U, t + q * dt, dt)
        else:
            g.rk3_steps(U, t, dt, n)
        return t + n * dt

    def barrier():
        torch.cuda.synchronize(dev)
        if dist:
            dist.barrier()
        torch.cuda.synchronize(dev)

    # ---------------- device-resident timing ----------------
    t = wl["t0"]
    t = steps(U, t, args.warmup)
    # The state the timed steps see.  Config 4 is a 500-step run in which the jet enters a quiescent domain and shocks
    # form: the MP limiter's slow path, almost idle at t = 0, costs more and more.  The timed
    # steps are therefore taken in the MIDDLE of the config's run (after `develop` untimed steps); the throughput of
    # the first steps is reported beside it as `startup`.
    develop = default_develop(wl, wl_name, args.develop)
    startup = None
    if develop > 0:
        barrier()
        s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        s0.record(stream)
        t = steps(U, t, args.steps)
        s1.record(stream)
        barrier()
        startup = max_over_ranks([s0.elapsed_time(s1)], dist, dev)[0]
        t = steps(U, t, max(0, develop - args.steps - args.warmup))
    # headline: K steps, no per-kernel events inside the timed region
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    t = steps(U, t, args.steps)
    e1.record(stream)
    barrier()
    ms = e0.elapsed_time(e1)
    # per-kernel breakdown: a second pass of K steps of the same (still developed, still warm) run with one CUDA event
    # pair around every kernel launch on the launching stream; its own wall time is reported as `profiled_ms_per_step`
    g.profile_enable(True)
    g.profile_read()
    barrier()
    p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    p0.record(stream)
    t = steps(U, t, args.steps)
    p1.record(stream)
    barrier()
    ms_prof = p0.elapsed_time(p1)
    clocks = sampler.stop() if rank == 0 else None
    prof = g.profile_read()
    g.profile_enable(False)
    finite = bool(torch.isfinite(U).all().item())

    # ---------------- end to end: host buffers, copies inside the timed region ----------------
    # (1) serial: ONE state, each step = copy in, meg6_rk3_step, copy out, one after the other on one stream
    Uh = torch.empty(U.shape, dtype=torch.float64).pin_memory()
    Uh.copy_(U)
    Ud = torch.empty_like(U)
    for _ in range(2):
        Ud.copy_(Uh, non_blocking=True); step(Ud, t, dt); Uh.copy_(Ud, non_blocking=True)
    barrier()
    f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    f0.record(stream)
    for _ in range(args.steps):
        Ud.copy_(Uh, non_blocking=True)          # host -> device copy of this step's input state
        step(Ud, t, dt)
        Uh.copy_(Ud, non_blocking=True)          # device -> host read of the step's result
        t += dt
    f1.record(stream)
    barrier()
    ms_e2e_serial = f0.elapsed_time(f1)
    # (2) pipelined: E2E_STATES independent states (an ensemble) in flight, every step still one copy in, one
    # meg6_rk3_step and one copy out of a whole state, but on three streams, so that the copies of one state overlap
    # the step of another (PCIe is full duplex and the copy engines run beside the SMs).  Not in slab mode.
    ms_e2e, e2e_states = ms_e2e_serial, 1
    if not stepper:
        e2e_states = E2E_STATES
        s_in, s_out = torch.cuda.Stream(dev), torch.cuda.Stream(dev)
        Uhs = [Uh] + [torch.empty(U.shape, dtype=torch.float64).pin_memory() for _ in range(e2e_states - 1)]
        Uds = [Ud] + [torch.empty_like(U) for _ in range(e2e_states - 1)]
        for h in Uhs[1:]:
            h.copy_(Uh)
        tb = [t] * e2e_states
        in_done = [torch.cuda.Event() for _ in range(e2e_states)]
        st_done = [torch.cuda.Event() for _ in range(e2e_states)]
        out_done = [torch.cuda.Event() for _ in range(e2e_states)]

        def pipelined(n):
            for i in range(n):
                b = i % e2e_states
                if i >= e2e_states:
                    s_in.wait_event(out_done[b])     # this state's previous result has arrived in its host buffer
                with torch.cuda.stream(s_in):
                    Uds[b].copy_(Uhs[b], non_blocking=True)
                    in_done[b].record(s_in)
                stream.wait_event(in_done[b])
                step(Uds[b], tb[b], dt)              # on the grid's stream
                tb[b] += dt
                st_done[b].record(stream)
                s_out.wait_event(st_done[b])
                with torch.cuda.stream(s_out):
                    Uhs[b].copy_(Uds[b], non_blocking=True)
                    out_done[b].record(s_out)
            for b in range(min(n, e2e_states)):
                stream.wait_event(out_done[b])       # the timed region ends when the last result is on the host

        barrier()
        pipelined(2 * e2e_states)
        barrier()
        f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        f0.record(stream)
        s_in.wait_event(f0)
        pipelined(args.steps)
        f1.record(stream)
        barrier()
        ms_e2e = f0.elapsed_time(f1)
        finite = finite and all(bool(torch.isfinite(h).all().item()) for h in Uhs)

    ms, ms_e2e, ms_e2e_serial = max_over_ranks([ms, ms_e2e, ms_e2e_serial], dist, dev)
    if rank != 0:
        if dist:
            dist.destroy_process_group()
        return

    value = whole_job_throughput(ncell_job / world, args.steps, world, ms)
    e2e_value = whole_job_throughput(ncell_job / world, args.steps, world, ms_e2e)
    hbm, sm_max, peak_src = peaks()
    bpc = bytes_per_cell_stage(prm, sponge_fraction(wl))
    stage_bytes = sum(bpc.values())
    # per-kernel breakdown measured live with CUDA events on the launching stream (the profiled pass)
    tot_prof = sum(v[0] for v in prof.values())
    kernels = {}
    launches = 0
    for k, (kms, kn) in prof.items():
        if kms == 0 and kn == 0:
            continue
        launches += kn
        per_stage = kms / (3 * args.steps)
        kernels[k] = {"ms_per_stage": per_stage, "share": kms / tot_prof, "launches": int(kn),
                      "algorithmic_GBps": (bpc.get(k, 0) * ncell / (per_stage * 1e-3) / 1e9) if per_stage else None}
    dom = max((k for k in kernels if k.startswith("flux")), key=lambda k: kernels[k]["ms_per_stage"])
    dsec = kernels[dom]["ms_per_stage"] * 1e-3
    ach = bpc[dom] * ncell / dsec / 1e9
    clk = (clocks or {}).get("sm_mhz") or sm_max
    from paper_2303_10785_b200 import fp64_peak
    dfma = fp64_peak(dev)                      # measured right after the timed steps: the clock the steps ended with
    ncu = NCU.get(wl["name"], {}).get(dom, {})
    roof = {"kernel": "k_flux3<%s,%s>" % (dom[5:], "visc" if prm["viscous"] else "inv"), "bound": "hbm",
            "achieved": ach, "peak": hbm, "unit": "GB/s", "frac": ach / hbm,
            "traffic": ncu.get("traffic"), "traffic_source": ncu.get("source"), "traffic_state": ncu.get("state"),
            "fp64_pipe_pct_ncu": ncu.get("fp64_pipe_pct"),
            "peak_source": peak_src, "bytes_per_cell": bpc[dom], "cells_per_launch": ncell,
            "avg_launch_ms": dsec * 1e3,
            "fp64_roof": {"measured_Tdfma_s": dfma / 1e12,
                          "how": "meg6_fp64_peak: register-resident DFMA loop on every SM, best of 3, run after the "
                                 "timed steps",
                          "nominal_Tdfma_s_at_sampled_clock": N_SM * FP64_LANES_PER_SM_CLK * clk * 1e6 / 1e12}}
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
            "scaling": "strong" if slabs else "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": make_config(wl, wl_name, prm, ncell_job if slabs else ncell, dt, world, slabs, develop, args.warmup),
            "clocks": clocks, "gpu_launches": int(launches), "finite": finite,
            "profiled_ms_per_step": ms_prof / args.steps, "inputs_sha256": input_hashes(wl),
            "sponge_cell_fraction": sponge_fraction(wl),
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(U.numel() * 8),
                    "d2h_bytes_per_step": int(U.numel() * 8), "ms_per_step": ms_e2e / args.steps,
                    "states_in_flight": e2e_states,
                    "how": ("every step: one whole state copied from pinned host memory, one meg6_rk3_step, the result "
                            "copied back; %d independent states in flight on three streams (copy in / step / copy out)"
                            % e2e_states) if e2e_states > 1 else "one state, copy in / step / copy out in sequence",
                    "serial": {"value": whole_job_throughput(ncell_job / world, args.steps, world, ms_e2e_serial),
                               "ms_per_step": ms_e2e_serial / args.steps,
                               "how": "one state, copy in / step / copy out one after the other on one stream"}},
            "roofline": roof,
            "hbm_roofline_step": {"bytes_per_cell_stage": stage_bytes,
                                  "achieved_GBps": stage_bytes * ncell_job * 3 * args.steps / (ms * 1e-3) / 1e9 / world,
                                  "frac": stage_bytes * ncell_job * 3 * args.steps / (ms * 1e-3) / 1e9 / world / hbm,
                                  "peak": hbm, "peak_source": peak_src},
            "kernels": kernels}
    if startup is not None:
        line["startup"] = {"value": whole_job_throughput(ncell_job / world, args.steps, world, startup), "unit": UNIT,
                           "ms_per_step": startup / args.steps,
                           "state": "the %d steps right after the %d warm-up steps from the initial state" % (args.steps, args.warmup)}
    if world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline()
    print(json.dumps(line))
    if dist:
        dist.destroy_process_group()


def run_metrics_only(args, g, wl, dev):
    """--metrics-only: times meg6_metrics_compute(t) alone (every RK stage on a moving mesh) --
    the command the geometry profiles under profiles/ are taken with."""
    import torch
    stream = torch.cuda.current_stream(dev)
    for r in range(max(3, args.warmup)):
        g.metrics_compute(0.01 * (r + 1))
    torch.cuda.synchronize(dev)
    g.profile_enable(True)
    g.profile_read()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for r in range(args.steps):
        g.metrics_compute(0.1 + 0.01 * r)
    e1.record(stream)
    torch.cuda.synchronize(dev)
    ms = e0.elapsed_time(e1) / args.steps
    prof = g.profile_read()
    prm = wl["params"]
    ncell = prm["ni"] * prm["nj"] * prm["nk"]
    bpc = bytes_per_cell_stage(prm, sponge_fraction(wl))["metrics"]
    hbm, _, peak_src = peaks()
    print(json.dumps({"metric": "meg6_metrics_compute ms per call", "value": ms, "unit": "ms", "higher_is_better": False,
                      "calls": args.steps, "dtype": "f64", "data": "synthetic",
                      "config": {"workload": wl["name"], "cells": ncell, "moving": prm["moving"],
                                 "scheme": "MIG4" if prm.get("scheme", 0) == 1 else "MEG6"},
                      "gpu_launches": int(prof["metrics"][1]),
                      "algorithmic_GBps": (bpc * ncell / (ms * 1e-3) / 1e9) if bpc else None, "hbm_peak": hbm,
                      "peak_source": peak_src}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c4")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--develop", type=int, default=None,
                    help="untimed steps that advance the flow before the timed ones (default: half of the config's step "
                         "count for c4, 0 otherwise)")
    ap.add_argument("--metrics-only", action="store_true",
                    help="time meg6_metrics_compute alone (moving-mesh workloads c2, c2_N): `--steps` calls")
    ap.add_argument("--decomp", default="replicas", choices=["replicas", "slabs"],
                    help="N > 1: independent replicas (weak scaling, default) or one workload cut into zeta slabs "
                         "with halo exchange (strong scaling)")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
