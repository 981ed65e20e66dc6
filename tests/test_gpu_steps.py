"""Step-count parity at the configs' own sizes (BASELINE.json north_star: "1e-9 after the config's step count"; SURVEY
8(d): full step counts on C1-C3, >= 20 steps on C4/C5 where the oracle is too slow for all of them).

The CPU oracle needs minutes for these (config 3: 128^3 x 200 steps ~ 7 min on 16 host cores; config 4: 20 steps of
12.8 M cells ~ 5 min), hence the extra marker `slow` -- they are part of `-m gpu`.  Every test reports, per step, the
number of interface-components that failed test E.1 on each side, and after the last right-hand side the branch records
(E.1 per component and side, branch of Eq. 26) are compared interface by interface: flipped decisions are listed.
"""
import time

import numpy as np
import pytest

import workloads as W
from test_gpu_parity import STEP_TOL, flip_report, mods, rel, strict_rel  # noqa: F401

pytestmark = [pytest.mark.gpu, pytest.mark.slow]


def run_both(torch, O, M, wl, U0, steps, t0=0.0, dt=None, label=""):
    import os
    O.set_threads(os.cpu_count() or 1)          # these runs are minutes of oracle time: every host core
    og = O.Grid(wl)
    og.metrics_compute(t0)
    g = M.Grid(wl)
    g.metrics_compute(t0)
    U = torch.as_tensor(U0, device="cuda").contiguous()
    if dt is None:
        dt = g.cfl_dt(U, wl["cfl"])
        assert dt == pytest.approx(og.cfl_dt(U0, wl["cfl"]), rel=1e-12)
    Uo = U0.copy()
    g.limiter_stats_enable(True)
    g.branch_masks_enable(True)
    og.branch_masks_enable(True)
    hist = []
    lo0 = lg0 = to0 = tg0 = 0
    t = t0
    wall = time.time()
    for s in range(steps):
        og.rk3_step(Uo, t, dt)
        g.rk3_step(U, t, dt)
        t += dt
        lo, to = og.limiter_stats()
        lg, tg = g.limiter_stats()
        hist.append((lo - lo0, lg - lg0))
        tested = to - to0
        assert tg - tg0 == tested
        lo0, lg0, to0, tg0 = lo, lg, to, tg
        if s in (0, 1, 4, 9, 19, 49, 99, 199) or s == steps - 1:
            print("%s step %d: rel %s, limited this step oracle %d gpu %d of %d" % (
                label, s + 1, rel(U.cpu().numpy(), Uo), hist[-1][0], hist[-1][1], tested), flush=True)
    wall = time.time() - wall
    Ug = U.cpu().numpy()
    rep, touched = flip_report(g, og, U0.shape[1:])
    diffs = [a - b for a, b in hist]
    print("%s: %d steps in %.0f s; per-step limited-count differences (oracle - gpu): min %d max %d, nonzero in %d steps"
          % (label, steps, wall, min(diffs), max(diffs), sum(1 for d in diffs if d)))
    print("%s: last right-hand side: %d flipped E.1 decisions, %d flipped decisive Eq. 26 branches (+ %d at the %d ties, "
          "R10) of %d interfaces; first: %s" % (label, rep["e1_flips"], rep["hllc_flips"], rep["hllc_flips_at_ties"],
                                                rep["ties"], rep["interfaces"], rep["flipped"]))
    print("%s: strict per-component rel %s" % (label, strict_rel(Ug, Uo)))
    g.close()
    return Ug, Uo, rep, touched, hist


def test_c3_128_200_steps(mods):
    """Config 3 as BASELINE.json states it: 128^3 wavy mesh, viscous TGV, CFL 0.2, all 200 RK3 steps, every cell."""
    torch, O, M = mods
    wl = W.c3_tgv(n=128)
    Ug, Uo, rep, touched, hist = run_both(torch, O, M, wl, wl["U0"], 200, label="c3 128^3")
    e = rel(Ug, Uo)
    assert np.all(e <= STEP_TOL), e
    assert hist[-1][0] > 0.02 * 30 * 128 ** 3 * 3       # 3.4 % of the interface-components are limited in every stage
    assert rep["e1_flips"] + rep["hllc_flips"] <= 20, rep


def test_c4_full_size_20_steps_from_the_developed_state(mods):
    """Config 4 at full size (320 x 200 x 200), 20 RK3 steps starting from the DEVELOPED jet: the GPU advances the
    initial state by 250 steps (the middle of the config's 500-step run, the state bench.py times: shocks at the nozzle
    lip, limiter active), both sides then take the same 20 steps from that state."""
    torch, O, M = mods
    wl = W.c4_jet()
    g = M.Grid(wl)
    g.metrics_compute(0.0)
    U = torch.as_tensor(wl["U0"], device="cuda").contiguous()
    for s in range(250):
        g.rk3_step(U, s * wl["dt"], wl["dt"])
    U250 = U.cpu().numpy()
    g.close()
    del U, g
    assert np.isfinite(U250).all()
    Ug, Uo, rep, touched, hist = run_both(torch, O, M, wl, U250, 20, t0=250 * wl["dt"], dt=wl["dt"], label="c4 developed")
    e = rel(Ug, Uo)
    assert np.all(e <= STEP_TOL), e
    assert hist[-1][0] > 1e-3 * 30 * 12.8e6 * 3           # the limiter is at work in the developed state
    assert rep["e1_flips"] + rep["hllc_flips"] <= 20, rep
    assert np.abs(Ug - U250).max() > 1e-3                  # and the 20 steps did something


def test_mig4_128_20_steps(mods):
    """Config 5's scheme (MIG4) and flow at 128^3 (the smallest grid of its sweep), 20 RK3 steps, every cell."""
    torch, O, M = mods
    wl = W.c5_tgv_mig4(n=128, steps=20)
    Ug, Uo, rep, touched, hist = run_both(torch, O, M, wl, wl["U0"], 20, label="c5 mig4 128^3")
    e = rel(Ug, Uo)
    assert np.all(e <= STEP_TOL), e


def test_mig4_256_3_steps(mods):
    """Config 5's scheme and flow at 256^3 (the middle of its 128^3..384^3 sweep; at 384^3 the oracle's arrays alone
    would take tens of GB of host memory): geometry of the implicit scheme on 16.8 M cells, dQ/dt and three RK3 steps,
    every cell."""
    torch, O, M = mods
    wl = W.c5_tgv_mig4(n=256, steps=3)
    Ug, Uo, rep, touched, hist = run_both(torch, O, M, wl, wl["U0"], 3, label="c5 mig4 256^3")
    e = rel(Ug, Uo)
    assert np.all(e <= STEP_TOL), e
    assert rep["e1_flips"] + rep["hllc_flips"] <= 20, rep


@pytest.mark.skipif(not __import__("os").environ.get("MEG6_LONG"), reason="2.5 hours of CPU oracle: set MEG6_LONG=1")
def test_c4_full_config_all_500_steps(mods):
    """Config 4 exactly as BASELINE.json states it: 320 x 200 x 200, all 500 RK3 steps from the initial state, GPU against
    the oracle, every cell (north_star: "1e-9 after the config's step count").  Not part of the default `-m gpu` run (the
    oracle needs about 13 s per step on 16 cores, and one call on the GPU pool is limited to an hour: round 2 ran it in two
    legs, steps 1-250 from the initial state and steps 251-500 from the GPU's state at step 250 -- MEG6_LONG_START=250
    MEG6_LONG_STEPS=250); the results are in profiles/r2_c4_500_steps.md.
    Progress goes to MEG6_LONG_LOG (a line every 25 steps), so an interrupted run still leaves its numbers."""
    import os
    torch, O, M = mods
    O.set_threads(os.cpu_count() or 1)
    wl = W.c4_jet()
    steps = int(os.environ.get("MEG6_LONG_STEPS", "500"))
    start = int(os.environ.get("MEG6_LONG_START", "0"))       # > 0: the GPU advances that many steps first, then both sides
    log = os.environ.get("MEG6_LONG_LOG")                     # continue from ITS state (a run in two legs)
    og = O.Grid(wl)
    og.metrics_compute(0.0)
    g = M.Grid(wl)
    g.metrics_compute(0.0)
    U = torch.as_tensor(wl["U0"], device="cuda").contiguous()
    dt = wl["dt"]
    for s in range(start):
        g.rk3_step(U, s * dt, dt)
    Uo = U.cpu().numpy().copy()
    g.limiter_stats_enable(True)
    g.branch_masks_enable(True)
    og.branch_masks_enable(True)
    lo0 = lg0 = 0
    worst = np.zeros(5)
    ndiff = 0
    t0 = time.time()
    for s in range(start, start + steps):
        og.rk3_step(Uo, s * dt, dt)
        g.rk3_step(U, s * dt, dt)
        lo, to = og.limiter_stats()
        lg, tg = g.limiter_stats()
        assert tg == to
        ndiff += int((lo - lo0) != (lg - lg0))
        if (s + 1) % 25 == 0 or s + 1 == start + steps:
            e = rel(U.cpu().numpy(), Uo)
            worst = np.maximum(worst, e)
            rep, _ = flip_report(g, og, wl["U0"].shape[1:])
            line = ("step %d: rel %s, limited in this step oracle %d gpu %d, steps with differing counts so far %d, last "
                    "right-hand side: %d flipped E.1, %d flipped decisive Eq. 26 (+ %d at %d ties), %.0f s"
                    % (s + 1, np.array2string(e, precision=2), lo - lo0, lg - lg0, ndiff, rep["e1_flips"],
                       rep["hllc_flips"], rep["hllc_flips_at_ties"], rep["ties"], time.time() - t0))
            print(line, flush=True)
            if log:
                with open(log, "a") as f:
                    f.write(line + "\n")
            assert np.all(e <= STEP_TOL), (s + 1, e)
        lo0, lg0 = lo, lg
    g.close()


@pytest.mark.skipif(not __import__("os").environ.get("MEG6_LONG"), reason="15 minutes of CPU oracle: set MEG6_LONG=1")
def test_mig4_256_all_50_steps(mods):
    """Config 5's scheme, flow and STEP COUNT (50) at 256^3 -- or, with MEG6_LONG_N=384, at the config's own 384^3 (the
    oracle then holds 64 GB of arrays and needs most of an hour on 16 cores).  Results of the round-2 runs in
    profiles/r2_c4_500_steps.md."""
    torch, O, M = mods
    n = int(__import__("os").environ.get("MEG6_LONG_N", "256"))
    wl = W.c5_tgv_mig4(n=n, steps=50)
    Ug, Uo, rep, touched, hist = run_both(torch, O, M, wl, wl["U0"], 50, label="c5 mig4 %d^3 x 50" % n)
    e = rel(Ug, Uo)
    assert np.all(e <= STEP_TOL), e
    assert rep["e1_flips"] + rep["hllc_flips"] <= 20, rep


def test_c2_mesh_and_step_count_with_a_nontrivial_flow(mods):
    """Config 2's mesh, motion, size and STEP COUNT (64^3 jittered mesh, nodes moving at omega = 1, 100 RK3 steps) with a
    smooth non-uniform flow instead of the freestream (whose parity is trivial: both sides stay uniform to 1e-12): 300
    geometry evaluations at the stage times, grid velocities, time metrics and GCL terms against the oracle's over the
    whole run (a minute of oracle time on 16 cores)."""
    torch, O, M = mods
    wl = W.c2_dynamic_freestream(n=64)
    xc, yc, zc = (W.cell_centres(wl[k]) for k in ("x", "y", "z"))
    s2 = lambda a: np.sin(2 * np.pi * a)
    U0 = W.conservative(1 + 0.1 * s2(xc) * s2(yc), 1 + 0.2 * s2(yc + 0.1), 0.1 * s2(zc) * s2(xc),
                        -0.15 * s2(xc + 0.3), (1 + 0.05 * s2(zc + 0.2)) / (1.4 * 0.25))
    Ug, Uo, rep, touched, hist = run_both(torch, O, M, wl, U0, 100, label="c2 mesh 64^3 x 100, smooth flow")
    e = rel(Ug, Uo)
    assert np.all(e <= STEP_TOL), e
    assert np.abs(Ug - U0).max() > 1e-2
    assert rep["e1_flips"] + rep["hllc_flips"] <= 20, rep

