"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle on the same seeded inputs.

Tolerances (BASELINE.json north_star): relative L-infinity <= 1e-11 on every single RHS and <= 1e-9 after
the step count, relative to max|field| per component; freestream deviation <= 1e-12.
"""
import numpy as np
import pytest

import workloads as W

pytestmark = pytest.mark.gpu

RHS_TOL = 1e-11
STEP_TOL = 1e-9
# the same right-hand sides in the norm of SURVEY 8(d) as written (per component, by that component's own maximum): the
# 1e-11 bound holds as it stands except for config 3, whose mass equation is 1e-3 of the flux scale at Ma 0.1 (its
# round-off is that of the fluxes: the bound is loosened by that factor)
STRICT_RHS_TOL = {"c1": 1e-11, "c2": 1e-11, "c3": 1e-8, "c4": 1e-11}


@pytest.fixture(scope="module")
def mods():
    import torch
    from oracle import meg6_oracle as O
    import paper_2303_10785_b200 as M
    assert torch.cuda.is_available()
    return torch, O, M


def rel(a, b):
    """per-component max |a-b| / max |b|; the three momentum components (one vector) share the scale of the
    largest of them, so that a component that is physically ~0 (w of a z-aligned vortex) is not normalised
    by its own round-off-sized magnitude ("Tolerances")."""
    n = a.shape[0]
    scale = np.abs(b).reshape(n, -1).max(1)
    if n == 5:
        scale[1:4] = scale[1:4].max()
    return np.abs(a - b).reshape(n, -1).max(1) / np.maximum(scale, 1e-300)


def rhs_err(a, b, U, gamma=1.4):
    """Parity norm of a right-hand side dQ/dt: per-component max |a-b| over the scale of that component,
    the scale being the largest component of the acoustically non-dimensionalised RHS vector
    (dQ_c/dt / ref_c, ref = (rho0, rho0 a0, rho0 a0, rho0 a0, rho0 a0^2)) brought back to the units of
    component c.  A component that is physically tiny (the mass equation of the nearly incompressible
    Taylor-Green vortex is 1e-3 of the flux scale) is thereby not normalised by its own cancellation
    residue.  tests/test_oracle_sensitivity.py measures how far FMA contraction alone moves the oracle on the
    same case (2.5e-11: more than the tolerance), which is why the metric kernels are bit-exact.
    DESIGN.md, "Tolerances"."""
    rho = U[0]
    p = (gamma - 1) * (U[4] - 0.5 * (U[1] ** 2 + U[2] ** 2 + U[3] ** 2) / rho)
    rho0, a0 = rho.mean(), np.sqrt(gamma * p / rho).mean()
    ref = np.array([rho0, rho0 * a0, rho0 * a0, rho0 * a0, rho0 * a0 * a0])
    mag = np.abs(b).reshape(5, -1).max(1) / ref
    scale = ref * mag.max()
    return np.abs(a - b).reshape(5, -1).max(1) / scale


def strict_rel(a, b):
    """SURVEY 8(d) as written: per-component max |a-b| / max |b_c|, every component by its own magnitude"""
    n = a.shape[0]
    return np.abs(a - b).reshape(n, -1).max(1) / np.maximum(np.abs(b).reshape(n, -1).max(1), 1e-300)


def flip_report(g, og, shape):
    """Branch records of the two sides after the same right-hand side (include/meg6.h: bits 0-9 test E.1 per
    characteristic component and side, bits 10-11 branch of Eq. 26), compared bit for bit.  Returns
    (report dict, boolean cell array: cells next to an interface whose record differs)."""
    nk, nj, ni = shape
    touched = np.zeros(shape, dtype=bool)
    rep = {"interfaces": 0, "e1_flips": 0, "hllc_flips": 0, "hllc_flips_at_ties": 0, "ties": 0, "flipped": []}
    for d in range(3):
        a, b = g.branch_mask_host(d), og.branch_mask(d)
        assert a.shape == b.shape
        rep["interfaces"] += a.size
        tie = (b >> 12) & 1          # oracle only: the cascade of Eq. 26 tested a wave speed that is zero to 1e-10 (R10)
        rep["ties"] += int(tie.sum())
        x = (a ^ b) & 0x0FFF
        hl = (x >> 10) != 0
        rep["e1_flips"] += int(sum(((x >> bit) & 1).sum() for bit in range(10)))
        rep["hllc_flips_at_ties"] += int((hl & (tie == 1)).sum())
        rep["hllc_flips"] += int((hl & (tie == 0)).sum())
        # listed and attributed: every differing E.1 decision and every differing DECISIVE branch of Eq. 26; a tie flips
        # with the rounding order and gives the same flux either way (counted above)
        idx = np.argwhere(((x & 0x3FF) != 0) | (hl & (tie == 0)))
        for k, j, i in idx:
            if len(rep["flipped"]) < 20:
                rep["flipped"].append((d, int(i), int(j), int(k), int(a[k, j, i]), int(b[k, j, i])))
            for off in (-1, 0):     # interface s of family d lies between cells s-1 and s
                c = [k, j, i]
                c[2 - d] += off
                if 0 <= c[2 - d] < shape[2 - d]:
                    touched[c[0], c[1], c[2]] = True
    return rep, touched


def small_cases():
    c1 = W.c1_vortex(n=32)
    c2 = W.c2_dynamic_freestream(n=24, steps=4)
    # the uniform state has a round-off-sized RHS (checked by the freestream test); parity of the moving-mesh
    # terms (xi_t in HLLC, (1/J)_t Q) needs a non-trivial state: smooth periodic perturbation
    xc, yc, zc = (W.cell_centres(c2[k]) for k in ("x", "y", "z"))
    s2 = lambda a: np.sin(2 * np.pi * a)
    c2["U0"] = W.conservative(1 + 0.1 * s2(xc) * s2(yc), 1 + 0.2 * s2(yc + 0.1), 0.1 * s2(zc) * s2(xc),
                              -0.15 * s2(xc + 0.3), (1 + 0.05 * s2(zc + 0.2)) / (1.4 * 0.25))
    c3 = W.c3_tgv(n=40, steps=3)
    c4 = W.c4_jet(ni=52, nj=37, nk=33, steps=3)   # ragged in every direction, several tiles
    # perturb the jet state so that the interior is not trivially uniform
    rng = np.random.default_rng(4)
    shape = c4["U0"].shape[1:]
    rho = 1.0 + 0.2 * rng.uniform(-1, 1, shape)
    u, v, w = (0.3 * rng.uniform(-1, 1, shape) for _ in range(3))
    p = (1.0 + 0.2 * rng.uniform(-1, 1, shape)) / 1.4
    c4["U0"] = W.conservative(rho, u, v, w, p)
    return {"c1": c1, "c2": c2, "c3": c3, "c4": c4}


@pytest.fixture(scope="module")
def cases():
    return small_cases()


@pytest.mark.parametrize("blocked", ["0", "1"])
@pytest.mark.parametrize("name", ["c1", "c2", "c3", "c4"])
def test_metrics_parity(mods, cases, name, blocked, monkeypatch):
    torch, O, M = mods
    wl = cases[name]
    # both forms of the coordinate-derivative / interface-metric kernels (one cell per thread, and blocks of six along the
    # grid line, which grids of 2 M cells and more take by default): the library reads the switch at every call
    monkeypatch.setenv("MEG6_GEOM_BLOCKED", blocked)
    t = 0.13 if wl["params"]["moving"] else 0.0
    og = O.Grid(wl)
    og.metrics_compute(t)
    g = M.Grid(wl)
    g.metrics_compute(t)
    # The metric kernels evaluate Eq. 17/19/16/36-38 in the order the paper states them, without FMA
    # contraction, so every geometric array must agree with the oracle BIT FOR BIT (index work and
    # rounding order are unique here); see DESIGN.md "Tolerances".
    names = []
    for q in list(range(10)) + [14, 15, 16]:
        names.append(("cell", q, g.get_array(0, q), og.cell(q)))
    for d in range(3):
        qs = range(10) if wl["params"]["viscous"] else range(3 * d, 3 * d + 3)
        for q in qs:
            names.append(("face%d" % d, q, g.get_array(1, 16 * d + q), og.face(d, q)))
    if wl["params"]["moving"]:
        for q in (10, 11, 12, 13):
            names.append(("cell", q, g.get_array(0, q), og.cell(q)))
        for d in range(3):
            names.append(("face%d" % d, 10, g.get_array(1, 16 * d + 10), og.face(d, 10)))
    for kind, q, a, b in names:
        assert np.array_equal(a, b), (name, kind, q, np.abs(a - b).max() / np.abs(b).max())
    g.close()


@pytest.mark.parametrize("name", ["c1", "c2", "c3", "c4"])
def test_rhs_parity(mods, cases, name):
    torch, O, M = mods
    wl = cases[name]
    t = 0.13 if wl["params"]["moving"] else 0.0
    og = O.Grid(wl)
    og.metrics_compute(t)
    og.branch_masks_enable(True)
    ref = og.rhs(wl["U0"])
    g = M.Grid(wl)
    g.metrics_compute(t)
    g.limiter_stats_enable(True)
    g.branch_masks_enable(True)
    U = torch.as_tensor(wl["U0"], device="cuda").contiguous()
    out = g.rhs(U).cpu().numpy()
    for f in range(6):
        a, b = g.get_array(2, f), og.prim(f)
        assert np.abs(a - b).max() <= 1e-14 * np.abs(b).max()
    e = rhs_err(out, ref, wl["U0"])
    assert np.all(e <= RHS_TOL), (name, e, rel(out, ref))
    # the norm of SURVEY 8(d) as written (every component by its own magnitude) is recorded and bounded as well: it
    # differs from the one above only where a component is physically tiny (mass equation of the Ma 0.1 TGV)
    es = strict_rel(out, ref)
    assert np.all(es <= STRICT_RHS_TOL[name]), (name, es)
    # branch decisions, interface by interface: same interfaces tested; every differing E.1 / Eq. 26 decision is listed
    lim_o, tst_o = og.limiter_stats()
    lim_g, tst_g = g.limiter_stats()
    assert tst_g == tst_o
    rep, touched = flip_report(g, og, wl["U0"].shape[1:])
    assert rep["e1_flips"] >= abs(lim_g - lim_o)
    assert rep["e1_flips"] + rep["hllc_flips"] <= 1e-5 * rep["interfaces"] + 2, rep
    if touched.any():   # the tolerance holds on the flipped cells too (the limiter and HLLC are continuous across
        ef = np.abs(out - ref)[:, touched].max(1) / np.abs(ref).reshape(5, -1).max(1)   # their switches)
        print("%s: %d cells next to flipped decisions, strict error there %s" % (name, int(touched.sum()), ef))
    print("%s: strict per-component rel Linf %s" % (name, es))
    print("%s: rel Linf %s, limited %d/%d (oracle %d); flipped E.1 decisions %d, flipped decisive Eq. 26 branches %d "
          "(+ %d at the %d ties) of %d interfaces: %s" % (name, e, lim_g, tst_g, lim_o, rep["e1_flips"],
                                                          rep["hllc_flips"], rep["hllc_flips_at_ties"], rep["ties"],
                                                          rep["interfaces"], rep["flipped"]))
    # time step formula
    assert g.cfl_dt(U, 0.2) == pytest.approx(og.cfl_dt(wl["U0"], 0.2), rel=1e-12)
    g.close()


@pytest.mark.parametrize("name", ["c1", "c2", "c3", "c4"])
def test_rk3_steps_parity(mods, cases, name):
    torch, O, M = mods
    wl = cases[name]
    og = O.Grid(wl)
    og.metrics_compute(0.0)
    dt = wl["dt"] if wl["dt"] else og.cfl_dt(wl["U0"], wl["cfl"])
    steps = min(wl["steps"], 4)
    Uo = wl["U0"].copy()
    g = M.Grid(wl)
    g.metrics_compute(0.0)
    U = torch.as_tensor(wl["U0"], device="cuda").contiguous()
    t = 0.0
    for s in range(steps):
        og.rk3_step(Uo, t, dt)
        g.rk3_step(U, t, dt)
        t += dt
    e = rel(U.cpu().numpy(), Uo)
    assert np.all(e <= STEP_TOL), (name, e)
    g.close()


def test_freestream_static_and_dynamic_on_gpu(mods):
    torch, O, M = mods
    for wl in (W.freestream_static(20, "random"), W.c2_dynamic_freestream(n=32, steps=10)):
        g = M.Grid(wl)
        g.metrics_compute(0.0)
        U = torch.as_tensor(wl["U0"], device="cuda").contiguous()
        dt = g.cfl_dt(U, 0.2)
        t = 0.0
        for s in range(10):
            g.rk3_step(U, t, dt)
            t += dt
        g.metrics_compute(t)
        r = g.rhs(U)
        assert float((dt * r).abs().max()) <= 1e-12
        Uh = U.cpu().numpy()
        p = 0.4 * (Uh[4] - 0.5 * (Uh[1] ** 2 + Uh[2] ** 2 + Uh[3] ** 2) / Uh[0])
        p0 = 1.0 / (1.4 * 0.25)
        dev = max(np.abs(Uh[0] - 1).max(), np.abs(Uh[1] / Uh[0] - 1).max(), np.abs(Uh[2] / Uh[0]).max(),
                  np.abs(Uh[3] / Uh[0]).max(), np.abs(p - p0).max() / p0)
        assert dev <= 1e-12, (wl["name"], dev)
        g.close()


def test_minimum_size_and_call_order(mods):
    torch, O, M = mods
    wl = W.c1_vortex(n=10)
    g = M.Grid(wl)
    U = torch.as_tensor(wl["U0"], device="cuda").contiguous()
    with pytest.raises(M.Meg6Error):
        g.rhs(U)                      # MEG6_ESTATE before metrics_compute
    g.metrics_compute(0.0)
    og = O.Grid(wl)
    og.metrics_compute(0.0)
    e = rhs_err(g.rhs(U).cpu().numpy(), og.rhs(wl["U0"]), wl["U0"])
    assert np.all(e <= RHS_TOL), e
    g.close()


def test_sponge_and_rk3_closed_form_on_gpu(mods):
    """dQ/dt = -sigma (Q - Qref) for a fluid at rest: one step multiplies by 1 + z + z^2/2 + z^3/6."""
    torch, O, M = mods
    n = 12
    x, y, z = W.wavy_periodic_grid(n, 6.0, 0.0)
    prm = W._base_params(n, n, n, period=[[6.0, 0, 0], [0, 6.0, 0], [0, 0, 6.0]])
    one = np.ones((n, n, n))
    Uref = W.conservative(one, 0 * one, 0 * one, 0 * one, one)
    U0 = W.conservative(1.3 * one, 0 * one, 0 * one, 0 * one, 1.2 * one)
    g = M.Grid(dict(params=prm, x=x, y=y, z=z, sigma=0.7 * one, U_ref=Uref))
    g.metrics_compute(0.0)
    U = torch.as_tensor(U0, device="cuda").contiguous()
    g.rk3_step(U, 0.0, 0.4)
    zz = -0.28
    amp = 1 + zz + zz ** 2 / 2 + zz ** 3 / 6
    assert np.allclose(U.cpu().numpy() - Uref, amp * (U0 - Uref), rtol=1e-12, atol=1e-13)
    g.close()


# ---------------------------------------------------------------------------------------------------------
# Full sizes of BASELINE.json, in the launch configuration bench.py times.

def test_c1_full_config_10_steps(mods):
    """Config 1 as BASELINE.json states it: 32^3 wavy mesh, CFL 0.5, 10 RK3 steps, against the oracle."""
    torch, O, M = mods
    wl = W.c1_vortex(n=32)
    og = O.Grid(wl)
    og.metrics_compute(0.0)
    dt = wl["dt"] if wl["dt"] else og.cfl_dt(wl["U0"], wl["cfl"])
    g = M.Grid(wl)
    g.metrics_compute(0.0)
    Uo = wl["U0"].copy()
    U = torch.as_tensor(wl["U0"], device="cuda").contiguous()
    t = 0.0
    for s in range(10):
        og.rk3_step(Uo, t, dt)
        g.rk3_step(U, t, dt)
        t += dt
    e = rel(U.cpu().numpy(), Uo)
    assert np.all(e <= STEP_TOL), e
    g.close()


def test_c2_full_config_freestream_100_steps(mods):
    """Config 2 as BASELINE.json states it (64^3 jittered moving mesh, 100 RK3 steps): the residual stays <= 1e-12.
    A property that holds at any size; no oracle run is needed at this length."""
    torch, O, M = mods
    wl = W.c2_dynamic_freestream(n=64)
    g = M.Grid(wl)
    g.metrics_compute(0.0)
    U = torch.as_tensor(wl["U0"], device="cuda").contiguous()
    dt = wl["dt"] if wl["dt"] else g.cfl_dt(U, wl["cfl"])
    t = 0.0
    worst = 0.0
    for s in range(100):
        if s % 20 == 0:
            g.metrics_compute(t)
            worst = max(worst, float((dt * g.rhs(U)).abs().max()))
        g.rk3_step(U, t, dt)
        t += dt
    Uh = U.cpu().numpy()
    p = 0.4 * (Uh[4] - 0.5 * (Uh[1] ** 2 + Uh[2] ** 2 + Uh[3] ** 2) / Uh[0])
    p0 = 1.0 / (1.4 * 0.25)
    dev = max(np.abs(Uh[0] - 1).max(), np.abs(Uh[1] / Uh[0] - 1).max(), np.abs(Uh[2] / Uh[0]).max(),
              np.abs(Uh[3] / Uh[0]).max(), np.abs(p - p0).max() / p0)
    assert worst <= 1e-12 and dev <= 1e-12, (worst, dev)
    g.close()


def test_c4_full_size_rhs_and_step(mods):
    """The bench workload itself (320 x 200 x 200 jet mesh, inflow/outflow, sponge, viscous): one dQ/dt and one
    RK3 step of a seeded randomised state against the oracle, every cell compared."""
    torch, O, M = mods
    wl = W.c4_jet()
    rng = np.random.default_rng(44)
    shape = wl["U0"].shape[1:]
    rho = 1.0 + 0.2 * rng.uniform(-1, 1, shape)
    u, v, w = (0.3 * rng.uniform(-1, 1, shape) for _ in range(3))
    p = (1.0 + 0.2 * rng.uniform(-1, 1, shape)) / 1.4
    U0 = W.conservative(rho, u, v, w, p)
    del rho, u, v, w, p
    og = O.Grid(wl)
    og.metrics_compute(0.0)
    ref = og.rhs(U0)
    g = M.Grid(wl)
    g.metrics_compute(0.0)
    U = torch.as_tensor(U0, device="cuda").contiguous()
    out = g.rhs(U).cpu().numpy()
    e = rhs_err(out, ref, U0)
    assert np.all(e <= RHS_TOL), (e, rel(out, ref))
    del out, ref
    Uo = U0.copy()
    og.rk3_step(Uo, 0.0, wl["dt"])
    g.rk3_step(U, 0.0, wl["dt"])
    e2 = rel(U.cpu().numpy(), Uo)
    assert np.all(e2 <= STEP_TOL), e2
    print("c4 full size: rhs %s, one step %s" % (e, e2))
    g.close()


@pytest.mark.parametrize("shape", [(10, 10, 10), (31, 17, 16), (61, 12, 46)])
def test_ragged_shapes_non_periodic_viscous(mods, shape):
    """Tile tails in every direction (xi tiles of 30 cells x 4 rows, eta/zeta tiles of 15 cells x 8 lanes), down to
    the minimum size, with inflow/outflow ghosts, sponge and viscous terms."""
    torch, O, M = mods
    wl = W.c4_jet(ni=shape[0], nj=shape[1], nk=shape[2], steps=2)
    rng = np.random.default_rng(sum(shape))
    sh = wl["U0"].shape[1:]
    wl["U0"] = W.conservative(1.0 + 0.2 * rng.uniform(-1, 1, sh), *(0.3 * rng.uniform(-1, 1, sh) for _ in range(3)),
                              (1.0 + 0.2 * rng.uniform(-1, 1, sh)) / 1.4)
    og = O.Grid(wl)
    og.metrics_compute(0.0)
    g = M.Grid(wl)
    g.metrics_compute(0.0)
    U = torch.as_tensor(wl["U0"], device="cuda").contiguous()
    e = rhs_err(g.rhs(U).cpu().numpy(), og.rhs(wl["U0"]), wl["U0"])
    assert np.all(e <= RHS_TOL), e
    Uo = wl["U0"].copy()
    t = 0.0
    for s in range(2):
        og.rk3_step(Uo, t, wl["dt"])
        g.rk3_step(U, t, wl["dt"])
        t += wl["dt"]
    assert np.all(rel(U.cpu().numpy(), Uo) <= STEP_TOL)
    g.close()


# ---------------------------------------------------------------------------------------------------------
# MIG4 variant (scheme = 1, Eq. 18; reading R26)

def mig4_cases():
    out = {}
    for name, wl in small_cases().items():
        wl = dict(wl)
        wl["params"] = dict(wl["params"], scheme=1)
        out[name] = wl
    return out


@pytest.mark.parametrize("name", ["c1", "c2", "c3", "c4"])
def test_mig4_metrics_parity(mods, name):
    """Geometry of the MIG4 variant (every gradient inside the metric evaluation is the implicit IG4 one): bit for
    bit, as for MEG6."""
    torch, O, M = mods
    wl = mig4_cases()[name]
    t = 0.13 if wl["params"]["moving"] else 0.0
    og = O.Grid(wl)
    og.metrics_compute(t)
    g = M.Grid(wl)
    g.metrics_compute(t)
    checks = [("cell", q, g.get_array(0, q), og.cell(q)) for q in range(10)]
    for d in range(3):
        qs = range(10) if wl["params"]["viscous"] else range(3 * d, 3 * d + 3)
        checks += [("face%d" % d, q, g.get_array(1, 16 * d + q), og.face(d, q)) for q in qs]
    if wl["params"]["moving"]:
        checks += [("cell", q, g.get_array(0, q), og.cell(q)) for q in (10, 11, 12, 13)]
        checks += [("face%d" % d, 10, g.get_array(1, 16 * d + 10), og.face(d, 10)) for d in range(3)]
    for kind, q, a, b in checks:
        assert np.array_equal(a, b), (name, kind, q, np.abs(a - b).max() / np.abs(b).max())
    g.close()


@pytest.mark.parametrize("name", ["c1", "c2", "c3", "c4"])
def test_mig4_rhs_and_steps_parity(mods, name):
    """dQ/dt and a few RK3 steps of the MIG4 variant against the oracle: implicit gradients in the reconstruction,
    in the viscous flux (normal and tangential) and in the metrics."""
    torch, O, M = mods
    wl = mig4_cases()[name]
    t = 0.13 if wl["params"]["moving"] else 0.0
    og = O.Grid(wl)
    og.metrics_compute(t)
    ref = og.rhs(wl["U0"])
    g = M.Grid(wl)
    g.metrics_compute(t)
    g.limiter_stats_enable(True)
    U = torch.as_tensor(wl["U0"], device="cuda").contiguous()
    out = g.rhs(U).cpu().numpy()
    e = rhs_err(out, ref, wl["U0"])
    assert np.all(e <= RHS_TOL), (name, e, rel(out, ref))
    lim_o, tst_o = og.limiter_stats()
    lim_g, tst_g = g.limiter_stats()
    assert tst_g == tst_o and abs(lim_g - lim_o) <= max(5, 1e-3 * lim_o), (lim_g, lim_o, tst_g, tst_o)
    og.metrics_compute(0.0)
    g.metrics_compute(0.0)
    dt = wl["dt"] if wl["dt"] else og.cfl_dt(wl["U0"], wl["cfl"])
    Uo = wl["U0"].copy()
    tt = 0.0
    for s in range(3):
        og.rk3_step(Uo, tt, dt)
        g.rk3_step(U, tt, dt)
        tt += dt
    e2 = rel(U.cpu().numpy(), Uo)
    assert np.all(e2 <= STEP_TOL), (name, e2)
    print("mig4 %s: rhs %s steps %s limited %d/%d" % (name, e, e2, lim_g, tst_g))
    g.close()


def test_mig4_freestream_static_and_dynamic_on_gpu(mods):
    """MIG4 keeps uniform flow to <= 1e-12 on a 20 %-randomised static mesh and on the moving jittered mesh: the
    metric identity holds for the implicit line operators as well (they commute), at a size beyond the oracle runs."""
    torch, O, M = mods
    for wl in (W.freestream_static(20, "random"), W.c2_dynamic_freestream(n=48, steps=10)):
        wl = dict(wl)
        wl["params"] = dict(wl["params"], scheme=1)
        g = M.Grid(wl)
        g.metrics_compute(0.0)
        U = torch.as_tensor(wl["U0"], device="cuda").contiguous()
        dt = g.cfl_dt(U, 0.2)
        t = 0.0
        for s in range(10):
            g.rk3_step(U, t, dt)
            t += dt
        g.metrics_compute(t)
        assert float((dt * g.rhs(U)).abs().max()) <= 1e-12
        Uh = U.cpu().numpy()
        assert max(np.abs(Uh[0] - 1).max(), np.abs(Uh[2] / Uh[0]).max(), np.abs(Uh[3] / Uh[0]).max()) <= 1e-12
        g.close()


@pytest.mark.parametrize("scheme", [0, 1])
def test_diagnostics_parity(mods, scheme):
    """Kinetic energy / enstrophy / volume (Eq. 54) on the viscous TGV and on the moving jittered mesh: sums of ~1e5
    positive terms in a different order on the two sides, hence 1e-12 relative."""
    torch, O, M = mods
    cases = mig4_cases() if scheme else small_cases()
    for name in ("c1", "c2", "c3"):
        wl = cases[name]
        og = O.Grid(wl)
        og.metrics_compute(0.05)
        g = M.Grid(wl)
        g.metrics_compute(0.05)
        U = torch.as_tensor(wl["U0"], device="cuda").contiguous()
        a, b = np.array(g.diagnostics(U)), og.diagnostics(wl["U0"])
        assert np.all(np.abs(a - b) <= 1e-12 * np.abs(b)), (name, a, b)
        g.close()


def test_abi_error_paths_on_device(mods):
    """Error behaviour the header promises: status codes, no exceptions, no partial handles."""
    import ctypes as C
    torch, O, M = mods
    from paper_2303_10785_b200 import binding as B
    L = B.lib()
    wl = W.c1_vortex(n=12)
    p = B.make_params(wl["params"])
    nb = L.meg6_workspace_bytes(C.byref(p))
    ws = torch.empty(nb + 512, dtype=torch.uint8, device="cuda")
    base = (ws.data_ptr() + 255) // 256 * 256
    x, y, z = (torch.as_tensor(wl[k], device="cuda").contiguous() for k in ("x", "y", "z"))
    h = C.c_void_p()
    args = lambda wsp, n: (C.byref(p), C.c_void_p(x.data_ptr()), C.c_void_p(y.data_ptr()), C.c_void_p(z.data_ptr()),
                           None, None, None, C.c_void_p(wsp), C.c_size_t(n), None, C.byref(h))
    saved = L.meg6_grid_create.argtypes
    L.meg6_grid_create.argtypes = None           # raw calls with deliberately wrong arguments; restored below
    assert L.meg6_grid_create(*args(base, nb - 1)) == 2 and not h.value        # MEG6_ENOMEM: workspace too small
    assert L.meg6_grid_create(*args(base + 8, nb)) == 1 and not h.value        # MEG6_EINVAL: misaligned workspace
    assert L.meg6_grid_create(C.byref(p), None, None, None, None, None, None, C.c_void_p(base), C.c_size_t(nb), None,
                              C.byref(h)) == 1                                  # null node arrays
    assert L.meg6_grid_create(*args(base, nb)) == 0 and h.value
    U = torch.as_tensor(wl["U0"], device="cuda").contiguous()
    out = torch.empty_like(U)
    assert L.meg6_rhs(h, C.c_void_p(U.data_ptr()), C.c_void_p(out.data_ptr())) == 4       # MEG6_ESTATE
    assert b"metrics_compute" in L.meg6_last_error()
    assert L.meg6_rhs(h, None, C.c_void_p(out.data_ptr())) == 1
    assert L.meg6_metrics_compute(h, C.c_double(0.0)) == 0
    assert L.meg6_rhs(h, C.c_void_p(U.data_ptr()), C.c_void_p(out.data_ptr())) == 0
    assert L.meg6_set_inflow(h, 0, C.c_void_p(U.data_ptr())) == 1               # periodic face: not an inflow face
    torch.cuda.synchronize()
    assert bool(torch.isfinite(out).all())
    L.meg6_grid_destroy(h)
    L.meg6_grid_create.argtypes = saved


# ------------------------------------------------------------------ walls (Table 1, R27)
def wall_cases():
    return {
        "channel_inviscid_wall": W.wall_channel(ni=37, nj=21, nk=26, wall=3, viscous=0, curved=True),
        "channel_slip_viscous": W.wall_channel(ni=24, nj=33, nk=20, wall=3, viscous=1, curved=True),
        "channel_adiabatic": W.wall_channel(ni=37, nj=21, nk=26, wall=4, viscous=1, curved=True),
        "box_mixed_walls": W.wall_box(),
        "box_mixed_walls_mig4": W.wall_box(ni=20, nj=23, nk=18, scheme=1),
        "channel_adiabatic_mig4": W.wall_channel(ni=24, nj=18, nk=20, wall=4, viscous=1, curved=True, scheme=1),
    }


@pytest.mark.parametrize("name", list(wall_cases()))
def test_wall_ghosts_rhs_and_steps_parity(mods, name):
    """Inviscid and adiabatic no-slip walls (bc 3 / 4): ghost primitives, one dQ/dt and three RK3 steps against the
    oracle; curved walls, ragged sizes, edges and corners of a closed box with walls of both kinds, MEG6 and MIG4."""
    torch, O, M = mods
    wl = wall_cases()[name]
    og = O.Grid(wl)
    og.metrics_compute(0.0)
    ref = og.rhs(wl["U0"])
    g = M.Grid(wl)
    g.metrics_compute(0.0)
    g.limiter_stats_enable(True)
    U = torch.as_tensor(wl["U0"], device="cuda").contiguous()
    out = g.rhs(U).cpu().numpy()
    for f in range(6):
        a, b = g.get_array(2, f), og.prim(f)
        assert np.abs(a - b).max() <= 1e-14 * np.abs(b).max()
    e = rhs_err(out, ref, wl["U0"])
    assert np.all(e <= RHS_TOL), (name, e, rel(out, ref))
    lim_o, tst_o = og.limiter_stats()
    lim_g, tst_g = g.limiter_stats()
    assert tst_g == tst_o
    assert abs(lim_g - lim_o) <= max(5, 1e-3 * lim_o), (lim_g, lim_o)
    dt = og.cfl_dt(wl["U0"], wl["cfl"])
    assert g.cfl_dt(U, wl["cfl"]) == pytest.approx(dt, rel=1e-12)
    Uo = wl["U0"].copy()
    t = 0.0
    for s in range(3):
        og.rk3_step(Uo, t, dt)
        g.rk3_step(U, t, dt)
        t += dt
    e = rel(U.cpu().numpy(), Uo)
    assert np.all(e <= STEP_TOL), (name, e)
    g.close()


INOUT_CASES = [(0, False, 1.0, 1, 0), (0, True, 0.5, 0, 0), (1, False, 1.0, 1, 0), (1, True, 1.6, 1, 1),
               (2, False, 0.5, 1, 1), (2, True, 1.0, 1, 0)]


@pytest.mark.parametrize("axis,flip,u_mean,viscous,scheme", INOUT_CASES)
def test_inflow_outflow_faces_in_every_direction_parity(mods, axis, flip, u_mean, viscous, scheme):
    """Inflow / outflow ghost rules (Table 1, R20) on each of the six faces, the other two directions
    periodic, non-uniform inflow data, sub- and supersonic outflow cells in one face (u_mean = 1): one dQ/dt and three
    RK3 steps against the oracle.  The inflow data of a ghost column of a periodic transverse direction are those of
    its periodic image (the corner ghost cells the viscous tangential gradients read)."""
    torch, O, M = mods
    n = [13, 11, 12]
    n[axis] = 21
    wl = W.inout_box(n=tuple(n), axis=axis, flip=flip, viscous=viscous, u_mean=u_mean, scheme=scheme)
    og = O.Grid(wl)
    og.metrics_compute(0.0)
    ref = og.rhs(wl["U0"])
    g = M.Grid(wl)
    g.metrics_compute(0.0)
    U = torch.as_tensor(wl["U0"], device="cuda").contiguous()
    out = g.rhs(U).cpu().numpy()
    e = rhs_err(out, ref, wl["U0"])
    assert np.all(e <= RHS_TOL), (wl["name"], e, rel(out, ref))
    dt = og.cfl_dt(wl["U0"], wl["cfl"])
    assert g.cfl_dt(U, wl["cfl"]) == pytest.approx(dt, rel=1e-12)
    Uo = wl["U0"].copy()
    t = 0.0
    for s in range(3):
        og.rk3_step(Uo, t, dt)
        g.rk3_step(U, t, dt)
        t += dt
    e = rel(U.cpu().numpy(), Uo)
    assert np.all(e <= STEP_TOL), (wl["name"], e)
    g.close()


def test_walls_on_a_moving_mesh_are_einval(mods):
    torch, O, M = mods
    wl = W.c2_dynamic_freestream(n=12, steps=1)
    wl["params"] = dict(wl["params"], periodic=[1, 0, 1], bc=[0, 0, 4, 4, 0, 0])
    with pytest.raises(Exception):
        M.Grid(wl)


# ------------------------------------------------------------------ block interfaces (NEXT-3, Sec. 6, R28)
def _block_sets():
    return {
        "cart_2x2_viscous": (W.cartesian_periodic(viscous=1), ((14, 10), (10, 10), (16,))),
        "cart_zeta_cut_inviscid": (W.cartesian_periodic(nk=22, viscous=0), ((24,), (20,), (12, 10))),
        "curved_box_walls_2x2x2": (W.wall_box(ni=26, nj=24, nk=22), ((14, 12), (11, 13), (10, 12))),
        "curved_box_walls_mig4": (W.wall_box(ni=26, nj=24, nk=22, scheme=1), ((14, 12), (24,), (10, 12))),
        # inflow / outflow faces across zeta with non-uniform P_in, cut in xi and eta: the corner ghost cells beyond the
        # block edges are the NEIGHBOUR's inflow ghosts (edge round of the fill, R28)
        "inout_zeta_cut_xi_eta": (W.inout_box(n=(23, 21, 21), axis=2, viscous=1, u_mean=1.0), ((12, 11), (10, 11), (21,))),
        "inout_eta_cut_xi": (W.inout_box(n=(23, 21, 12), axis=1, flip=True, viscous=1, u_mean=0.5), ((12, 11), (21,), (12,))),
    }


@pytest.mark.parametrize("name", list(_block_sets()))
def test_blocks_rhs_and_steps_parity(mods, name):
    """meg6_rhs_blocks / meg6_rk3_step_blocks against the oracle's multi-block calls, block by block: Cartesian cuts
    (where the oracle pins say cut == uncut) and curved blocks with walls of both kinds on the outer faces, edges and
    corners through diagonal neighbours, MEG6 and MIG4."""
    torch, O, M = mods
    wl, cuts = _block_sets()[name]
    blocks, links = W.split_blocks(wl, cuts)
    og = [O.Grid(b) for b in blocks]
    gg = [M.Grid(b) for b in blocks]
    W.link_all(og, blocks, links)
    W.link_all(gg, blocks, links)
    O.metrics_compute_blocks(og, 0.0)
    M.metrics_compute_blocks(gg, 0.0)
    for a, b in zip(og, gg):        # geometry of every block, ghost coordinates from the neighbours: bit for bit
        for q in range(10):
            assert np.array_equal(b.get_array(0, q), a.cell(q)), (name, q)
    ref = O.rhs_blocks(og, [b["U0"] for b in blocks])
    Us = [torch.as_tensor(b["U0"], device="cuda").contiguous() for b in blocks]
    out = M.rhs_blocks(gg, Us)
    for b, r, o in zip(blocks, ref, out):
        e = rhs_err(o.cpu().numpy(), r, b["U0"])
        assert np.all(e <= RHS_TOL), (name, b["name"], e)
    dt = min(g.cfl_dt(b["U0"], 0.4) for g, b in zip(og, blocks))
    Uo = [b["U0"].copy() for b in blocks]
    for s in range(3):
        O.rk3_step_blocks(og, Uo, s * dt, dt)
        M.rk3_step_blocks(gg, Us, s * dt, dt)
    for b, uo, u in zip(blocks, Uo, Us):
        e = rel(u.cpu().numpy(), uo)
        assert np.all(e <= STEP_TOL), (name, b["name"], e)
    if wl["params"].get("scheme", 0) == 0:
        # and the cut run equals the uncut one on the GPU as well, curved meshes included (ghost coordinates of an
        # interface face are the neighbour's cell centres, R28); walls of both kinds on the outer faces.  Not for MIG4:
        # its implicit gradients are line solves, and a cut line is two systems with their own closures (R26)
        g1 = M.Grid(wl)
        g1.metrics_compute(0.0)
        U1 = torch.as_tensor(wl["U0"], device="cuda").contiguous()
        for s in range(3):
            g1.rk3_step(U1, s * dt, dt)
        U1 = U1.cpu().numpy()
        for b, u in zip(blocks, Us):
            e = rel(u.cpu().numpy(), U1[(slice(None),) + b["slices"]])
            assert np.all(e <= 1e-11), (name, b["name"], e)
        g1.close()
    for g in gg:
        g.close()


def test_blocks_call_order_errors(mods):
    torch, O, M = mods
    wl = W.cartesian_periodic(ni=20, nj=12, nk=12, viscous=0)
    blocks, links = W.split_blocks(wl, ((10, 10), (12,), (12,)))
    gg = [M.Grid(b) for b in blocks]
    Us = [torch.as_tensor(b["U0"], device="cuda").contiguous() for b in blocks]
    with pytest.raises(M.Meg6Error):
        M.metrics_compute_blocks(gg, 0.0)          # interfaces not linked yet
    W.link_all(gg, blocks, links)
    with pytest.raises(M.Meg6Error):
        gg[0].metrics_compute(0.0)                 # single-grid call on a block with a foreign neighbour
    with pytest.raises(M.Meg6Error):
        M.rhs_blocks(gg, Us)                       # before the metrics
    M.metrics_compute_blocks(gg, 0.0)
    with pytest.raises(M.Meg6Error):
        gg[0].rhs(Us[0])                           # single-grid call on a block with a foreign neighbour
    with pytest.raises(M.Meg6Error):
        M.rhs_blocks(gg[:1], Us[:1])               # neighbour missing from the list
    with pytest.raises(M.Meg6Error):
        M.Grid(wl).link(0, gg[0])                  # not an interface face
    M.rhs_blocks(gg, Us)
    for g in gg:
        g.close()


def test_staged_api_with_packed_layers_equals_linked_blocks(mods):
    """The staged calls (meg6_stage_prim / _pack / _ghosts / _sweeps with meg6_set_interface_buffer), driven here for
    two blocks in one process with the packed layers copied by hand, are the path paper_2303_10785_b200.slabs runs
    between ranks: bit for bit the result of meg6_rk3_step_blocks on linked blocks (same kernels, same data)."""
    torch, O, M = mods
    wl = W.wall_box(ni=26, nj=24, nk=22)
    cuts = ((26,), (11, 13), (10, 12))      # eta and zeta interfaces: edge ghosts travel inside the packed layers
    blocks, links = W.split_blocks(wl, cuts)
    ref = [M.Grid(b) for b in blocks]
    W.link_all(ref, blocks, links)
    M.metrics_compute_blocks(ref, 0.0)
    gg = [M.Grid(b) for b in blocks]
    send, recv, gsend, grecv = {}, {}, {}, {}
    for home, face, nb in links:
        send[(home, face)] = gg[home].new_interface_buffer(face)
        recv[(home, face)] = gg[home].new_interface_buffer(face)
        gg[home].set_interface_buffer(face, recv[(home, face)])
        gsend[(home, face)] = gg[home].new_geom_interface_buffer(face)
        grecv[(home, face)] = gg[home].new_geom_interface_buffer(face)
        gg[home].set_geom_interface_buffer(face, grecv[(home, face)], blocks[home]["link_offset"].get(face))
    # staged geometry: centres, then per direction pack / hand over / extend, then the metrics
    for g in gg:
        g.stage_geom_centres(0.0)
    for d in range(3):
        for home, face, nb in links:
            if face // 2 == d:
                gg[home].stage_geom_pack(face, gsend[(home, face)])
        for home, face, nb in links:
            if face // 2 == d:
                grecv[(nb, face ^ 1)].copy_(gsend[(home, face)])
        for g in gg:
            g.stage_geom_extend(d)
    for g in gg:
        g.stage_geom_finish()
    for a, b in zip(gg, ref):
        for q in range(10):
            assert np.array_equal(a.get_array(0, q), b.get_array(0, q))
    Ur = [torch.as_tensor(b["U0"], device="cuda").contiguous() for b in blocks]
    Us = [u.clone() for u in Ur]
    dt = 1.5e-3

    def ghosts(s):
        for d in range(3):
            for home, face, nb in links:
                if face // 2 == d:
                    gg[home].stage_pack(s, face, send[(home, face)])
            for home, face, nb in links:
                if face // 2 == d:
                    recv[(nb, face ^ 1)].copy_(send[(home, face)])
            for g in gg:
                g.stage_ghosts(s, d)

    # right-hand side
    want = M.rhs_blocks(ref, Ur)
    got = [torch.empty_like(u) for u in Us]
    for g, u in zip(gg, Us):
        g.stage_prim(u)
    ghosts(0)
    for g, u, o in zip(gg, Us, got):
        g.stage_sweeps(u, 0, 0.0, out=o)
    for a, b in zip(got, want):
        assert torch.equal(a, b)
    # two RK3 steps
    for step in range(2):
        M.rk3_step_blocks(ref, Ur, step * dt, dt)
        for s in range(3):
            if s == 0:
                for g, u in zip(gg, Us):
                    g.stage_prim(u)
            ghosts(s)
            for g, u in zip(gg, Us):
                g.stage_sweeps(u, s, dt)
    for a, b, blk in zip(Us, Ur, blocks):
        assert torch.equal(a, b)
        assert (a.cpu().numpy() - blk["U0"]).__abs__().max() > 1e-5
    for g in ref + gg:
        g.close()


def test_tgv_kinetic_energy_budget_on_gpu(mods):
    """Physics-level check of the whole GPU path with no oracle in it: for the nearly
    incompressible Taylor-Green vortex the kinetic energy obeys -dE_k/dt = 2 nu * enstrophy, both sides
    measured with meg6_diagnostics while meg6_rk3_step advances the flow on the wavy mesh.  Re = 100 so that the
    physical dissipation dominates the scheme's own; Ma = 0.1 leaves an O(Ma^2) pressure-dilatation term."""
    torch, O, M = mods
    re = 100.0
    wl = W.c3_tgv(n=64, re=re)
    g = M.Grid(wl)
    g.metrics_compute(0.0)
    U = torch.as_tensor(wl["U0"], device="cuda").contiguous()
    ke0, en0, vol = g.diagnostics(U)
    assert ke0 == pytest.approx(0.125, rel=2e-3) and en0 == pytest.approx(0.375, rel=2e-3)
    assert vol == pytest.approx((2 * np.pi) ** 3, rel=1e-12)
    dt = g.cfl_dt(U, 0.4)
    every, t, hist = 25, 0.0, [(0.0, ke0, en0)]
    for s in range(1, 12 * every + 1):
        g.rk3_step(U, t, dt)
        t += dt
        if s % every == 0:
            ke, en, _ = g.diagnostics(U)
            hist.append((t, ke, en))
    h = np.array(hist)
    assert np.all(np.diff(h[:, 1]) < 0)                       # energy decays monotonically
    eps = -(h[2:, 1] - h[:-2, 1]) / (h[2:, 0] - h[:-2, 0])    # central differences at the interior samples
    visc = 2.0 / re * h[1:-1, 2]
    assert np.all(np.abs(eps / visc - 1.0) < 0.03), (eps / visc)
    g.close()


def test_c3_full_size_conservation_and_symmetry_of_the_step(mods):
    """Config 3 at BASELINE.json's full size (128^3, the launch configuration bench.py --workload c3 times), checked
    through properties that hold at any size: the sum over cells of (1/J) dQ/dt telescopes to zero on the periodic
    mesh (Eq. 8-9), and ten RK3 steps conserve the (1/J)-weighted totals of mass, momentum and energy."""
    torch, O, M = mods
    wl = W.c3_tgv(n=128)
    g = M.Grid(wl)
    g.metrics_compute(0.0)
    U = torch.as_tensor(wl["U0"], device="cuda").contiguous()
    rj = torch.as_tensor(g.get_array(0, 9), device="cuda")
    r = g.rhs(U)
    tot = (r * rj).reshape(5, -1).sum(1)
    scale = (r.abs() * rj).reshape(5, -1).sum(1)
    assert bool(torch.all(tot.abs() <= 1e-11 * torch.clamp(scale, min=1.0))), (tot, scale)
    q0 = (U * rj).reshape(5, -1).sum(1)
    dt = g.cfl_dt(U, wl["cfl"])
    for s in range(10):
        g.rk3_step(U, s * dt, dt)
    q1 = (U * rj).reshape(5, -1).sum(1)
    ref = (U.abs() * rj).reshape(5, -1).sum(1)
    assert bool(torch.isfinite(U).all())
    assert bool(torch.all((q1 - q0).abs() <= 1e-11 * ref)), (q1 - q0, ref)
    g.close()


def test_full_step_counts_of_configs_3_4_5_stay_finite_and_bounded(mods):
    """BASELINE.json's step counts at full size on the GPU: config 3 (128^3, 200 RK3 steps), config 4 (320x200x200,
    500 steps: the jet starts up, shocks form at the nozzle lip, the limiter becomes active) and the MIG4 variant
    (config 5 in full: 384^3, 50 steps).  The oracle would need hours for these; the checks are properties: finite
    state, positive density and pressure, kinetic energy of the Taylor-Green vortex decaying."""
    torch, O, M = mods

    def run(wl, steps, cfl=None):
        g = M.Grid(wl)
        g.metrics_compute(0.0)
        U = torch.as_tensor(wl["U0"], device="cuda").contiguous()
        dt = wl["dt"] if wl["dt"] else g.cfl_dt(U, cfl or wl["cfl"])
        ke0 = g.diagnostics(U)[0]
        for s in range(steps):
            g.rk3_step(U, s * dt, dt)
        assert bool(torch.isfinite(U).all())
        rho = U[0]
        p = 0.4 * (U[4] - 0.5 * (U[1] ** 2 + U[2] ** 2 + U[3] ** 2) / rho)
        assert float(rho.min()) > 0.0 and float(p.min()) > 0.0
        ke1 = g.diagnostics(U)[0]
        g.limiter_stats_enable(True)
        g.rk3_step(U, steps * dt, dt)
        lim, tst = g.limiter_stats()
        g.close()
        return ke0, ke1, lim / tst

    ke0, ke1, _ = run(W.c3_tgv(n=128), 200)
    assert 0.9 * ke0 < ke1 < ke0
    ke0, ke1, _ = run(W.c5_tgv_mig4(n=384), 50)      # config 5 at its own size: 56.6 M cells, 50 GB of workspace
    assert 0.95 * ke0 < ke1 < ke0
    ke0, ke1, frac = run(W.c4_jet(), 500)
    assert ke1 > ke0                     # the jet has entered the quiescent domain
    assert frac > 1e-4                   # and the limiter is at work
    print("C4 after 500 steps: limited fraction %.4f" % frac)


# ------------------------------------------------------------------ ghost coordinates from the neighbour, rotated blocks
def test_cut_stretched_jet_mesh_equals_the_uncut_one_on_gpu(mods):
    """Config-4-type mesh (tanh-stretched, inflow / outflow / sponge, viscous) cut into 2 x 2 x 2 blocks: the metrics of
    every block are those of the uncut mesh BIT FOR BIT (ghost coordinates of an interface face = the neighbour's cell
    centres), dQ/dt and three RK3 steps agree with the uncut run to round-off, and with the oracle's blocks."""
    torch, O, M = mods
    wl = small_cases()["c4"]
    cuts = ((26, 26), (20, 17), (17, 16))
    blocks, links = W.split_blocks(wl, cuts)
    gg = [M.Grid(b) for b in blocks]
    W.link_all(gg, blocks, links)
    M.metrics_compute_blocks(gg, 0.0)
    g1 = M.Grid(wl)
    g1.metrics_compute(0.0)
    for b, g in zip(blocks, gg):
        for q in range(10):
            assert np.array_equal(g.get_array(0, q), g1.get_array(0, q)[b["slices"]]), (b["name"], q)
        for d in range(3):
            fsl = list(b["slices"])
            fsl[2 - d] = slice(fsl[2 - d].start, fsl[2 - d].stop + 1)
            for q in range(10):
                assert np.array_equal(g.get_array(1, 16 * d + q), g1.get_array(1, 16 * d + q)[tuple(fsl)])
    U1 = torch.as_tensor(wl["U0"], device="cuda").contiguous()
    Us = [torch.as_tensor(b["U0"], device="cuda").contiguous() for b in blocks]
    r1 = g1.rhs(U1).cpu().numpy()
    out = M.rhs_blocks(gg, Us)
    for b, o in zip(blocks, out):
        e = rhs_err(o.cpu().numpy(), r1[(slice(None),) + b["slices"]], b["U0"])
        assert np.all(e <= 1e-12), (b["name"], e)
    for s in range(3):
        g1.rk3_step(U1, s * wl["dt"], wl["dt"])
        M.rk3_step_blocks(gg, Us, s * wl["dt"], wl["dt"])
    U1 = U1.cpu().numpy()
    for b, u in zip(blocks, Us):
        assert np.all(rel(u.cpu().numpy(), U1[(slice(None),) + b["slices"]]) <= 1e-12)
    for g in gg + [g1]:
        g.close()


def _link_oriented(grids, blocks, periods=()):
    for home, face, nb, nb_face, swap, fa, fb, off in W.auto_links(blocks, periods):
        grids[home].link(face, grids[nb], nb_face=nb_face, swap=swap, flip_a=fa, flip_b=fb, offset=off)


@pytest.mark.parametrize("case", ["wavy_periodic_3d", "jet_mesh_quadrants", "mig4_quadrants"])
def test_blocks_with_rotated_coordinate_systems_on_gpu(mods, case):
    """Sec. 6 (SURVEY NEXT-3 "4-block butterfly"): blocks stored in frames rotated against their neighbours'
    (quarter turns about zeta: the four wings of a butterfly-type section; cyclic and x-axis rotations in the 3-D case),
    linked by node matching.  Against the oracle's blocks (same links): geometry bit for bit, dQ/dt <= 1e-11, three
    steps <= 1e-9; and turned back, against the UNCUT single block on the GPU, which never sees a link."""
    torch, O, M = mods
    if case == "wavy_periodic_3d":
        wl = W.c3_tgv(n=24)
        cuts, rots = ((12, 12), (10, 14), (14, 10)), ["id", "z90", "cyc", "x90", "z270", "id", "z180", "cyc"]
        periods = wl["params"]["period"]
    else:
        # outflow faces around, four quadrant blocks about the jet axis direction (here zeta), each turned by a quarter
        wl = W.c4_jet(ni=26, nj=24, nk=22)
        wl["params"] = dict(wl["params"], bc=[2, 2, 2, 2, 2, 2], scheme=1 if case == "mig4_quadrants" else 0)
        wl["inflow"] = {}
        rng = np.random.default_rng(12)
        sh = wl["U0"].shape[1:]
        wl["U0"] = W.conservative(1.0 + 0.1 * rng.uniform(-1, 1, sh), *(0.2 * rng.uniform(-1, 1, sh) for _ in range(3)),
                                  (1.0 + 0.1 * rng.uniform(-1, 1, sh)) / 1.4)
        cuts, rots = ((14, 12), (12, 12), (22,)), ["id", "z90", "z270", "z180"]
        periods = ()
    plain, _ = W.split_blocks(wl, cuts)
    blocks = [W.rotate_block(b, r) for b, r in zip(plain, rots)]
    og = [O.Grid(b) for b in blocks]
    gg = [M.Grid(b) for b in blocks]
    _link_oriented(og, blocks, periods)
    _link_oriented(gg, blocks, periods)
    O.metrics_compute_blocks(og, 0.0)
    M.metrics_compute_blocks(gg, 0.0)
    for a, b in zip(og, gg):
        for q in range(10):
            assert np.array_equal(b.get_array(0, q), a.cell(q)), (case, q)
    ref = O.rhs_blocks(og, [b["U0"] for b in blocks])
    Us = [torch.as_tensor(b["U0"], device="cuda").contiguous() for b in blocks]
    out = [o.cpu().numpy() for o in M.rhs_blocks(gg, Us)]
    for b, r, o in zip(blocks, ref, out):
        e = rhs_err(o, r, b["U0"])
        assert np.all(e <= RHS_TOL), (case, b["name"], e)
    # turned back: the uncut block
    g1 = M.Grid(wl)
    g1.metrics_compute(0.0)
    U1 = torch.as_tensor(wl["U0"], device="cuda").contiguous()
    r1 = g1.rhs(U1).cpu().numpy()
    tol = 1e-10 if case == "wavy_periodic_3d" else 1e-11     # Ma 0.1: see tests/test_oracle_blocks.py
    if case != "jet_mesh_quadrants" and case != "mig4_quadrants":
        for b, p, o in zip(blocks, plain, out):
            e = rhs_err(W.unrotate_state(o, b["rotation"]), r1[(slice(None),) + p["slices"]], p["U0"])
            assert np.all(e <= tol), (case, b["name"], e)
    dt = min(g.cfl_dt(b["U0"], 0.4) for g, b in zip(og, blocks))
    Uo = [b["U0"].copy() for b in blocks]
    for s in range(3):
        O.rk3_step_blocks(og, Uo, s * dt, dt)
        M.rk3_step_blocks(gg, Us, s * dt, dt)
    for b, uo, u in zip(blocks, Uo, Us):
        assert np.all(rel(u.cpu().numpy(), uo) <= STEP_TOL), (case, b["name"])
    for g in gg + [g1]:
        g.close()


def test_slab_stepper_on_two_cuda_grids_through_an_in_process_transport(mods, monkeypatch):
    """paper_2303_10785_b200.slabs.SlabStepper itself (geometry exchange, per-direction pack / exchange / ghost fill,
    sweeps) driven for two zeta slabs of the stretched jet mesh on the ONE device: torch.distributed's point-to-point
    calls are replaced by a shim that hands the tensors over with device-to-device copies (NCCL cannot put two ranks
    on one GPU; the NCCL leg itself stays unexecuted on this pool).  Result: bit for bit meg6_rk3_step_blocks."""
    torch, O, M = mods
    from paper_2303_10785_b200 import slabs
    wl = small_cases()["c4"]
    blocks, links = W.split_blocks(wl, ((52,), (37,), (17, 16)))
    ref = [M.Grid(b) for b in blocks]
    W.link_all(ref, blocks, links)
    M.metrics_compute_blocks(ref, 0.0)
    gg = [M.Grid(b) for b in blocks]

    import threading

    class Shim:
        """mailbox transport for ranks that are threads of this process: a send parks a copy of the tensor, a receive
        waits for it and copies it in (device-to-device, on the one stream both grids use)"""
        isend, irecv = "send", "recv"

        def __init__(self):
            self.tls, self.box, self.cv = threading.local(), {}, threading.Condition()

        def P2POp(self, op, tensor, peer, group=None, tag=0):
            return (op, tensor, peer, tag)

        def batch_isend_irecv(self, ops):
            me, works = self.tls.rank, []
            for op, t, peer, tag in ops:
                if op == "send":
                    with self.cv:
                        self.box[(me, peer, tag)] = t.clone()
                        self.cv.notify_all()
                else:
                    works.append(self._Recv(self, (peer, me, tag), t))
            return works

        class _Recv:
            def __init__(self, shim, key, t):
                self.shim, self.key, self.t = shim, key, t

            def wait(self):
                with self.shim.cv:
                    assert self.shim.cv.wait_for(lambda: self.key in self.shim.box, timeout=60)
                    src = self.shim.box.pop(self.key)
                self.t.copy_(src)
    shim = Shim()
    monkeypatch.setattr(slabs, "dist", shim)
    steppers = []
    for r in range(2):
        remote = {face: nb for home, face, nb in links if home == r}
        steppers.append(slabs.SlabStepper(gg[r], remote, offsets=blocks[r]["link_offset"]))

    def on_ranks(fn):
        """fn(rank) on one thread per rank, as torchrun would on one process per rank"""
        errs = []

        def body(r):
            shim.tls.rank = r
            try:
                with torch.cuda.device(0):
                    fn(r)
            except BaseException as e:   # noqa: BLE001
                errs.append(e)
        th = [threading.Thread(target=body, args=(r,)) for r in range(2)]
        for t in th:
            t.start()
        for t in th:
            t.join()
        if errs:
            raise errs[0]
    on_ranks(lambda r: steppers[r].metrics_compute(0.0))
    for a, b in zip(gg, ref):
        for q in range(10):
            assert np.array_equal(a.get_array(0, q), b.get_array(0, q))
    Ur = [torch.as_tensor(b["U0"], device="cuda").contiguous() for b in blocks]
    Us = [u.clone() for u in Ur]
    for n in range(2):
        M.rk3_step_blocks(ref, Ur, n * wl["dt"], wl["dt"])
        on_ranks(lambda r: steppers[r].rk3_step(Us[r], n * wl["dt"], wl["dt"]))
    for a, b, blk in zip(Us, Ur, blocks):
        assert torch.equal(a, b)
        assert (a.cpu().numpy() - blk["U0"]).__abs__().max() > 1e-6
    for g in ref + gg:
        g.close()


@pytest.mark.parametrize("name", ["c2", "c3", "c4"])
def test_rk3_steps_equals_repeated_rk3_step_bit_for_bit(mods, cases, name):
    """meg6_rk3_steps(n) = n x meg6_rk3_step: same kernels on the same data (the primitive conversion of U^{n+1} moves
    from its own kernel into the last sweep of step n), static and moving meshes, odd step count (buffer parity)."""
    torch, O, M = mods
    wl = cases[name]
    side = torch.cuda.Stream()                    # graphs need a stream of the caller's own
    torch.cuda.current_stream().synchronize()
    with torch.cuda.stream(side):
        _rk3_steps_body(torch, M, wl)
    side.synchronize()


def _rk3_steps_body(torch, M, wl):
    g = M.Grid(wl)
    g.metrics_compute(0.0)
    U = torch.as_tensor(wl["U0"], device="cuda").contiguous()
    dt = wl["dt"] if wl["dt"] else g.cfl_dt(U, wl["cfl"])
    Ua, Ub = U.clone(), U.clone()
    for s in range(5):
        g.rk3_step(Ua, s * dt, dt)
    g.rk3_steps(Ub, 0.0, dt, 5)
    assert torch.equal(Ua, Ub)
    g.rk3_steps(Ub, 5 * dt, dt, 0)
    assert torch.equal(Ua, Ub)
    # again from the new state (static meshes replay the captured two-step graph), then with another dt (re-captured)
    for dt2, n in ((dt, 6), (0.5 * dt, 4)):
        for s in range(n):
            g.rk3_step(Ua, s * dt2, dt2)
        g.rk3_steps(Ub, 0.0, dt2, n)
        assert torch.equal(Ua, Ub)
    g.close()


@pytest.mark.parametrize("scheme", [0, 1])
def test_butterfly_section_on_gpu(mods, scheme):
    """Butterfly-type O-grid section (Fig. 13b): square core + four outer blocks in frames a quarter turn apart,
    three blocks around each corner edge of the core, sixteen oriented links found by node matching.  Against the
    oracle's blocks: geometry bit for bit, dQ/dt <= 1e-11, three RK3 steps <= 1e-9, MEG6 and MIG4; and a uniform viscous
    flow stays uniform to <= 1e-12 on the GPU (Sec. 7: freestream preservation on any mesh)."""
    torch, O, M = mods
    blocks = W.butterfly(n=14, nr=12, nk=10, scheme=scheme)
    og = [O.Grid(b) for b in blocks]
    gg = [M.Grid(b) for b in blocks]
    _link_oriented(og, blocks)
    _link_oriented(gg, blocks)
    O.metrics_compute_blocks(og, 0.0)
    M.metrics_compute_blocks(gg, 0.0)
    for a, b in zip(og, gg):
        for q in range(10):
            assert np.array_equal(b.get_array(0, q), a.cell(q)), q
    ref = O.rhs_blocks(og, [b["U0"] for b in blocks])
    Us = [torch.as_tensor(b["U0"], device="cuda").contiguous() for b in blocks]
    out = [o.cpu().numpy() for o in M.rhs_blocks(gg, Us)]
    for b, r, o in zip(blocks, ref, out):
        e = rhs_err(o, r, b["U0"])
        assert np.all(e <= RHS_TOL), (b["name"], e)
    dt = min(g.cfl_dt(b["U0"], 0.4) for g, b in zip(og, blocks))
    Uo = [b["U0"].copy() for b in blocks]
    for s in range(3):
        O.rk3_step_blocks(og, Uo, s * dt, dt)
        M.rk3_step_blocks(gg, Us, s * dt, dt)
    for b, uo, u in zip(blocks, Uo, Us):
        assert np.all(rel(u.cpu().numpy(), uo) <= STEP_TOL), b["name"]
    for g in gg:
        g.close()
    # freestream on the GPU
    blocks = W.butterfly(n=14, nr=12, nk=10, scheme=scheme, uniform=True)
    gg = [M.Grid(b) for b in blocks]
    _link_oriented(gg, blocks)
    M.metrics_compute_blocks(gg, 0.0)
    Us = [torch.as_tensor(b["U0"], device="cuda").contiguous() for b in blocks]
    dt = min(g.cfl_dt(u, 0.4) for g, u in zip(gg, Us))
    assert max(float((dt * o).abs().max()) for o in M.rhs_blocks(gg, Us)) <= 1e-12
    for s in range(3):
        M.rk3_step_blocks(gg, Us, s * dt, dt)
    assert max(np.abs(u.cpu().numpy() - b["U0"]).max() for u, b in zip(Us, blocks)) <= 1e-12
    for g in gg:
        g.close()


@pytest.mark.parametrize("name", ["c3", "c4"])
def test_one_launch_ghost_fill_equals_the_three_passes_bit_for_bit(mods, cases, name):
    """meg6_rhs fills the ghost cells of a fully periodic block in ONE launch (k_ghost_periodic: the interior cell at the
    wrapped index); the staged calls run the three direction-ordered passes of k_ghost.  dQ/dt must be identical, edge and
    corner ghosts (viscous cross terms) included.  (c4: inflow / outflow faces, three passes on both sides -- the staged
    calls against meg6_rhs.  Composing the three passes per ghost cell for such faces too was measured SLOWER than the
    three launches, 0.086 against 0.075 ms per stage on C4, and is not in the library.)"""
    torch, O, M = mods
    wl = cases[name]
    g = M.Grid(wl)
    g.metrics_compute(0.0)
    U = torch.as_tensor(wl["U0"], device="cuda").contiguous()
    a = g.rhs(U)
    b = torch.empty_like(U)
    g.stage_prim(U)
    for d in range(3):
        g.stage_ghosts(0, d)
    g.stage_sweeps(U, 0, 0.0, out=b)
    assert torch.equal(a, b)
    g.close()
