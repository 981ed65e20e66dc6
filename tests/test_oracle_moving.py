"""Pins of the oracle's grid-velocity path: node velocities, time metrics Eq. 11, the interface time
metric in the Riemann flux (Eq. 24, 26-27), the GCL term Eq. 14 and the RK stage times of Eq. B.1 (R17).

CPU only.  The freestream test of tests/test_oracle_rhs.py cannot see xi_t (it cancels identically between the flux
and (1/J)_t Q); the references here are
  * a rigidly translating mesh (displacement mode = one constant vector): the grid velocity is the known vector
    2 pi omega cos(2 pi omega t) c everywhere, so xi_t = -x_t . grad(xi) is a closed form on a Cartesian mesh, the
    mesh does not deform ((1/J)_t = 0), and a flow observed from it is the same flow (Galilean shift of the frame);
  * the paper's own check, Sec. 8.2.2: a stationary isentropic vortex on a deforming mesh is an exact
    steady solution, whatever the mesh does;
  * third-order accuracy in time of SSP-RK3 (Eq. B.1) on a deforming mesh.
"""
import numpy as np
import pytest

import workloads as W
from oracle import meg6_oracle as O

TWO_PI = 2.0 * np.pi


def translating_box(n=(12, 10, 14), h=(0.5, 0.25, 0.125), c=(0.3, -0.2, 0.5), omega=0.7, wavy=0.0):
    """periodic box, spacing h (powers of two: exactly representable), every node displaced by s(t) c"""
    L = tuple(n[d] * h[d] for d in range(3))
    X, E, Z = W._comp_coords(n, L)
    x, y, z = X - L[0] / 2, E - L[1] / 2, Z - L[2] / 2
    if wavy:
        s = lambda a, l: np.sin(TWO_PI * a / l)
        x = x + wavy * s(E, L[1]) * s(Z, L[2])
        y = y + wavy * s(Z, L[2]) * s(X, L[0])
        z = z + wavy * s(X, L[0]) * s(E, L[1])
    one = np.ones_like(X)
    prm = W._base_params(n[0], n[1], n[2], period=[[L[0], 0, 0], [0, L[1], 0], [0, 0, L[2]]], moving=1, omega=omega)
    return dict(params=prm, x=np.ascontiguousarray(x), y=np.ascontiguousarray(y), z=np.ascontiguousarray(z),
                dx_mode=c[0] * one, dy_mode=c[1] * one, dz_mode=c[2] * one), L


def test_rigid_translation_time_metrics_closed_form():
    """Eq. 11 with the analytic grid velocity: on a Cartesian mesh translating as s(t) c the hatted
    metrics are the face areas (h_eta h_zeta, ...), so xi^_t = -x_t h_eta h_zeta with x_t = 2 pi omega cos(2 pi omega t) c_x
    at every cell centre AND at every interface, the boundary ones included (the ghost grid velocities are plain
    periodic copies); the mesh does not deform, so (1/J)_t of Eq. 14 vanishes."""
    n, h, c, om, t = (12, 10, 14), (0.5, 0.25, 0.125), (0.3, -0.2, 0.5), 0.7, 0.13
    wl, L = translating_box(n, h, c, om)
    g = O.Grid(wl)
    g.metrics_compute(t)
    s, sd = np.sin(TWO_PI * om * t), TWO_PI * om * np.cos(TWO_PI * om * t)
    xc0 = W.cell_centres(wl["x"])
    assert np.allclose(g.cell(14), xc0 + s * c[0], rtol=0, atol=1e-14)          # the mesh really is displaced
    area = (h[1] * h[2], h[0] * h[2], h[0] * h[1])
    for d in range(3):
        want = -sd * c[d] * area[d]
        assert np.allclose(g.cell(10 + d), want, rtol=1e-12, atol=0), d          # sign and 2 pi omega of Eq. 11 / P:166
        assert np.allclose(g.face(d, 10), want, rtol=1e-12, atol=0), d           # interfaces, first and last included
    assert np.abs(g.cell(13)).max() <= 1e-13 * abs(sd) * max(area)               # rigid motion: no volume change


def test_rigid_translation_of_a_wavy_mesh():
    """The same on a curved mesh: x_t is still the one known vector, so xi^_t = -(x_t . xi^_x) with the oracle's own
    static metrics, cell by cell and (by linearity of the interpolation, Eq. 38) interface by interface; periodicity
    of the interface arrays (first interface = last interface) sees any offset in the ghost grid velocities."""
    om, t, c = 1.3, 0.21, (0.25, 0.4, -0.35)
    wl, L = translating_box((12, 12, 12), (0.5, 0.5, 0.5), c, om, wavy=0.08)
    g = O.Grid(wl)
    g.metrics_compute(t)
    sd = TWO_PI * om * np.cos(TWO_PI * om * t)
    for d in range(3):
        want = -sd * sum(c[q] * g.cell(3 * d + q) for q in range(3))
        assert np.allclose(g.cell(10 + d), want, rtol=1e-12, atol=1e-15)
        wantf = -sd * sum(c[q] * g.face(d, 3 * d + q) for q in range(3))
        f = g.face(d, 10)
        assert np.allclose(f, wantf, rtol=1e-11, atol=1e-14)
        first = np.take(f, 0, axis=2 - d)
        last = np.take(f, -1, axis=2 - d)
        assert np.allclose(first, last, rtol=1e-12, atol=1e-15)
    assert np.abs(g.cell(13)).max() <= 1e-12 * abs(sd) * np.abs(g.cell(0)).max()


def vortex_at(xc, yc, x0, y0, L):
    """stationary isentropic vortex (strength 5) centred at (x0, y0) on the periodic box of side L"""
    xs = (xc - x0 + L / 2) % L - L / 2
    ys = (yc - y0 + L / 2) % L - L / 2
    return W.conservative(*W.isentropic_vortex(xs, ys, mach=0.0))


def deforming_vortex_mesh(n, L=10.0, amp=0.45):
    """mesh of Sec. 8.2.1-8.2.2 in form (Eq. 49): x = xi + A sin(2 pi omega t) sin sin, periodic"""
    x, y, z = W.wavy_periodic_grid(n, L, 0.0)
    X, E, Z = x + L / 2, y + L / 2, z + L / 2
    s = lambda a: np.sin(TWO_PI * a / L)
    prm = W._base_params(n, n, n, period=[[L, 0, 0], [0, L, 0], [0, 0, L]], moving=1, omega=1.0)
    return dict(params=prm, x=x, y=y, z=z, dx_mode=amp * s(E) * s(Z), dy_mode=amp * s(Z) * s(X),
                dz_mode=amp * s(X) * s(E))


def run_vortex(wl, U, T, cfl=0.4):
    g = O.Grid(wl)
    g.metrics_compute(0.0)
    dt0 = g.cfl_dt(U, cfl)
    ns = int(np.ceil(T / dt0))
    dt = T / ns
    for s in range(ns):
        g.rk3_step(U, s * dt, dt)
    g.metrics_compute(T)
    return g


@pytest.mark.parametrize("centre", [(0.0, 0.0), (5.0, 5.0)])
def test_stationary_vortex_on_deforming_mesh(centre):
    """Sec. 8.2.2: a stationary vortex stays what it is while the mesh deforms under it.  After a quarter
    period (the mesh at its largest displacement, 1.4 cells at 32^3) the solution at the DISPLACED cell centres is the
    exact vortex there: error at the level of the static-mesh run, second-order convergence.  A wrong sign of
    xi_t (Eq. 11), a grid velocity without its 2 pi omega or a stage-3 geometry at t + dt instead of t + dt/2
    (R17) each leave an O(displacement x gradient) error, 10-100 times the bound.  centre (5, 5): the vortex sits on
    the periodic corner of the box, so the ghost coordinates and ghost grid velocities carry the core."""
    L, T = 10.0, 0.25
    errs, stat = [], []
    for n in (16, 32):
        wl = deforming_vortex_mesh(n, L)
        xc, yc = W.cell_centres(wl["x"]), W.cell_centres(wl["y"])
        U = vortex_at(xc, yc, centre[0], centre[1], L)
        g = run_vortex(wl, U, T)
        xe, ye = g.cell(14), g.cell(15)
        assert np.abs(xe - xc).max() > 0.3                       # the mesh moved
        ex = vortex_at(xe, ye, centre[0], centre[1], L)
        errs.append(np.sqrt(np.mean((U[0] - ex[0]) ** 2)))
        # the same vortex on the mesh at rest
        ws = dict(wl, params=dict(wl["params"], moving=0))
        Us = vortex_at(xc, yc, centre[0], centre[1], L)
        run_vortex(ws, Us, T)
        stat.append(np.sqrt(np.mean((Us[0] - vortex_at(xc, yc, centre[0], centre[1], L)[0]) ** 2)))
    rate = np.log2(errs[0] / errs[1])
    assert rate > 1.9, (errs, rate)
    assert errs[1] < 4.0 * stat[1] + 1e-5 and errs[1] < 4e-4, (errs, stat)


def test_vortex_seen_from_a_translating_mesh_is_the_advected_vortex():
    """Galilean shift of the observer: a vortex advected at Mach 0.5 on a Cartesian mesh that translates rigidly
    (mode = constant vector, peak mesh speed 1.6 a_inf along a diagonal) is the exact translated vortex at the moving
    cell centres.  Uniform flow cannot see this (xi_t cancels); the vortex core does."""
    L, T, n = 10.0, 0.5, 32
    x, y, z = W.wavy_periodic_grid(n, L, 0.0)
    one = np.ones_like(x)
    c = (0.35, -0.25, 0.2)
    prm = W._base_params(n, n, n, period=[[L, 0, 0], [0, L, 0], [0, 0, L]], moving=1, omega=0.8)
    wl = dict(params=prm, x=x, y=y, z=z, dx_mode=c[0] * one, dy_mode=c[1] * one, dz_mode=c[2] * one)
    xc, yc = W.cell_centres(x), W.cell_centres(y)
    U = W.conservative(*W.isentropic_vortex(xc, yc, mach=0.5))
    g = run_vortex(wl, U, T)
    s = np.sin(TWO_PI * 0.8 * T)
    assert np.allclose(g.cell(14), xc + s * c[0], atol=1e-13)
    shift = 0.5 * np.sqrt(1.4) * T
    xs = (g.cell(14) - shift + L / 2) % L - L / 2
    ys = (g.cell(15) + L / 2) % L - L / 2
    ex = W.conservative(*W.isentropic_vortex(xs, ys, mach=0.5))
    err = np.sqrt(np.mean((U[0] - ex[0]) ** 2))
    # static-mesh run of tests/test_oracle_rhs.py::test_isentropic_vortex_advection_order: < 3e-4 at 32^3
    assert err < 4e-4, err


def test_rk3_is_third_order_in_time_on_a_deforming_mesh():
    """Eq. B.1 with the geometry of each stage at its own time t, t + dt, t + dt/2 (R17): the step-size
    error of a smooth flow on a strongly deforming mesh falls as dt^3 (self-convergence on one mesh: the spatial error
    is common to all runs).  A stage geometry taken at another time degrades this to first order."""
    n, L, T = 12, 10.0, 0.32
    wl = deforming_vortex_mesh(n, L, amp=0.6)
    xc, yc, zc = (W.cell_centres(wl[k]) for k in ("x", "y", "z"))
    k = TWO_PI / L
    U0 = W.conservative(1 + 0.1 * np.sin(k * xc) * np.cos(k * yc), 0.3 + 0.1 * np.sin(k * yc + 0.5),
                        -0.2 + 0.1 * np.cos(k * zc), 0.1 * np.sin(k * (xc + zc)), 1 + 0.05 * np.cos(k * yc) * np.sin(k * zc))
    g = O.Grid(wl)
    sols = {}
    for ns in (2, 4, 8, 32):
        U = U0.copy()
        dt = T / ns
        for s in range(ns):
            g.rk3_step(U, s * dt, dt)
        sols[ns] = U
    e = [np.abs(sols[ns] - sols[32]).max() for ns in (2, 4, 8)]
    rates = np.log2(np.array(e[:-1]) / np.array(e[1:]))
    assert np.all(rates > 2.6), (e, rates)
