"""Pins of the oracle's time-step formula, Eq. B.2 / B.3.  CPU only.

On a Cartesian mesh the un-hatted metrics are grad(xi) = (1/h_xi, 0, 0) etc., so the contravariant speeds are
|U| = |u|/h_xi, c |grad xi| = c/h_xi and Eq. B.2 has the closed form CFL min_d h_d / (|u_d| + c); Eq. B.3 adds
h_d^2 / (alpha mu) (alpha read as alpha^D = 4, R25 -- the reading is unpinned, the formula around it is pinned here).
"""
import numpy as np
import pytest

import workloads as W
from oracle import meg6_oracle as O
from test_oracle_moving import translating_box, TWO_PI

G = 1.4


def cart_box(n, h, **kw):
    L = tuple(n[d] * h[d] for d in range(3))
    X, E, Z = W._comp_coords(n, L)
    prm = W._base_params(n[0], n[1], n[2], period=[[L[0], 0, 0], [0, L[1], 0], [0, 0, L[2]]], **kw)
    return dict(params=prm, x=np.ascontiguousarray(X - L[0] / 2), y=np.ascontiguousarray(E - L[1] / 2),
                z=np.ascontiguousarray(Z - L[2] / 2))


@pytest.mark.parametrize("vel", [(0.9, 0.1, -0.05), (0.05, -1.7, 0.3), (0.0, 0.2, 2.5)])
def test_inviscid_dt_closed_form_uniform_flow(vel):
    """Eq. B.2: dt = CFL min_d h_d / (|u_d| + c); the three velocities make each direction the binding one in turn
    (h = 0.5, 0.25, 0.125 alone would always pick zeta)."""
    n, h = (12, 10, 14), (0.5, 0.25, 0.125)
    wl = cart_box(n, h)
    g = O.Grid(wl)
    g.metrics_compute(0.0)
    shp = (n[2], n[1], n[0])
    rho, p = 1.3, 0.9
    U = W.conservative(*(np.full(shp, v) for v in (rho, vel[0], vel[1], vel[2], p)))
    c = np.sqrt(G * p / rho)
    want = 0.37 * min(h[d] / (abs(vel[d]) + c) for d in range(3))
    assert g.cfl_dt(U, 0.37) == pytest.approx(want, rel=1e-12)


def test_dt_is_the_minimum_over_cells():
    """non-uniform state on the uniform mesh: Eq. B.2 cell by cell in numpy, and the cell that binds is a known one"""
    n, h = (10, 12, 11), (0.25, 0.25, 0.25)
    wl = cart_box(n, h)
    g = O.Grid(wl)
    g.metrics_compute(0.0)
    shp = (n[2], n[1], n[0])
    rng = np.random.default_rng(11)
    rho = 1.0 + 0.3 * rng.uniform(-1, 1, shp)
    u, v, w = (0.5 * rng.uniform(-1, 1, shp) for _ in range(3))
    p = 1.0 + 0.3 * rng.uniform(-1, 1, shp)
    w[7, 3, 5] = -3.0                                        # the binding cell and direction
    U = W.conservative(rho, u, v, w, p)
    c = np.sqrt(G * p / rho)
    per_cell = np.minimum(np.minimum(h[0] / (np.abs(u) + c), h[1] / (np.abs(v) + c)), h[2] / (np.abs(w) + c))
    assert np.unravel_index(per_cell.argmin(), shp) == (7, 3, 5)
    assert g.cfl_dt(U, 0.2) == pytest.approx(0.2 * per_cell.min(), rel=1e-12)


def test_viscous_dt_closed_form():
    """Eq. B.3: min( inviscid, min_d h_d^2 / (alpha mu) ), alpha = 4 (R25).  mu large: the viscous limit binds and picks
    the finest direction; mu small: the inviscid one binds."""
    n, h = (12, 10, 14), (0.5, 0.25, 0.125)
    shp = (n[2], n[1], n[0])
    U = W.conservative(*(np.full(shp, v) for v in (1.0, 0.3, 0.0, 0.0, 1.0)))
    c = np.sqrt(G)
    inv = min(h[0] / (0.3 + c), h[1] / c, h[2] / c)
    for mu in (0.5, 1e-4):
        wl = cart_box(n, h, viscous=1, mu_ref=mu, s_suth=-1.0)
        g = O.Grid(wl)
        g.metrics_compute(0.0)
        want = 0.2 * min(inv, min(hd * hd for hd in h) / (4.0 * mu))
        assert g.cfl_dt(U, 0.2) == pytest.approx(want, rel=1e-12)
    assert min(hd * hd for hd in h) / (4.0 * 0.5) < inv < min(hd * hd for hd in h) / (4.0 * 1e-4)


def test_viscous_dt_uses_sutherland_of_the_local_temperature():
    """mu of Eq. B.3 is mu(T) of the cell: one hot cell binds"""
    n, h = (10, 10, 10), (0.25, 0.25, 0.25)
    shp = (n[2], n[1], n[0])
    wl = cart_box(n, h, viscous=1, mu_ref=0.2, t_ref=1.0, s_suth=0.4, r_gas=1.0)
    g = O.Grid(wl)
    g.metrics_compute(0.0)
    rho = np.ones(shp)
    p = np.ones(shp)
    p[2, 6, 4] = 3.0                                          # T = 3
    U = W.conservative(rho, 0 * rho, 0 * rho, 0 * rho, p)
    mu_hot = 0.2 * 3.0 ** 1.5 * (1.0 + 0.4) / (3.0 + 0.4)
    want = 0.2 * min(0.25 / np.sqrt(G * 3.0), 0.25 ** 2 / (4.0 * mu_hot))
    assert g.cfl_dt(U, 0.2) == pytest.approx(want, rel=1e-12)


def test_stretched_mesh_binding_cell():
    """smoothly clustered periodic mesh along xi, x_xi = h (1 - A cos(2 pi (xi - xi0)/N)): the finest cell (centre at
    xi0 = 20.5) binds.  The metric is the consistent derivative (Eq. 41) of the 2-node-mean cell centres, i.e. the
    derivative of xc(xi) = (x(xi - 1/2) + x(xi + 1/2))/2 up to its fourth-order error h^4 f^(5)/720 ~ 1e-6 here."""
    ni, A, h, xi0 = 40, 0.6, 0.25, 20.5
    kk = TWO_PI / ni
    xi = np.arange(ni + 1.0)
    xn = h * (xi - A / kk * np.sin(kk * (xi - xi0)))
    Lx = xn[-1] - xn[0]
    Z, E, X = np.meshgrid(np.arange(11) * 0.5, np.arange(11) * 0.5, xn - xn[0] - Lx / 2, indexing="ij")
    prm = W._base_params(ni, 10, 10, period=[[Lx, 0, 0], [0, 5.0, 0], [0, 0, 5.0]])
    wl = dict(params=prm, x=np.ascontiguousarray(X), y=np.ascontiguousarray(E), z=np.ascontiguousarray(Z))
    g = O.Grid(wl)
    g.metrics_compute(0.0)
    shp = (10, 10, ni)
    U = W.conservative(*(np.full(shp, v) for v in (1.0, 0.4, 0.0, 0.0, 1.0)))
    x_xi = h * (1.0 - A * np.cos(kk * 0.5))                   # mean of x_xi at xi0 -+ 1/2
    want = 0.2 * x_xi / (0.4 + np.sqrt(G))
    assert g.cfl_dt(U, 0.2) == pytest.approx(want, rel=1e-4)
    nxt = h * (1.0 - A * (np.cos(kk * 0.5) + np.cos(kk * 1.5)) / 2)   # the neighbouring cells are coarser by more than that
    assert g.cfl_dt(U, 0.2) < 0.2 * nxt / (0.4 + np.sqrt(G)) * (1 - 1e-3)


def test_moving_mesh_dt_sees_the_relative_velocity():
    """Eq. B.2 with U = xi_t + u xi_x + ... (Eq. 4): on a mesh translating with velocity x_t the speed that
    counts is |u - x_t|.  Here the mesh moves with the flow along xi at t = 0 (relative speed zero there)."""
    om, c = 0.5, (0.25, 0.0, 0.0)
    n, h = (12, 10, 14), (0.25, 0.25, 0.25)
    wl, L = translating_box(n, h, c, om)
    g = O.Grid(wl)
    shp = (n[2], n[1], n[0])
    a = np.sqrt(G)
    for t in (0.0, 0.3):
        g.metrics_compute(t)
        xt = TWO_PI * om * np.cos(TWO_PI * om * t) * c[0]
        u = TWO_PI * om * c[0]                                  # = x_t at t = 0
        U = W.conservative(*(np.full(shp, v) for v in (1.0, u, 0.1, -0.2, 1.0)))
        want = 0.2 * min(h[0] / (abs(u - xt) + a), h[1] / (0.1 + a), h[2] / (0.2 + a))
        assert g.cfl_dt(U, 0.2) == pytest.approx(want, rel=1e-12)


def test_stored_time_steps_of_the_configs():
    """tests/golden/dt.json (written by tests/golden/make_dt.py, which calls only oracle/) holds Eq. B.2/B.3 of configs
    1-3 at t = 0; the closed forms above pin the function, this pins the stored numbers to it."""
    import json
    import os
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "dt.json")) as f:
        stored = json.load(f)
    for wl in (W.c1_vortex(n=32), W.c2_dynamic_freestream(n=64)):
        g = O.Grid(wl)
        g.metrics_compute(wl["t0"])
        assert g.cfl_dt(wl["U0"], wl["cfl"]) == pytest.approx(stored[wl["name"]], rel=1e-13)
    # config 1, order of magnitude by hand: h = 10/32, max |u| + c ~ 0.5 sqrt(1.4) + 0.8 + 1.18
    assert stored["c1_vortex_32"] == pytest.approx(0.5 * (10 / 32) / (0.5 * np.sqrt(1.4) + 0.8 + np.sqrt(1.4)), rel=0.25)
