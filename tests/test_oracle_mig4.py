"""Pins of the oracle's MIG4 variant (scheme = 1): implicit fourth-order gradients IG4, Eq. 18 (R2),
used wherever MEG6 uses E6 -- reconstruction, viscous flux and metrics.  CPU only.

The paper does not say where the tridiagonal systems end; reading R26: a system spans every cell of
the padded grid line whose right-hand side exists and is closed at both ends with the explicit fourth-order
difference of Eq. D.2.  The pins: an independent dense-matrix restatement of that system, polynomial exactness
and fourth-order convergence, machine-zero freestream (the metric identity holds for any commuting line
operators), convergence of the assembled right-hand side to the analytic Navier-Stokes terms."""
import numpy as np
import pytest

import workloads as W
from oracle import meg6_oracle as O

ALPHA = 5.0 / 14.0


def dense_ig4(f):
    """Eq. 18 with the Eq. D.2 closure as ONE dense linear system (numpy.linalg.solve)."""
    n = f.size
    m = n - 4                      # unknowns at cells 2 .. n-3
    A = np.zeros((m, m))
    r = np.zeros(m)
    c4 = lambda i: 2.0 / 3.0 * (f[i + 1] - f[i - 1]) - 1.0 / 12.0 * (f[i + 2] - f[i - 2])
    for q in range(m):
        i = q + 2
        if q in (0, m - 1):
            A[q, q] = 1.0
            r[q] = c4(i)
        else:
            A[q, q - 1] = A[q, q + 1] = ALPHA
            A[q, q] = 1.0
            r[q] = (2 + ALPHA) / 3 * (f[i + 1] - f[i - 1]) + (4 * ALPHA - 1) / 12 * (f[i + 2] - f[i - 2])
    out = np.full(n, np.nan)
    out[2:n - 2] = np.linalg.solve(A, r)
    return out


def test_ig4_equals_dense_solve_of_eq18():
    rng = np.random.default_rng(18)
    f = rng.standard_normal(37)
    a, b = O.line_op("IG4", f), dense_ig4(f)
    assert np.array_equal(np.isnan(a), np.isnan(b))
    assert np.nanmax(np.abs(a - b)) <= 1e-13


def test_ig4_is_exact_to_degree_4_and_fourth_order():
    i = np.arange(40.0)
    for k in range(5):
        d = O.line_op("IG4", (i / 10) ** k)
        ex = k * (i / 10) ** (k - 1) / 10 if k else 0 * i
        assert np.nanmax(np.abs(d - ex)) <= 1e-12
    assert np.nanmax(np.abs(O.line_op("IG4", (i / 10) ** 5) - 5 * (i / 10) ** 4 / 10)) > 1e-6   # not degree 5
    errs = []
    for n in (32, 64, 128):
        x = np.arange(n + 8) * (2 * np.pi / n)
        d = O.line_op("IG4", np.sin(x)) / (2 * np.pi / n)
        errs.append(np.nanmax(np.abs(d - np.cos(x))[8:-8]))
    rates = np.log2(np.array(errs[:-1]) / np.array(errs[1:]))
    assert np.all(rates > 3.8), (errs, rates)


def test_ig4_beats_e6_nowhere_but_is_implicit():
    """sanity of the variant switch: the two gradient schemes differ at truncation level, not at round-off."""
    x = np.arange(48) * 0.3
    a, b = O.line_op("IG4", np.sin(x)), O.line_op("D1", np.sin(x))
    d = np.nanmax(np.abs(a - b))
    assert 1e-7 < d < 1e-2


def _with_scheme(wl, scheme=1):
    wl = dict(wl)
    wl["params"] = dict(wl["params"], scheme=scheme)
    return wl


@pytest.mark.parametrize("kind", ["wavy", "random"])
def test_mig4_freestream_static(kind):
    wl = _with_scheme(W.freestream_static(20, kind))
    g = O.Grid(wl)
    g.metrics_compute(0.0)
    dt = g.cfl_dt(wl["U0"], 0.2)
    assert np.abs(dt * g.rhs(wl["U0"])).max() <= 1e-12
    U = wl["U0"].copy()
    for s in range(5):
        g.rk3_step(U, s * dt, dt)
    assert np.abs(U[0] - 1).max() <= 1e-12 and np.abs(U[2] / U[0]).max() <= 1e-12


def test_mig4_freestream_dynamic_and_nonperiodic():
    wl = _with_scheme(W.c2_dynamic_freestream(n=16, steps=6))
    U = wl["U0"].copy()
    g = O.Grid(wl)
    g.metrics_compute(0.0)
    dt = g.cfl_dt(U, 0.2)
    t = 0.0
    for s in range(6):
        g.rk3_step(U, t, dt)
        t += dt
    g.metrics_compute(t)
    assert np.abs(dt * g.rhs(U)).max() <= 1e-12
    wl = _with_scheme(W.c4_jet(ni=24, nj=14, nk=12))
    shape = wl["U0"].shape[1:]
    one = np.ones(shape)
    U0 = W.conservative(one, 0.3 * one, -0.2 * one, 0.1 * one, one / 1.4)
    wl["inflow"] = {0: np.stack([np.ones(shape[:2]), 0.3 * np.ones(shape[:2]), -0.2 * np.ones(shape[:2]),
                                 0.1 * np.ones(shape[:2]), np.ones(shape[:2]) / 1.4])}
    wl["sigma"] = None
    g = O.Grid(wl)
    g.metrics_compute(0.0)
    r = g.rhs(U0)
    assert np.abs(wl["dt"] * r).max() <= 1e-12


@pytest.mark.parametrize("viscous", [0, 1])
def test_mig4_rhs_converges_to_analytic_navier_stokes(viscous):
    """Same reference as tests/test_oracle_rhs.py (spectral evaluation of the analytic right-hand side on a wavy
    periodic mesh): the MIG4 assembly converges at the order the paper states for non-linear problems."""
    from test_oracle_rhs import spectral_rhs, smooth_state, relmax, l2
    L = 10.0
    errs = []
    for n in (16, 32):
        x, y, z = W.wavy_periodic_grid(n, L, 0.25)
        xc, yc, zc = W.cell_centres(x), W.cell_centres(y), W.cell_centres(z)
        prim = smooth_state(xc, yc, zc, L)
        prm = W._base_params(n, n, n, period=[[L, 0, 0], [0, L, 0], [0, 0, L]], viscous=viscous,
                             mu_ref=0.05, s_suth=0.4, t_ref=1.0, r_gas=1.0, scheme=1)
        g = O.Grid(dict(params=prm, x=x, y=y, z=z))
        g.metrics_compute(0.0)
        num = g.rhs(W.conservative(*prim))
        ref = spectral_rhs(xc, yc, zc, L, prim, prm)
        errs.append(l2(num - ref) / relmax(ref))
    errs = np.array(errs)
    assert np.all(errs[1] < 1e-3), errs
    assert np.all(np.log2(errs[0] / errs[1]) > 1.8), errs


def test_mig4_conservation_on_periodic_mesh_up_to_the_closure():
    """R26 closes every line system inside the ghost layers, so the periodic images of an interface see slightly
    different implicit gradients: the telescoping sum of Eq. 8-9 is no longer zero to round-off but to the closure
    influence (decay 0.42 per cell x fourth-order closure mismatch).  Bounded here so that a regression shows."""
    wl = _with_scheme(W.c1_vortex(n=16))
    g = O.Grid(wl)
    g.metrics_compute(0.0)
    r = g.rhs(wl["U0"])
    rj = g.cell(9)
    tot = (r * rj).reshape(5, -1).sum(axis=1)
    scale = (np.abs(r) * rj).reshape(5, -1).sum(axis=1)
    print("relative conservation defect:", np.abs(tot) / scale)
    assert np.all(np.abs(tot) <= 5e-4 * scale)
