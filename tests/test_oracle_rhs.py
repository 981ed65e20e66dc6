"""Pins of the oracle's assembled right-hand side and time stepping.

CPU only.  The references are: machine-zero freestream residuals with the paper's magnitudes (Table 2,
Fig. 10c) and the App. D negative control; telescoping conservation; a spectral (numpy FFT) evaluation of
the analytic Navier-Stokes right-hand side in physical space via the chain rule; the closed-form RK3
amplification factor; the exact (translated) isentropic vortex.
"""
import numpy as np
import pytest

import workloads as W
from oracle import meg6_oracle as O


def relmax(a):
    return np.abs(a).reshape(a.shape[0], -1).max(axis=1)


def l2(a):
    return np.sqrt((a ** 2).reshape(a.shape[0], -1).mean(axis=1))


# ------------------------------------------------------------------ P2 freestream
@pytest.mark.parametrize("kind", ["wavy", "random"])
def test_freestream_static_and_negative_control(kind):
    """Sec. 8.1.1 / Table 2: conservative consistent metrics keep uniform flow to machine zero;
    the App. D non-conservative metrics do not (1e-3..1e-1)."""
    wl = W.freestream_static(20, kind)
    U0 = wl["U0"]
    g = O.Grid(wl)
    g.metrics_compute(0.0)
    dt = g.cfl_dt(U0, 0.2)
    assert np.abs(dt * g.rhs(U0)).max() <= 1e-12
    U = U0.copy()
    for s in range(10):
        g.rk3_step(U, s * dt, dt)
    rho, v, w = U[0], U[2] / U[0], U[3] / U[0]
    assert np.abs(rho - 1).max() <= 1e-12 and np.abs(v).max() <= 1e-12 and np.abs(w).max() <= 1e-12
    bad = O.Grid(wl, metric_form=1)
    bad.metrics_compute(0.0)
    Ub = U0.copy()
    for s in range(10):
        bad.rk3_step(Ub, s * dt, dt)
    assert np.abs(Ub[2] / Ub[0]).max() > (1e-6 if kind == "wavy" else 1e-3)


def test_freestream_dynamic_mesh_gcl():
    """Sec. 8.2.1 / Fig. 10c: uniform flow on a deforming jittered mesh stays uniform to
    <= 1e-12 with xi_t and (1/J)_t from Eq. 11/14."""
    wl = W.c2_dynamic_freestream(n=16, steps=12)
    U = wl["U0"].copy()
    g = O.Grid(wl)
    g.metrics_compute(0.0)
    dt = g.cfl_dt(U, 0.2)
    t = 0.0
    for s in range(wl["steps"]):
        g.rk3_step(U, t, dt)
        t += dt
    g.metrics_compute(t)
    assert np.abs(dt * g.rhs(U)).max() <= 1e-12
    p = 0.4 * (U[4] - 0.5 * (U[1] ** 2 + U[2] ** 2 + U[3] ** 2) / U[0])
    p0 = 1.0 / (1.4 * 0.25)
    dev = max(np.abs(U[0] - 1).max(), np.abs(U[1] / U[0] - 1).max(), np.abs(U[2] / U[0]).max(),
              np.abs(U[3] / U[0]).max(), np.abs(p - p0).max() / p0)
    assert dev <= 1e-12
    # the mesh really moves and the GCL term is not trivially zero
    assert np.abs(g.cell(13)).max() > 1e-6 and np.abs(g.cell(10)).max() > 1e-6


def test_freestream_nonperiodic_stretched_mesh_R13():
    """R13: ghost coordinates by linear extrapolation + interior formulas everywhere keep the metric
    identity on a non-periodic stretched mesh; uniform inflow/outflow data => RHS at round-off."""
    wl = W.c4_jet(ni=24, nj=16, nk=16)
    prm = dict(wl["params"], viscous=0)
    n = (16, 16, 24)
    rho, u, v, w, p = np.ones(n), 0.4 * np.ones(n), 0.2 * np.ones(n), -0.1 * np.ones(n), np.ones(n) / 1.4
    U0 = W.conservative(rho, u, v, w, p)
    pin = np.zeros((5, 16, 16))
    for f, val in enumerate((1.0, 0.4, 0.2, -0.1, 1 / 1.4)):
        pin[f] = val
    wl2 = dict(wl, params=prm, U0=U0, inflow={0: pin}, sigma=None)
    g = O.Grid(wl2)
    g.metrics_compute(0.0)
    dt = g.cfl_dt(U0, 0.2)
    assert np.abs(dt * g.rhs(U0)).max() <= 1e-12


# ------------------------------------------------------------------ P8 conservation
@pytest.mark.parametrize("viscous", [0, 1])
def test_discrete_conservation_on_periodic_mesh(viscous):
    """Eq. 8-9: sum over cells of (1/J) dQ/dt telescopes to zero on a static periodic mesh."""
    wl = W.c3_tgv(n=16) if viscous else W.c1_vortex(n=16)
    g = O.Grid(wl)
    g.metrics_compute(0.0)
    r = g.rhs(wl["U0"])
    rj = g.cell(9)
    tot = (r * rj).reshape(5, -1).sum(axis=1)
    scale = (np.abs(r) * rj).reshape(5, -1).sum(axis=1) + 1e-300
    assert np.all(np.abs(tot) <= 1e-12 * np.maximum(scale, 1.0))


# ------------------------------------------------------------------ P11 spectral reference
def spectral_rhs(xc, yc, zc, L, prim, cfg):
    """Analytic dQ/dt = -div(F - Fv) of Eq. 1 in physical space, evaluated at the cell centres with FFT
    derivatives along the (periodic, unit-spaced) computational coordinates and the chain rule with the
    inverse of the spectral coordinate Jacobian.  Independent of every stencil in the oracle."""
    nk, nj, ni = xc.shape
    n = (ni, nj, nk)

    def dcomp(f, d, linear=0.0):
        ax = 2 - d
        k = 2j * np.pi * np.fft.fftfreq(n[d])
        shp = [1, 1, 1]
        shp[ax] = n[d]
        fh = np.fft.fft(f, axis=ax) * k.reshape(shp)
        if n[d] % 2 == 0:
            sl = [slice(None)] * 3
            sl[ax] = n[d] // 2
            fh[tuple(sl)] = 0.0
        return np.real(np.fft.ifft(fh, axis=ax)) + linear
    idx = np.meshgrid(np.arange(nk), np.arange(nj), np.arange(ni), indexing="ij")
    A = np.empty((3, 3) + xc.shape)    # A[c][d] = d x_c / d xi_d
    for c, X in enumerate((xc, yc, zc)):
        h = L / n[c]
        per = X - h * idx[2 - c]
        for d in range(3):
            A[c, d] = dcomp(per, d, h if c == d else 0.0)
    Ai = np.linalg.inv(np.moveaxis(A, (0, 1), (-2, -1)))   # Ai[..., d, c] = d xi_d / d x_c

    def grad(f):
        gc = [dcomp(f, d) for d in range(3)]
        return [sum(Ai[..., d, c] * gc[d] for d in range(3)) for c in range(3)]
    rho, u, v, w, p = prim
    gam = cfg["gamma"]
    E = p / (gam - 1) + 0.5 * rho * (u * u + v * v + w * w)
    vel = (u, v, w)
    Fc = []     # Fc[c][q]: flux of equation q along x_c
    if cfg["viscous"]:
        T = p / (rho * cfg["r_gas"])
        r_ = T / cfg["t_ref"]
        mu = cfg["mu_ref"] * r_ ** 1.5 * (cfg["t_ref"] + cfg["s_suth"]) / (T + cfg["s_suth"]) if cfg["s_suth"] >= 0 \
            else cfg["mu_ref"] + 0 * T
        kap = mu * gam * cfg["r_gas"] / ((gam - 1) * cfg["prandtl"])
        gu, gv, gw, gT = grad(u), grad(v), grad(w), grad(T)
        gvel = (gu, gv, gw)
        div = gu[0] + gv[1] + gw[2]
        tau = [[mu * (gvel[a][b] + gvel[b][a]) - (2.0 / 3.0 * mu * div if a == b else 0.0) for b in range(3)]
               for a in range(3)]
    for c in range(3):
        f = [rho * vel[c], rho * u * vel[c], rho * v * vel[c], rho * w * vel[c], (E + p) * vel[c]]
        f[1 + c] = f[1 + c] + p
        if cfg["viscous"]:
            for a in range(3):
                f[1 + a] = f[1 + a] - tau[a][c]
            f[4] = f[4] - (u * tau[0][c] + v * tau[1][c] + w * tau[2][c] + kap * gT[c])
        Fc.append(f)
    out = np.zeros((5,) + xc.shape)
    for q in range(5):
        for c in range(3):
            out[q] -= grad(Fc[c][q])[c]
    return out


def smooth_state(xc, yc, zc, L):
    k = 2 * np.pi / L
    rho = 1.0 + 0.15 * np.sin(k * xc + 0.3) * np.cos(k * yc) + 0.05 * np.cos(k * zc + 1.0)
    u = 0.5 + 0.2 * np.sin(k * yc + 0.5) * np.cos(k * zc)
    v = -0.3 + 0.2 * np.cos(k * xc) * np.sin(k * zc + 0.2)
    w = 0.2 + 0.2 * np.sin(k * xc + 1.1) * np.sin(k * yc)
    p = 1.0 + 0.1 * np.cos(k * xc + 0.7) * np.cos(k * yc + 0.1) * np.cos(k * zc)
    return rho, u, v, w, p


@pytest.mark.parametrize("wavy,viscous", [(False, 0), (True, 0), (True, 1)])
def test_rhs_converges_to_analytic_navier_stokes(wavy, viscous):
    """The assembled RHS (metrics, gradients, reconstruction, HLLC, alpha-damping, Eq. 9 assembly) must
    converge to the analytic -div(F - Fv) for smooth data: second order for the non-linear system
    (point-value reconstruction of P, then F(P); "fourth order for linear, second
    for non-linear"), with small absolute error.  A wrong sign, index or transposed metric gives O(1)."""
    L = 10.0
    errs = []
    for n in (16, 32):
        x, y, z = W.wavy_periodic_grid(n, L, 0.25 if wavy else 0.0)
        xc, yc, zc = W.cell_centres(x), W.cell_centres(y), W.cell_centres(z)
        prim = smooth_state(xc, yc, zc, L)
        prm = W._base_params(n, n, n, period=[[L, 0, 0], [0, L, 0], [0, 0, L]], viscous=viscous,
                             mu_ref=0.05, s_suth=0.4, t_ref=1.0, r_gas=1.0)
        wl = dict(params=prm, x=x, y=y, z=z)
        g = O.Grid(wl)
        g.metrics_compute(0.0)
        U = W.conservative(*prim)
        num = g.rhs(U)
        ref = spectral_rhs(xc, yc, zc, L, prim, prm)
        scale = relmax(ref)
        errs.append(l2(num - ref) / scale)
        linf = relmax(num - ref) / scale
    errs = np.array(errs)
    rate = np.log2(errs[0] / errs[1])
    # L2 norm for the rate: the MP limiter clips isolated smooth extrema, which makes L-infinity noisy
    assert np.all(errs[1] < 5e-4) and np.all(linf < 1.5e-2), (errs, linf)
    assert np.all(rate > 1.8), (errs, rate)


def test_viscous_terms_alone_converge():
    """difference (viscous RHS - inviscid RHS) against the spectral viscous divergence alone, so that the
    alpha-damping path is not hidden behind the larger inviscid terms."""
    L = 10.0
    errs = []
    for n in (16, 32):
        x, y, z = W.wavy_periodic_grid(n, L, 0.25)
        xc, yc, zc = W.cell_centres(x), W.cell_centres(y), W.cell_centres(z)
        prim = smooth_state(xc, yc, zc, L)
        U = W.conservative(*prim)
        res = []
        for viscous in (0, 1):
            prm = W._base_params(n, n, n, period=[[L, 0, 0], [0, L, 0], [0, 0, L]], viscous=viscous,
                                 mu_ref=0.05, s_suth=0.4, t_ref=1.0, r_gas=1.0)
            g = O.Grid(dict(params=prm, x=x, y=y, z=z))
            g.metrics_compute(0.0)
            res.append((g.rhs(U), spectral_rhs(xc, yc, zc, L, prim, prm)))
        num = res[1][0] - res[0][0]
        ref = res[1][1] - res[0][1]
        errs.append(l2(num[1:] - ref[1:]) / relmax(ref[1:]))
        assert np.abs(num[0]).max() < 1e-12   # no viscous mass flux (Eq. 3)
    errs = np.array(errs)
    assert np.all(errs[1] < 5e-3) and np.all(np.log2(errs[0] / errs[1]) > 1.8), errs


# ------------------------------------------------------------------ P10 RK3
def test_rk3_amplification_factor_closed_form():
    """Eq. B.1 on dQ/dt = -sigma (Q - Qref) (fluid at rest, uniform => Res = 0): one step
    multiplies Q - Qref by 1 + z + z^2/2 + z^3/6, z = -sigma dt."""
    n = 12
    x, y, z = W.wavy_periodic_grid(n, 6.0, 0.0)
    prm = W._base_params(n, n, n, period=[[6.0, 0, 0], [0, 6.0, 0], [0, 0, 6.0]])
    shape = (n, n, n)
    one = np.ones(shape)
    Uref = W.conservative(one, 0 * one, 0 * one, 0 * one, one)
    U = W.conservative(1.3 * one, 0 * one, 0 * one, 0 * one, 1.2 * one)
    sigma = 0.7 * one
    g = O.Grid(dict(params=prm, x=x, y=y, z=z, sigma=sigma, U_ref=Uref))
    g.metrics_compute(0.0)
    dt = 0.4
    zz = -0.7 * dt
    amp = 1 + zz + zz ** 2 / 2 + zz ** 3 / 6
    U1 = U.copy()
    g.rk3_step(U1, 0.0, dt)
    assert np.allclose(U1 - Uref, amp * (U - Uref), rtol=1e-13, atol=1e-14)


# ------------------------------------------------------------------ P7 vortex
@pytest.mark.parametrize("wavy", [False, True])
def test_isentropic_vortex_advection_order(wavy):
    """Sec. 8.1.2-style check: the advected isentropic vortex is an exact solution; the
    scheme converges at order >= 2 (fourth order for linear, second for non-linear)."""
    L, T = 10.0, 0.5
    errs = []
    for n in (16, 32):
        wl = W.c1_vortex(n=n, wavy=wavy)
        g = O.Grid(wl)
        g.metrics_compute(0.0)
        U = wl["U0"].copy()
        dt0 = g.cfl_dt(U, 0.4)
        ns = int(np.ceil(T / dt0))
        dt = T / ns
        for s in range(ns):
            g.rk3_step(U, s * dt, dt)
        xc, yc = W.cell_centres(wl["x"]), W.cell_centres(wl["y"])
        shift = 0.5 * np.sqrt(1.4) * T
        xs = (xc - shift + L / 2) % L - L / 2
        ex = W.conservative(*W.isentropic_vortex(xs, yc))
        errs.append(np.sqrt(np.mean((U[0] - ex[0]) ** 2)))
    rate = np.log2(errs[0] / errs[1])
    assert rate > 1.9, (errs, rate)
    assert errs[1] < 3e-4


# ------------------------------------------------------------------ branch record (per-interface E.1 / Eq. 26 decisions)
def test_branch_record_matches_counters_and_hllc_regimes():
    """The per-interface branch record the parity tests compare with the GPU's (bits 0-9: E.1 failed per characteristic
    component and side, bits 10-11: branch of Eq. 26, bit 12: tie): its population count is the limiter counter; a
    uniform supersonic stream takes branch 0 (S_L >= 0: F_L) everywhere along +x and branch 3 against it, a subsonic one
    the star branches 1 / 2 by the sign of S* = the contravariant velocity; fluid at rest is a tie (R10)."""
    n = 12
    x, y, z = W.wavy_periodic_grid(n, 6.0, 0.0)
    prm = W._base_params(n, n, n, period=[[6.0, 0, 0], [0, 6.0, 0], [0, 0, 6.0]])
    one = np.ones((n, n, n))
    g = O.Grid(dict(params=prm, x=x, y=y, z=z))
    g.metrics_compute(0.0)
    g.branch_masks_enable(True)
    a = np.sqrt(1.4)
    for u, want_x, tie in ((2.0 * a, 0, 0), (-2.0 * a, 3, 0), (0.5 * a, 1, 0), (-0.5 * a, 2, 0), (0.0, None, 1)):
        g.rhs(W.conservative(one, u * one, 0.3 * a * one, 0 * one, one))
        m = g.branch_mask(0)
        assert np.all((m & 0x3FF) == 0)                          # uniform state: nothing limited
        assert np.all(((m >> 12) & 1) == tie)
        if want_x is not None:
            assert np.all(((m >> 10) & 3) == want_x), (u, np.unique((m >> 10) & 3))
        assert np.all(((g.branch_mask(1) >> 10) & 3) == 1)       # v = +0.3 a: subsonic, S* > 0 along eta
        assert np.all(((g.branch_mask(2) >> 12) & 1) == 1)       # w = 0: tie along zeta
    # a state with a density step: some components limited; bits = counters
    wl = W.c1_vortex(n=16)
    U = wl["U0"].copy()
    U[0, :, :, 8:] *= 1.5
    g2 = O.Grid(wl)
    g2.metrics_compute(0.0)
    g2.branch_masks_enable(True)
    l0, t0 = g2.limiter_stats()
    g2.rhs(U)
    l1, t1 = g2.limiter_stats()
    bits = sum(int(((g2.branch_mask(d) >> b) & 1).sum()) for d in range(3) for b in range(10))
    assert l1 - l0 == bits > 0
    assert t1 - t0 == 10 * sum(g2.branch_mask(d).size for d in range(3))
