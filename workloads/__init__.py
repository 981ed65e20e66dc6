"""Seeded synthetic inputs for the five BASELINE.json configs (and reduced-size variants).

This module serves BOTH the CPU oracle and the CUDA path and therefore holds none of the method's
arithmetic: it only builds node coordinates, initial states and boundary data (numpy, seeded with
numpy.random.default_rng).  The inputs are synthetic stand-ins with the shapes, sizes and value ranges of
the paper's workloads; the paper's own
grids and data are not in the container and nothing here reproduces them.

Every generator returns a dict:
  params   plain dict with the fields of the params struct (ni,nj,nk,periodic,period,viscous,...)
  x,y,z    node coordinates, shape (nk+1, nj+1, ni+1), float64
  dx_mode,dy_mode,dz_mode   node displacement modes (moving meshes only)
  U0       initial conservative state, shape (5, nk, nj, ni)
  inflow   {face: P_in (5, n2, n1)}       (optional)
  sigma, U_ref                            (optional sponge)
  dt (None: CFL-based, from `cfl` by Eq. B.2/B.3 on the solver's side), cfl, steps, name, t0
"""
import hashlib

import numpy as np

GAMMA = 1.4


def cell_centres(a):
    """8-vertex mean of a node array -- geometry preprocessing for the initial data."""
    return 0.125 * (a[:-1, :-1, :-1] + a[:-1, :-1, 1:] + a[:-1, 1:, :-1] + a[:-1, 1:, 1:]
                    + a[1:, :-1, :-1] + a[1:, :-1, 1:] + a[1:, 1:, :-1] + a[1:, 1:, 1:])


def conservative(rho, u, v, w, p, gamma=GAMMA):
    """(rho,u,v,w,p) -> Q of Eq. 5; input packing only."""
    E = p / (gamma - 1.0) + 0.5 * rho * (u * u + v * v + w * w)
    return np.ascontiguousarray(np.stack([rho, rho * u, rho * v, rho * w, E]))


def sha256(*arrays):
    h = hashlib.sha256()
    for a in arrays:
        h.update(np.ascontiguousarray(a).tobytes())
    return h.hexdigest()


def _base_params(ni, nj, nk, **kw):
    p = dict(ni=ni, nj=nj, nk=nk, periodic=[1, 1, 1], period=[[0.0] * 3 for _ in range(3)], scheme=0,
             viscous=0, gamma=GAMMA, r_gas=1.0, prandtl=0.71, mu_ref=0.0, t_ref=1.0, s_suth=-1.0,
             mp_alpha=4.0, moving=0, omega=0.0, bc=[0] * 6, p_out=0.0)
    p.update(kw)
    return p


def _comp_coords(n, L):
    """computational coordinates of the nodes, (nk+1,nj+1,ni+1) each, spanning [0,L]"""
    ni, nj, nk = n
    xi = np.arange(ni + 1) * (L[0] / ni)
    et = np.arange(nj + 1) * (L[1] / nj)
    ze = np.arange(nk + 1) * (L[2] / nk)
    Z, E, X = np.meshgrid(ze, et, xi, indexing="ij")
    return X, E, Z


# --------------------------------------------------------------------------------------------------
def wavy_periodic_grid(n, L, amp, centre=True):
    """x = xi + amp sin(2 pi eta/L) sin(2 pi zeta/L) and cyclic (config 1; form of Eq. 45)."""
    X, E, Z = _comp_coords((n, n, n), (L, L, L))
    s = lambda a: np.sin(2.0 * np.pi * a / L)
    x = X + amp * s(E) * s(Z)
    y = E + amp * s(Z) * s(X)
    z = Z + amp * s(X) * s(E)
    if centre:
        x, y, z = x - L / 2, y - L / 2, z - L / 2
    return x, y, z


def random_periodic_grid(n, L, frac, seed, centre=True):
    """uniform grid with every node moved by U(-frac,frac) x spacing, identical on periodic images."""
    X, E, Z = _comp_coords((n, n, n), (L, L, L))
    rng = np.random.default_rng(seed)
    out = []
    for base in (X, E, Z):
        r = rng.uniform(-frac, frac, size=(n, n, n)) * (L / n)
        full = np.empty((n + 1, n + 1, n + 1))
        full[:n, :n, :n] = r
        full[n, :, :] = full[0, :, :]
        full[:, n, :] = full[:, 0, :]
        full[:, :, n] = full[:, :, 0]
        out.append(base + full - (L / 2 if centre else 0.0))
    return out


def isentropic_vortex(xc, yc, mach=0.5, eps=5.0, gamma=GAMMA):
    """z-aligned isentropic vortex on a Mach `mach` +x stream, rho_inf = p_inf = 1 (config 1)."""
    r2 = xc * xc + yc * yc
    f = eps / (2.0 * np.pi) * np.exp(0.5 * (1.0 - r2))
    u = mach * np.sqrt(gamma) - yc * f
    v = xc * f
    T = 1.0 - (gamma - 1.0) * eps * eps / (8.0 * gamma * np.pi ** 2) * np.exp(1.0 - r2)
    rho = T ** (1.0 / (gamma - 1.0))
    p = rho ** gamma
    return rho, u, v, np.zeros_like(u), p


def c1_vortex(n=32, wavy=True, steps=10):
    """Config 1: inviscid isentropic vortex, periodic [-5,5]^3, wavy mesh amplitude 0.1, CFL 0.5."""
    L = 10.0
    x, y, z = wavy_periodic_grid(n, L, 0.1 if wavy else 0.0)
    rho, u, v, w, p = isentropic_vortex(cell_centres(x), cell_centres(y))
    prm = _base_params(n, n, n, period=[[L, 0, 0], [0, L, 0], [0, 0, L]])
    name = "c1_vortex_%d%s" % (n, "" if wavy else "_cart")
    return dict(name=name, params=prm, x=x, y=y, z=z, U0=conservative(rho, u, v, w, p), dt=None,
                cfl=0.5, steps=steps, t0=0.0)


def freestream_state(shape, mach=0.5, gamma=GAMMA):
    """(rho,u,v,w,p) = (1,1,0,0,1/(gamma M^2))"""
    one = np.ones(shape)
    return one, one.copy(), 0 * one, 0 * one, one / (gamma * mach * mach)


def freestream_static(n=20, kind="wavy", seed=7):
    """Sec. 8.1.1 analogue: uniform flow on a sinusoidal or 20%-randomised periodic grid, L=4."""
    L = 4.0
    if kind == "wavy":
        # Eq. 45: amplitude = one grid spacing, half-wave sin(pi ...) over [0,L] made periodic
        X, E, Z = _comp_coords((n, n, n), (L, L, L))
        h = L / n
        s = lambda a: np.sin(2.0 * np.pi * a / L)
        x = X + h * s(E) * s(Z) - L / 2
        y = E + h * s(Z) * s(X) - L / 2
        z = Z + h * s(X) * s(E) - L / 2
    else:
        x, y, z = random_periodic_grid(n, L, 0.2, seed)
    prm = _base_params(n, n, n, period=[[L, 0, 0], [0, L, 0], [0, 0, L]])
    U0 = conservative(*freestream_state((n, n, n)))
    return dict(name="freestream_%s_%d" % (kind, n), params=prm, x=x, y=y, z=z, U0=U0, dt=None, cfl=0.2,
                steps=10, t0=0.0)


def c2_dynamic_freestream(n=64, steps=100, seed=20231):
    """Config 2: uniform Mach 0.5 flow, periodic unit cube, nodes move as 0.08 sin(2 pi t) sin sin (+-2% jitter)."""
    L = 1.0
    X, E, Z = _comp_coords((n, n, n), (L, L, L))
    xj, yj, zj = random_periodic_grid(n, L, 0.02, seed)
    s = lambda a: np.sin(2.0 * np.pi * a)
    dxm = 0.08 * s(E) * s(Z)
    dym = 0.08 * s(Z) * s(X)
    dzm = 0.08 * s(X) * s(E)
    prm = _base_params(n, n, n, period=[[L, 0, 0], [0, L, 0], [0, 0, L]], moving=1, omega=1.0)
    U0 = conservative(*freestream_state((n, n, n)))
    name = "c2_dynfree_%d" % n
    return dict(name=name, params=prm, x=xj, y=yj, z=zj, dx_mode=dxm, dy_mode=dym, dz_mode=dzm, U0=U0,
                dt=None, cfl=0.2, steps=steps, t0=0.0)


def tgv_state(xc, yc, zc, mach=0.1, gamma=GAMMA):
    p0 = 1.0 / (gamma * mach * mach)
    u = np.sin(xc) * np.cos(yc) * np.cos(zc)
    v = -np.cos(xc) * np.sin(yc) * np.cos(zc)
    w = np.zeros_like(u)
    p = p0 + (np.cos(2 * xc) + np.cos(2 * yc)) * (np.cos(2 * zc) + 2.0) / 16.0
    rho = p / p0
    return rho, u, v, w, p


def c3_tgv(n=128, steps=200, seed=1600, amp=0.05, scheme=0, re=1600.0):
    """Config 3 (and 5 with scheme=1): viscous Taylor-Green vortex, Re 1600, Ma 0.1, wavy periodic mesh."""
    L = 2.0 * np.pi
    X, E, Z = _comp_coords((n, n, n), (L, L, L))
    rng = np.random.default_rng(seed)
    k = rng.integers(1, 4, size=(3, 2))
    ph = rng.uniform(0.0, 2.0 * np.pi, size=(3, 2))
    x = X - np.pi + amp * np.sin(k[0, 0] * E + ph[0, 0]) * np.sin(k[0, 1] * Z + ph[0, 1])
    y = E - np.pi + amp * np.sin(k[1, 0] * Z + ph[1, 0]) * np.sin(k[1, 1] * X + ph[1, 1])
    z = Z - np.pi + amp * np.sin(k[2, 0] * X + ph[2, 0]) * np.sin(k[2, 1] * E + ph[2, 1])
    mach = 0.1
    p0 = 1.0 / (GAMMA * mach * mach)
    prm = _base_params(n, n, n, period=[[L, 0, 0], [0, L, 0], [0, 0, L]], viscous=1, r_gas=p0,
                       mu_ref=1.0 / re, t_ref=1.0, s_suth=110.4 / 293.0, scheme=scheme)
    rho, u, v, w, p = tgv_state(cell_centres(x), cell_centres(y), cell_centres(z), mach)
    name = "c%d_tgv_%d" % (5 if scheme else 3, n)
    return dict(name=name, params=prm, x=x, y=y, z=z, U0=conservative(rho, u, v, w, p), dt=None,
                cfl=0.2, steps=steps, t0=0.0)


def jet_exit_state(mj=1.35, tn=1.0, gamma=GAMMA):
    """Eq. 55 in units rho_inf = a_inf = 1."""
    pe = (1.0 / gamma) * ((2.0 + (gamma - 1.0) * mj * mj) / (gamma + 1.0)) ** (gamma / (gamma - 1.0))
    rhoe = gamma * (gamma + 1.0) * pe / (2.0 * tn)
    ue = np.sqrt(2.0 * tn / (gamma + 1.0))
    return rhoe, ue, pe


def c4_jet(ni=320, nj=200, nk=200, steps=500, seed=135, re=1.0e4):
    """Config 4: under-expanded Mach 1.35 jet on a tanh-stretched Cartesian-topology mesh, inflow/outflow,
    sponge, viscous Re_D = 1e4.  Constant dt = 2e-3 (the paper's dt a_inf/D)."""
    Lx, bx, Lr, br = 25.0, 2.0, 8.0, 2.0
    s = np.arange(ni + 1) / ni
    xs = Lx * (1.0 - np.tanh(bx * (1.0 - s)) / np.tanh(bx))

    def radial(n):
        sg = 2.0 * np.arange(n + 1) / n - 1.0
        return np.sign(sg) * Lr * (1.0 - np.tanh(br * (1.0 - np.abs(sg))) / np.tanh(br))

    ys, zs = radial(nj), radial(nk)
    z, y, x = np.meshgrid(zs, ys, xs, indexing="ij")
    x, y, z = (np.ascontiguousarray(a) for a in (x, y, z))
    g = GAMMA
    rhoe, ue, pe = jet_exit_state()
    shape = (nk, nj, ni)
    amb = (np.ones(shape), np.zeros(shape), np.zeros(shape), np.zeros(shape), np.full(shape, 1.0 / g))
    U0 = conservative(*amb)
    # inflow face imin: top-hat of diameter 1, 1% seeded velocity perturbation
    yc = 0.5 * (ys[:-1] + ys[1:])
    zc = 0.5 * (zs[:-1] + zs[1:])
    ZC, YC = np.meshgrid(zc, yc, indexing="ij")
    core = (YC * YC + ZC * ZC) < 0.25
    rng = np.random.default_rng(seed)
    pert = 1.0 + 0.01 * rng.uniform(-1.0, 1.0, size=core.shape)
    pin = np.zeros((5, nk, nj))
    pin[0] = np.where(core, rhoe, 1.0)
    pin[1] = np.where(core, ue * pert, 0.0)
    pin[4] = np.where(core, pe, 1.0 / g)
    # sponge: sigma = 2 s^2 over the last 15% of x and the outer 15% of |y|,|z|
    xc3, yc3, zc3 = cell_centres(x), cell_centres(y), cell_centres(z)
    ramp = lambda a, L: np.clip((a - 0.85 * L) / (0.15 * L), 0.0, 1.0)
    sp = np.maximum(ramp(xc3, Lx), np.maximum(ramp(np.abs(yc3), Lr), ramp(np.abs(zc3), Lr)))
    sigma = 2.0 * sp * sp
    # viscosity: Re_D = rho_e u_e D / mu(T_e) with Sutherland (t_ref = T_inf = 1, S = 110.4/293)
    r_gas = 1.0 / g
    Te = pe / (rhoe * r_gas)
    S = 110.4 / 293.0
    mu_e = rhoe * ue / re
    mu_ref = mu_e / (Te ** 1.5 * (1.0 + S) / (Te + S))
    prm = _base_params(ni, nj, nk, periodic=[0, 0, 0], viscous=1, r_gas=r_gas, mu_ref=mu_ref, t_ref=1.0,
                       s_suth=S, bc=[1, 2, 2, 2, 2, 2], p_out=1.0 / g)
    return dict(name="c4_jet_%dx%dx%d" % (ni, nj, nk), params=prm, x=x, y=y, z=z, U0=U0, inflow={0: pin},
                sigma=sigma, U_ref=U0.copy(), dt=2.0e-3, cfl=None, steps=steps, t0=0.0)


def c5_tgv_mig4(n=384, steps=50):
    return c3_tgv(n=n, steps=steps, scheme=1)


# --------------------------------------------------------------------------------------------------
# Walls (Table 1).  Synthetic channel / closed-box inputs; no paper grid is reproduced.
def _smooth_state(xc, yc, zc, L, seed, mach=0.3, amp=0.05, gamma=GAMMA):
    """(rho,u,v,w,p): Mach `mach` stream along x plus seeded smooth perturbations of every primitive variable."""
    rng = np.random.default_rng(seed)
    ph = rng.uniform(0.0, 2.0 * np.pi, size=(5, 3))
    kx, ky, kz = 2.0 * np.pi / L[0], 2.0 * np.pi / L[1], 2.0 * np.pi / L[2]
    f = lambda q: np.sin(kx * xc + ph[q, 0]) * np.cos(ky * yc + ph[q, 1]) * np.sin(kz * zc + ph[q, 2])
    a0 = 1.0
    rho = 1.0 + amp * f(0)
    u = mach * a0 * (1.0 + 2.0 * amp * f(1))
    v = mach * a0 * 2.0 * amp * f(2)
    w = mach * a0 * 2.0 * amp * f(3)
    p = (1.0 / gamma) * (1.0 + amp * f(4))
    return rho, u, v, w, p


def wall_channel(ni=24, nj=16, nk=20, wall=3, viscous=0, scheme=0, seed=4242, curved=True, amp=0.05):
    """Channel between two eta walls (bc 3 inviscid / 4 adiabatic no-slip), periodic in xi and zeta.
    curved=False: y = eta with spacing 2/nj (a power of two for nj = 16, 32), x and z wavy in (xi, zeta) only --
    the mesh of the reflection-principle pin; curved=True: the walls themselves are wavy (non-trivial normals)."""
    L = (4.0, 2.0, 3.0)
    X, E, Z = _comp_coords((ni, nj, nk), L)
    s = lambda a, l: np.sin(2.0 * np.pi * a / l)
    x = X + 0.08 * s(Z, L[2])
    z = Z + 0.06 * s(X, L[0])
    y = E + (0.05 * s(X, L[0]) * np.cos(2.0 * np.pi * Z / L[2]) * (1.0 + 0.5 * E) if curved else 0.0)
    x, y, z = (np.ascontiguousarray(a) for a in (x, y, z))
    rho, u, v, w, p = _smooth_state(cell_centres(x), cell_centres(y), cell_centres(z), L, seed, amp=amp)
    prm = _base_params(ni, nj, nk, periodic=[1, 0, 1], period=[[L[0], 0, 0], [0, 0, 0], [0, 0, L[2]]], scheme=scheme,
                       viscous=viscous, bc=[0, 0, wall, wall, 0, 0], p_out=1.0 / GAMMA)
    if viscous:
        prm.update(mu_ref=0.3 * 1.0 / 200.0, t_ref=1.0 / GAMMA, s_suth=0.4 / GAMMA)   # Re ~ 200 on the unit length
    return dict(name="wall_channel_%dx%dx%d_bc%d%s" % (ni, nj, nk, wall, "" if curved else "_flat"), params=prm,
                x=x, y=y, z=z, U0=conservative(rho, u, v, w, p), dt=None, cfl=0.4, steps=3, t0=0.0)


def wall_box(ni=22, nj=19, nk=17, bc=(3, 4, 3, 3, 4, 3), viscous=1, scheme=0, seed=515):
    """Closed box, walls of mixed kind on all six faces of a smoothly distorted non-periodic mesh (edges and
    corners: ghost cells of ghost cells)."""
    L = (2.0, 1.5, 1.0)
    X, E, Z = _comp_coords((ni, nj, nk), L)
    s = lambda a, l: np.sin(2.0 * np.pi * a / l)
    x = X + 0.04 * s(E, L[1]) * s(Z, L[2])
    y = E + 0.03 * s(Z, L[2]) * s(X, L[0])
    z = Z + 0.02 * s(X, L[0]) * s(E, L[1])
    x, y, z = (np.ascontiguousarray(a) for a in (x, y, z))
    rho, u, v, w, p = _smooth_state(cell_centres(x), cell_centres(y), cell_centres(z), L, seed)
    prm = _base_params(ni, nj, nk, periodic=[0, 0, 0], scheme=scheme, viscous=viscous, bc=list(bc), p_out=1.0 / GAMMA)
    if viscous:
        prm.update(mu_ref=0.3 * 1.0 / 200.0, t_ref=1.0 / GAMMA, s_suth=0.4 / GAMMA)
    return dict(name="wall_box_%dx%dx%d" % (ni, nj, nk), params=prm, x=x, y=y, z=z,
                U0=conservative(rho, u, v, w, p), dt=None, cfl=0.4, steps=3, t0=0.0)


# --------------------------------------------------------------------------------------------------
def inout_box(n=(18, 9, 8), axis=0, flip=False, viscous=0, u_mean=1.0, scheme=0, seed=77, h=0.1):
    """Uniform Cartesian box with an inflow and an outflow face (bc 1 / 2, Table 1) across direction `axis`
    (flip: inflow on the max side, flow towards the min side), periodic in the two other directions; smooth + seeded
    state with the stream along `axis` at mean Mach number u_mean (sound speed ~ 1: u_mean = 1 puts sub- and supersonic
    outflow cells into one face), non-uniform inflow data.  wl["P0"] = the primitive state (rho, u, v, w, p)."""
    ni, nj, nk = n
    X, E, Z = _comp_coords(n, (ni * h, nj * h, nk * h))
    rng = np.random.default_rng(seed)
    xc, yc, zc = cell_centres(X), cell_centres(E), cell_centres(Z)
    cc = (xc, yc, zc)
    kk = [2 * np.pi / (m * h) for m in n]
    kk[axis] = 3.0                                                # not periodic along the stream
    wob = lambda ph: np.sin(kk[0] * xc + ph) * np.cos(kk[1] * yc + ph) * np.cos(kk[2] * zc - ph)
    sgn = -1.0 if flip else 1.0
    rho = 1.0 + 0.08 * wob(0.3) + 0.01 * rng.uniform(-1, 1, xc.shape)
    vel = [0.10 * wob(2.0), -0.07 * wob(0.7), 0.05 * wob(1.4)]
    vel[axis] = sgn * (u_mean + 0.12 * wob(1.1) + 0.01 * rng.uniform(-1, 1, xc.shape))
    p = (1.0 + 0.08 * wob(1.9) + 0.01 * rng.uniform(-1, 1, xc.shape)) / GAMMA
    ta, tb = [d for d in range(3) if d != axis]                   # transverse directions, storage order: tb slow
    take = [slice(None)] * 3
    take[2 - axis] = 0
    ca, cb = cc[ta][tuple(take)], cc[tb][tuple(take)]             # (n_tb, n_ta)
    pin = np.empty((5,) + ca.shape)
    pin[0] = 1.0 + 0.05 * np.cos(kk[ta] * ca)
    pin[1:4] = 0.0
    pin[1 + ta] = 0.03 * np.sin(kk[ta] * ca)
    pin[1 + tb] = -0.02 * np.sin(kk[tb] * cb)
    pin[1 + axis] = sgn * (u_mean + 0.05 * np.cos(kk[tb] * cb))
    pin[4] = (1.0 + 0.04 * np.cos(kk[ta] * ca + kk[tb] * cb)) / GAMMA
    periodic, bc = [1, 1, 1], [0] * 6
    periodic[axis] = 0
    bc[2 * axis + (1 if flip else 0)] = 1
    bc[2 * axis + (0 if flip else 1)] = 2
    period = [[0.0] * 3 for _ in range(3)]
    for d in (ta, tb):
        period[d][d] = n[d] * h
    prm = _base_params(ni, nj, nk, periodic=periodic, period=period, viscous=viscous, scheme=scheme,
                       mu_ref=2e-3 if viscous else 0.0, bc=bc, p_out=0.93 / GAMMA)
    P0 = np.stack([rho, vel[0], vel[1], vel[2], p])
    return dict(name="inout_box_%dx%dx%d_axis%d%s" % (ni, nj, nk, axis, "_flip" if flip else ""), params=prm,
                x=np.ascontiguousarray(X), y=np.ascontiguousarray(E), z=np.ascontiguousarray(Z), U0=conservative(*P0),
                P0=P0, inflow={2 * axis + (1 if flip else 0): pin}, sigma=None, dt=None, cfl=0.4, steps=3, t0=0.0)


# --------------------------------------------------------------------------------------------------
# Multi-block inputs (Sec. 6): a single-block workload cut into aligned blocks.
def cartesian_periodic(ni=24, nj=20, nk=16, viscous=1, seed=77, scheme=0):
    """Uniform Cartesian periodic box (spacing 1/8: exactly representable coordinates) with a seeded smooth state:
    the mesh on which linearly extrapolated ghost coordinates (R13) equal the neighbour block's true ones."""
    h = 0.125
    L = (ni * h, nj * h, nk * h)
    X, E, Z = _comp_coords((ni, nj, nk), L)
    x, y, z = (np.ascontiguousarray(a) for a in (X, E, Z))
    rho, u, v, w, p = _smooth_state(cell_centres(x), cell_centres(y), cell_centres(z), L, seed)
    prm = _base_params(ni, nj, nk, period=[[L[0], 0, 0], [0, L[1], 0], [0, 0, L[2]]], viscous=viscous, scheme=scheme)
    if viscous:
        prm.update(mu_ref=0.3 * 1.0 / 200.0, t_ref=1.0 / GAMMA, s_suth=0.4 / GAMMA)
    return dict(name="cart_periodic_%dx%dx%d" % (ni, nj, nk), params=prm, x=x, y=y, z=z,
                U0=conservative(rho, u, v, w, p), dt=None, cfl=0.4, steps=3, t0=0.0)


def split_blocks(wl, cuts):
    """Cuts a static single-block workload into aligned blocks (each block dict carries `link_offset`: per linked face
    the vector added to the neighbour's coordinates seen from the block -- the period across a wrap-around link).  cuts = (cells of the xi pieces, eta pieces, zeta
    pieces), e.g. ((12, 12), (20,), (16,)).  Returns (blocks, links): blocks in storage order (xi piece fastest),
    links = [(home, face, neighbour)].  Cut directions become non-periodic with bc 5 on the cut faces; a periodic
    direction that is cut wraps around through links; outer faces of non-periodic directions keep their bc."""
    prm = wl["params"]
    assert not prm["moving"]
    n = (prm["ni"], prm["nj"], prm["nk"])
    for d in range(3):
        assert sum(cuts[d]) == n[d]
    starts = [np.concatenate([[0], np.cumsum(cuts[d])]) for d in range(3)]
    nb = [len(cuts[d]) for d in range(3)]
    idx = lambda a, b, c: (c * nb[1] + b) * nb[0] + a
    blocks, links = [], []
    for c in range(nb[2]):
        for b in range(nb[1]):
            for a in range(nb[0]):
                pos = (a, b, c)
                lo = [int(starts[d][pos[d]]) for d in range(3)]
                hi = [int(starts[d][pos[d] + 1]) for d in range(3)]
                p = dict(prm)
                p["ni"], p["nj"], p["nk"] = (hi[d] - lo[d] for d in range(3))
                p["periodic"] = list(prm["periodic"])
                p["bc"] = list(prm["bc"])
                link_offset = {}
                for d in range(3):
                    if nb[d] == 1:
                        continue
                    p["periodic"][d] = 0
                    for side in range(2):
                        q = pos[d] + (1 if side else -1)
                        if 0 <= q < nb[d] or prm["periodic"][d]:
                            p["bc"][2 * d + side] = 5
                            npos = list(pos)
                            npos[d] = q % nb[d]
                            links.append((idx(*pos), 2 * d + side, idx(*npos)))
                            # what is added to the neighbour's coordinates seen from here: the period vector where
                            # the link wraps around a periodic direction, else nothing
                            wrap = (1.0 if q >= nb[d] else -1.0 if q < 0 else 0.0)
                            link_offset[2 * d + side] = [wrap * float(v) for v in prm["period"][d]]
                sl_n = tuple(slice(lo[d], hi[d] + 1) for d in (2, 1, 0))
                sl_c = tuple(slice(lo[d], hi[d]) for d in (2, 1, 0))
                extra = {}
                if wl.get("sigma") is not None:
                    extra["sigma"] = np.ascontiguousarray(wl["sigma"][sl_c])
                    extra["U_ref"] = np.ascontiguousarray(wl["U_ref"][(slice(None),) + sl_c])
                inflow = {}
                for face, pin in wl.get("inflow", {}).items():   # pin[5][n2][n1], transverse axes in storage order
                    d = int(face) // 2
                    if p["bc"][int(face)] != 1:
                        continue
                    t1, t2 = [e for e in range(3) if e != d]
                    inflow[int(face)] = np.ascontiguousarray(pin[:, lo[t2]:hi[t2], lo[t1]:hi[t1]])
                if inflow:
                    extra["inflow"] = inflow
                blocks.append(dict(extra, name="%s_block%d" % (wl["name"], idx(*pos)), params=p, link_offset=link_offset,
                                   x=np.ascontiguousarray(wl["x"][sl_n]), y=np.ascontiguousarray(wl["y"][sl_n]),
                                   z=np.ascontiguousarray(wl["z"][sl_n]),
                                   U0=np.ascontiguousarray(wl["U0"][(slice(None),) + sl_c]),
                                   dt=wl.get("dt"), cfl=wl.get("cfl"), steps=wl.get("steps"), t0=0.0, slices=sl_c))
    return blocks, links


def link_all(grids, blocks, links):
    """plumbing: grids[home].link(face, grids[nb]) for every link of split_blocks, with its coordinate offset"""
    for home, face, nb in links:
        grids[home].link(face, grids[nb], offset=blocks[home]["link_offset"].get(face))


# --------------------------------------------------------------------------------------------------
# Blocks with their own coordinate systems (Sec. 6): index plumbing only.
ROTATIONS = {
    # name: (source axis of the new xi, eta, zeta; +1 forwards / -1 backwards) -- proper rotations (right-handed)
    "id": ((0, 1), (1, 1), (2, 1)),
    "z90": ((1, 1), (0, -1), (2, 1)),      # new xi = old eta, new eta = -old xi
    "z180": ((0, -1), (1, -1), (2, 1)),
    "z270": ((1, -1), (0, 1), (2, 1)),
    "cyc": ((1, 1), (2, 1), (0, 1)),       # new (xi, eta, zeta) = old (eta, zeta, xi)
    "x90": ((0, 1), (2, 1), (1, -1)),      # new eta = old zeta, new zeta = -old eta
}


def _reindex(a, rot, lead=0):
    """array with trailing axes (k, j, i) re-expressed in the rotated computational frame"""
    # numpy axis of computational direction e is lead + 2 - e
    src = [lead + 2 - rot[e][0] for e in range(3)]          # numpy source axis of new direction e
    out = np.transpose(a, list(range(lead)) + [src[2], src[1], src[0]])
    for e in range(3):
        if rot[e][1] < 0:
            out = np.flip(out, axis=lead + 2 - e)
    return np.ascontiguousarray(out)


def rotate_block(blk, name):
    """The same block of cells stored in another computational frame: node arrays, state and boundary data re-indexed,
    face numbers and periodicity permuted.  Cartesian vector components (u, v, w; x, y, z) are untouched."""
    rot = ROTATIONS[name]
    p = dict(blk["params"])
    n_old = (p["ni"], p["nj"], p["nk"])
    p["ni"], p["nj"], p["nk"] = (n_old[rot[e][0]] for e in range(3))
    p["periodic"] = [blk["params"]["periodic"][rot[e][0]] for e in range(3)]
    p["period"] = [[rot[e][1] * v for v in blk["params"]["period"][rot[e][0]]] for e in range(3)]
    bc, link_offset, face_map = [0] * 6, {}, {}
    for e in range(3):
        for side in range(2):
            old_face = 2 * rot[e][0] + (side if rot[e][1] > 0 else 1 - side)
            bc[2 * e + side] = blk["params"]["bc"][old_face]
            face_map[old_face] = 2 * e + side
            if old_face in blk.get("link_offset", {}):
                link_offset[2 * e + side] = blk["link_offset"][old_face]
    p["bc"] = bc
    out = dict(blk, params=p, link_offset=link_offset, face_map=face_map, rotation=name,
               name=blk["name"] + "_" + name)
    for key in ("x", "y", "z", "dx_mode", "dy_mode", "dz_mode"):
        if blk.get(key) is not None:
            out[key] = _reindex(blk[key], rot)
    out["U0"] = _reindex(blk["U0"], rot, lead=1)
    if blk.get("sigma") is not None:
        out["sigma"] = _reindex(blk["sigma"], rot)
        out["U_ref"] = _reindex(blk["U_ref"], rot, lead=1)
    assert not blk.get("inflow"), "rotate_block: inflow faces are not re-indexed"
    return out


def unrotate_state(a, name):
    """inverse of the re-indexing of rotate_block for a state array (5, nk, nj, ni)"""
    rot = ROTATIONS[name]
    out = a
    for e in range(3):
        if rot[e][1] < 0:
            out = np.flip(out, axis=1 + 2 - e)
    src = [1 + 2 - rot[e][0] for e in range(3)]
    perm = [0, src[2], src[1], src[0]]
    inv = np.argsort(perm)
    return np.ascontiguousarray(np.transpose(out, inv))


def _face_nodes(blk, face):
    """node coordinates of a block face, shape (nb+1, na+1, 3), transverse axes in storage order (a fast)"""
    d, side = face // 2, face % 2
    sl = [slice(None)] * 3
    sl[2 - d] = -1 if side else 0
    return np.stack([blk[k][tuple(sl)] for k in ("x", "y", "z")], axis=-1)


def auto_links(blocks, periods=()):
    """Finds, for every block-interface face (bc 5), the neighbour block, its face and the orientation of its axes by
    matching the node coordinates of the faces (up to one of the given period vectors).  Returns
    [(home, face, nb, nb_face, swap, flip_a, flip_b, offset)]: the arguments of the oriented link call."""
    offs = [np.zeros(3)] + [s * np.asarray(v, dtype=float) for v in periods for s in (1.0, -1.0)]
    faces = [(b, f, _face_nodes(blk, f)) for b, blk in enumerate(blocks) for f in range(6)
             if not blk["params"]["periodic"][f // 2] and blk["params"]["bc"][f] == 5]
    links = []
    for b, f, N in faces:
        h = np.linalg.norm(N[1, 1] - N[0, 0]) if min(N.shape[:2]) > 1 else 1.0
        found = None
        for c, g, M in faces:
            if (c, g) == (b, f) and not periods:
                continue
            for swap in (0, 1):
                Ms = np.swapaxes(M, 0, 1) if swap else M     # home a runs along the neighbour's b' when swapped
                if Ms.shape != N.shape:
                    continue
                for fa in (0, 1):
                    for fb in (0, 1):
                        T = Ms[:, ::-1] if fa else Ms
                        T = T[::-1] if fb else T
                        for off in offs:
                            if (c, g) == (b, f) and not off.any():
                                continue
                            if np.abs(T + off - N).max() <= 1e-9 * max(h, 1e-30) + 1e-12:
                                found = (b, f, c, g, swap, fa, fb, [float(v) for v in off])
                        if found:
                            break
                    if found:
                        break
                if found:
                    break
            if found:
                break
        if found is None:
            raise ValueError("auto_links: no partner for block %d face %d" % (b, f))
        links.append(found)
    return links


def butterfly(n=12, nr=12, nk=10, a=0.5, R=2.0, Lz=1.0, viscous=1, scheme=0, seed=627, uniform=False):
    """Butterfly-type O-grid section (Fig. 13b "to avoid singularity at the axis"), synthetic: a square core block
    of n x n cells and four outer blocks of nr x n cells between the square and a circle of radius R, each in its own
    frame (xi radial, eta along the core's side; quarter turns about the axis from one to the next), extruded along a
    periodic zeta.  Three blocks meet along each of the core's four corner edges.  Returns the five block workloads
    (interfaces bc 5, outer rim outflow); link them with auto_links.  (The paper's jet grid has four blocks and is not
    in the container; this one only has its topology class: rotated frames around a core, singular corner edges.)"""
    s = np.linspace(-1.0, 1.0, n + 1)
    r = np.linspace(0.0, 1.0, nr + 1)
    zk = np.linspace(-Lz / 2, Lz / 2, nk + 1)

    def extrude(X2, Y2):
        shp = (nk + 1,) + X2.shape
        return (np.ascontiguousarray(np.broadcast_to(X2, shp)), np.ascontiguousarray(np.broadcast_to(Y2, shp)),
                np.ascontiguousarray(np.broadcast_to(zk[:, None, None], shp)))
    X, Y = np.meshgrid(a * s, a * s, indexing="xy")
    grids = [extrude(X, Y)]
    P0 = np.stack([a * np.ones_like(s), a * s], -1)                                  # the core's east side
    P1 = np.stack([R * np.cos(s * np.pi / 4), R * np.sin(s * np.pi / 4)], -1)        # the rim arc facing it
    N = (1 - r)[None, :, None] * P0[:, None, :] + r[None, :, None] * P1[:, None, :]  # (eta = s, xi = r, 2)
    for q in range(4):
        c, sn = np.cos(q * np.pi / 2), np.sin(q * np.pi / 2)
        c, sn = round(c), round(sn)                                                  # exact quarter turns
        grids.append(extrude(c * N[..., 0] - sn * N[..., 1], sn * N[..., 0] + c * N[..., 1]))
    rng = np.random.default_rng(seed)
    ph = rng.uniform(0.0, 2.0 * np.pi, size=(5, 3))
    blocks = []
    for b, (x, y, z) in enumerate(grids):
        nj_, ni_ = x.shape[1] - 1, x.shape[2] - 1
        bc = [5, 5, 5, 5, 0, 0] if b == 0 else [5, 2, 5, 5, 0, 0]
        prm = _base_params(ni_, nj_, nk, periodic=[0, 0, 1], period=[[0, 0, 0], [0, 0, 0], [0, 0, Lz]], bc=bc,
                           viscous=viscous, scheme=scheme, p_out=1.0 / GAMMA)
        if viscous:
            prm.update(mu_ref=0.3 * 1.0 / 200.0, t_ref=1.0 / GAMMA, s_suth=0.4 / GAMMA)
        xc, yc, zc = cell_centres(x), cell_centres(y), cell_centres(z)
        if uniform:
            one = np.ones_like(xc)
            prim = (one, 0.3 * one, 0.2 * one, -0.1 * one, one / GAMMA)
        else:
            f = lambda qq: np.sin(1.3 * xc + ph[qq, 0]) * np.cos(1.1 * yc + ph[qq, 1]) * np.sin(2 * np.pi * zc / Lz + ph[qq, 2])
            prim = (1.0 + 0.05 * f(0), 0.3 * (1.0 + 0.1 * f(1)), 0.03 * f(2), 0.03 * f(3), (1.0 + 0.05 * f(4)) / GAMMA)
        blocks.append(dict(name="butterfly_block%d" % b, params=prm, x=x, y=y, z=z, U0=conservative(*prim), dt=None,
                           cfl=0.4, steps=3, t0=0.0))
    return blocks
