"""Pins of the oracle's inflow and outflow ghost rules (Table 1, garbled in PAPER.md; reading R20).

CPU only.  The reading itself (what the garbled table meant) cannot be pinned; what CAN be fixed independently of the
oracle's ghost-fill code is that the right-hand side it produces next to such a face is the one the reading defines:
  * extension principle: ten ghost layers are all any interior cell's dQ/dt depends on (6-point limiter window of an
    interface + E6 gradients of the two cells beside it), so a box with an inflow and an outflow face IS the
    inner part of a longer PERIODIC box whose extra cells hold the ghost states -- evaluated through the oracle's
    periodic wrap, a code path that never sees a boundary rule;
  * reflection about the inflow state: with ghost = 2 P_in - P_mirror the linear interface values of Eq. 16 on the two
    sides of the inflow face satisfy P^L + P^R = 2 P_in identically, so for interior data equal to P_in the face is
    transparent, and a wrong mirror index (off by one cell) breaks the extension test at the first interior cells;
  * the outflow switch: supersonic outflow must not see p_out at all, subsonic outflow must.
"""
import numpy as np
import pytest

import workloads as W
from oracle import meg6_oracle as O

GP = 10            # ghost layers the method needs
NI, NJ, NK = 18, 9, 8
H = 0.1


def box(viscous, u_mean, seed=77):
    """Uniform Cartesian box, inflow at imin, outflow at imax, periodic in eta and zeta; smooth + random data"""
    X, E, Z = W._comp_coords((NI, NJ, NK), (NI * H, NJ * H, NK * H))
    rng = np.random.default_rng(seed)
    xc, yc, zc = W.cell_centres(X), W.cell_centres(E), W.cell_centres(Z)
    ky, kz = 2 * np.pi / (NJ * H), 2 * np.pi / (NK * H)
    wob = lambda ph: np.sin(3.0 * xc + ph) * np.cos(ky * yc + ph) * np.cos(kz * zc - ph)
    rho = 1.0 + 0.08 * wob(0.3) + 0.01 * rng.uniform(-1, 1, xc.shape)
    u = u_mean + 0.12 * wob(1.1) + 0.01 * rng.uniform(-1, 1, xc.shape)
    v = 0.10 * wob(2.0)
    w = -0.07 * wob(0.7)
    p = (1.0 + 0.08 * wob(1.9) + 0.01 * rng.uniform(-1, 1, xc.shape)) / W.GAMMA
    pin = np.empty((5, NK, NJ))
    yy, zz = yc[:, :, 0], zc[:, :, 0]
    pin[0] = 1.0 + 0.05 * np.cos(ky * yy)
    pin[1] = u_mean + 0.05 * np.cos(kz * zz)
    pin[2] = 0.03 * np.sin(ky * yy)
    pin[3] = -0.02 * np.sin(kz * zz)
    pin[4] = (1.0 + 0.04 * np.cos(ky * yy + kz * zz)) / W.GAMMA
    prm = W._base_params(NI, NJ, NK, periodic=[0, 1, 1], period=[[0, 0, 0], [0, NJ * H, 0], [0, 0, NK * H]],
                         viscous=viscous, mu_ref=2e-3 if viscous else 0.0, bc=[1, 2, 0, 0, 0, 0], p_out=0.93 / W.GAMMA)
    return dict(name="inout_box", params=prm, x=X, y=E, z=Z, U0=W.conservative(rho, u, v, w, p), inflow={0: pin},
                sigma=None), (rho, u, v, w, p)


def extended_periodic_twin(wl, prim):
    """The box with GP more cells at each end of xi, periodic in xi over the longer length; the extra cells hold what
    reading R20 says the ghost cells hold (written out here on the primitive variables, cell by cell)."""
    P = np.stack(prim)                                            # (5, nk, nj, ni)
    pin = wl["inflow"][0]
    g = W.GAMMA
    lo = np.empty((5, NK, NJ, GP))
    hi = np.empty((5, NK, NJ, GP))
    for q in range(1, GP + 1):
        lo[..., GP - q] = 2.0 * pin - P[..., q - 1]              # layer q outside imin mirrors the q-th interior cell
    last = P[..., NI - 1].copy()
    mach = last[1] / np.sqrt(g * last[4] / last[0])               # outward normal = +x on this mesh
    last[4] = np.where(mach < 1.0, wl["params"]["p_out"], last[4])
    for q in range(GP):
        hi[..., q] = last
    P2 = np.concatenate([lo, P, hi], axis=3)
    assert P2[0].min() > 0.2 and P2[4].min() > 0.2
    n2 = NI + 2 * GP
    X, E, Z = W._comp_coords((n2, NJ, NK), (n2 * H, NJ * H, NK * H))
    prm = dict(wl["params"])
    prm.update(ni=n2, periodic=[1, 1, 1], bc=[0] * 6, period=[[n2 * H, 0, 0], [0, NJ * H, 0], [0, 0, NK * H]])
    twin = dict(wl, params=prm, x=X - GP * H, y=E, z=Z, U0=W.conservative(*P2))
    twin.pop("inflow")
    return twin, mach


def relerr(a, b):
    s = np.abs(b).reshape(5, -1).max(axis=1)
    s = np.maximum(s, s.max() * 1e-3)
    return (np.abs(a - b).reshape(5, -1).max(axis=1) / s).max()


@pytest.mark.parametrize("viscous", [0, 1])
@pytest.mark.parametrize("u_mean", [0.5, 1.0, 1.6])
def test_inflow_outflow_box_is_the_inner_part_of_the_extended_periodic_box(viscous, u_mean):
    wl, prim = box(viscous, u_mean)
    twin, mach = extended_periodic_twin(wl, prim)
    if u_mean == 1.0:
        assert (mach < 1.0).any() and (mach >= 1.0).any()         # both branches of the outflow rule in one face
    g, g2 = O.Grid(wl), O.Grid(twin)
    g.metrics_compute(0.0)
    g2.metrics_compute(0.0)
    r, r2 = g.rhs(wl["U0"]), g2.rhs(twin["U0"])
    assert np.abs(r).max() > 1e-1
    assert relerr(r, r2[..., GP:GP + NI]) <= 1e-12
    # negative control: the same comparison with the mirror index shifted by one cell is far off
    P = np.stack(prim)
    bad = dict(twin)
    U2 = twin["U0"].copy()
    shifted = [2.0 * wl["inflow"][0] - P[..., min(q, NI - 1)] for q in range(1, GP + 1)]
    U2[..., :GP] = W.conservative(*np.stack(shifted[::-1], axis=-1))
    bad["U0"] = U2
    g3 = O.Grid(bad)
    g3.metrics_compute(0.0)
    assert relerr(r, g3.rhs(U2)[..., GP:GP + NI]) > 1e-4
    # and ten layers are what the interior depends on: junk in the wrap region beyond them changes nothing inside --
    # here the two ends of the twin meet with a jump (outflow copies against inflow reflections)
    assert np.abs(r2[..., :2]).max() > 0.0


def test_inflow_face_is_transparent_for_the_inflow_state_and_supersonic_outflow_ignores_p_out():
    wl, prim = box(0, 1.6)
    pin = wl["inflow"][0]
    uni = [np.broadcast_to(pin[f, 0, 0], prim[0].shape).copy() for f in range(5)]
    pin_u = np.broadcast_to(pin[:, :1, :1], pin.shape).copy()
    wl_u = dict(wl, U0=W.conservative(*uni), inflow={0: pin_u})
    g = O.Grid(wl_u)
    g.metrics_compute(0.0)
    assert np.abs(g.rhs(wl_u["U0"])).max() <= 1e-12              # supersonic everywhere: p_out != p is never applied
    # subsonic: the same uniform state now meets p_out at the outflow face and only there
    uni[1][:] = 0.5
    pin_u[1] = 0.5
    wl_s = dict(wl, U0=W.conservative(*uni), inflow={0: pin_u})
    g = O.Grid(wl_s)
    g.metrics_compute(0.0)
    r = g.rhs(wl_s["U0"])
    assert np.abs(r[..., :NI - 6]).max() <= 1e-12
    assert np.abs(r[..., NI - 1]).max() > 1e-2
    # p_out equal to the state's own pressure: transparent again
    prm = dict(wl["params"], p_out=float(pin_u[4, 0, 0]))
    g = O.Grid(dict(wl_s, params=prm))
    g.metrics_compute(0.0)
    assert np.abs(g.rhs(wl_s["U0"])).max() <= 1e-12
