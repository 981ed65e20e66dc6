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
N = (18, 9, 8)     # 18 cells along the stream (the mirror of ten ghost layers needs ten interior cells), ragged across
H = 0.1


def dims(axis):
    n = [9, 8, 9]
    n[(axis + 1) % 3] = 8 if axis != 2 else 9
    n[axis] = 18
    return tuple(n)


def extended_periodic_twin(wl):
    """The box with GP more cells at each end of the stream direction, periodic in it over the longer length; the extra
    cells hold what reading R20 says the ghost cells hold (written out here on the primitive variables, layer by
    layer).  Returns the twin, the slice of the box inside it and the outward normal Mach numbers of the outflow face."""
    prm = wl["params"]
    axis = [d for d in range(3) if not prm["periodic"][d]][0]
    (fin, pin), = wl["inflow"].items()
    flip = fin % 2 == 1
    ax = 3 - axis                                                  # array axis of the stream in (5, nk, nj, ni)
    P = np.moveaxis(wl["P0"], ax, -1)                              # stream index last
    if flip:
        P = P[..., ::-1]                                           # ... counted from the inflow face
    n = P.shape[-1]
    g = W.GAMMA
    lo = np.empty(P.shape[:-1] + (GP,))
    for q in range(1, GP + 1):
        lo[..., GP - q] = 2.0 * pin - P[..., q - 1]               # layer q outside the inflow face mirrors the q-th interior cell
    last = P[..., n - 1].copy()
    mach = (-1.0 if flip else 1.0) * last[1 + axis] / np.sqrt(g * last[4] / last[0])   # outward normal of the outflow face
    last[4] = np.where(mach < 1.0, prm["p_out"], last[4])
    hi = np.repeat(last[..., None], GP, axis=-1)
    P2 = np.concatenate([lo, P, hi], axis=-1)
    if flip:
        P2 = P2[..., ::-1]
    P2 = np.ascontiguousarray(np.moveaxis(P2, -1, ax))
    assert P2[0].min() > 0.2 and P2[4].min() > 0.2
    nb = (prm["ni"], prm["nj"], prm["nk"])
    n2 = list(nb)
    n2[axis] += 2 * GP
    X = list(W._comp_coords(tuple(n2), tuple(m * H for m in n2)))
    X[axis] = X[axis] - GP * H
    period = [list(r) for r in prm["period"]]
    period[axis][axis] = n2[axis] * H
    p2 = dict(prm)
    p2.update(ni=n2[0], nj=n2[1], nk=n2[2], periodic=[1, 1, 1], bc=[0] * 6, period=period)
    twin = dict(wl, params=p2, x=X[0], y=X[1], z=X[2], U0=W.conservative(*P2), P0=P2)
    twin.pop("inflow")
    inner = [slice(None)] * 4
    inner[ax] = slice(GP, GP + nb[axis])
    return twin, tuple(inner), mach, axis, flip


def relerr(a, b):
    s = np.abs(b).reshape(5, -1).max(axis=1)
    s = np.maximum(s, s.max() * 1e-3)
    return (np.abs(a - b).reshape(5, -1).max(axis=1) / s).max()


def rhs_of(wl):
    g = O.Grid(wl)
    g.metrics_compute(0.0)
    return g.rhs(wl["U0"])


@pytest.mark.parametrize("viscous", [0, 1])
@pytest.mark.parametrize("axis,flip,u_mean", [(0, False, 0.5), (0, False, 1.0), (0, False, 1.6), (0, True, 1.0),
                                              (1, False, 1.0), (1, True, 0.5), (2, False, 1.6), (2, True, 1.0)])
def test_inflow_outflow_box_is_the_inner_part_of_the_extended_periodic_box(viscous, axis, flip, u_mean):
    wl = W.inout_box(n=dims(axis), axis=axis, flip=flip, viscous=viscous, u_mean=u_mean, h=H)
    twin, inner, mach, _, _ = extended_periodic_twin(wl)
    if u_mean == 1.0:
        assert (mach < 1.0).any() and (mach >= 1.0).any()         # both branches of the outflow rule in one face
    r, r2 = rhs_of(wl), rhs_of(twin)
    assert np.abs(r).max() > 1e-1
    assert relerr(r, r2[inner]) <= 1e-12
    # negative control: the same comparison with the mirror cell of the inflow rule shifted by one is far off
    if axis == 0 and not flip:
        P = wl["P0"]
        pin = wl["inflow"][0]
        shifted = [2.0 * pin - P[..., min(q, N[0] - 1)] for q in range(1, GP + 1)]
        U2 = twin["U0"].copy()
        U2[..., :GP] = W.conservative(*np.stack(shifted[::-1], axis=-1))
        assert relerr(r, rhs_of(dict(twin, U0=U2))[inner]) > 1e-4


def test_inflow_face_is_transparent_for_the_inflow_state_and_supersonic_outflow_ignores_p_out():
    NI = N[0]
    wl = W.inout_box(n=N, u_mean=1.6, h=H)
    prim = list(wl["P0"])
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
