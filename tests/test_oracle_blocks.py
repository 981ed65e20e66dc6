"""Pins of the oracle's block interfaces (Table 1 last column; R28).

CPU only.  What fixes the exchange independently of the oracle's own copy loop: a domain cut into blocks must give
the result of the uncut domain.  That holds to round-off where the per-block geometry equals the single-block one,
i.e. on a uniform Cartesian mesh (linearly extrapolated ghost coordinates, R13, are then the neighbour's true ones);
the uncut run goes through the periodic wrap and never sees a block interface.  With a 2 x 2 cut and the viscous
flux (tangential gradients in ghost cells) the edge ghosts must arrive from the diagonal neighbour.  On curved
blocks, whose ghost geometry differs from the neighbour's ("metric terms are non-existent" there), the pin is
the paper's own: uniform flow stays uniform to machine zero.
"""
import numpy as np
import pytest

import workloads as W
from oracle import meg6_oracle as O


def make_blocks(wl, cuts):
    blocks, links = W.split_blocks(wl, cuts)
    grids = [O.Grid(b) for b in blocks]
    for home, face, nb in links:
        grids[home].link(face, grids[nb])
    for g in grids:
        g.metrics_compute(0.0)
    return blocks, grids


def gather(blocks, arrays, shape):
    out = np.empty(shape)
    for b, a in zip(blocks, arrays):
        out[(slice(None),) + b["slices"]] = a
    return out


def relerr(a, b):
    s = np.abs(b).reshape(5, -1).max(axis=1)
    s = np.maximum(s, s.max() * 1e-3)
    return (np.abs(a - b).reshape(5, -1).max(axis=1) / s).max()


@pytest.mark.parametrize("cuts,viscous", [(((14, 10), (20,), (16,)), 0), (((14, 10), (12, 8), (16,)), 1),
                                          (((24,), (20,), (10, 6)), 1)])
def test_cut_periodic_cartesian_box_equals_the_uncut_one(cuts, viscous):
    wl = W.cartesian_periodic(viscous=viscous)
    g1 = O.Grid(wl)
    g1.metrics_compute(0.0)
    ref = g1.rhs(wl["U0"])
    blocks, grids = make_blocks(wl, cuts)
    out = O.rhs_blocks(grids, [b["U0"] for b in blocks])
    assert relerr(gather(blocks, out, ref.shape), ref) <= 1e-12
    dt = g1.cfl_dt(wl["U0"], 0.4)
    U = wl["U0"].copy()
    Us = [b["U0"].copy() for b in blocks]
    for s in range(2):
        g1.rk3_step(U, s * dt, dt)
        O.rk3_step_blocks(grids, Us, s * dt, dt)
    assert np.abs(U - wl["U0"]).max() > 1e-4
    assert relerr(gather(blocks, Us, U.shape), U) <= 1e-12


def test_block_linked_to_itself_is_the_periodic_wrap():
    wl = W.cartesian_periodic(ni=16, nj=12, nk=12, viscous=1)
    g1 = O.Grid(wl)
    g1.metrics_compute(0.0)
    ref = g1.rhs(wl["U0"])
    wl2 = dict(wl, params=dict(wl["params"], periodic=[0, 1, 1], bc=[5, 5, 0, 0, 0, 0]))
    g2 = O.Grid(wl2)
    g2.link(0, g2)
    g2.link(1, g2)
    g2.metrics_compute(0.0)
    assert relerr(g2.rhs(wl["U0"]), ref) <= 1e-12


def test_freestream_across_curved_block_interfaces():
    """Sec. 7 applied per block: each block's metrics satisfy the identities with its own (extrapolated)
    ghost geometry, and the exchanged ghost state of a uniform flow is that uniform flow."""
    wl = W.wall_box(ni=24, nj=20, nk=18, bc=(2, 2, 2, 2, 2, 2), viscous=1)
    rho, u, v, w, p = W.freestream_state(wl["U0"].shape[1:])
    wl["U0"] = W.conservative(rho, u, 0.3 * u, -0.2 * u, p)
    wl["params"]["p_out"] = float(p.flat[0])
    blocks, grids = make_blocks(wl, ((12, 12), (10, 10), (18,)))
    Us = [b["U0"].copy() for b in blocks]
    out = O.rhs_blocks(grids, Us)
    dt = min(g.cfl_dt(b["U0"], 0.4) for g, b in zip(grids, blocks))
    assert max(np.abs(dt * o).max() for o in out) <= 1e-12
    for s in range(3):
        O.rk3_step_blocks(grids, Us, s * dt, dt)
    for U, b in zip(Us, blocks):
        assert np.abs(U - b["U0"]).max() <= 1e-12


def test_link_validation():
    wl = W.cartesian_periodic(ni=16, nj=12, nk=12, viscous=0)
    blocks, _ = W.split_blocks(wl, ((10, 6), (12,), (12,)))
    a, b = O.Grid(blocks[0]), O.Grid(blocks[1])
    a.link(1, b)
    with pytest.raises(ValueError):
        O.Grid(wl).link(1, b)                       # face of a periodic direction
    other, _ = W.split_blocks(W.cartesian_periodic(ni=16, nj=14, nk=12, viscous=0), ((10, 6), (14,), (12,)))
    with pytest.raises(ValueError):
        a.link(1, O.Grid(other[1]))                 # transverse sizes differ
