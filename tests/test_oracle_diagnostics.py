"""Pins of the oracle's kinetic-energy / enstrophy integrals (Eq. 54): closed forms
of the Taylor-Green field u = sin x cos y cos z, v = -cos x sin y cos z, w = 0 at unit density on [0, 2 pi]^3:
E_k = 1/8 and enstrophy = 3/8 (|omega|^2 averages to 1/8 + 1/8 + 4/8), volume (2 pi)^3 -- on a Cartesian and on a
wavy mesh, with the sixth-order (MEG6) and the fourth-order implicit (MIG4) shared gradients."""
import numpy as np
import pytest

import workloads as W
from oracle import meg6_oracle as O


def tgv_unit_density(n, amp, scheme):
    L = 2 * np.pi
    x, y, z = W.wavy_periodic_grid(n, L, amp)
    xc, yc, zc = W.cell_centres(x), W.cell_centres(y), W.cell_centres(z)
    one = np.ones_like(xc)
    u = np.sin(xc) * np.cos(yc) * np.cos(zc)
    v = -np.cos(xc) * np.sin(yc) * np.cos(zc)
    prm = W._base_params(n, n, n, period=[[L, 0, 0], [0, L, 0], [0, 0, L]], scheme=scheme)
    return dict(params=prm, x=x, y=y, z=z), W.conservative(one, u, v, 0 * one, 100 * one)


@pytest.mark.parametrize("amp", [0.0, 0.05])
@pytest.mark.parametrize("scheme,order", [(0, 6), (1, 4)])
def test_kinetic_energy_enstrophy_volume_closed_forms(amp, scheme, order):
    errs = []
    for n in (16, 32):
        wl, U = tgv_unit_density(n, amp, scheme)
        g = O.Grid(wl)
        g.metrics_compute(0.0)
        ke, en, vol = g.diagnostics(U)
        assert abs(vol - (2 * np.pi) ** 3) <= 1e-9
        assert abs(ke - 0.125) <= 1e-10
        errs.append(abs(en - 0.375))
    assert errs[1] < 1e-4
    assert np.log2(errs[0] / errs[1]) > order - 0.6, errs
