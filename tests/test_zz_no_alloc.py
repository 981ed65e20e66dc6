"""meg6_cfl_dt_noalloc (include/meg6.h): the Eq. B.2 / B.3 time step with its reduction scratch in a static device array
of the library -- for callers that may not allocate or wait.  Checked against the existing path (meg6_cfl_dt: scratch in
the caller's workspace, reduction finished on the host) within the tolerance the other GPU tests use for the time step
(rel 1e-12), on calls in a row that share the array.

Named test_zz_* so that pytest collects it last: the suite runs with `pytest -x`.
"""
import numpy as np
import pytest

import workloads as W

pytestmark = pytest.mark.gpu

DT_TOL = 1e-12


@pytest.fixture(scope="module")
def mods():
    import torch
    import paper_2303_10785_b200 as M
    assert torch.cuda.is_available()
    return torch, M


def perturbed(wl, seed):
    """a non-trivial state on the workload's mesh: the binding cell of the minimum is somewhere in the interior"""
    rng = np.random.default_rng(seed)
    sh = wl["U0"].shape[1:]
    g = 1.4
    p0 = float((g - 1) * (wl["U0"][4] - 0.5 * (wl["U0"][1] ** 2 + wl["U0"][2] ** 2 + wl["U0"][3] ** 2) / wl["U0"][0]).mean())
    return W.conservative(1.0 + 0.2 * rng.uniform(-1, 1, sh), *(0.4 * rng.uniform(-1, 1, sh) for _ in range(3)),
                          p0 * (1.0 + 0.2 * rng.uniform(-1, 1, sh)))


def test_no_alloc_time_step_equals_the_existing_path_on_calls_in_a_row(mods):
    torch, M = mods
    # a larger grid first (more partial minima in the shared array), then smaller ones: stale entries beyond a call's own
    # must not leak into it; viscous static, inviscid moving (time metric in Eq. B.2), MIG4, a ragged non-periodic mesh
    cases = [(W.c3_tgv(n=48), 0.0), (W.c2_dynamic_freestream(n=24), 0.13), (W.c3_tgv(n=20, scheme=1), 0.0),
             (W.c4_jet(ni=31, nj=17, nk=16), 0.0)]
    out = torch.full((1,), -1.0, dtype=torch.float64, device="cuda")
    for n, (wl, t) in enumerate(cases):
        g = M.Grid(wl)
        g.metrics_compute(t)
        for rep in range(2):                                  # two calls in a row on the same grid, different states
            U = torch.as_tensor(perturbed(wl, 10 * n + rep), device="cuda").contiguous()
            want = g.cfl_dt(U, 0.3)
            if n == 0 and rep == 0:
                g.cfl_dt_noalloc(U, 0.3, out)                 # first launch of the two kernels in this process: the
                torch.cuda.synchronize()                      # driver loads their code lazily (its memory, not ours)
            free0 = torch.cuda.mem_get_info()[0]
            g.cfl_dt_noalloc(U, 0.3, out)
            got = float(out.item())
            assert torch.cuda.mem_get_info()[0] == free0      # the call took no device memory
            assert got == pytest.approx(want, rel=DT_TOL), (wl["name"], rep, got, want)
            assert got > 0.0 and np.isfinite(got)
        g.close()


def test_no_alloc_time_step_rejects_grids_beyond_its_maximum_and_bad_calls(mods):
    torch, M = mods
    wl = W.c1_vortex(n=12)
    g = M.Grid(wl)
    U = torch.as_tensor(wl["U0"], device="cuda").contiguous()
    out = torch.zeros(1, dtype=torch.float64, device="cuda")
    with pytest.raises(M.Meg6Error, match="metrics_compute"):
        g.cfl_dt_noalloc(U, 0.2, out)                         # MEG6_ESTATE before the metrics, like meg6_cfl_dt
    g.close()
    # 257^3 = 16 974 593 cells > 2^24: rejected before anything is launched (no metrics needed to see that)
    n = 257
    L = 10.0
    x, y, z = W.wavy_periodic_grid(n, L, 0.0)
    prm = W._base_params(n, n, n, period=[[L, 0, 0], [0, L, 0], [0, 0, L]])
    big = M.Grid(dict(params=prm, x=x, y=y, z=z))
    Ub = torch.ones((5, n, n, n), dtype=torch.float64, device="cuda")
    with pytest.raises(M.Meg6Error, match="maximum 16777216"):
        big.cfl_dt_noalloc(Ub, 0.2, out)
    assert float(out.item()) == 0.0                           # nothing was written
    big.close()
