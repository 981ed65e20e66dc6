"""Slab decomposition over ranks (paper_2303_10785_b200/slabs.py): the host logic -- which interface layers go to
which rank, in which order, at which point of an RK stage -- exercised with two gloo ranks on CPU.  The compute
backend of this test is an adapter around the CPU oracle with the staged methods of the CUDA Grid; the expected result
is the oracle's single-process multi-block step on the same cut (itself pinned: cut == uncut, test_oracle_blocks)."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import workloads as W  # noqa: E402


class OracleBlock:
    """the staged interface of paper_2303_10785_b200.Grid on top of oracle.meg6_oracle.Grid (numpy state)"""

    def __init__(self, wl):
        from oracle import meg6_oracle as O
        self.g = O.Grid(wl)
        self.U0 = None

    def new_geom_interface_buffer(self, face):
        return torch.zeros(self.g.geom_interface_doubles(face), dtype=torch.float64)

    def set_geom_interface_buffer(self, face, layers, offset=None):
        self.g.set_geom_interface_buffer(face, layers.numpy(), offset)

    def stage_geom_centres(self, t):
        self.g.stage_geom_centres(t)

    def stage_geom_pack(self, face, layers):
        self.g.stage_geom_pack(face, layers.numpy())

    def stage_geom_extend(self, d):
        self.g.stage_geom_extend(d)

    def stage_geom_finish(self):
        self.g.stage_geom_finish()

    def new_interface_buffer(self, face):
        return torch.zeros(self.g.interface_doubles(face), dtype=torch.float64)

    def set_interface_buffer(self, face, layers):
        self.g.set_interface_buffer(face, layers.numpy())     # shares the tensor's memory

    def stage_prim(self, U):
        self.g.stage_prim(U)

    def stage_pack(self, s, face, layers):
        self.g.stage_pack(face, layers.numpy())

    def stage_ghosts(self, s, d):
        self.g.stage_ghosts(d)

    def stage_sweeps(self, U, s, dt, out=None):
        L = self.g.stage_rhs(U)
        if out is not None:
            out[...] = L
            return
        if s == 0:
            self.U0 = U.copy()
            U[...] = self.U0 + dt * L
        elif s == 1:
            U[...] = 3.0 / 4.0 * self.U0 + 1.0 / 4.0 * (U + dt * L)
        else:
            U[...] = 1.0 / 3.0 * self.U0 + 2.0 / 3.0 * (U + dt * L)
        self.g.stage_prim(U)      # the CUDA sweeps leave the primitives of the new state behind; so does this


def _case(kind):
    if kind == "periodic_zeta":      # two slabs, wrap-around: both faces of a rank talk to the same peer
        return W.cartesian_periodic(ni=12, nj=10, nk=22, viscous=1), ((12,), (10,), (12, 10))
    return W.wall_box(ni=14, nj=12, nk=22, viscous=1), ((14,), (12,), (10, 12))   # curved, walls outside, one interface


def _worker(rank, world, port, kind, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2303_10785_b200.slabs import SlabStepper
    wl, cuts = _case(kind)
    blocks, links = W.split_blocks(wl, cuts)
    blk = OracleBlock(blocks[rank])
    remote = {face: nb for home, face, nb in links if home == rank}
    st = SlabStepper(blk, remote, offsets=blocks[rank]["link_offset"])
    st.metrics_compute(0.0)
    U = blocks[rank]["U0"].copy()
    rhs = np.empty_like(U)
    st.rhs(U, rhs)
    dt = 2.0e-3
    for s in range(2):
        st.rk3_step(U, s * dt, dt)
    out[rank] = (rhs, U)
    dist.barrier()
    dist.destroy_process_group()


def _reference(kind):
    from oracle import meg6_oracle as O
    wl, cuts = _case(kind)
    blocks, links = W.split_blocks(wl, cuts)
    grids = [O.Grid(b) for b in blocks]
    W.link_all(grids, blocks, links)
    O.metrics_compute_blocks(grids, 0.0)
    rhs = O.rhs_blocks(grids, [b["U0"] for b in blocks])
    Us = [b["U0"].copy() for b in blocks]
    dt = 2.0e-3
    for s in range(2):
        O.rk3_step_blocks(grids, Us, s * dt, dt)
    return rhs, Us


def _run(kind, port):
    world = 2
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, kind, out), nprocs=world, join=True)
        res = dict(out)
    rhs, Us = _reference(kind)
    for r in range(world):
        assert np.array_equal(res[r][0], rhs[r])          # same arithmetic, same data: bit for bit
        assert np.array_equal(res[r][1], Us[r])
        assert np.abs(res[r][1] - _case(kind)[0]["U0"][(slice(None),) + W.split_blocks(*_case(kind))[0][r]["slices"]]).max() > 1e-5


def test_two_ranks_periodic_wrap_matches_single_process_blocks():
    _run("periodic_zeta", 29541)


def test_two_ranks_curved_blocks_with_walls_match_single_process_blocks():
    _run("curved_walls", 29542)


def test_slab_cuts():
    from paper_2303_10785_b200.slabs import slab_cuts
    assert slab_cuts(200, 8) == (25,) * 8
    assert slab_cuts(200, 3) == (67, 67, 66)
    assert sum(slab_cuts(384, 7)) == 384
