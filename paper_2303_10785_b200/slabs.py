"""Slab decomposition over ranks: one block per process, interface layers carried by torch.distributed.

Host logic only -- which layers go where, in which order, at which point of an RK stage.  Every kernel is the
library's (include/meg6.h, "Staged stepping"); the exchange is point-to-point (`batch_isend_irecv`: NCCL over
NVLink for CUDA tensors, gloo for the CPU tests), one message per interface face and stage: six cell layers of the
six primitive fields over the padded transverse extent, i.e. (ni+16)(nj+12) * 36 doubles per zeta face.

A `block` is any object with the staged methods of `paper_2303_10785_b200.Grid` (new_interface_buffer,
set_interface_buffer, stage_prim, stage_pack, stage_ghosts, stage_sweeps, and for the geometry
new_geom_interface_buffer, set_geom_interface_buffer, stage_geom_centres / _pack / _extend / _finish) -- the tests drive the same
class with an adapter around the CPU oracle on two gloo ranks.
"""
import torch.distributed as dist


def slab_cuts(n, parts):
    """cell counts of `parts` nearly equal slabs of n cells (larger ones first)"""
    q, r = divmod(n, parts)
    return tuple(q + (1 if p < r else 0) for p in range(parts))


class SlabStepper:
    """Advances one block whose interface faces `remote` = {face: peer rank} belong to blocks of other ranks.

    Message order per pair of ranks is fixed (faces in increasing order on the sending side, their opposite faces in
    that same order on the receiving side), so the two messages a rank pair exchanges across a periodic wrap with two
    ranks cannot be confused; gloo additionally gets tags.
    """

    def __init__(self, block, remote, moving=False, group=None, offsets=None):
        self.block = block
        self.remote = dict(remote)
        self.moving = moving
        self.group = group
        self.send = {f: block.new_interface_buffer(f) for f in self.remote}
        self.recv = {f: block.new_interface_buffer(f) for f in self.remote}
        for f, buf in self.recv.items():
            block.set_interface_buffer(f, buf)
        # geometry: the ten ghost layers of cell-centre coordinates (and grid velocities) beyond an interface face are
        # the neighbour's own cell centres (+ the period across a wrap-around link), so that both ranks difference the
        # same coordinates across the cut; static meshes exchange them once, moving ones at every stage time
        offsets = offsets or {}
        self.gsend = {f: block.new_geom_interface_buffer(f) for f in self.remote}
        self.grecv = {f: block.new_geom_interface_buffer(f) for f in self.remote}
        for f, buf in self.grecv.items():
            block.set_geom_interface_buffer(f, buf, offsets.get(f))

    def _swap(self, faces, send, recv):
        ops = []
        for f in faces:                       # my layers next to face f feed the peer's ghosts of its face f ^ 1
            ops.append(dist.P2POp(dist.isend, send[f], self.remote[f], group=self.group, tag=f ^ 1))
        for f in sorted(faces, key=lambda f: f ^ 1):   # the peer sent them in the order of ITS faces
            ops.append(dist.P2POp(dist.irecv, recv[f], self.remote[f], group=self.group, tag=f))
        for w in dist.batch_isend_irecv(ops):
            w.wait()

    def metrics_compute(self, t=0.0):
        """meg6_metrics_compute for a block with remote neighbours: centres, then per direction [exchange the
        cell-centre layers of that direction's interface faces, extend], then the metrics"""
        self.block.stage_geom_centres(t)
        for d in range(3):
            faces = [f for f in sorted(self.remote) if f // 2 == d]
            for f in faces:
                self.block.stage_geom_pack(f, self.gsend[f])
            if faces:
                self._swap(faces, self.gsend, self.grecv)
            self.block.stage_geom_extend(d)
        self.block.stage_geom_finish()

    def _exchange(self, s, d):
        faces = [f for f in sorted(self.remote) if f // 2 == d]
        if not faces:
            return
        for f in faces:
            self.block.stage_pack(s, f, self.send[f])
        self._swap(faces, self.send, self.recv)

    def _ghosts(self, s):
        for d in range(3):
            self._exchange(s, d)
            self.block.stage_ghosts(s, d)

    def rhs(self, U, out):
        self.block.stage_prim(U)
        self._ghosts(0)
        self.block.stage_sweeps(U, 0, 0.0, out=out)
        return out

    def rk3_step(self, U, t, dt):
        ts = (t, t + dt, t + 0.5 * dt)
        for s in range(3):
            if self.moving:
                self.metrics_compute(ts[s])
            if s == 0:
                self.block.stage_prim(U)
            self._ghosts(s)
            self.block.stage_sweeps(U, s, dt)
