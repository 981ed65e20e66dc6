"""ctypes binding of the CPU ORACLE (oracle/meg6_oracle.cpp).

Test infrastructure, NOT the product: only tests/, bench.py's cpu_baseline / --impl reference legs and
__graft_entry__.smoke() may import this module.  It imports nothing from paper_2303_10785_b200.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
# MEG6_ORACLE_SO: load another build of the SAME source (tests/test_oracle_sensitivity.py builds one with FMA
# contraction switched on to measure how far rounding order alone moves the oracle)
_SO = os.environ.get("MEG6_ORACLE_SO") or os.path.join(_HERE, "libmeg6_oracle.so")
_SRC = [os.path.join(_HERE, "meg6_oracle.cpp"), os.path.join(_HERE, "meg6_oracle.h")]


def build(force=False):
    """Compile the oracle with the system g++ (-O2 -ffp-contract=off, OpenMP if available)."""
    if os.environ.get("MEG6_ORACLE_SO"):
        return _SO
    if not force and os.path.exists(_SO) and all(os.path.getmtime(_SO) >= os.path.getmtime(s) for s in _SRC):
        return _SO
    base = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fPIC", "-shared", "-o", _SO, _SRC[0]]
    r = subprocess.run(base[:4] + ["-fopenmp"] + base[4:], capture_output=True, text=True)
    if r.returncode != 0:
        r = subprocess.run(base, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("oracle build failed:\n" + r.stderr)
    return _SO


class Params(C.Structure):
    _fields_ = [("ni", C.c_int), ("nj", C.c_int), ("nk", C.c_int),
                ("periodic", C.c_int * 3), ("period", (C.c_double * 3) * 3),
                ("scheme", C.c_int), ("viscous", C.c_int),
                ("gamma", C.c_double), ("r_gas", C.c_double), ("prandtl", C.c_double),
                ("mu_ref", C.c_double), ("t_ref", C.c_double), ("s_suth", C.c_double),
                ("mp_alpha", C.c_double), ("moving", C.c_int), ("omega", C.c_double),
                ("bc", C.c_int * 6), ("p_out", C.c_double), ("metric_form", C.c_int)]


_lib = None
_dp = C.POINTER(C.c_double)


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_SO)
        L.meg6o_create.restype = C.c_void_p
        L.meg6o_create.argtypes = [C.POINTER(Params)] + [_dp] * 6
        L.meg6o_destroy.argtypes = [C.c_void_p]
        L.meg6o_set_threads.argtypes = [C.c_int]
        L.meg6o_get_threads.restype = C.c_int
        L.meg6o_metrics_compute.argtypes = [C.c_void_p, C.c_double]
        L.meg6o_set_centres.argtypes = [C.c_void_p, _dp, _dp, _dp]
        L.meg6o_set_inflow.argtypes = [C.c_void_p, C.c_int, _dp]
        L.meg6o_set_sponge.argtypes = [C.c_void_p, _dp, _dp]
        L.meg6o_rhs.argtypes = [C.c_void_p, _dp, _dp]
        L.meg6o_rk3_step.argtypes = [C.c_void_p, _dp, C.c_double, C.c_double]
        L.meg6o_link_blocks.restype = C.c_int
        L.meg6o_link_blocks.argtypes = [C.c_void_p, C.c_int, C.c_void_p]
        L.meg6o_link_blocks_oriented.restype = C.c_int
        L.meg6o_link_blocks_oriented.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, _dp]
        L.meg6o_metrics_compute_blocks.argtypes = [C.c_int, C.POINTER(C.c_void_p), C.c_double]
        L.meg6o_geom_interface_doubles.restype = C.c_size_t
        L.meg6o_geom_interface_doubles.argtypes = [C.c_void_p, C.c_int]
        L.meg6o_set_geom_interface_buffer.argtypes = [C.c_void_p, C.c_int, C.c_void_p, _dp]
        L.meg6o_stage_geom_centres.argtypes = [C.c_void_p, C.c_double]
        L.meg6o_stage_geom_pack.argtypes = [C.c_void_p, C.c_int, C.c_void_p]
        L.meg6o_stage_geom_extend.argtypes = [C.c_void_p, C.c_int]
        L.meg6o_stage_geom_finish.argtypes = [C.c_void_p]
        L.meg6o_rhs_blocks.argtypes = [C.c_int, C.POINTER(C.c_void_p), C.POINTER(C.c_void_p), C.POINTER(C.c_void_p)]
        L.meg6o_rk3_step_blocks.argtypes = [C.c_int, C.POINTER(C.c_void_p), C.POINTER(C.c_void_p), C.c_double, C.c_double]
        L.meg6o_interface_doubles.restype = C.c_size_t
        L.meg6o_interface_doubles.argtypes = [C.c_void_p, C.c_int]
        L.meg6o_set_interface_buffer.argtypes = [C.c_void_p, C.c_int, C.c_void_p]
        L.meg6o_stage_prim.argtypes = [C.c_void_p, _dp]
        L.meg6o_stage_ghosts.argtypes = [C.c_void_p, C.c_int]
        L.meg6o_stage_pack.argtypes = [C.c_void_p, C.c_int, C.c_void_p]
        L.meg6o_stage_rhs.argtypes = [C.c_void_p, _dp, _dp]
        L.meg6o_cfl_dt.restype = C.c_double
        L.meg6o_cfl_dt.argtypes = [C.c_void_p, _dp, C.c_double]
        L.meg6o_diagnostics.argtypes = [C.c_void_p, _dp, _dp]
        L.meg6o_limiter_stats.argtypes = [C.c_void_p, C.POINTER(C.c_ulonglong), C.POINTER(C.c_ulonglong)]
        L.meg6o_branch_masks_enable.argtypes = [C.c_void_p, C.c_int]
        L.meg6o_get_branch_mask.restype = C.c_size_t
        L.meg6o_get_branch_mask.argtypes = [C.c_void_p, C.c_int, C.c_void_p]
        L.meg6o_get_cell.argtypes = [C.c_void_p, C.c_int, _dp]
        L.meg6o_get_face.argtypes = [C.c_void_p, C.c_int, C.c_int, _dp]
        L.meg6o_get_prim.argtypes = [C.c_void_p, C.c_int, _dp]
        L.meg6o_get_grad.argtypes = [C.c_void_p, C.c_int, C.c_int, _dp]
        L.meg6o_line_op.argtypes = [C.c_int, C.c_int, _dp, _dp]
        L.meg6o_eigen.argtypes = [_dp, C.c_double, C.c_double, _dp, _dp]
        L.meg6o_mp_limit.restype = C.c_double
        L.meg6o_mp_limit.argtypes = [C.c_double] * 7 + [C.POINTER(C.c_int)]
        L.meg6o_hllc.restype = C.c_int
        L.meg6o_hllc.argtypes = [_dp, _dp, _dp, C.c_double, _dp]
        L.meg6o_inviscid_face.argtypes = [_dp, _dp, _dp, _dp, C.c_double, C.c_double, _dp]
        L.meg6o_viscous_face.argtypes = [C.c_int, _dp, _dp, _dp, C.c_double, C.POINTER(Params), _dp]
        L.meg6o_sutherland.restype = C.c_double
        L.meg6o_sutherland.argtypes = [C.POINTER(Params), C.c_double]
        _lib = L
    return _lib


def _p(a):
    return a.ctypes.data_as(_dp)


def _c(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def make_params(cfg, metric_form=0):
    """cfg: the plain dict produced by workloads.* (keys = fields of the params struct)."""
    p = Params()
    p.ni, p.nj, p.nk = cfg.get("ni", 1), cfg.get("nj", 1), cfg.get("nk", 1)
    for d in range(3):
        p.periodic[d] = int(cfg.get("periodic", [1, 1, 1])[d])
        for c in range(3):
            p.period[d][c] = float(cfg.get("period", [[0.0] * 3] * 3)[d][c])
    p.scheme = int(cfg.get("scheme", 0))
    p.viscous = int(cfg.get("viscous", 0))
    p.gamma = cfg.get("gamma", 1.4)
    p.r_gas = cfg.get("r_gas", 1.0)
    p.prandtl = cfg.get("prandtl", 0.71)
    p.mu_ref = cfg.get("mu_ref", 0.0)
    p.t_ref = cfg.get("t_ref", 1.0)
    p.s_suth = cfg.get("s_suth", -1.0)
    p.mp_alpha = cfg.get("mp_alpha", 4.0)
    p.moving = int(cfg.get("moving", 0))
    p.omega = cfg.get("omega", 0.0)
    for f in range(6):
        p.bc[f] = int(cfg.get("bc", [0] * 6)[f])
    p.p_out = cfg.get("p_out", 0.0)
    p.metric_form = metric_form
    return p


def set_threads(n):
    lib().meg6o_set_threads(int(n))


def get_threads():
    return lib().meg6o_get_threads()


class Grid:
    """Oracle solver handle.  Arrays are numpy float64, U/dUdt shaped (5, nk, nj, ni)."""

    def __init__(self, wl, metric_form=0):
        L = lib()
        self.cfg = wl["params"]
        self.p = make_params(self.cfg, metric_form)
        self.shape = (self.cfg["nk"], self.cfg["nj"], self.cfg["ni"])
        x, y, z = (_c(wl["x"]), _c(wl["y"]), _c(wl["z"]))
        if self.p.moving:
            m = [_c(wl["dx_mode"]), _c(wl["dy_mode"]), _c(wl["dz_mode"])]
            self.h = L.meg6o_create(C.byref(self.p), _p(x), _p(y), _p(z), _p(m[0]), _p(m[1]), _p(m[2]))
        else:
            self.h = L.meg6o_create(C.byref(self.p), _p(x), _p(y), _p(z), None, None, None)
        if not self.h:
            raise ValueError("meg6o_create rejected the parameters (walls need a static mesh)")
        for face, pin in wl.get("inflow", {}).items():
            pin = _c(pin)
            L.meg6o_set_inflow(self.h, int(face), _p(pin))
        if wl.get("sigma") is not None:
            s, ur = _c(wl["sigma"]), _c(wl["U_ref"])
            L.meg6o_set_sponge(self.h, _p(s), _p(ur))

    def __del__(self):
        if getattr(self, "h", None):
            lib().meg6o_destroy(self.h)
            self.h = None

    def set_centres(self, xc, yc, zc):
        """tests only: padded (ghost 10) cell-centre coordinate arrays, shape (nk+20, nj+20, ni+20)"""
        a = [_c(xc), _c(yc), _c(zc)]
        lib().meg6o_set_centres(self.h, _p(a[0]), _p(a[1]), _p(a[2]))

    def metrics_compute(self, t=0.0):
        lib().meg6o_metrics_compute(self.h, float(t))

    def rhs(self, U):
        U = _c(U)
        out = np.empty_like(U)
        lib().meg6o_rhs(self.h, _p(U), _p(out))
        return out

    def rk3_step(self, U, t, dt):
        """In place on a contiguous float64 array."""
        assert U.flags.c_contiguous and U.dtype == np.float64
        lib().meg6o_rk3_step(self.h, _p(U), float(t), float(dt))

    def link(self, face, neighbour, nb_face=None, swap=0, flip_a=0, flip_b=0, offset=None):
        """block interface: ghost cells of `face` come from `neighbour` (its face nb_face, default the opposite one;
        orientation of the transverse axes: swap / flip_a / flip_b; offset added to its coordinates seen from here)"""
        off = _c(offset if offset is not None else [0.0, 0.0, 0.0])
        if nb_face is None and not (swap or flip_a or flip_b):
            rc = lib().meg6o_link_blocks(self.h, int(face), neighbour.h)
            if rc == 0 and offset is not None:
                rc = lib().meg6o_link_blocks_oriented(self.h, int(face), neighbour.h, int(face) ^ 1, 0, 0, 0, _p(off))
        else:
            rc = lib().meg6o_link_blocks_oriented(self.h, int(face), neighbour.h,
                                                  int(face) ^ 1 if nb_face is None else int(nb_face), int(swap),
                                                  int(flip_a), int(flip_b), _p(off))
        if rc != 0:
            raise ValueError("meg6o_link_blocks rejected the pair")
        self._links = getattr(self, "_links", []) + [neighbour]

    # staged geometry (blocks in different processes)
    def geom_interface_doubles(self, face):
        return int(lib().meg6o_geom_interface_doubles(self.h, int(face)))

    def set_geom_interface_buffer(self, face, layers, offset=None):
        assert layers.dtype == np.float64 and layers.flags["C_CONTIGUOUS"]
        off = _c(offset if offset is not None else [0.0, 0.0, 0.0])
        lib().meg6o_set_geom_interface_buffer(self.h, int(face), layers.ctypes.data, _p(off))

    def stage_geom_centres(self, t):
        lib().meg6o_stage_geom_centres(self.h, float(t))

    def stage_geom_pack(self, face, layers):
        assert layers.dtype == np.float64 and layers.flags["C_CONTIGUOUS"]
        lib().meg6o_stage_geom_pack(self.h, int(face), layers.ctypes.data)

    def stage_geom_extend(self, d):
        lib().meg6o_stage_geom_extend(self.h, int(d))

    def stage_geom_finish(self):
        lib().meg6o_stage_geom_finish(self.h)

    # staged evaluation (blocks in different processes); `layers` are numpy float64 arrays kept alive by the caller
    def interface_doubles(self, face):
        return int(lib().meg6o_interface_doubles(self.h, int(face)))

    def set_interface_buffer(self, face, layers):
        assert layers.dtype == np.float64 and layers.flags["C_CONTIGUOUS"]
        lib().meg6o_set_interface_buffer(self.h, int(face), layers.ctypes.data)

    def stage_prim(self, U):
        lib().meg6o_stage_prim(self.h, _p(U))

    def stage_ghosts(self, d):
        lib().meg6o_stage_ghosts(self.h, int(d))

    def stage_pack(self, face, layers):
        assert layers.dtype == np.float64 and layers.flags["C_CONTIGUOUS"]
        lib().meg6o_stage_pack(self.h, int(face), layers.ctypes.data)

    def stage_rhs(self, U):
        out = np.empty_like(U)
        lib().meg6o_stage_rhs(self.h, _p(U), _p(out))
        return out

    def diagnostics(self, U):
        """(kinetic energy, enstrophy, volume), Eq. 54"""
        U = _c(U)
        out = np.empty(3)
        lib().meg6o_diagnostics(self.h, _p(U), _p(out))
        return out

    def cfl_dt(self, U, cfl):
        U = _c(U)
        return lib().meg6o_cfl_dt(self.h, _p(U), float(cfl))

    def limiter_stats(self):
        a, b = C.c_ulonglong(), C.c_ulonglong()
        lib().meg6o_limiter_stats(self.h, C.byref(a), C.byref(b))
        return a.value, b.value

    def branch_masks_enable(self, on=True):
        lib().meg6o_branch_masks_enable(self.h, int(on))

    def branch_mask(self, d):
        """uint16 per interface of family d after the last rhs: bits 0-4 / 5-9 E.1 failed (left / right state of the
        five characteristic components), bits 10-11 branch of Eq. 26; shape as face(d, .)"""
        shp = list(self.shape)
        shp[2 - d] += 1
        out = np.empty(shp, dtype=np.uint16)
        n = lib().meg6o_get_branch_mask(self.h, int(d), out.ctypes.data)
        assert n == out.size, (n, out.size)
        return out

    def cell(self, which):
        out = np.empty(self.shape)
        lib().meg6o_get_cell(self.h, which, _p(out))
        return out

    def face(self, d, q):
        shp = list(self.shape)
        shp[2 - d] += 1
        out = np.empty(shp)
        lib().meg6o_get_face(self.h, d, q, _p(out))
        return out

    def prim(self, f):
        out = np.empty(self.shape)
        lib().meg6o_get_prim(self.h, f, _p(out))
        return out

    def grad(self, d, f):
        out = np.empty(self.shape)
        lib().meg6o_get_grad(self.h, d, f, _p(out))
        return out


def _vps(ptrs):
    return (C.c_void_p * len(ptrs))(*ptrs)


def metrics_compute_blocks(grids, t=0.0):
    """geometry of several linked blocks together (meg6o_metrics_compute_blocks)"""
    lib().meg6o_metrics_compute_blocks(len(grids), _vps([g.h for g in grids]), float(t))


def rhs_blocks(grids, Us):
    """dQ/dt of several linked blocks (meg6o_rhs_blocks)"""
    Us = [_c(U) for U in Us]
    outs = [np.empty_like(U) for U in Us]
    lib().meg6o_rhs_blocks(len(grids), _vps([g.h for g in grids]), _vps([U.ctypes.data for U in Us]),
                           _vps([o.ctypes.data for o in outs]))
    return outs


def rk3_step_blocks(grids, Us, t, dt):
    """in place; every U must be a contiguous float64 array"""
    for U in Us:
        assert U.flags["C_CONTIGUOUS"] and U.dtype == np.float64
    lib().meg6o_rk3_step_blocks(len(grids), _vps([g.h for g in grids]), _vps([U.ctypes.data for U in Us]),
                                float(t), float(dt))


# ---- fine-grained pieces ----
OPS = {"D1": 0, "D2": 1, "Lft": 2, "Rgt": 3, "H": 4, "delta": 5, "alpha_damp": 6, "C4": 7, "IG4": 8,
       "delta_IG4": 9, "H_IG4": 10}


def line_op(op, f):
    f = _c(f)
    out = np.empty_like(f)
    lib().meg6o_line_op(OPS[op], f.size, _p(f), _p(out))
    return out


def eigen(n, rho, a):
    n = _c(n)
    L, R = np.empty(25), np.empty(25)
    lib().meg6o_eigen(_p(n), float(rho), float(a), _p(L), _p(R))
    return L.reshape(5, 5), R.reshape(5, 5)


def mp_limit(w, c0, cm, cp, dm_near, dm_far, alpha=4.0):
    fl = C.c_int()
    v = lib().meg6o_mp_limit(w, c0, cm, cp, dm_near, dm_far, alpha, C.byref(fl))
    return v, fl.value


def hllc(PL, PR, m, gamma=1.4):
    PL, PR, m = _c(PL), _c(PR), _c(m)
    F = np.empty(5)
    br = lib().meg6o_hllc(_p(PL), _p(PR), _p(m), gamma, _p(F))
    return F, br


def inviscid_face(Pc, P1, P2, m, gamma=1.4, alpha=4.0):
    Pc, P1, P2, m = _c(Pc), _c(P1), _c(P2), _c(m)
    assert Pc.shape == (4, 5) and P1.shape == (2, 5) and P2.shape == (4, 5)
    F = np.empty(5)
    lib().meg6o_inviscid_face(_p(Pc), _p(P1), _p(P2), _p(m), gamma, alpha, _p(F))
    return F


def viscous_face(d, phi, g, mh, rj, cfg):
    phi, g, mh = _c(phi), _c(g), _c(mh)
    assert phi.shape == (2, 4) and g.shape == (2, 3, 4) and mh.shape == (9,)
    p = make_params(cfg)
    F = np.empty(5)
    lib().meg6o_viscous_face(d, _p(phi), _p(g), _p(mh), float(rj), C.byref(p), _p(F))
    return F


def sutherland(cfg, T):
    p = make_params(cfg)
    return lib().meg6o_sutherland(C.byref(p), float(T))
