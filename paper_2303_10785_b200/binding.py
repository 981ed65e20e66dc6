"""ctypes binding of csrc/libmeg6.so -- same names as include/meg6.h, argument marshalling only.

PyTorch is used for device memory and streams.  Nothing here computes: every method forwards to the C ABI.
"""
import ctypes as C
import os

from . import build as _build

EXPORTS = ["meg6_workspace_bytes", "meg6_grid_create", "meg6_grid_destroy", "meg6_metrics_compute",
           "meg6_set_inflow", "meg6_set_sponge", "meg6_rhs", "meg6_rk3_step", "meg6_rk3_steps", "meg6_cfl_dt", "meg6_cfl_dt_noalloc",
           "meg6_diagnostics",
           "meg6_limiter_stats_enable", "meg6_limiter_stats", "meg6_set_branch_masks", "meg6_get_array", "meg6_profile_enable",
           "meg6_profile_read", "meg6_fp64_peak", "meg6_last_error",
           "meg6_version", "meg6_link_blocks", "meg6_link_blocks_oriented", "meg6_metrics_compute_blocks", "meg6_rhs_blocks",
           "meg6_rk3_step_blocks", "meg6_geom_interface_doubles", "meg6_set_geom_interface_buffer",
           "meg6_stage_geom_centres", "meg6_stage_geom_pack", "meg6_stage_geom_extend", "meg6_stage_geom_finish",
           "meg6_interface_doubles", "meg6_set_interface_buffer", "meg6_stage_prim", "meg6_stage_pack",
           "meg6_stage_ghosts", "meg6_stage_sweeps"]


class Meg6Error(RuntimeError):
    pass


class Params(C.Structure):
    _fields_ = [("ni", C.c_int), ("nj", C.c_int), ("nk", C.c_int),
                ("periodic", C.c_int * 3), ("period", (C.c_double * 3) * 3),
                ("scheme", C.c_int), ("viscous", C.c_int),
                ("gamma", C.c_double), ("r_gas", C.c_double), ("prandtl", C.c_double),
                ("mu_ref", C.c_double), ("t_ref", C.c_double), ("s_suth", C.c_double),
                ("mp_alpha", C.c_double), ("moving", C.c_int), ("omega", C.c_double),
                ("bc", C.c_int * 6), ("p_out", C.c_double)]


def make_params(cfg):
    p = Params()
    p.ni, p.nj, p.nk = cfg["ni"], cfg["nj"], cfg["nk"]
    for d in range(3):
        p.periodic[d] = int(cfg["periodic"][d])
        for c in range(3):
            p.period[d][c] = float(cfg["period"][d][c])
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
    return p


_lib = None
_vp = C.c_void_p


def lib_path():
    return _build.SO


def lib():
    """Loads (building first if the sources are newer) the CUDA library.  Raises if it cannot."""
    global _lib
    if _lib is None:
        so = _build.build()
        L = C.CDLL(so)
        L.meg6_workspace_bytes.restype = C.c_size_t
        L.meg6_workspace_bytes.argtypes = [C.POINTER(Params)]
        L.meg6_grid_create.restype = C.c_int
        L.meg6_grid_create.argtypes = [C.POINTER(Params)] + [_vp] * 6 + [_vp, C.c_size_t, _vp, C.POINTER(_vp)]
        L.meg6_grid_destroy.argtypes = [_vp]
        L.meg6_metrics_compute.restype = C.c_int
        L.meg6_metrics_compute.argtypes = [_vp, C.c_double]
        L.meg6_set_inflow.restype = C.c_int
        L.meg6_set_inflow.argtypes = [_vp, C.c_int, _vp]
        L.meg6_set_sponge.restype = C.c_int
        L.meg6_set_sponge.argtypes = [_vp, _vp, _vp]
        L.meg6_rhs.restype = C.c_int
        L.meg6_rhs.argtypes = [_vp, _vp, _vp]
        L.meg6_rk3_step.restype = C.c_int
        L.meg6_rk3_step.argtypes = [_vp, _vp, C.c_double, C.c_double]
        L.meg6_rk3_steps.restype = C.c_int
        L.meg6_rk3_steps.argtypes = [_vp, _vp, C.c_double, C.c_double, C.c_int]
        L.meg6_diagnostics.restype = C.c_int
        L.meg6_diagnostics.argtypes = [_vp, _vp, C.POINTER(C.c_double)]
        L.meg6_cfl_dt.restype = C.c_int
        L.meg6_cfl_dt.argtypes = [_vp, _vp, C.c_double, C.POINTER(C.c_double)]
        L.meg6_cfl_dt_noalloc.restype = C.c_int
        L.meg6_cfl_dt_noalloc.argtypes = [_vp, _vp, C.c_double, _vp]
        L.meg6_limiter_stats_enable.restype = C.c_int
        L.meg6_limiter_stats_enable.argtypes = [_vp, C.c_int]
        L.meg6_limiter_stats.restype = C.c_int
        L.meg6_limiter_stats.argtypes = [_vp, C.POINTER(C.c_ulonglong), C.POINTER(C.c_ulonglong)]
        L.meg6_set_branch_masks.restype = C.c_int
        L.meg6_set_branch_masks.argtypes = [_vp, _vp, _vp, _vp]
        L.meg6_get_array.restype = C.c_int
        L.meg6_get_array.argtypes = [_vp, C.c_int, C.c_int, _vp]
        L.meg6_profile_enable.restype = C.c_int
        L.meg6_profile_enable.argtypes = [_vp, C.c_int]
        L.meg6_profile_read.restype = C.c_int
        L.meg6_profile_read.argtypes = [_vp, C.POINTER(C.c_double), C.POINTER(C.c_ulonglong)]
        L.meg6_link_blocks.restype = C.c_int
        L.meg6_link_blocks.argtypes = [_vp, C.c_int, _vp]
        L.meg6_link_blocks_oriented.restype = C.c_int
        L.meg6_link_blocks_oriented.argtypes = [_vp, C.c_int, _vp, C.c_int, C.c_int, C.c_int, C.c_int,
                                                C.POINTER(C.c_double)]
        L.meg6_metrics_compute_blocks.restype = C.c_int
        L.meg6_metrics_compute_blocks.argtypes = [C.c_int, C.POINTER(_vp), C.c_double]
        L.meg6_geom_interface_doubles.restype = C.c_size_t
        L.meg6_geom_interface_doubles.argtypes = [_vp, C.c_int]
        L.meg6_set_geom_interface_buffer.restype = C.c_int
        L.meg6_set_geom_interface_buffer.argtypes = [_vp, C.c_int, _vp, C.POINTER(C.c_double)]
        L.meg6_stage_geom_centres.restype = C.c_int
        L.meg6_stage_geom_centres.argtypes = [_vp, C.c_double]
        L.meg6_stage_geom_pack.restype = C.c_int
        L.meg6_stage_geom_pack.argtypes = [_vp, C.c_int, _vp]
        L.meg6_stage_geom_extend.restype = C.c_int
        L.meg6_stage_geom_extend.argtypes = [_vp, C.c_int]
        L.meg6_stage_geom_finish.restype = C.c_int
        L.meg6_stage_geom_finish.argtypes = [_vp]
        L.meg6_rhs_blocks.restype = C.c_int
        L.meg6_rhs_blocks.argtypes = [C.c_int, C.POINTER(_vp), C.POINTER(_vp), C.POINTER(_vp)]
        L.meg6_rk3_step_blocks.restype = C.c_int
        L.meg6_rk3_step_blocks.argtypes = [C.c_int, C.POINTER(_vp), C.POINTER(_vp), C.c_double, C.c_double]
        L.meg6_interface_doubles.restype = C.c_size_t
        L.meg6_interface_doubles.argtypes = [_vp, C.c_int]
        L.meg6_set_interface_buffer.restype = C.c_int
        L.meg6_set_interface_buffer.argtypes = [_vp, C.c_int, _vp]
        L.meg6_stage_prim.restype = C.c_int
        L.meg6_stage_prim.argtypes = [_vp, _vp]
        L.meg6_stage_pack.restype = C.c_int
        L.meg6_stage_pack.argtypes = [_vp, C.c_int, C.c_int, _vp]
        L.meg6_stage_ghosts.restype = C.c_int
        L.meg6_stage_ghosts.argtypes = [_vp, C.c_int, C.c_int]
        L.meg6_stage_sweeps.restype = C.c_int
        L.meg6_stage_sweeps.argtypes = [_vp, _vp, _vp, C.c_int, C.c_double]
        L.meg6_fp64_peak.restype = C.c_int
        L.meg6_fp64_peak.argtypes = [_vp, _vp, C.POINTER(C.c_double)]
        L.meg6_last_error.restype = C.c_char_p
        L.meg6_version.restype = C.c_int
        _lib = L
    return _lib


def _check(status, what):
    if status != 0:
        raise Meg6Error("%s failed (status %d): %s" % (what, status, lib().meg6_last_error().decode()))


class Grid:
    """Handle around meg6_grid.  All tensors are torch CUDA float64; U is (5, nk, nj, ni) contiguous."""

    def __init__(self, wl, device="cuda:0", stream=None):
        import torch
        if not torch.cuda.is_available():
            raise Meg6Error("no CUDA device: the MEG6 path has no CPU fallback")
        L = lib()
        self.torch = torch
        self.device = torch.device(device)
        self.cfg = wl["params"]
        self.p = make_params(self.cfg)
        self.shape = (self.cfg["nk"], self.cfg["nj"], self.cfg["ni"])
        nbytes = L.meg6_workspace_bytes(C.byref(self.p))
        if nbytes == 0:
            raise Meg6Error("meg6_workspace_bytes: " + L.meg6_last_error().decode())
        self.workspace_bytes = nbytes
        with torch.cuda.device(self.device):
            self.ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            base = (self.ws.data_ptr() + 255) // 256 * 256
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            dev = lambda a: torch.as_tensor(a, dtype=torch.float64).contiguous().to(self.device)
            x, y, z = dev(wl["x"]), dev(wl["y"]), dev(wl["z"])
            modes = [None, None, None]
            if self.p.moving:
                modes = [dev(wl["dx_mode"]), dev(wl["dy_mode"]), dev(wl["dz_mode"])]
            h = _vp()
            _check(L.meg6_grid_create(C.byref(self.p), x.data_ptr(), y.data_ptr(), z.data_ptr(),
                                      *(m.data_ptr() if m is not None else None for m in modes),
                                      base, nbytes, self.stream.cuda_stream, C.byref(h)), "meg6_grid_create")
            self.h = h
            for face, pin in wl.get("inflow", {}).items():
                t = dev(pin)
                _check(L.meg6_set_inflow(self.h, int(face), t.data_ptr()), "meg6_set_inflow")
            self.sigma = self.uref = None
            if wl.get("sigma") is not None:
                self.sigma, self.uref = dev(wl["sigma"]), dev(wl["U_ref"])
                _check(L.meg6_set_sponge(self.h, self.sigma.data_ptr(), self.uref.data_ptr()), "meg6_set_sponge")
            self.stream.synchronize()   # node / inflow staging copies done before the temporaries die

    def close(self):
        if getattr(self, "h", None):
            self.torch.cuda.synchronize(self.device)
            lib().meg6_grid_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _chk_state(self, U):
        assert U.is_cuda and U.dtype == self.torch.float64 and U.is_contiguous() and tuple(U.shape) == (5,) + self.shape

    def metrics_compute(self, t=0.0):
        _check(lib().meg6_metrics_compute(self.h, float(t)), "meg6_metrics_compute")

    def rhs(self, U, out=None):
        self._chk_state(U)
        if out is None:
            out = self.torch.empty_like(U)
        _check(lib().meg6_rhs(self.h, U.data_ptr(), out.data_ptr()), "meg6_rhs")
        return out

    def rk3_step(self, U, t, dt):
        self._chk_state(U)
        _check(lib().meg6_rk3_step(self.h, U.data_ptr(), float(t), float(dt)), "meg6_rk3_step")

    def rk3_steps(self, U, t, dt, nsteps):
        self._chk_state(U)
        _check(lib().meg6_rk3_steps(self.h, U.data_ptr(), float(t), float(dt), int(nsteps)), "meg6_rk3_steps")

    def link(self, face, neighbour, nb_face=None, swap=0, flip_a=0, flip_b=0, offset=None):
        """block interface (bc 5): ghost cells of `face` come from `neighbour` (its face nb_face, default the opposite
        one; orientation of the transverse axes: swap / flip_a / flip_b; offset added to its coordinates seen from here)"""
        if nb_face is None and not (swap or flip_a or flip_b) and offset is None:
            _check(lib().meg6_link_blocks(self.h, int(face), neighbour.h), "meg6_link_blocks")
        else:
            off = (C.c_double * 3)(*(offset if offset is not None else (0.0, 0.0, 0.0)))
            _check(lib().meg6_link_blocks_oriented(self.h, int(face), neighbour.h,
                                                   int(face) ^ 1 if nb_face is None else int(nb_face), int(swap),
                                                   int(flip_a), int(flip_b), off), "meg6_link_blocks_oriented")
        self._links = getattr(self, "_links", []) + [neighbour]   # keep the neighbour alive

    # ---- staged geometry (include/meg6.h): the pieces paper_2303_10785_b200.slabs drives ----
    def new_geom_interface_buffer(self, face):
        n = lib().meg6_geom_interface_doubles(self.h, int(face))
        return self.torch.zeros(n, dtype=self.torch.float64, device=self.device)

    def set_geom_interface_buffer(self, face, layers, offset=None):
        assert layers.is_cuda and layers.dtype == self.torch.float64 and layers.is_contiguous()
        off = (C.c_double * 3)(*(offset if offset is not None else (0.0, 0.0, 0.0)))
        _check(lib().meg6_set_geom_interface_buffer(self.h, int(face), layers.data_ptr(), off),
               "meg6_set_geom_interface_buffer")
        if not hasattr(self, "_gbufs"):
            self._gbufs = {}
        self._gbufs[int(face)] = layers   # keep it alive

    def stage_geom_centres(self, t):
        _check(lib().meg6_stage_geom_centres(self.h, float(t)), "meg6_stage_geom_centres")

    def stage_geom_pack(self, face, layers):
        _check(lib().meg6_stage_geom_pack(self.h, int(face), layers.data_ptr()), "meg6_stage_geom_pack")

    def stage_geom_extend(self, d):
        _check(lib().meg6_stage_geom_extend(self.h, int(d)), "meg6_stage_geom_extend")

    def stage_geom_finish(self):
        _check(lib().meg6_stage_geom_finish(self.h), "meg6_stage_geom_finish")

    # ---- staged stepping (include/meg6.h "Staged stepping"): the pieces paper_2303_10785_b200.slabs drives ----
    def new_interface_buffer(self, face):
        n = lib().meg6_interface_doubles(self.h, int(face))
        return self.torch.zeros(n, dtype=self.torch.float64, device=self.device)

    def set_interface_buffer(self, face, layers):
        assert layers.is_cuda and layers.dtype == self.torch.float64 and layers.is_contiguous()
        _check(lib().meg6_set_interface_buffer(self.h, int(face), layers.data_ptr()), "meg6_set_interface_buffer")
        if not hasattr(self, "_ibufs"):
            self._ibufs = {}
        self._ibufs[int(face)] = layers   # keep it alive

    def stage_prim(self, U):
        self._chk_state(U)
        _check(lib().meg6_stage_prim(self.h, U.data_ptr()), "meg6_stage_prim")

    def stage_pack(self, s, face, layers):
        _check(lib().meg6_stage_pack(self.h, int(s), int(face), layers.data_ptr()), "meg6_stage_pack")

    def stage_ghosts(self, s, d):
        _check(lib().meg6_stage_ghosts(self.h, int(s), int(d)), "meg6_stage_ghosts")

    def stage_sweeps(self, U, s, dt, out=None):
        self._chk_state(U)
        _check(lib().meg6_stage_sweeps(self.h, U.data_ptr(), out.data_ptr() if out is not None else None, int(s),
                                       float(dt)), "meg6_stage_sweeps")

    def diagnostics(self, U):
        """(kinetic energy, enstrophy, volume) of the state U, Eq. 54"""
        out = (C.c_double * 3)()
        _check(lib().meg6_diagnostics(self.h, U.data_ptr(), out), "meg6_diagnostics")
        return [out[0], out[1], out[2]]

    def cfl_dt(self, U, cfl):
        self._chk_state(U)
        dt = C.c_double()
        _check(lib().meg6_cfl_dt(self.h, U.data_ptr(), float(cfl), C.byref(dt)), "meg6_cfl_dt")
        return dt.value

    def cfl_dt_noalloc(self, U, cfl, out):
        """meg6_cfl_dt_noalloc: the time step into `out`, a one-element CUDA float64 tensor of the caller's (no
        allocation, no host copy, no synchronisation; grids of at most 2^24 cells)"""
        self._chk_state(U)
        assert out.is_cuda and out.dtype == self.torch.float64 and out.numel() == 1
        _check(lib().meg6_cfl_dt_noalloc(self.h, U.data_ptr(), float(cfl), out.data_ptr()), "meg6_cfl_dt_noalloc")
        return out

    def limiter_stats_enable(self, on=True):
        _check(lib().meg6_limiter_stats_enable(self.h, int(on)), "meg6_limiter_stats_enable")

    def limiter_stats(self):
        a, b = C.c_ulonglong(), C.c_ulonglong()
        _check(lib().meg6_limiter_stats(self.h, C.byref(a), C.byref(b)), "meg6_limiter_stats")
        return a.value, b.value

    def branch_masks_enable(self, on=True):
        """allocates (or drops) the three per-interface branch-record arrays and hands them to the library"""
        if on:
            t = self.torch
            nk, nj, ni = self.shape
            self.branch_mask = [t.zeros((nk, nj, ni + 1), dtype=t.int16, device=self.device),
                                t.zeros((nk, nj + 1, ni), dtype=t.int16, device=self.device),
                                t.zeros((nk + 1, nj, ni), dtype=t.int16, device=self.device)]
            ptrs = [m.data_ptr() for m in self.branch_mask]
        else:
            self.branch_mask, ptrs = None, [None, None, None]
        _check(lib().meg6_set_branch_masks(self.h, *ptrs), "meg6_set_branch_masks")

    def branch_mask_host(self, d):
        """numpy uint16 copy of the record of family d (bits: include/meg6.h)"""
        import numpy as np
        return self.branch_mask[d].cpu().numpy().view(np.uint16)

    PROFILE_KINDS = ["metrics", "prim", "ghost", "grad", "flux_xi", "flux_eta", "flux_zeta", "update",
                     "copy_Un", "cfl"]

    def profile_enable(self, on=True):
        _check(lib().meg6_profile_enable(self.h, int(on)), "meg6_profile_enable")

    def profile_read(self):
        """{kind: (milliseconds, kernel launches)} since the last read"""
        ms = (C.c_double * 16)()
        n = (C.c_ulonglong * 16)()
        _check(lib().meg6_profile_read(self.h, ms, n), "meg6_profile_read")
        return {k: (ms[i], n[i]) for i, k in enumerate(self.PROFILE_KINDS)}

    def get_array(self, kind, which):
        import numpy as np
        shp = list(self.shape)
        if kind == 1:
            shp[2 - which // 16] += 1
        out = np.empty(shp, dtype=np.float64)
        _check(lib().meg6_get_array(self.h, kind, which, out.ctypes.data), "meg6_get_array")
        return out


def fp64_peak(device="cuda:0"):
    """measured FP64-pipe roof of the device in DFMA thread-instructions per second (meg6_fp64_peak)"""
    import torch
    dev = torch.device(device)
    with torch.cuda.device(dev):
        scratch = torch.zeros(1, dtype=torch.float64, device=dev)
        r = C.c_double()
        _check(lib().meg6_fp64_peak(torch.cuda.current_stream(dev).cuda_stream, scratch.data_ptr(), C.byref(r)),
               "meg6_fp64_peak")
    return r.value


def _ptr_array(ptrs):
    return (_vp * len(ptrs))(*ptrs)


def metrics_compute_blocks(grids, t=0.0):
    """geometry of several linked blocks together (meg6_metrics_compute_blocks)"""
    _check(lib().meg6_metrics_compute_blocks(len(grids), _ptr_array([g.h.value for g in grids]), float(t)),
           "meg6_metrics_compute_blocks")


def rhs_blocks(grids, Us, outs=None):
    """dQ/dt of several linked blocks (meg6_rhs_blocks); returns the list of output tensors"""
    for g, U in zip(grids, Us):
        g._chk_state(U)
    if outs is None:
        outs = [g.torch.empty_like(U) for g, U in zip(grids, Us)]
    _check(lib().meg6_rhs_blocks(len(grids), _ptr_array([g.h.value for g in grids]),
                                 _ptr_array([U.data_ptr() for U in Us]), _ptr_array([o.data_ptr() for o in outs])),
           "meg6_rhs_blocks")
    return outs


def rk3_step_blocks(grids, Us, t, dt):
    """one SSP-RK3 step of several linked blocks, in place (meg6_rk3_step_blocks)"""
    for g, U in zip(grids, Us):
        g._chk_state(U)
    _check(lib().meg6_rk3_step_blocks(len(grids), _ptr_array([g.h.value for g in grids]),
                                      _ptr_array([U.data_ptr() for U in Us]), float(t), float(dt)),
           "meg6_rk3_step_blocks")
