"""ctypes binding of oracle/libsfh_oracle.so (test infrastructure only; see sfh_oracle.cpp).

The oracle keeps GHOSTED 12^3 blocks in host memory, in the caller's block order (20^3 for the build with blocks
of 16^3 cells, ncell = 16: the same source compiled with -DSFH_ORACLE_N=16).
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

N, G, M, NV = 8, 2, 12, 5


class Config(C.Structure):
    _fields_ = [("nb0", C.c_int32 * 3), ("ncell", C.c_int32), ("nghost", C.c_int32), ("max_level", C.c_int32),
                ("bc", (C.c_int32 * 2) * 3), ("box_len", C.c_double * 3), ("gamma", C.c_double), ("cfl", C.c_double),
                ("nscalar", C.c_int32)]


_libs = {}


def lib(ncell=N):
    if ncell not in _libs:
        path = _build.build(ncell=ncell)
        L = C.CDLL(path)
        L.orc_create_mesh.argtypes = [C.POINTER(Config), C.c_int64, C.c_void_p, C.c_void_p, C.POINTER(C.c_void_p)]
        L.orc_destroy_mesh.argtypes = [C.c_void_p]
        L.orc_last_error.argtypes = [C.c_void_p]
        L.orc_last_error.restype = C.c_char_p
        L.orc_bind.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_set_reflux.argtypes = [C.c_void_p, C.c_int]
        L.orc_is_leaf.argtypes = [C.c_void_p, C.c_int64]
        L.orc_cell_width.argtypes = [C.c_void_p, C.c_int]
        L.orc_cell_width.restype = C.c_double
        L.orc_num_registers.argtypes = [C.c_void_p, C.c_int]
        L.orc_num_registers.restype = C.c_int64
        L.orc_fill_ghosts.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_double]
        L.orc_predictor.argtypes = [C.c_void_p, C.c_int, C.c_double]
        L.orc_corrector.argtypes = [C.c_void_p, C.c_int, C.c_double]
        L.orc_zero_registers.argtypes = [C.c_void_p, C.c_int]
        L.orc_restrict.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int]
        L.orc_reflux.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_double]
        L.orc_copy_level.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int]
        L.orc_cfl_dt.argtypes = [C.c_void_p, C.c_int, C.c_int]
        L.orc_cfl_dt.restype = C.c_double
        L.orc_max_speed.argtypes = [C.c_void_p, C.c_int, C.c_int]
        L.orc_max_speed.restype = C.c_double
        L.orc_substep_exponent.argtypes = [C.c_double, C.c_double]
        L.orc_time_interp.argtypes = [C.c_double] * 4
        L.orc_time_interp.restype = C.c_double
        L.orc_hllc.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_double, C.c_void_p]
        L.orc_roe.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_double, C.c_void_p]
        L.orc_set_riemann.argtypes = [C.c_void_p, C.c_int]
        L.orc_minmod.argtypes = [C.c_double, C.c_double]
        L.orc_minmod.restype = C.c_double
        L.orc_get.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_void_p]
        L.orc_advance.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_double, C.POINTER(C.c_double), C.c_void_p]
        L.orc_status.argtypes = [C.c_void_p, C.c_int]
        L.orc_refine_indicator.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_double, C.c_void_p]
        L.orc_transfer_state.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_int]
        L.orc_status.restype = C.c_int64
        L.orc_regrid.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_double, C.c_double, C.POINTER(C.c_void_p)]
        L.orc_num_blocks.argtypes = [C.c_void_p]
        L.orc_num_blocks.restype = C.c_int64
        L.orc_block_list.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        _libs[ncell] = L
    return _libs[ncell]


def make_config(nb0, max_level, bc, box_len, gamma, cfl, nscalar=0, ncell=N):
    cfg = Config()
    cfg.nscalar = int(nscalar)
    for d in range(3):
        cfg.nb0[d] = int(nb0[d])
        cfg.box_len[d] = float(box_len[d])
        for s in range(2):
            cfg.bc[d][s] = int(bc[d][s])
    cfg.ncell, cfg.nghost, cfg.max_level = int(ncell), G, int(max_level)
    cfg.gamma, cfg.cfl = float(gamma), float(cfl)
    return cfg


def hllc(WL, WR, d, gamma):
    WL = np.ascontiguousarray(WL, dtype=np.float64)
    WR = np.ascontiguousarray(WR, dtype=np.float64)
    F = np.zeros(NV)
    lib().orc_hllc(WL.ctypes.data, WR.ctypes.data, int(d), float(gamma), F.ctypes.data)
    return F


def roe(WL, WR, d, gamma):
    WL = np.ascontiguousarray(WL, dtype=np.float64)
    WR = np.ascontiguousarray(WR, dtype=np.float64)
    F = np.zeros(NV)
    lib().orc_roe(WL.ctypes.data, WR.ctypes.data, int(d), float(gamma), F.ctypes.data)
    return F


class OracleMesh:
    """Oracle mesh + three ghosted state copies (0: U^n, 1: U^{n+1/2}, 2: U^{n+1})."""

    def __init__(self, nb0, max_level, bc, box_len, gamma, cfl, level, ijk, nscalar=0, handle=None, ncell=N):
        self.L = lib(ncell)
        self.n = int(ncell)                  # cells per block edge; ghosted blocks are (n + 4)^3
        self.nv = NV + int(nscalar)          # 5 hydro variables + passive scalars rho*s
        self.cfg = make_config(nb0, max_level, bc, box_len, gamma, cfl, nscalar, ncell)
        if handle is None:
            self.level = np.ascontiguousarray(level, dtype=np.int32)
            self.ijk = np.ascontiguousarray(ijk, dtype=np.int32).reshape(-1, 3)
            self.nb = len(self.level)
            self.h = C.c_void_p()
            rc = self.L.orc_create_mesh(C.byref(self.cfg), self.nb, self.level.ctypes.data, self.ijk.ctypes.data,
                                        C.byref(self.h))
            if rc != 0:
                raise ValueError("orc_create_mesh failed: %d" % rc)
        else:                                # a mesh the oracle built itself (orc_regrid): read its block list back
            self.h = handle
            self.nb = int(self.L.orc_num_blocks(self.h))
            self.level = np.zeros(self.nb, dtype=np.int32)
            self.ijk = np.zeros((self.nb, 3), dtype=np.int32)
            self.L.orc_block_list(self.h, self.level.ctypes.data, self.ijk.ctypes.data)
        self.U = [np.zeros((self.nb, self.nv) + (self.n + 2 * G,) * 3) for _ in range(3)]
        self.L.orc_bind(self.h, *[u.ctypes.data for u in self.U])
        self.max_level = int(max_level)
        self.t = C.c_double(0.0)
        self.nupd = np.zeros(self.max_level + 1, dtype=np.int64)

    def __del__(self):
        if getattr(self, "h", None):
            self.L.orc_destroy_mesh(self.h)
            self.h = None

    def _chk(self, rc):
        if rc != 0:
            raise RuntimeError("oracle error %d: %s" % (rc, self.L.orc_last_error(self.h).decode()))

    # state access (interior cells, [nb][5][8][8][8] indexed [b][v][k][j][i])
    def set_state(self, Uint, copy=0):
        n = self.n
        self.U[copy][:, :, G:G + n, G:G + n, G:G + n] = Uint

    def get_state(self, copy=0):
        n = self.n
        return self.U[copy][:, :, G:G + n, G:G + n, G:G + n].copy()

    def is_leaf(self):
        return np.array([self.L.orc_is_leaf(self.h, b) for b in range(self.nb)], dtype=bool)

    def cell_width(self, l):
        return self.L.orc_cell_width(self.h, l)

    def fill_ghosts(self, level=-1, which=0, interp=0, tau=0.0):
        self._chk(self.L.orc_fill_ghosts(self.h, level, which, interp, tau))

    def predictor(self, level, dt):
        self._chk(self.L.orc_predictor(self.h, level, dt))

    def corrector(self, level, dt):
        self._chk(self.L.orc_corrector(self.h, level, dt))

    def zero_registers(self, coarse_level=-1):
        self.L.orc_zero_registers(self.h, coarse_level)

    def restrict(self, coarse_level, src_copy=0, dst_copy=0):
        self.L.orc_restrict(self.h, coarse_level, src_copy, dst_copy)

    def restrict_all(self, copy=0):
        for l in range(self.max_level - 1, -1, -1):
            self.restrict(l, copy, copy)

    def reflux(self, coarse_level, copy, dt_coarse):
        self.L.orc_reflux(self.h, coarse_level, copy, dt_coarse)

    def copy_level(self, level, src, dst):
        self.L.orc_copy_level(self.h, level, src, dst)

    def cfl_dt(self, level=-1, copy=0):
        return self.L.orc_cfl_dt(self.h, level, copy)

    def max_speed(self, level, copy=0):
        return self.L.orc_max_speed(self.h, level, copy)

    def set_reflux(self, on):
        self.L.orc_set_reflux(self.h, int(on))

    def set_riemann(self, solver):
        """0 / "hllc": HLLC, 1 / "roe": Roe."""
        self._chk(self.L.orc_set_riemann(self.h, {"hllc": 0, "roe": 1}.get(solver, solver)))

    def advance(self, nsteps, mode=0, dt_fixed=0.0):
        self._chk(self.L.orc_advance(self.h, nsteps, mode, dt_fixed, C.byref(self.t), self.nupd.ctypes.data))
        return self.t.value

    def status(self, copy=0):
        return self.L.orc_status(self.h, copy)

    def transfer_from(self, src, which=0):
        """State copy `which` of this (new) mesh from the old mesh `src` after a regrid: copies and prolongations."""
        self._chk(self.L.orc_transfer_state(src.h, which, self.h, which))

    def regrid(self, criterion, threshold, which=0, G=1.0):
        """The regridded mesh (blocks flagged where the indicator >= threshold get children, 2:1 padded) holding the
        state of copy `which` moved onto it (orc_regrid + orc_transfer_state)."""
        h = C.c_void_p()
        self._chk(self.L.orc_regrid(self.h, which, criterion, float(G), float(threshold), C.byref(h)))
        c = self.cfg
        new = OracleMesh(tuple(c.nb0), c.max_level, [tuple(b) for b in c.bc], tuple(c.box_len), c.gamma, c.cfl, None, None,
                         nscalar=c.nscalar, handle=h)
        new.transfer_from(self, which)
        return new

    def refine_indicator(self, criterion=0, which=0, G=1.0):
        """Per-block refinement indicator (0: eq. 33-34 curvature, 1: h / Jeans length); ghosts must be filled."""
        out = np.zeros(self.nb)
        self._chk(self.L.orc_refine_indicator(self.h, which, criterion, float(G), out.ctypes.data))
        return out

    def get(self, level, I, J, K, which=0):
        out = np.zeros(self.nv)
        rc = self.L.orc_get(self.h, level, I, J, K, which, out.ctypes.data)
        if rc != 0:
            raise RuntimeError("orc_get: unresolved cell")
        return out


def oracle_for(p, U=None):
    """OracleMesh of a problem description `p` (fields nb0, max_level, bc, box_len, gamma, cfl, level, ijk, U:
    sfh_inputs.Problem), holding U (default p.U) as its copy 0."""
    U = p.U if U is None else U
    m = OracleMesh(p.nb0, p.max_level, p.bc, p.box_len, p.gamma, p.cfl, p.level, p.ijk, nscalar=U.shape[1] - NV,
                   ncell=U.shape[-1])
    m.set_state(U)
    return m
