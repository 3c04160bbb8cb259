"""ctypes binding of libsfh.so (include/sfh.h).  Argument marshalling only."""
import ctypes as C
import os
import re

import numpy as np

from . import build as _build

N, NV = 8, 5
BLK = NV * N * N * N
HERE = os.path.dirname(os.path.abspath(__file__))
HEADER = os.path.join(os.path.dirname(HERE), "include", "sfh.h")

ERRORS = {-1: "SFH_EINVAL", -2: "SFH_EMESH", -3: "SFH_ENOMEM", -4: "SFH_ECUDA", -5: "SFH_ESTATE"}


class SfhError(RuntimeError):
    def __init__(self, code, text):
        super().__init__("%s (%d): %s" % (ERRORS.get(code, "SFH_E?"), code, text))
        self.code = code


class SfhConfig(C.Structure):
    _fields_ = [("nb0", C.c_int32 * 3), ("ncell", C.c_int32), ("nghost", C.c_int32), ("max_level", C.c_int32),
                ("bc", (C.c_int32 * 2) * 3), ("box_len", C.c_double * 3), ("gamma", C.c_double), ("cfl", C.c_double),
                ("nscalar", C.c_int32)]


def library_path():
    return _build.lib_path()


def declared_symbols():
    """Names of the functions include/sfh.h declares."""
    text = open(HEADER).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(sfh_[a-z_0-9]+)\s*\(", text)))


_lib = None


def load_library(path=None):
    """Loads libsfh.so (building it with nvcc if it is missing or stale).  Raises if that fails:
    there is no fallback implementation."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    if path is None:
        path = _build.build()
    L = C.CDLL(path)
    vp, i64, i32, dbl = C.c_void_p, C.c_int64, C.c_int, C.c_double
    sig = {
        "sfh_create_mesh": (i32, [C.POINTER(SfhConfig), i64, vp, vp, C.POINTER(vp)]),
        "sfh_destroy_mesh": (i32, [vp]),
        "sfh_set_riemann": (i32, [vp, i32]),
        "sfh_num_blocks": (i64, [vp]),
        "sfh_level_range": (i32, [vp, i32, C.POINTER(i64), C.POINTER(i64)]),
        "sfh_block_order": (i32, [vp, vp]),
        "sfh_num_faces": (i32, [vp, C.POINTER(i64), C.POINTER(i64)]),
        "sfh_cell_width": (dbl, [vp, i32]),
        "sfh_state_bytes": (i64, [vp]),
        "sfh_work_bytes": (i64, [vp]),
        "sfh_bind": (i32, [vp, vp, vp, vp, vp]),
        "sfh_set_state": (i32, [vp, i32, vp, vp]),
        "sfh_get_state": (i32, [vp, i32, vp, vp]),
        "sfh_fill_ghosts": (i32, [vp, i32, i32, i32, dbl, vp]),
        "sfh_get_ghosted": (i32, [vp, i32, vp, vp]),
        "sfh_cfl_dt": (i32, [vp, i32, C.POINTER(dbl), vp]),
        "sfh_cfl_dt_noalloc": (i32, [vp, i64, dbl, dbl, dbl, vp, vp]),
        "sfh_refine_indicator": (i32, [vp, i32, i32, dbl, vp, vp]),
        "sfh_transfer_state": (i32, [vp, i32, vp, i32, vp]),
        "sfh_regrid": (i32, [vp, i32, i32, dbl, dbl, C.POINTER(vp), vp]),
        "sfh_regrid_from_indicator": (i32, [vp, vp, dbl, C.POINTER(vp)]),
        "sfh_block_list": (i32, [vp, vp, vp]),
        "sfh_hydro_step": (i32, [vp, i32, dbl, i32, dbl, dbl, vp]),
        "sfh_flux_correct": (i32, [vp, i32, dbl, vp]),
        "sfh_restrict": (i32, [vp, i32, i32, i32, vp]),
        "sfh_end_step": (i32, [vp, i32]),
        "sfh_advance": (i32, [vp, i32, i32, dbl, C.POINTER(dbl), vp, vp]),
        "sfh_advance_host": (i32, [vp, vp, vp, i32, i32, dbl, C.POINTER(dbl), vp, vp]),
        "sfh_status": (i32, [vp, i32, C.POINTER(i64), vp]),
        "sfh_launch_count": (i64, [vp]),
        "sfh_profile": (i32, [vp, i32]),
        "sfh_kernel_times": (i32, [vp, vp, vp]),
        "sfh_measure_fp64_rate": (i32, [i32, C.POINTER(dbl), vp]),
        "sfh_last_error": (C.c_char_p, []),
    }
    for name, (res, args) in sig.items():
        fn = getattr(L, name)
        fn.restype = res
        fn.argtypes = args
    if path == _build.lib_path():
        _lib = L
    return L


def _stream():
    import torch
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def measure_fp64_rate(chains=8):
    """Thread-level DFMA instructions per second of the current device (sfh_measure_fp64_rate)."""
    L = load_library()
    r = C.c_double()
    rc = L.sfh_measure_fp64_rate(int(chains), C.byref(r), _stream())
    if rc != 0:
        raise SfhError(rc, L.sfh_last_error().decode())
    return r.value


def cfl_dt_noalloc(U, gamma, cfl, h, out=None):
    """sfh_cfl_dt_noalloc: the CFL step of one level for callers that may not allocate device memory (a memory pool
    owns the GPU, a loop that must not stall on cudaMalloc, a host program that forbids it): no mesh, no work buffer;
    the reduction's intermediates live in an array built into libsfh.so (at most SFH_NOALLOC_MAX_BLOCKS = 65536
    blocks; shared by all calls, so calls that overlap on the GPU race).  U: CUDA float64 tensor [nb][5][8][8][8];
    `out`: CUDA float64 tensor of 2 elements to receive (dt, max speed) -- pass one you already own, since the one
    torch creates when it is None is an allocation of the caller's (never of the library).  Asynchronous on
    torch's current stream; returns `out`."""
    import torch
    L = load_library()
    assert U.is_cuda and U.dtype == torch.float64 and U.is_contiguous() and U.numel() % BLK == 0
    if out is None:
        out = torch.empty(2, dtype=torch.float64, device=U.device)
    assert out.is_cuda and out.dtype == torch.float64 and out.numel() >= 2 and out.is_contiguous()
    with torch.cuda.device(U.device):
        rc = L.sfh_cfl_dt_noalloc(U.data_ptr(), U.numel() // BLK, float(gamma), float(cfl), float(h), out.data_ptr(),
                                  _stream())
    if rc != 0:
        raise SfhError(rc, L.sfh_last_error().decode())
    return out


class Mesh:
    """An octree block mesh bound to three device state buffers and a work buffer (torch tensors).

    level[nb], ijk[nb,3]: the caller's block list; states cross this interface in caller layout
    double [nb][5][8][8][8] (interior cells, [block][var][k][j][i])."""

    def __init__(self, nb0, max_level, bc, box_len, gamma, cfl, level, ijk, device="cuda:0", bind=True, lib=None,
                 nscalar=0, handle=None, ncell=N):
        self.L = lib or load_library()
        cfg = SfhConfig()
        for d in range(3):
            cfg.nb0[d] = int(nb0[d])
            cfg.box_len[d] = float(box_len[d])
            for s in range(2):
                cfg.bc[d][s] = int(bc[d][s])
        cfg.ncell, cfg.nghost, cfg.max_level = int(ncell), 2, int(max_level)
        self.ncell = int(ncell)              # 8, or 16: states cross the interface as [nb][nv][16][16][16] (sfh.h)
        cfg.gamma, cfg.cfl = float(gamma), float(cfl)
        cfg.nscalar = int(nscalar)
        self.nv = NV + int(nscalar)          # variables per cell in the caller layout
        self.cfg = cfg
        self.max_level = int(max_level)
        if handle is None:
            self.level = np.ascontiguousarray(level, dtype=np.int32)
            self.ijk = np.ascontiguousarray(ijk, dtype=np.int32).reshape(-1, 3)
            self.nb = len(self.level)
            self.h = C.c_void_p()
            self._chk(self.L.sfh_create_mesh(C.byref(cfg), self.nb, self.level.ctypes.data, self.ijk.ctypes.data,
                                             C.byref(self.h)))
        else:                                # a mesh the library built itself (sfh_regrid): read its block list back
            self.h = handle
            self.nb = int(self.L.sfh_num_blocks(self.h))
            self.level = np.zeros(self.nb, dtype=np.int32)
            self.ijk = np.zeros((self.nb, 3), dtype=np.int32)
            self._chk(self.L.sfh_block_list(self.h, self.level.ctypes.data, self.ijk.ctypes.data))
        self.t = C.c_double(0.0)
        self.nupd = np.zeros(self.max_level + 1, dtype=np.int64)
        self.device = device
        self.bound = False
        if bind:
            self.bind()

    @classmethod
    def from_problem(cls, p, **kw):
        kw.setdefault("nscalar", p.U.shape[1] - NV)
        kw.setdefault("ncell", p.U.shape[-1])
        return cls(p.nb0, p.max_level, p.bc, p.box_len, p.gamma, p.cfl, p.level, p.ijk, **kw)

    def __del__(self):
        if getattr(self, "h", None) and self.h.value:
            self.L.sfh_destroy_mesh(self.h)
            self.h = C.c_void_p()

    def _chk(self, rc):
        if rc != 0:
            raise SfhError(rc, self.L.sfh_last_error().decode())

    # ---- host-only queries
    def nentries(self):
        """Blocks as the library counts them: self.nb, or 8 * self.nb (the octants) for ncell = 16 (sfh.h)."""
        return int(self.L.sfh_num_blocks(self.h))

    def level_range(self, l):
        a, b = C.c_int64(), C.c_int64()
        self._chk(self.L.sfh_level_range(self.h, l, C.byref(a), C.byref(b)))
        return a.value, b.value

    def block_order(self):
        perm = np.zeros(self.nentries(), dtype=np.int64)
        self._chk(self.L.sfh_block_order(self.h, perm.ctypes.data))
        return perm

    def num_faces(self):
        a, b = C.c_int64(), C.c_int64()
        self._chk(self.L.sfh_num_faces(self.h, C.byref(a), C.byref(b)))
        return a.value, b.value

    def cell_width(self, l):
        return self.L.sfh_cell_width(self.h, l)

    def state_bytes(self):
        return self.L.sfh_state_bytes(self.h)

    def work_bytes(self):
        return self.L.sfh_work_bytes(self.h)

    def launch_count(self):
        return self.L.sfh_launch_count(self.h)

    def set_riemann(self, solver):
        """0 / "hllc" or 1 / "roe"."""
        self._chk(self.L.sfh_set_riemann(self.h, {"hllc": 0, "roe": 1}.get(solver, solver)))

    # ---- device
    def bind(self, guard=0, poison=False):
        """Allocates the three state buffers and the work buffer and binds them.  Debugging aids (compute-sanitizer
        is not available on every pool): guard > 0 puts `guard` doubles of a canary pattern before and after every
        buffer (check_guards() tells whether any kernel wrote outside its buffer); poison fills everything the
        library does not initialise itself with NaN, so that a read of never-written memory shows up in the results."""
        import torch
        if not torch.cuda.is_available():
            raise SfhError(-4, "no CUDA device: libsfh has no CPU fallback")
        dev = torch.device(self.device)
        torch.cuda.set_device(dev)
        guard = (int(guard) + 31) // 32 * 32        # keeps the 256-byte alignment sfh_bind asks for
        sizes = [self.state_bytes() // 8] * 3 + [self.work_bytes() // 8]
        self._guard = guard
        self._raw = [torch.empty(n + 2 * guard, dtype=torch.float64, device=dev) for n in sizes]
        for r in self._raw:
            if poison:
                r.fill_(float("nan"))
            if guard:
                r[:guard] = self._CANARY
                r[r.numel() - guard:] = self._CANARY
        bufs = [r[guard:r.numel() - guard] for r in self._raw]
        self.state, self.work = bufs[:3], bufs[3]
        torch.cuda.synchronize()
        self._chk(self.L.sfh_bind(self.h, self.state[0].data_ptr(), self.state[1].data_ptr(),
                                  self.state[2].data_ptr(), self.work.data_ptr()))
        if poison:      # sfh_bind zeroes the work buffer; only its last 4 KB (device scalars: time, dt, counters) must stay
            self.work[: self.work.numel() - 512] = float("nan")
            torch.cuda.synchronize()
        self.bound = True

    _CANARY = -6.02214076e23

    def check_guards(self):
        """True if the canaries around the four buffers are intact (bind(guard=n))."""
        import torch
        torch.cuda.synchronize()
        g = self._guard
        return all(bool((r[:g] == self._CANARY).all()) and bool((r[r.numel() - g:] == self._CANARY).all())
                   for r in self._raw) if g else True

    def _dev_state(self, U):
        import torch
        if isinstance(U, np.ndarray):
            U = torch.from_numpy(np.ascontiguousarray(U, dtype=np.float64))
        U = U.to(device=self.device, dtype=torch.float64).contiguous()
        assert U.numel() == self.nb * self.nv * self.ncell ** 3, "state must be [nb][5 + nscalar][ncell]^3"
        return U

    def set_state(self, U, which=0):
        U = self._dev_state(U)
        self._chk(self.L.sfh_set_state(self.h, which, U.data_ptr(), _stream()))
        import torch
        torch.cuda.current_stream().synchronize()   # U may be a temporary

    def get_state(self, which=0):
        """torch tensor [nb][5][8][8][8] on the device."""
        import torch
        out = torch.empty((self.nb, self.nv) + (self.ncell,) * 3, dtype=torch.float64, device=self.device)
        self._chk(self.L.sfh_get_state(self.h, which, out.data_ptr(), _stream()))
        return out

    def get_ghosted(self, which=0):
        import torch
        out = torch.empty((self.nentries(), NV, N + 4, N + 4, N + 4), dtype=torch.float64, device=self.device)
        self._chk(self.L.sfh_get_ghosted(self.h, which, out.data_ptr(), _stream()))
        return out

    def fill_ghosts(self, level=-1, which=0, interp=0, tau=0.0):
        self._chk(self.L.sfh_fill_ghosts(self.h, level, which, interp, tau, _stream()))

    def cfl_dt(self, level=-1):
        dt = C.c_double()
        self._chk(self.L.sfh_cfl_dt(self.h, level, C.byref(dt), _stream()))
        return dt.value

    def hydro_step(self, level, dt, interp=0, tau=0.0, dtau=0.0):
        self._chk(self.L.sfh_hydro_step(self.h, level, dt, interp, tau, dtau, _stream()))

    def flux_correct(self, coarse_level, dt_coarse):
        self._chk(self.L.sfh_flux_correct(self.h, coarse_level, dt_coarse, _stream()))

    def restrict(self, coarse_level, src_role=0, dst_role=0):
        self._chk(self.L.sfh_restrict(self.h, coarse_level, src_role, dst_role, _stream()))

    def restrict_all(self, role=0):
        for l in range(self.max_level - 1, -1, -1):
            self.restrict(l, role, role)

    def end_step(self, level=-1):
        self._chk(self.L.sfh_end_step(self.h, level))

    def advance(self, nsteps, mode=0, dt_fixed=0.0):
        self._chk(self.L.sfh_advance(self.h, nsteps, mode, dt_fixed, C.byref(self.t), self.nupd.ctypes.data,
                                     _stream()))
        return self.t.value

    def advance_host(self, h_in, h_out, nsteps, mode=0, dt_fixed=0.0):
        """h_in, h_out: host tensors/arrays in caller layout (pinned for full PCIe speed)."""
        pin = h_in.data_ptr() if hasattr(h_in, "data_ptr") else h_in.ctypes.data
        pout = h_out.data_ptr() if hasattr(h_out, "data_ptr") else h_out.ctypes.data
        self._chk(self.L.sfh_advance_host(self.h, pin, pout, nsteps, mode, dt_fixed, C.byref(self.t),
                                          self.nupd.ctypes.data, _stream()))
        return self.t.value

    KERNEL_CLASSES = ("predictor", "corrector", "prolong", "restrict", "reflux", "max_speed", "scalars")

    def profile(self, enable=True):
        self._chk(self.L.sfh_profile(self.h, int(enable)))

    def kernel_times(self):
        """{class: (total ms, launches)} since the last call (synchronises)."""
        ms = np.zeros(len(self.KERNEL_CLASSES), dtype=np.float64)
        cnt = np.zeros(len(self.KERNEL_CLASSES), dtype=np.int64)
        self._chk(self.L.sfh_kernel_times(self.h, ms.ctypes.data, cnt.ctypes.data))
        return {k: (float(ms[i]), int(cnt[i])) for i, k in enumerate(self.KERNEL_CLASSES)}

    def transfer_from(self, src, which=0):
        """Regrid: state copy `which` of this (new) mesh from the old mesh `src` (copies and prolongations); fill
        the old mesh's ghosts of `which` first."""
        self._chk(self.L.sfh_transfer_state(src.h, which, self.h, which, _stream()))

    def _derived(self, handle, bind):
        """Wrapper of a mesh the library derived from this one (sfh_regrid*).  Such a mesh always has 8^3 blocks: from
        a mesh of 16^3 blocks the library derives the mesh of the octants (sfh.h, "Blocks of 16^3 cells"), whose root
        grid counts twice as many blocks per axis; states then cross the interface as [nb][nv][8][8][8]."""
        c = self.cfg
        k = self.ncell // N
        return Mesh(tuple(k * n for n in c.nb0), c.max_level, [tuple(b) for b in c.bc], tuple(c.box_len), c.gamma,
                    c.cfl, None, None, device=self.device, lib=self.L, nscalar=c.nscalar, handle=handle, bind=bind,
                    ncell=N)

    def regrid_from_indicator(self, indicator, threshold, bind=False):
        """The new mesh from a host indicator array (caller order); host only unless bind=True."""
        ind = np.ascontiguousarray(indicator, dtype=np.float64)
        assert ind.shape == (self.nentries(),)
        h = C.c_void_p()
        self._chk(self.L.sfh_regrid_from_indicator(self.h, ind.ctypes.data, float(threshold), C.byref(h)))
        return self._derived(h, bind)

    def regrid(self, criterion, threshold, which=0, G=1.0):
        """The regridded mesh (sfh_regrid: blocks with indicator >= threshold get children, 2:1 closure), bound to new
        buffers, holding the state of copy `which` moved onto it (sfh_transfer_state)."""
        h = C.c_void_p()
        self._chk(self.L.sfh_regrid(self.h, which, criterion, float(G), float(threshold), C.byref(h), _stream()))
        new = self._derived(h, True)
        new.transfer_from(self, which)
        return new

    def refine_indicator(self, criterion=0, which=0, G=1.0):
        """Per-block refinement indicator (0: eq. 33-34 curvature, 1: h / Jeans length), caller order."""
        import torch
        out = torch.empty(self.nentries(), dtype=torch.float64, device=self.device)
        self._chk(self.L.sfh_refine_indicator(self.h, which, criterion, float(G), out.data_ptr(), _stream()))
        return out

    def status(self, which=0):
        n = C.c_int64()
        self._chk(self.L.sfh_status(self.h, which, C.byref(n), _stream()))
        return n.value
