"""Thin ctypes binding of libvlasov_b200.so -- same names as include/vlasov.h, argument marshalling only.

Every step of the path runs in the library's CUDA kernels.  torch is used for device memory and
streams.  There is NO CPU fallback: a missing library raises at import of the symbols, a missing GPU
makes vlasov_init return VLASOV_ECUDA (raised as VlasovError).
"""
import ctypes as C
import os

HERE = os.path.dirname(os.path.abspath(__file__))
# VLASOV_B200_LIB: another build of the same library (A/B measurements of kernel variants); default: the in-tree build
LIB_PATH = os.environ.get("VLASOV_B200_LIB") or os.path.join(HERE, "libvlasov_b200.so")

OK, EINVAL, EALIGN, ESHIFT, EDOMAIN, ECUDA, ETOOBIG = 0, -1, -2, -3, -4, -5, -6
FLUID_STATIC_SCRATCH_BYTES = 4 << 20
BC_PERIODIC, BC_REFLECT, BC_FLUID = 0, 1, 2
ORDER_XVX, ORDER_VXV = 0, 1
STAGE_X1, STAGE_V, STAGE_X2, STAGE_GHOST, STAGE_MOMENTS, STAGE_ALL = 1, 2, 4, 8, 16, 31

EXPORTS = ["vlasov_scratch_bytes", "vlasov_init", "vlasov_set_boundary", "vlasov_step", "vlasov_step_host",
           "vlasov_moments", "vlasov_current", "vlasov_maxwell", "vlasov_touch", "vlasov_set_option", "vlasov_check",
           "vlasov_launch_count", "vlasov_free", "vlasov_strerror", "vlasov_cycle", "vlasov_cycle_host",
           "vlasov_timing_enable", "vlasov_timing_read", "vlasov_fluid_boundary_mark", "vlasov_fluid_boundary",
           "vlasov_fluid_scratch_bytes", "vlasov_fluid_step", "vlasov_fluid_from_moments", "vlasov_fluid_to_boundary",
           "vlasov_fluid_step_static"]
FLUID_BC_PERIODIC, FLUID_BC_WALL, FLUID_BC_COUPLED = 0, 1, 2
OPT_FUSE_XY = 1
OPT_FUSE_MOMENTS = 2
KINDS = ["sweep_x", "sweep_y", "table", "vsweep_x", "vsweep_yz", "moments", "ghost_table", "current", "maxwell", "sweep_xy", "sweep_yx",
         "ghost_vsweep_x", "ghost_vsweep_yz", "ghost_moments", "ghost_sweep_x", "sweep_z"]


class vlasov_species(C.Structure):
    _fields_ = [("q", C.c_double), ("m", C.c_double), ("nv", C.c_int32 * 3), ("vmin", C.c_double * 3),
                ("vmax", C.c_double * 3), ("f_inf", C.c_double)]


class vlasov_config(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nghost_y", C.c_int32), ("nspecies", C.c_int32),
                ("lx", C.c_double), ("ly", C.c_double), ("bc_y_lo", C.c_int32), ("bc_y_hi", C.c_int32),
                ("order", C.c_int32), ("limiter", C.c_int32), ("fields_yee", C.c_int32), ("nz", C.c_int32),
                ("c", C.c_double), ("mu0", C.c_double), ("lz", C.c_double), ("stream", C.c_void_p)]


class vlasov_fluid_config(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nspecies", C.c_int32), ("bc_y_lo", C.c_int32),
                ("bc_y_hi", C.c_int32), ("reserved", C.c_int32), ("dx", C.c_double), ("dy", C.c_double),
                ("q", C.c_double * 8), ("m", C.c_double * 8), ("stream", C.c_void_p)]


class VlasovError(RuntimeError):
    def __init__(self, code, where):
        self.code = code
        super().__init__(f"{where}: {strerror(code)} ({code})")


_lib = None


def lib():
    """Load the C-ABI library (fails loudly when it has not been built)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise OSError(f"{LIB_PATH} is missing: run `python -m paper_1406_5445_b200.build` "
                          "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp, dp = C.c_void_p, C.c_void_p
        L.vlasov_scratch_bytes.restype = C.c_size_t
        L.vlasov_scratch_bytes.argtypes = [C.POINTER(vlasov_config), C.POINTER(vlasov_species)]
        L.vlasov_init.restype = C.c_int
        L.vlasov_init.argtypes = [C.POINTER(vlasov_config), C.POINTER(vlasov_species), C.POINTER(C.c_void_p),
                                  vp, C.c_size_t, C.POINTER(C.c_void_p)]
        L.vlasov_set_boundary.restype = C.c_int
        L.vlasov_set_boundary.argtypes = [vp, C.c_int, C.c_int, C.c_int, dp]
        L.vlasov_step.restype = C.c_int
        L.vlasov_step.argtypes = [vp, C.c_double, dp, dp, C.c_uint32]
        L.vlasov_step_host.restype = C.c_int
        L.vlasov_step_host.argtypes = [vp, C.c_double, dp, dp, C.c_uint32, dp]
        L.vlasov_moments.restype = C.c_int
        L.vlasov_moments.argtypes = [vp, C.c_int, dp]
        L.vlasov_fluid_boundary_mark.restype = C.c_int
        L.vlasov_fluid_boundary_mark.argtypes = [vp]
        L.vlasov_fluid_boundary.restype = C.c_int
        L.vlasov_fluid_boundary.argtypes = [vp, C.c_int, C.c_int, C.c_double, dp]
        L.vlasov_current.restype = C.c_int
        L.vlasov_current.argtypes = [vp, dp]
        L.vlasov_maxwell.restype = C.c_int
        L.vlasov_maxwell.argtypes = [vp, C.c_double, C.c_int, dp, dp, dp, dp]
        L.vlasov_cycle.restype = C.c_int
        L.vlasov_cycle.argtypes = [vp, C.c_double, C.c_int, dp, dp]
        L.vlasov_cycle_host.restype = C.c_int
        L.vlasov_cycle_host.argtypes = [vp, C.c_double, C.c_int, dp, dp, dp]
        L.vlasov_timing_enable.restype = C.c_int
        L.vlasov_timing_enable.argtypes = [vp, C.c_int]
        L.vlasov_timing_read.restype = C.c_int
        L.vlasov_timing_read.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(C.c_int64), C.c_int]
        L.vlasov_set_option.restype = C.c_int
        L.vlasov_set_option.argtypes = [vp, C.c_int, C.c_int]
        L.vlasov_touch.restype = C.c_int
        L.vlasov_touch.argtypes = [vp]
        L.vlasov_check.restype = C.c_int
        L.vlasov_check.argtypes = [vp]
        L.vlasov_launch_count.restype = C.c_int64
        L.vlasov_launch_count.argtypes = [vp]
        L.vlasov_free.restype = None
        L.vlasov_free.argtypes = [vp]
        L.vlasov_strerror.restype = C.c_char_p
        L.vlasov_strerror.argtypes = [C.c_int]
        L.vlasov_fluid_scratch_bytes.restype = C.c_size_t
        L.vlasov_fluid_scratch_bytes.argtypes = [C.POINTER(vlasov_fluid_config)]
        L.vlasov_fluid_step.restype = C.c_int
        L.vlasov_fluid_step.argtypes = [C.POINTER(vlasov_fluid_config), C.c_double, dp, dp, dp, dp, dp, vp, C.c_size_t]
        L.vlasov_fluid_step_static.restype = C.c_int
        L.vlasov_fluid_step_static.argtypes = [C.POINTER(vlasov_fluid_config), C.c_double, dp, dp, dp, dp, dp]
        L.vlasov_fluid_from_moments.restype = C.c_int
        L.vlasov_fluid_from_moments.argtypes = [dp, C.c_double, dp, C.c_long, vp]
        L.vlasov_fluid_to_boundary.restype = C.c_int
        L.vlasov_fluid_to_boundary.argtypes = [dp, C.c_double, dp, C.c_long, vp]
        _lib = L
    return _lib


def strerror(code):
    return lib().vlasov_strerror(int(code)).decode()


def _chk(code, where):
    if code != OK:
        raise VlasovError(code, where)


def _ptr(t):
    """Device (or pinned host) address of a torch tensor / numpy array, or None."""
    if t is None:
        return None
    if hasattr(t, "data_ptr"):
        return C.c_void_p(t.data_ptr())
    return C.c_void_p(t.ctypes.data)


def make_config(nx, ny, nghost_y, nspecies, lx, ly, bc_y_lo, bc_y_hi, order=ORDER_XVX, limiter=1, fields_yee=0,
                c=1.0, mu0=1.0, stream=0, nz=1, lz=1.0):
    cfg = vlasov_config()
    cfg.nx, cfg.ny, cfg.nghost_y, cfg.nspecies = nx, ny, nghost_y, nspecies
    cfg.lx, cfg.ly = lx, ly
    cfg.bc_y_lo, cfg.bc_y_hi = bc_y_lo, bc_y_hi
    cfg.order, cfg.limiter, cfg.fields_yee, cfg.nz = order, limiter, fields_yee, int(nz)
    cfg.c, cfg.mu0, cfg.lz = c, mu0, float(lz)
    cfg.stream = stream
    return cfg


def make_species(specs):
    """specs: iterable of objects with q, m, nv, vmin, vmax, f_inf (e.g. inputs.SpeciesSpec)."""
    specs = list(specs)
    arr = (vlasov_species * len(specs))()
    for k, s in enumerate(specs):
        arr[k].q, arr[k].m = float(s.q), float(s.m)
        for d in range(3):
            arr[k].nv[d] = int(s.nv[d])
            arr[k].vmin[d] = float(s.vmin[d])
            arr[k].vmax[d] = float(s.vmax[d])
        arr[k].f_inf = float(s.f_inf)
    return arr


def vlasov_scratch_bytes(cfg, species_arr):
    return int(lib().vlasov_scratch_bytes(C.byref(cfg), species_arr))


class Context:
    """Owns a vlasov_ctx*.  f_list: torch cuda float64 tensors [ny_g, nx, nvx, nvy, nvz] ([nz, ny, nx, ...] for 3D3V),
    kept alive here."""

    def __init__(self, cfg, species_arr, f_list, scratch=None):
        import torch
        self.cfg, self.species_arr = cfg, species_arr
        self.f = list(f_list)
        for t in self.f:
            if not (t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
                raise ValueError("f must be contiguous float64 CUDA tensors")
        nbytes = vlasov_scratch_bytes(cfg, species_arr)
        if nbytes == 0:
            raise VlasovError(EINVAL, "vlasov_scratch_bytes")
        self.scratch = scratch if scratch is not None else torch.empty(nbytes, dtype=torch.uint8, device=self.f[0].device)
        self.scratch_bytes = nbytes
        fp = (C.c_void_p * len(self.f))(*[t.data_ptr() for t in self.f])
        h = C.c_void_p()
        _chk(lib().vlasov_init(C.byref(cfg), species_arr, fp, C.c_void_p(self.scratch.data_ptr()),
                               C.c_size_t(self.scratch.numel()), C.byref(h)), "vlasov_init")
        self.h = h
        self._keep = []

    def vlasov_set_boundary(self, species, side, kind, fluid5=None):
        if fluid5 is not None:
            self._keep.append(fluid5)
            self._keep = self._keep[-16:]
        _chk(lib().vlasov_set_boundary(self.h, species, side, kind, _ptr(fluid5)), "vlasov_set_boundary")

    def vlasov_step(self, dt, E, B, stages=STAGE_ALL):
        _chk(lib().vlasov_step(self.h, float(dt), _ptr(E), _ptr(B), stages), "vlasov_step")

    def vlasov_step_host(self, dt, E_host, B_host, stages=STAGE_ALL, mom_host=None):
        _chk(lib().vlasov_step_host(self.h, float(dt), _ptr(E_host), _ptr(B_host), stages, _ptr(mom_host)),
             "vlasov_step_host")

    def vlasov_moments(self, species, mom):
        _chk(lib().vlasov_moments(self.h, species, _ptr(mom)), "vlasov_moments")

    def vlasov_fluid_boundary_mark(self):
        _chk(lib().vlasov_fluid_boundary_mark(self.h), "vlasov_fluid_boundary_mark")

    def vlasov_fluid_boundary(self, species, side, theta, out):
        _chk(lib().vlasov_fluid_boundary(self.h, int(species), int(side), float(theta), _ptr(out)), "vlasov_fluid_boundary")

    def vlasov_current(self, J):
        _chk(lib().vlasov_current(self.h, _ptr(J)), "vlasov_current")

    def vlasov_maxwell(self, dt, nsub, E, B, J, Bavg=None):
        _chk(lib().vlasov_maxwell(self.h, float(dt), int(nsub), _ptr(E), _ptr(B), _ptr(J), _ptr(Bavg)), "vlasov_maxwell")

    def vlasov_cycle(self, dt, nsub, E, B):
        _chk(lib().vlasov_cycle(self.h, float(dt), int(nsub), _ptr(E), _ptr(B)), "vlasov_cycle")

    def vlasov_cycle_host(self, dt, nsub, E_host, B_host, mom_host=None):
        _chk(lib().vlasov_cycle_host(self.h, float(dt), int(nsub), _ptr(E_host), _ptr(B_host), _ptr(mom_host)),
             "vlasov_cycle_host")

    def vlasov_timing_enable(self, on):
        _chk(lib().vlasov_timing_enable(self.h, 1 if on else 0), "vlasov_timing_enable")

    def vlasov_timing_read(self):
        """{kind name: (milliseconds, launches)} since timing was enabled / last read."""
        n = len(KINDS)
        ms = (C.c_double * n)()
        cnt = (C.c_int64 * n)()
        _chk(lib().vlasov_timing_read(self.h, ms, cnt, n), "vlasov_timing_read")
        return {KINDS[k]: (float(ms[k]), int(cnt[k])) for k in range(n)}

    def vlasov_set_option(self, option, value):
        _chk(lib().vlasov_set_option(self.h, int(option), int(value)), "vlasov_set_option")

    def vlasov_touch(self):
        _chk(lib().vlasov_touch(self.h), "vlasov_touch")

    def vlasov_check(self):
        """Synchronise; raise on an asynchronously recorded error."""
        _chk(lib().vlasov_check(self.h), "vlasov_check")

    def check_code(self):
        return int(lib().vlasov_check(self.h))

    def launch_count(self):
        return int(lib().vlasov_launch_count(self.h))

    def close(self):
        if getattr(self, "h", None):
            lib().vlasov_free(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def context_for(workload, f_list, order=ORDER_XVX, limiter=1, stream=None):
    """Context for an inputs.Workload (marshalling only)."""
    import torch
    if stream is None:
        stream = torch.cuda.current_stream().cuda_stream
    cfg = make_config(workload.nx, workload.ny, workload.nghost_y, len(workload.species), workload.lx, workload.ly,
                      workload.bc_y_lo, workload.bc_y_hi, order=order, limiter=limiter,
                      fields_yee=workload.fields_yee, c=workload.c, mu0=workload.mu0, stream=stream,
                      nz=getattr(workload, "nz", 1), lz=getattr(workload, "lz", 1.0))
    return Context(cfg, make_species(workload.species), f_list)


class FluidBlock:
    """Arguments of vlasov_fluid_step for one fluid block (marshalling only).  U: torch cuda float64
    [nspecies, 5, ny + 4, nx]."""

    def __init__(self, nx, ny, dx, dy, q, m, bc_y_lo, bc_y_hi, stream=None):
        import torch
        if stream is None:
            stream = torch.cuda.current_stream().cuda_stream
        cfg = vlasov_fluid_config()
        cfg.nx, cfg.ny, cfg.nspecies = int(nx), int(ny), len(q)
        cfg.bc_y_lo, cfg.bc_y_hi, cfg.reserved = int(bc_y_lo), int(bc_y_hi), 0
        cfg.dx, cfg.dy = float(dx), float(dy)
        for s in range(len(q)):
            cfg.q[s], cfg.m[s] = float(q[s]), float(m[s])
        cfg.stream = stream
        self.cfg = cfg
        nbytes = int(lib().vlasov_fluid_scratch_bytes(C.byref(cfg)))
        if nbytes == 0:
            raise VlasovError(EINVAL, "vlasov_fluid_scratch_bytes")
        self.scratch = torch.empty(nbytes, dtype=torch.uint8, device="cuda")

    def vlasov_fluid_step(self, dt, U, E, B, ghost_lo=None, ghost_hi=None):
        _chk(lib().vlasov_fluid_step(C.byref(self.cfg), float(dt), _ptr(U), _ptr(E), _ptr(B), _ptr(ghost_lo), _ptr(ghost_hi),
                                     C.c_void_p(self.scratch.data_ptr()), C.c_size_t(self.scratch.numel())), "vlasov_fluid_step")

    def vlasov_fluid_step_static(self, dt, U, E, B, ghost_lo=None, ghost_hi=None):
        """The same step with the stage buffers in the library's static device array: no allocation (include/vlasov.h)."""
        _chk(lib().vlasov_fluid_step_static(C.byref(self.cfg), float(dt), _ptr(U), _ptr(E), _ptr(B), _ptr(ghost_lo),
                                            _ptr(ghost_hi)), "vlasov_fluid_step_static")


def vlasov_fluid_from_moments(mom10, m, U5, stream=None):
    import torch
    st = torch.cuda.current_stream().cuda_stream if stream is None else stream
    _chk(lib().vlasov_fluid_from_moments(_ptr(mom10), float(m), _ptr(U5), C.c_long(mom10.numel() // 10), C.c_void_p(st)),
         "vlasov_fluid_from_moments")


def vlasov_fluid_to_boundary(U5, m, fluid5, stream=None):
    import torch
    st = torch.cuda.current_stream().cuda_stream if stream is None else stream
    _chk(lib().vlasov_fluid_to_boundary(_ptr(U5), float(m), _ptr(fluid5), C.c_long(U5.numel() // 5), C.c_void_p(st)),
         "vlasov_fluid_to_boundary")
