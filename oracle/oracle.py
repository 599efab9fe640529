"""ORACLE -- TEST INFRASTRUCTURE ONLY (ctypes face of oracle/vlasov_oracle.cpp).

Plain fp64 CPU implementation of the Vlasov hot path of arXiv 1406.5445, written from PAPER.md.
Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this module.  It shares nothing with paper_1406_5445_b200/ (the CUDA path) and never imports it.

The five-moment fluid step of the coupling lives in oracle/fluid.py (numpy).  cycle() below composes the time-stepping
cycle of section 4.3 from these functions (pinned by tests/test_oracle_cycle.py).

Arrays are numpy float64, C-contiguous, laid out as the interface says:
  f[ny_g, nx, nvx, nvy, nvz];  E, B, J: [3, ny_g, nx];  moments: [10, ny_g, nx].
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "vlasov_oracle.cpp")
_LIB = os.path.join(_HERE, "liboracle.so")

BC_PERIODIC, BC_REFLECT, BC_FLUID = 0, 1, 2
ORDER_XVX, ORDER_VXV = 0, 1
STAGE_X1, STAGE_V, STAGE_X2, STAGE_GHOST, STAGE_MOMENTS, STAGE_ALL = 1, 2, 4, 8, 16, 31
ERR_SHIFT, ERR_DOMAIN = -3, -4


def build(force=False):
    """Compile the oracle's C++ (g++ -O2, no FMA contraction, OpenMP)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
                               _SRC, "-o", _LIB])
    return _LIB


_lib = None
_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int)


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_vfoot.restype = C.c_double
    return _lib


def _d(a):
    return None if a is None else a.ctypes.data_as(_dp)


def _f64(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a


def _i3(nv):
    return (C.c_int * 3)(*[int(x) for x in nv])


def _d3(v):
    return (C.c_double * 3)(*[float(x) for x in v])


def num_threads():
    return int(lib().orc_num_threads())


def remap1d(f, sigma, bc="periodic", f_inf=1.0, limiter=1):
    """8(c)-1.  f: N cell averages; sigma: N+1 face shifts (face k between cells k-1 and k)."""
    f = _f64(f)
    n = f.shape[0]
    sigma = np.asarray(sigma, dtype=np.float64)
    if sigma.ndim == 0:
        sigma = np.full(n + 1, float(sigma))
    sigma = _f64(sigma)
    assert sigma.shape == (n + 1,)
    out = np.empty_like(f)
    lib().orc_remap1d(_d(f), C.c_long(n), _d(sigma), C.c_int(0 if bc == "periodic" else 1),
                      C.c_double(f_inf), C.c_int(limiter), _d(out))
    return out


class Species:
    def __init__(self, q, m, nv, vmin, vmax, f_inf):
        self.q, self.m = float(q), float(m)
        self.nv = tuple(int(x) for x in nv)
        self.vmin = tuple(float(x) for x in vmin)
        self.vmax = tuple(float(x) for x in vmax)
        self.f_inf = float(f_inf)


def sweep_x(f, sp, nx, ny, g, dx, dts, limiter=1):
    assert f.flags.c_contiguous and f.dtype == np.float64
    lib().orc_sweep_x(_d(f), nx, ny, g, _i3(sp.nv), _d3(sp.vmin), _d3(sp.vmax), C.c_double(dx),
                      C.c_double(dts), C.c_double(sp.f_inf), C.c_int(limiter))


def sweep_y(f, sp, nx, ny, g, dy, dts, bc_lo, bc_hi, limiter=1):
    assert f.flags.c_contiguous and f.dtype == np.float64
    return lib().orc_sweep_y(_d(f), nx, ny, g, _i3(sp.nv), _d3(sp.vmin), _d3(sp.vmax),
                             C.c_double(dy), C.c_double(dts), C.c_double(sp.f_inf), C.c_int(limiter),
                             C.c_int(bc_lo), C.c_int(bc_hi))


def boris_coeffs(Ec, Bc, q, m, dt):
    t = np.zeros(3)
    s = np.zeros(3)
    h = np.zeros(3)
    err = lib().orc_boris_coeffs(_d(_f64(Ec)), _d(_f64(Bc)), C.c_double(q), C.c_double(m),
                                 C.c_double(dt), _d(t), _d(s), _d(h))
    return t, s, h, err


def vfoot(direction, face, w1, w2, t, s, h):
    return float(lib().orc_vfoot(C.c_int(direction), C.c_double(face), C.c_double(w1), C.c_double(w2),
                                 _d(_f64(t)), _d(_f64(s)), _d(_f64(h))))


def boris_back(vnp1, t, s, h):
    out = np.zeros(3)
    lib().orc_boris_back(_d(_f64(vnp1)), _d(_f64(t)), _d(_f64(s)), _d(_f64(h)), _d(out))
    return out


def vsweeps_block(fb, sp, t, s, h, limiter=1, order_reversed=False):
    assert fb.flags.c_contiguous and fb.dtype == np.float64 and fb.shape == sp.nv
    lib().orc_vsweeps_block(_d(fb), _i3(sp.nv), _d3(sp.vmin), _d3(sp.vmax), _d(_f64(t)), _d(_f64(s)),
                            _d(_f64(h)), C.c_double(sp.f_inf), C.c_int(limiter),
                            C.c_int(1 if order_reversed else 0))


def vstep(f, sp, nx, ny, g, dt, E, B, fields_yee=0, wall=0, limiter=1):
    assert f.flags.c_contiguous and f.dtype == np.float64
    return lib().orc_vstep(_d(f), nx, ny, g, _i3(sp.nv), _d3(sp.vmin), _d3(sp.vmax), C.c_double(sp.q),
                           C.c_double(sp.m), C.c_double(dt), _d(_f64(E)), _d(_f64(B)),
                           C.c_int(fields_yee), C.c_int(wall), C.c_double(sp.f_inf), C.c_int(limiter))


def field_at_cell(E, B, fields_yee, wall, ix, j):
    E = _f64(E)
    B = _f64(B)
    _, nyg, nx = E.shape
    Ec = np.zeros(3)
    Bc = np.zeros(3)
    lib().orc_field_at_cell(_d(E), _d(B), nx, nyg, C.c_int(fields_yee), C.c_int(wall), ix, j, _d(Ec), _d(Bc))
    return Ec, Bc


def moments_block(fb, sp):
    out = np.zeros(10)
    fb = _f64(fb)
    lib().orc_moments_block(_d(fb), _i3(sp.nv), _d3(sp.vmin), _d3(sp.vmax), _d(out))
    return out


def moments(f, sp, nx, ny, g):
    assert f.flags.c_contiguous and f.dtype == np.float64
    mom = np.zeros((10, ny + 2 * g, nx))
    lib().orc_moments(_d(f), nx, ny, g, _i3(sp.nv), _d3(sp.vmin), _d3(sp.vmax), _d(mom))
    return mom


def fluid_boundary(f_t, f_t1, sp, nx, ny, g, side, theta):
    """Section 4.1: boundary data for the two-fluid code.  The raw moments, eqs. (2)-(4), of the g
    kinetic rows next to the border `side` (0: rows 0..g-1 of the interior, 1: rows ny-g..ny-1; reading R22: the fluid
    block's ghost cells are as deep as the kinetic block's), at time t + theta dt "by linear interpolation in time"
    between the Vlasov data at t (f_t) and at t + dt (f_t1).  Returns [10][g][nx]."""
    assert g >= 1 and ny >= g and side in (0, 1)
    j0 = g if side == 0 else ny            # ghost-inclusive index of the first of those rows
    m_t = moments(f_t, sp, nx, ny, g)[:, j0:j0 + g, :]
    m_t1 = moments(f_t1, sp, nx, ny, g)[:, j0:j0 + g, :]
    return (1.0 - theta) * m_t + theta * m_t1


def ghost_fill(f, sp, nx, ny, g, side, fluid5, limiter=1):
    assert f.flags.c_contiguous and f.dtype == np.float64
    fluid5 = _f64(fluid5)
    assert fluid5.shape == (5, g, nx)
    return lib().orc_ghost_fill(_d(f), nx, ny, g, _i3(sp.nv), _d3(sp.vmin), _d3(sp.vmax),
                                C.c_double(sp.m), C.c_int(side), _d(fluid5), C.c_int(limiter))


def current(mom_list, q_list, fields_yee=0, wall=0):
    mom = _f64(np.stack(mom_list))
    ns, _, nyg, nx = mom.shape
    q = _f64(np.array(q_list, dtype=np.float64))
    J = np.zeros((3, nyg, nx))
    lib().orc_current(_d(mom), ns, _d(q), nx, nyg, C.c_int(fields_yee), C.c_int(wall), _d(J))
    return J


def maxwell(E, B, J, dx, dy, c, mu0, dt, nsub, wall, want_bavg=False):
    """In place on E, B (float64 [3, ny_g, nx]).  Returns B at the final E time if want_bavg."""
    assert E.flags.c_contiguous and B.flags.c_contiguous
    _, nyg, nx = E.shape
    Bavg = np.zeros_like(B) if want_bavg else None
    lib().orc_maxwell(_d(E), _d(B), _d(_f64(J)), nx, nyg, C.c_double(dx), C.c_double(dy), C.c_double(c),
                      C.c_double(mu0), C.c_double(dt), C.c_int(nsub), C.c_int(wall), _d(Bavg))
    return Bavg


def step(f, sp, nx, ny, g, lx, ly, dt, E, B, fields_yee=0, limiter=1, bc_lo=BC_PERIODIC,
         bc_hi=BC_PERIODIC, fluid_lo=None, fluid_hi=None, order=ORDER_XVX, stages=STAGE_ALL,
         want_moments=True):
    """One full step of one species, 8(c)-2.  f updated in place.  Returns (err, moments or None)."""
    assert f.flags.c_contiguous and f.dtype == np.float64
    mom = np.zeros((10, ny + 2 * g, nx)) if (want_moments and stages & STAGE_MOMENTS) else None
    fl = None if fluid_lo is None else _f64(fluid_lo)
    fh = None if fluid_hi is None else _f64(fluid_hi)
    err = lib().orc_step(_d(f), nx, ny, g, _i3(sp.nv), _d3(sp.vmin), _d3(sp.vmax), C.c_double(sp.q),
                         C.c_double(sp.m), C.c_double(lx), C.c_double(ly), C.c_double(dt), _d(_f64(E)),
                         _d(_f64(B)), C.c_int(fields_yee), C.c_double(sp.f_inf), C.c_int(limiter),
                         C.c_int(bc_lo), C.c_int(bc_hi), _d(fl), _d(fh), C.c_int(order),
                         C.c_uint(stages), _d(mom))
    return err, mom


def cycle(f_list, sp_list, mom_list, E, B, nx, ny, g, lx, ly, dt, nsub, c, mu0, fields_yee=0, bc_lo=BC_PERIODIC,
          bc_hi=BC_PERIODIC, fluid=None, order=ORDER_XVX, limiter=1):
    """One time-stepping cycle of section 4.3 (Fig. 2) without the fluid step (item 4):
      1. "the currents are calculated from the Vlasov data" (eq. 11) from the moments of f at time t (mom_list);
      2. the fields are advanced half a step with these currents (nsub FDTD sub-steps of dt/(2 nsub), eqs. 9, 10);
         the magnetic field is "interpolated to the time of the electric field";
      3. one complete Vlasov step with the new E and that B (held fixed over the step, R11), every species;
      5. the currents are calculated again from the new Vlasov data;
      6. the fields are advanced another half step.
    f_list, E, B are advanced in place ("B" stays half a sub-step ahead of "E", 8(c)-5).  fluid: None, or per species a
    pair (fluid_lo, fluid_hi) of [5][g][nx] states for FLUID sides.  Returns the new list of moments [10][ny_g][nx]."""
    wall = 0 if bc_lo == BC_PERIODIC else 1
    q = [sp.q for sp in sp_list]
    J = current(mom_list, q, fields_yee, wall)
    Bavg = maxwell(E, B, J, lx / nx, ly / ny, c, mu0, dt / 2, nsub, wall, want_bavg=True)
    new_mom = []
    for s, sp in enumerate(sp_list):
        fl = (None, None) if fluid is None else fluid[s]
        err, m = step(f_list[s], sp, nx, ny, g, lx, ly, dt, E, Bavg, fields_yee=fields_yee, limiter=limiter,
                      bc_lo=bc_lo, bc_hi=bc_hi, fluid_lo=fl[0], fluid_hi=fl[1], order=order)
        if err:
            raise RuntimeError(f"oracle step error {err}")
        new_mom.append(m)
    J = current(new_mom, q, fields_yee, wall)
    maxwell(E, B, J, lx / nx, ly / ny, c, mu0, dt / 2, nsub, wall)
    return new_mom


# ------------------------------------------------------------------------------------------------
# 3D3V: f[nz, ny, nx, nvx, nvy, nvz]; fields, moments [.., nz, ny, nx]
# ------------------------------------------------------------------------------------------------
def sweep_z(f, sp, nx, nyg, nz, dz, dts, limiter=1):
    assert f.flags.c_contiguous and f.dtype == np.float64
    lib().orc_sweep_z(_d(f), nx, nyg, nz, _i3(sp.nv), _d3(sp.vmin), _d3(sp.vmax), C.c_double(dz), C.c_double(dts),
                      C.c_double(sp.f_inf), C.c_int(limiter))


def field_at_cell3d(E, B, fields_yee, wall, ix, j, k):
    E = _f64(E)
    B = _f64(B)
    _, nz, nyg, nx = E.shape
    Ec = np.zeros(3)
    Bc = np.zeros(3)
    lib().orc_field_at_cell3d(_d(E), _d(B), nx, nyg, nz, C.c_int(fields_yee), C.c_int(wall), ix, j, k, _d(Ec), _d(Bc))
    return Ec, Bc


def moments3d(f, sp, nx, ny, nz):
    """[10, nz, ny, nx]: the moments are local to a spatial cell."""
    return moments(f, sp, nx, ny * nz, 0).reshape(10, nz, ny, nx)


def current3d(mom_list, q_list, fields_yee=0, wall=0):
    mom = _f64(np.stack(mom_list))
    ns, _, nz, nyg, nx = mom.shape
    q = _f64(np.array(q_list, dtype=np.float64))
    J = np.zeros((3, nz, nyg, nx))
    lib().orc_current3d(_d(mom), ns, _d(q), nx, nyg, nz, C.c_int(fields_yee), C.c_int(wall), _d(J))
    return J


def maxwell3d(E, B, J, dx, dy, dz, c, mu0, dt, nsub, wall, want_bavg=False):
    assert E.flags.c_contiguous and B.flags.c_contiguous
    _, nz, nyg, nx = E.shape
    Bavg = np.zeros_like(B) if want_bavg else None
    lib().orc_maxwell3d(_d(E), _d(B), _d(_f64(J)), nx, nyg, nz, C.c_double(dx), C.c_double(dy), C.c_double(dz),
                        C.c_double(c), C.c_double(mu0), C.c_double(dt), C.c_int(nsub), C.c_int(wall), _d(Bavg))
    return Bavg


def step3d(f, sp, nx, ny, nz, lx, ly, lz, dt, E, B, fields_yee=0, limiter=1, bc_lo=BC_PERIODIC, bc_hi=BC_PERIODIC,
           order=ORDER_XVX, stages=STAGE_ALL, want_moments=True):
    """One full 3D3V step of one species (no ghost rows).  f updated in place.  Returns (err, moments [10,nz,ny,nx] or None)."""
    assert f.flags.c_contiguous and f.dtype == np.float64
    mom = np.zeros((10, nz, ny, nx)) if (want_moments and stages & STAGE_MOMENTS) else None
    err = lib().orc_step3d(_d(f), nx, ny, nz, _i3(sp.nv), _d3(sp.vmin), _d3(sp.vmax), C.c_double(sp.q), C.c_double(sp.m),
                           C.c_double(lx), C.c_double(ly), C.c_double(lz), C.c_double(dt), _d(_f64(E)), _d(_f64(B)),
                           C.c_int(fields_yee), C.c_double(sp.f_inf), C.c_int(limiter), C.c_int(bc_lo), C.c_int(bc_hi),
                           C.c_int(order), C.c_uint(stages), _d(mom))
    return err, mom


def cycle3d(f_list, sp_list, mom_list, E, B, nx, ny, nz, lx, ly, lz, dt, nsub, c, mu0, fields_yee=0, bc_lo=BC_PERIODIC,
            bc_hi=BC_PERIODIC, order=ORDER_XVX, limiter=1):
    """The cycle of section 4.3 (see cycle()) on the 3D grid."""
    wall = 0 if bc_lo == BC_PERIODIC else 1
    q = [sp.q for sp in sp_list]
    J = current3d(mom_list, q, fields_yee, wall)
    Bavg = maxwell3d(E, B, J, lx / nx, ly / ny, lz / nz, c, mu0, dt / 2, nsub, wall, want_bavg=True)
    new_mom = []
    for s, sp in enumerate(sp_list):
        err, m = step3d(f_list[s], sp, nx, ny, nz, lx, ly, lz, dt, E, Bavg, fields_yee=fields_yee, limiter=limiter,
                        bc_lo=bc_lo, bc_hi=bc_hi, order=order)
        if err:
            raise RuntimeError(f"oracle step error {err}")
        new_mom.append(m)
    J = current3d(new_mom, q, fields_yee, wall)
    maxwell3d(E, B, J, lx / nx, ly / ny, lz / nz, c, mu0, dt / 2, nsub, wall)
    return new_mom
