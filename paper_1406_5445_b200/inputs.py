"""Seeded synthetic inputs.  Serves BOTH the CUDA path and the oracle.

This module holds none of the method's arithmetic: it only evaluates closed-form initial profiles
(Landau perturbation, GEM Harris sheet: Birn et al. set-up as used in PAPER.md:427) plus a
counter-based hash noise, and describes the five BASELINE.json workloads as plain numbers.
It imports neither the CUDA binding nor the oracle.
"""
from dataclasses import dataclass, field
from typing import List, Tuple

import numpy as np

BC_PERIODIC, BC_REFLECT, BC_FLUID = 0, 1, 2


@dataclass
class SpeciesSpec:
    name: str
    q: float
    m: float
    nv: Tuple[int, int, int]
    vmin: Tuple[float, float, float]
    vmax: Tuple[float, float, float]
    vth: float = 1.0
    drift_z: float = 0.0      # Harris drift u_sz of the sheet population
    f_inf: float = 0.0        # filled by the generators: max of the initial f (reading R6)

    @property
    def dv(self):
        return tuple((self.vmax[d] - self.vmin[d]) / self.nv[d] for d in range(3))

    @property
    def ncell_v(self):
        return self.nv[0] * self.nv[1] * self.nv[2]

    def centres(self, d):
        return self.vmin[d] + (np.arange(self.nv[d]) + 0.5) * self.dv[d]


@dataclass
class Workload:
    name: str
    nx: int
    ny: int
    nghost_y: int
    lx: float
    ly: float
    x0: float
    y0: float
    bc_y_lo: int
    bc_y_hi: int
    dt: float
    steps: int
    species: List[SpeciesSpec] = field(default_factory=list)
    c: float = 1.0
    mu0: float = 1.0
    nsub: int = 1
    fields_yee: int = 1
    seed: int = 1
    kind: str = "gem"     # "landau" | "gem" | "band"
    y_centre_offset: float = 0.0
    nz: int = 1           # 3D3V (NEXT-4): cells along z, periodic
    lz: float = 1.0

    @property
    def ny_g(self):
        return self.ny + 2 * self.nghost_y

    @property
    def dx(self):
        return self.lx / self.nx

    @property
    def dy(self):
        return self.ly / self.ny

    @property
    def interior_cells(self):
        return sum(self.nx * self.ny * s.ncell_v for s in self.species)

    def x_centres(self):
        return self.x0 + (np.arange(self.nx) + 0.5) * self.dx

    def y_centres_g(self):
        """Centres of all rows, ghost rows included."""
        return self.y0 + (np.arange(self.ny_g) - self.nghost_y + 0.5) * self.dy


# ------------------------------------------------------------------------------------------------
# counter-based noise: splitmix64 of (seed, species, linear cell index) -> xi in [-1, 1)
# ------------------------------------------------------------------------------------------------
def hash_noise(seed: int, stream: int, start: int, count: int) -> np.ndarray:
    with np.errstate(over="ignore"):
        z = np.arange(start, start + count, dtype=np.uint64)
        z += np.uint64((seed * 0x9E3779B97F4A7C15 + stream * 0xD1B54A32D192ED03 + 0x632BE59BD9B4E019) % (1 << 64))
        z += np.uint64(0x9E3779B97F4A7C15)
        z ^= z >> np.uint64(30)
        z *= np.uint64(0xBF58476D1CE4E5B9)
        z ^= z >> np.uint64(27)
        z *= np.uint64(0x94D049BB133111EB)
        z ^= z >> np.uint64(31)
        z >>= np.uint64(11)
    xi = z.astype(np.float64)
    xi *= 2.0 / float(1 << 53)
    xi -= 1.0
    return xi


def _maxwellian_1d(v, u, vth):
    return np.exp(-0.5 * ((v - u) / vth) ** 2) / (np.sqrt(2.0 * np.pi) * vth)


def _maxwellian_3d(sp: SpeciesSpec, uz: float):
    mx = _maxwellian_1d(sp.centres(0), 0.0, sp.vth)
    my = _maxwellian_1d(sp.centres(1), 0.0, sp.vth)
    mz = _maxwellian_1d(sp.centres(2), uz, sp.vth)
    return mx[:, None, None] * my[None, :, None] * mz[None, None, :]


# ------------------------------------------------------------------------------------------------
# config 1: Landau damping (BASELINE.json configs[0])
# ------------------------------------------------------------------------------------------------
def landau_workload(nx=32, ny=2, nv=(64, 8, 8), dt=0.05, steps=100, k=0.5, amp=0.01) -> Workload:
    sp = SpeciesSpec("electrons", q=-1.0, m=1.0, nv=tuple(nv), vmin=(-6.0,) * 3, vmax=(6.0,) * 3, vth=1.0)
    w = Workload("landau", nx=nx, ny=ny, nghost_y=0, lx=2.0 * np.pi / k, ly=1.0, x0=0.0, y0=0.0,
                 bc_y_lo=BC_PERIODIC, bc_y_hi=BC_PERIODIC, dt=dt, steps=steps, species=[sp],
                 c=1.0, mu0=1.0, nsub=1, fields_yee=0, seed=0, kind="landau")
    w.landau_k = k
    w.landau_amp = amp
    return w


def landau_f(w: Workload) -> np.ndarray:
    sp = w.species[0]
    M = _maxwellian_3d(sp, 0.0)
    x = w.x_centres()
    prof = 1.0 + w.landau_amp * np.cos(w.landau_k * x)
    f = np.empty((w.ny_g, w.nx) + sp.nv)
    f[:] = prof[None, :, None, None, None] * M[None, None]
    sp.f_inf = float(f.max())
    return f


# ------------------------------------------------------------------------------------------------
# configs 2, 3, 5: GEM Harris sheet (units d_i, 1/Omega_ci, v_A, B0, n0, m_i = e = mu0 = 1)
# ------------------------------------------------------------------------------------------------
GEM_LAMBDA = 0.5
GEM_NB = 0.2
GEM_PSI0 = 0.1
GEM_TI = 5.0 / 12.0
GEM_TE = 1.0 / 12.0
GEM_MI = 1.0
GEM_ME = 1.0 / 25.0
GEM_C = 20.0


def gem_species(nv) -> List[SpeciesSpec]:
    if isinstance(nv, int):
        nv = (nv, nv, nv)
    vthe = float(np.sqrt(GEM_TE / GEM_ME))
    vthi = float(np.sqrt(GEM_TI / GEM_MI))
    # Harris current j_z = -(B0/lambda) sech^2, shared as u_iz/T_i = -u_ez/T_e
    uiz = -2.0 * GEM_TI / GEM_LAMBDA
    uez = +2.0 * GEM_TE / GEM_LAMBDA
    el = SpeciesSpec("electrons", q=-1.0, m=GEM_ME, nv=tuple(nv), vmin=(-6 * vthe,) * 3, vmax=(6 * vthe,) * 3,
                     vth=vthe, drift_z=uez)
    io = SpeciesSpec("ions", q=+1.0, m=GEM_MI, nv=tuple(nv), vmin=(-6 * vthi,) * 3, vmax=(6 * vthi,) * 3,
                     vth=vthi, drift_z=uiz)
    return [el, io]


def _nsub_for(c, dt_half, dx, dy, cfl=0.75):
    n = 1
    while c * (dt_half / n) * np.sqrt(2.0) / min(dx, dy) > cfl:
        n *= 2
    return n


def gem_workload(nx=64, ny=32, nv=32, steps=50, dt=0.005, seed=1, name=None, lx=25.6, ly=12.8) -> Workload:
    w = Workload(name or f"gem_{nx}x{ny}x{nv}^3", nx=nx, ny=ny, nghost_y=0, lx=lx, ly=ly, x0=-lx / 2, y0=-ly / 2,
                 bc_y_lo=BC_REFLECT, bc_y_hi=BC_REFLECT, dt=dt, steps=steps, species=gem_species(nv),
                 c=GEM_C, mu0=1.0, fields_yee=1, seed=seed, kind="gem")
    w.nsub = _nsub_for(w.c, dt / 2, w.dx, w.dy)
    return w


def band_workload(nx=256, ny_band=32, ny_domain=128, nv=40, g=3, steps=20, dt=0.005, seed=2,
                  lx=25.6, ly=12.8) -> Workload:
    """Config 4: the ny_band central rows of a (nx x ny_domain) GEM domain, g FLUID ghost rows per side."""
    dy = ly / ny_domain
    lyb = ny_band * dy
    w = Workload(f"band_{nx}x{ny_band}x{nv}^3", nx=nx, ny=ny_band, nghost_y=g, lx=lx, ly=lyb, x0=-lx / 2, y0=-lyb / 2,
                 bc_y_lo=BC_FLUID, bc_y_hi=BC_FLUID, dt=dt, steps=steps, species=gem_species(nv),
                 c=GEM_C, mu0=1.0, fields_yee=1, seed=seed, kind="band")
    w.nsub = _nsub_for(w.c, dt / 2, w.dx, w.dy)
    w.ly_domain = ly
    return w


def harris_density(y):
    return 1.0 / np.cosh(y / GEM_LAMBDA) ** 2


def gem_f(w: Workload, s: int, rows=None) -> np.ndarray:
    """f_s on rows `rows` (default: all ghost-inclusive rows):
    [sech^2(y/l) M(v; u_sz z, vth) + 0.2 M(v; 0, vth)] (1 + 1e-6 xi)."""
    sp = w.species[s]
    yc = w.y_centres_g()
    if rows is None:
        rows = range(w.ny_g)
    rows = list(rows)
    Md = _maxwellian_3d(sp, sp.drift_z)
    M0 = _maxwellian_3d(sp, 0.0)
    nvt = sp.ncell_v
    f = np.empty((len(rows), w.nx) + sp.nv)
    for k, r in enumerate(rows):
        blk = harris_density(yc[r]) * Md + GEM_NB * M0
        xi = hash_noise(w.seed, s, r * w.nx * nvt, w.nx * nvt).reshape((w.nx,) + sp.nv)
        xi *= 1e-6
        xi += 1.0
        np.multiply(xi, blk[None], out=f[k])
    return f


def gem_f_inf(w: Workload, s: int) -> float:
    """Upper bound of the initial f (reading R6): sheet centre value times the largest noise factor."""
    sp = w.species[s]
    peak = (_maxwellian_3d(sp, sp.drift_z) + GEM_NB * _maxwellian_3d(sp, 0.0)).max()
    return float(peak * (1.0 + 1e-6))


def gem_fields(w: Workload):
    """E = 0, B_x = tanh(y/l) - d_y psi, B_y = d_x psi, psi = psi0 cos(2 pi x/Lx) cos(pi y/Ly_domain).
    Sampled at the Yee positions of reading R17 if w.fields_yee else at cell centres."""
    ly_dom = getattr(w, "ly_domain", w.ly)
    lx = w.lx
    xi_ = w.x0 + np.arange(w.nx) * w.dx              # integer (node) x positions
    xh = xi_ + 0.5 * w.dx                            # half positions
    yj = w.y0 + (np.arange(w.ny_g) - w.nghost_y) * w.dy
    yh = yj + 0.5 * w.dy

    def bx(x, y):
        return np.tanh(y / GEM_LAMBDA) + GEM_PSI0 * (np.pi / ly_dom) * np.cos(2 * np.pi * x / lx) * np.sin(np.pi * y / ly_dom)

    def by(x, y):
        return -GEM_PSI0 * (2 * np.pi / lx) * np.sin(2 * np.pi * x / lx) * np.cos(np.pi * y / ly_dom)

    E = np.zeros((3, w.ny_g, w.nx))
    B = np.zeros((3, w.ny_g, w.nx))
    if w.fields_yee:
        B[0] = bx(xi_[None, :], yh[:, None])          # Bx(i, j+1/2)
        B[1] = by(xh[None, :], yj[:, None])           # By(i+1/2, j)
        if w.bc_y_lo != BC_PERIODIC:
            B[1, 0, :] = 0.0                            # PEC wall row
    else:
        B[0] = bx(xh[None, :], yh[:, None])
        B[1] = by(xh[None, :], yh[:, None])
    return E, B


def band_fluid_state(w: Workload, s: int, side: int, step_index: int) -> np.ndarray:
    """Config 4: seeded 5-moment state [5][g][nx] = n, ux, uy, uz, p of the ghost cells of one side,
    Harris-profile moments times (1 + 0.01 xi), redrawn per step.  Layer l counts outward."""
    sp = w.species[s]
    g = w.nghost_y
    yc = w.y_centres_g()
    out = np.zeros((5, g, w.nx))
    T = sp.m * sp.vth ** 2
    for l in range(g):
        row = g - 1 - l if side == 0 else g + w.ny + l
        sh = harris_density(yc[row])
        n = sh + GEM_NB
        base = [n, 0.0, 0.0, sh * sp.drift_z / n, n * T]
        for k in range(5):
            xi = hash_noise(w.seed, 1000 + 100 * s + 10 * side + k, (step_index * g + l) * w.nx, w.nx)
            out[k, l, :] = base[k] * (1.0 + 0.01 * xi)
    return out


def band_fluid_block(w: Workload, nyf: int, side: int):
    """A five-moment fluid block of nyf rows below (side 0) or above (side 1) the kinetic band of workload w, same dx, dy
    (the fluid region of the coupled set-up): the Harris-sheet moments per species as conserved variables
    U[ns][5][nyf + 4][nx] = rho, momentum density (3), energy density (eqs. 2-4, 8; two ghost rows per side), and the
    fields E, B [3][nyf + 4][nx] at the cell centres."""
    import copy
    wf = copy.deepcopy(w)
    wf.ny, wf.nghost_y, wf.fields_yee = nyf, 2, 0
    wf.ly = nyf * w.dy
    wf.y0 = w.y0 - nyf * w.dy if side == 0 else w.y0 + w.ny * w.dy
    wf.ly_domain = getattr(w, "ly_domain", w.ly)
    E, B = gem_fields(wf)
    yc = wf.y_centres_g()
    U = np.zeros((len(w.species), 5, nyf + 4, w.nx))
    for s, sp in enumerate(w.species):
        sh = harris_density(yc)[:, None] + 0 * np.arange(w.nx)[None, :]
        n = sh + GEM_NB
        T = sp.m * sp.vth ** 2
        uz = sh * sp.drift_z / n
        U[s, 0] = sp.m * n
        U[s, 3] = sp.m * n * uz
        U[s, 4] = 1.5 * n * T + 0.5 * sp.m * n * uz ** 2
    return U, E, B


# ------------------------------------------------------------------------------------------------
# 3D3V (NEXT-4): the Harris sheet extruded along z (uniform in z up to the noise), z periodic
# ------------------------------------------------------------------------------------------------
def gem3d_workload(nx=32, ny=32, nz=8, nv=32, steps=10, dt=0.005, seed=1, lx=25.6, ly=12.8, lz=6.4, name=None) -> Workload:
    w = gem_workload(nx=nx, ny=ny, nv=nv, steps=steps, dt=dt, seed=seed, lx=lx, ly=ly,
                     name=name or f"gem3d_{nx}x{ny}x{nz}x{nv}^3_x2species")
    w.nz, w.lz = nz, lz
    w.nsub = _nsub_for(w.c, dt / 2, min(w.dx, lz / nz), w.dy)
    w.kind = "gem3d"
    return w


def gem3d_f(w: Workload, s: int, k: int) -> np.ndarray:
    """Slab k of f_s [ny, nx, nvx, nvy, nvz]: the 2D Harris state with its own noise stream."""
    seed = w.seed
    w.seed = seed + 7919 * (k + 1)
    try:
        return gem_f(w, s)
    finally:
        w.seed = seed


def gem3d_fields(w: Workload):
    """[3, nz, ny, nx]: the 2D fields at every z (they do not depend on z)."""
    E, B = gem_fields(w)
    rep = lambda A: np.ascontiguousarray(np.broadcast_to(A[:, None], (3, w.nz) + A.shape[1:]))
    return rep(E), rep(B)
