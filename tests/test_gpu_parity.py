"""GPU parity: the CUDA path (through the C ABI) against the oracle, element by element, on the same
seeded inputs.  Tolerances are north_star's: relative L2 <= 1e-12 after one step, <= 1e-10 after 50
steps, relative mass drift <= 1e-13; moments <= 1e-12."""
import numpy as np
import pytest

from paper_1406_5445_b200 import inputs

pytestmark = pytest.mark.gpu

TOL1 = 1e-12
TOL50 = 1e-10


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1406_5445_b200 import binding
    binding.lib()           # fails loudly when the library is missing
    return binding


def rel_l2(a, b):
    a = np.asarray(a, dtype=np.float64).ravel()
    b = np.asarray(b, dtype=np.float64).ravel()
    d = np.linalg.norm(a - b)
    n = np.linalg.norm(b)
    return d / n if n > 0 else d


def local_scale(a, radius=3):
    """max |a| over the cells within `radius` along each velocity axis and within 1 along x and y (wrap-around)."""
    sc = np.abs(a)
    for ax, r in ((a.ndim - 1, radius), (a.ndim - 2, radius), (a.ndim - 3, radius), (1, 1), (0, 1)):
        if a.shape[ax] == 1:
            continue
        m = sc.copy()
        for k in range(1, r + 1):
            np.maximum(m, np.roll(sc, k, axis=ax), out=m)
            np.maximum(m, np.roll(sc, -k, axis=ax), out=m)
        sc = m
    return sc


def tail_check(got, want, tol=1e-10, what="", rel_tol=1e-9):
    """Element-wise check that sees the tails.  A global norm cannot see the corners of the velocity box of a
    Harris-sheet state (f ~ 1e-20 of the peak), where the multi-cell electron walks run.  Two bounds per cell:
      |got - want| <= tol * (largest |want| among the cells a sweep can bring in: the local scale), everywhere --
        eq. (38) forms f + (Phi - Phi), so a cell may legitimately be a cancellation residue of its neighbours;
      |got - want| <= rel_tol * |want| for the cells that are no such residue (|want| >= 1e-3 of the local scale).
    Prints the worst cell of each."""
    got = np.asarray(got); want = np.asarray(want)
    sc = local_scale(want)
    err = np.abs(got - want)
    pos = sc > 0
    a = np.zeros(want.shape); a[pos] = err[pos] / sc[pos]
    k = np.unravel_index(int(np.argmax(a)), a.shape)
    solid = np.abs(want) >= 1e-3 * sc
    solid &= pos
    r = np.zeros(want.shape); r[solid] = err[solid] / np.abs(want[solid])
    j = np.unravel_index(int(np.argmax(r)), r.shape)
    print(f"tail_check {what}: worst vs local scale {a[k]:.2e} at {tuple(int(i) for i in k)} (got {got[k]!r}, want {want[k]!r}, "
          f"scale {sc[k]:.2e}); worst relative {r[j]:.2e} at {tuple(int(i) for i in j)} (want {want[j]!r}); "
          f"smallest |want| checked {np.abs(want[solid]).min():.2e}")
    assert (err[~pos] == 0).all(), what
    assert a[k] <= tol, (what, k, got[k], want[k], sc[k])
    assert r[j] <= rel_tol, (what, j, got[j], want[j])


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def osp(orc, s):
    return orc.Species(s.q, s.m, s.nv, s.vmin, s.vmax, s.f_inf)


def random_workload(rng, nx, ny, nv, g=0, bc=inputs.BC_PERIODIC, nspecies=1, fields_yee=0, vmax=(4.0, 3.0, 2.0)):
    sp = []
    for s in range(nspecies):
        q = -1.0 if s == 0 else 1.0
        m = 1.0 if s == 0 else 4.0
        sp.append(inputs.SpeciesSpec(f"s{s}", q=q, m=m, nv=tuple(nv), vmin=tuple(-x for x in vmax), vmax=tuple(vmax), f_inf=1.0))
    w = inputs.Workload("random", nx=nx, ny=ny, nghost_y=g, lx=1.7, ly=0.9, x0=0.0, y0=0.0, bc_y_lo=bc, bc_y_hi=bc,
                        dt=0.05, steps=1, species=sp, c=3.0, mu0=1.0, nsub=1, fields_yee=fields_yee, seed=3)
    return w


def smooth_random_f(rng, w, s):
    """Positive, bounded by f_inf = 1, rough enough to exercise the limiters."""
    sp = w.species[s]
    shape = (w.ny_g, w.nx) + sp.nv
    c = [sp.centres(d) for d in range(3)]
    M = np.exp(-0.5 * ((c[0][:, None, None] / 1.3) ** 2 + (c[1][None, :, None] / 1.1) ** 2 + (c[2][None, None, :] / 0.8) ** 2))
    f = 0.9 * M[None, None] * (0.3 + 0.7 * rng.random(shape))
    f[rng.random(shape) < 0.05] = 0.0
    f[rng.random(shape) < 0.02] = 1.0
    return np.ascontiguousarray(f)


def run_both(gpu, orc, w, f0, E, B, dt, stages, order=0, limiter=1, fluid=None, fuse=None, mark_theta=None):
    """One vlasov_step on both sides.  Returns (f_gpu list, f_orc list, mom_gpu list, mom_orc list, code).
    mark_theta: also take the fluid boundary data of section 4.1 around the step (run_both.boundary[s][side] = (gpu, oracle))."""
    import torch
    fg = [dev(f) for f in f0]
    ctx = gpu.context_for(w, fg, order=order, limiter=limiter)
    if fuse is not None:
        ctx.vlasov_set_option(gpu.OPT_FUSE_XY, fuse)
    ctx.vlasov_timing_enable(True)
    keep = []
    if fluid is not None:
        for s in range(len(w.species)):
            for side in (0, 1):
                t = dev(fluid[s][side])
                keep.append(t)
                ctx.vlasov_set_boundary(s, side, inputs.BC_FLUID, t)
    Ed, Bd = dev(E), dev(B)
    if mark_theta is not None:
        ctx.vlasov_fluid_boundary_mark()
    ctx.vlasov_step(dt, Ed, Bd, stages)
    code = ctx.check_code()
    run_both.kinds = ctx.vlasov_timing_read()
    ctx.vlasov_timing_enable(False)
    momg = []
    for s in range(len(w.species)):
        m = torch.empty((10, w.ny_g, w.nx), dtype=torch.float64, device="cuda")
        ctx.vlasov_moments(s, m)
        momg.append(m.cpu().numpy())
    fo, momo = [], []
    for s, spec in enumerate(w.species):
        f = f0[s].copy()
        fl = (None, None) if fluid is None else fluid[s]
        err, _ = orc.step(f, osp(orc, spec), w.nx, w.ny, w.nghost_y, w.lx, w.ly, dt, E, B, fields_yee=w.fields_yee,
                          limiter=limiter, bc_lo=w.bc_y_lo, bc_hi=w.bc_y_hi, fluid_lo=fl[0], fluid_hi=fl[1], order=order,
                          stages=stages, want_moments=False)
        fo.append(f)
        momo.append(orc.moments(f, osp(orc, spec), w.nx, w.ny, w.nghost_y))
    if mark_theta is not None:
        run_both.boundary = []
        for s, spec in enumerate(w.species):
            per_side = []
            for side in (0, 1):
                b = torch.empty((10, w.nghost_y, w.nx), dtype=torch.float64, device="cuda")
                ctx.vlasov_fluid_boundary(s, side, mark_theta, b)
                per_side.append((b.cpu().numpy(), orc.fluid_boundary(f0[s], fo[s], osp(orc, spec), w.nx, w.ny, w.nghost_y,
                                                                     side, mark_theta)))
            run_both.boundary.append(per_side)
    out = [t.cpu().numpy() for t in fg]
    ctx.close()
    return out, fo, momg, momo, code


@pytest.mark.parametrize("bc", [inputs.BC_PERIODIC, inputs.BC_REFLECT])
@pytest.mark.parametrize("stages", [1, 4])
def test_spatial_half_steps(gpu, orc, bc, stages):
    """a1+a2 / a7+a8 on ragged sizes: shifts of both signs, several cells (|sigma| up to ~3.5), wrap-around."""
    rng = np.random.default_rng(1)
    w = random_workload(rng, nx=13, ny=9, nv=(6, 8, 10), bc=bc)
    f0 = [smooth_random_f(rng, w, 0)]
    Z = np.zeros((3, w.ny_g, w.nx))
    dt = 0.23         # sigma_x = vx * dt/2 / (1.7/13) up to 3.2 cells; sigma_y up to 3.0 cells
    fg, fo, mg, mo, code = run_both(gpu, orc, w, f0, Z, Z, dt, stages)
    assert code == 0
    assert rel_l2(fg[0], fo[0]) <= TOL1
    assert np.abs(fg[0] - fo[0]).max() <= 1e-13
    assert rel_l2(mg[0], mo[0]) <= TOL1


@pytest.mark.parametrize("bc,g", [(inputs.BC_PERIODIC, 0), (inputs.BC_REFLECT, 0), (inputs.BC_FLUID, 2), (inputs.BC_FLUID, 3)])
@pytest.mark.parametrize("nx,nv", [(13, (6, 8, 10)), (12, (4, 4, 8)), (16, (6, 8, 16)), (24, (3, 6, 32)),
                                   (64, (24, 24, 24)), (64, (32, 32, 32)), (128, (32, 32, 32)),
                                   (64, (48, 48, 48)), (256, (40, 40, 40)), (320, (4, 4, 8))])
@pytest.mark.parametrize("stages", [1, 4])
def test_fused_spatial_stage(gpu, orc, bc, g, nx, nv, stages):
    """a1+a2 / a7+a8 as ONE fused pass (all |sigma| < 1): x blocks of 1 and 4 cells, chunks of 2..32 velocity cells
    made of part of a v_z row / several rows, every y boundary kind; against the oracle and against the general
    one-direction kernels.  The shapes with nx = 64 / 128 / 256 are the compile-time-shape kernels of the benchmark
    configs (32^3 with nx = 64 / 128; 24^3 and 48^3 of config 5 with nx = 64; 40^3 of config 4 with nx = 256); nx = 320: a
    row wider than one TMA box (256 rows) arrives as two boxes."""
    rng = np.random.default_rng(5)
    w = random_workload(rng, nx=nx, ny=7 if nx < 64 else 3, nv=nv, g=g, bc=bc)
    if nx >= 64:
        w.lx = 3.4 * nx / 24      # full velocity grids reach |v_x| = 3.9: keeps |sigma_x| <= 0.7
    f0 = [smooth_random_f(rng, w, 0)]
    Z = np.zeros((3, w.ny_g, w.nx))
    dt = 0.05          # |sigma_x| <= 4 * 0.025 / (1.7/24) = 0.71 ... 0.38; |sigma_y| <= 3 * 0.025 / (0.9/7) = 0.58
    fg, fo, mg, mo, code = run_both(gpu, orc, w, f0, Z, Z, dt, stages, fuse=1)
    assert code == 0
    fused = run_both.kinds["sweep_xy" if stages == 1 else "sweep_yx"][1]
    assert fused == 1 and run_both.kinds["sweep_y"][1] == 0                              # the fused kernel ran
    assert run_both.kinds["ghost_sweep_x"][1] == (2 if g else 0) and run_both.kinds["sweep_x"][1] == 0   # ghost rows: x sweep only
    assert rel_l2(fg[0], fo[0]) <= TOL1
    assert np.abs(fg[0] - fo[0]).max() <= 1e-13
    assert rel_l2(mg[0], mo[0]) <= TOL1
    fu, _, _, _, code = run_both(gpu, orc, w, f0, Z, Z, dt, stages, fuse=0)
    assert code == 0
    assert run_both.kinds["sweep_xy"][1] + run_both.kinds["sweep_yx"][1] == 0 and run_both.kinds["sweep_y"][1] == 1
    assert rel_l2(fg[0], fu[0]) <= TOL1


@pytest.mark.parametrize("nv", [(12, 10, 14), (8, 16, 32), (32, 32, 32), (24, 24, 24), (4, 40, 40), (6, 48, 48), (16, 16, 16),
                                (40, 40, 40), (48, 48, 48), (6, 8, 8), (9, 8, 8), (12, 4, 8), (9, 4, 4)])
@pytest.mark.parametrize("fields_yee", [0, 1])
def test_velocity_step_multicell_shifts(gpu, orc, fields_yee, nv):
    """a3-a6: strong fields give sign-changing shifts of several cells; Yee gather vs cell-centred.  (12,10,14):
    ragged segments, the general face walk; (8,16,32) and 32^3: 8-cell segments, the register-window walk wherever a
    whole warp has |sigma| < 1 (and for 32^3 the compile-time-shape, TMA-staged kernels); the
    other shapes are the remaining compile-time-shape kernels (16, 24, 40: TMA-staged vy+vz; 48: plain; 16^3: TMA vx);
    (6,8,8), (9,8,8), (12,4,8), (9,4,4): small planes, where the generic vx kernel has more threads per column than
    segments of the line (trailing work items are empty and must neither read nor write)."""
    rng = np.random.default_rng(2)
    big = nv[0] * nv[1] * nv[2] > 8000
    w = random_workload(rng, nx=3 if big else 5, ny=2 if big else 4, nv=nv, bc=inputs.BC_REFLECT,
                        fields_yee=fields_yee)
    f0 = [smooth_random_f(rng, w, 0)]
    E = 6.0 * rng.standard_normal((3, w.ny_g, w.nx))
    B = 8.0 * rng.standard_normal((3, w.ny_g, w.nx))
    B *= 0.9 / (np.abs(B).max() * 0.5 * 0.1)        # |t| = |q/m dt/2 B| up to 0.9 per component? keep D1, D2 > 0
    B *= 0.5
    fg, fo, mg, mo, code = run_both(gpu, orc, w, f0, E, B, 0.1, 2)
    assert code == 0
    assert rel_l2(fg[0], fo[0]) <= TOL1
    assert np.abs(fg[0] - fo[0]).max() <= 2e-13          # element-wise: data of size <= 1
    assert rel_l2(mg[0], mo[0]) <= TOL1
    # the sweep really moved things by more than a cell somewhere
    assert np.abs(fg[0] - f0[0]).max() > 0.1


@pytest.mark.parametrize("nv", [(32, 32, 32), (24, 24, 24), (16, 16, 16), (48, 48, 48), (8, 16, 32)])
@pytest.mark.parametrize("limiter", [1, 0])
def test_velocity_step_moderate_rotation(gpu, orc, limiter, nv):
    """a3-a6 in the regime of the GEM electrons: rotation angles of 0.03 .. 0.25 per step, so sigma is nearly constant
    along a line (slope of a few hundredths per face) but reaches 0.5 .. 4 cells at the edge of the box, changes sign
    inside segments, and floor|sigma| steps by one inside segments.  This is what the flow-ordered walk for
    multi-cell shifts (shift identity) takes: box faces with floor|sigma| = 1, 2 (the whole
    cells added back at the outflow face), crossing lanes, both limiter settings (without the limiter the flux of
    the inflow box face is zeroed explicitly); 32 / 16: TMA kernels with whole warps, 24: partial warps, 48 and
    (8,16,32): the plain kernels, which admit one cell less before a line."""
    rng = np.random.default_rng(11)
    w = random_workload(rng, nx=4, ny=2, nv=nv, bc=inputs.BC_REFLECT, fields_yee=1)
    f0 = [smooth_random_f(rng, w, 0)]
    E = 2.0 * rng.standard_normal((3, w.ny_g, w.nx))
    B = rng.standard_normal((3, w.ny_g, w.nx))
    B *= rng.uniform(0.3, 2.5, size=(1, w.ny_g, w.nx)) / np.sqrt((B ** 2).sum(0, keepdims=True))
    fg, fo, mg, mo, code = run_both(gpu, orc, w, f0, E, B, 0.1, 2, limiter=limiter)
    assert code == 0
    assert rel_l2(fg[0], fo[0]) <= TOL1
    assert np.abs(fg[0] - fo[0]).max() <= 1e-13
    assert rel_l2(mg[0], mo[0]) <= TOL1
    m0 = f0[0].sum()
    assert abs(fg[0].sum() - m0) / m0 <= 1e-13      # zero flux through the box faces (R7)
    assert np.abs(fg[0] - f0[0]).max() > 0.1


@pytest.mark.parametrize("order", [0, 1])
@pytest.mark.parametrize("bc", [inputs.BC_PERIODIC, inputs.BC_REFLECT])
@pytest.mark.parametrize("nv,dt", [((6, 5, 7), 0.07), ((5, 3, 3), 0.07), ((4, 4, 5), 0.23), ((8, 6, 9), 0.02), ((6, 4, 1), 0.07)])
def test_full_step_odd_velocity_grids(gpu, orc, order, bc, nv, dt):
    """Velocity grids with an odd nv[2] (and an odd block, 5x3x3; a single v_z cell, 6x4x1): nothing in the method asks
    for an even count, only the 16-byte paths of the kernels do -- these shapes take one cell per thread in the spatial
    sweeps and the moments and column-by-column tile loads in the vx sweep.  dt = 0.02: all spatial shifts below one
    cell (the fused stage has no shape for an odd nv[2]: the general kernels run); 0.23: multi-cell shifts."""
    rng = np.random.default_rng(17)
    w = random_workload(rng, nx=7, ny=5, nv=nv, bc=bc, nspecies=2, fields_yee=1)
    f0 = [smooth_random_f(rng, w, s) for s in range(2)]
    E = rng.standard_normal((3, w.ny_g, w.nx))
    B = 2.0 * rng.standard_normal((3, w.ny_g, w.nx))
    fg, fo, mg, mo, code = run_both(gpu, orc, w, f0, E, B, dt, 31, order=order)
    assert code == 0
    assert run_both.kinds["sweep_xy"][1] + run_both.kinds["sweep_yx"][1] == 0
    for s in range(2):
        assert rel_l2(fg[s], fo[s]) <= TOL1
        assert np.abs(fg[s] - fo[s]).max() <= 2e-13
        assert rel_l2(mg[s], mo[s]) <= TOL1
        m0 = f0[s].sum()
        assert abs(fg[s].sum() - m0) / m0 <= 1e-13
        assert np.abs(fg[s] - f0[s]).max() > 0.05


@pytest.mark.parametrize("order", [0, 1])
@pytest.mark.parametrize("limiter", [1, 0])
def test_full_step_two_species(gpu, orc, order, limiter):
    rng = np.random.default_rng(3)
    w = random_workload(rng, nx=9, ny=6, nv=(8, 8, 8), bc=inputs.BC_REFLECT, nspecies=2, fields_yee=1)
    f0 = [smooth_random_f(rng, w, s) for s in range(2)]
    E = rng.standard_normal((3, w.ny_g, w.nx))
    B = 2.0 * rng.standard_normal((3, w.ny_g, w.nx))
    fg, fo, mg, mo, code = run_both(gpu, orc, w, f0, E, B, 0.07, 31, order=order, limiter=limiter)
    assert code == 0
    for s in range(2):
        assert rel_l2(fg[s], fo[s]) <= TOL1
        assert rel_l2(mg[s], mo[s]) <= TOL1
        m0 = f0[s].sum()
        assert abs(fg[s].sum() - m0) / m0 <= 1e-13


def test_gem_cut_one_step(gpu, orc):
    """A 16x8 spatial cut of config 2 (GEM Harris sheet, 16^3 velocity cells, both species, Yee fields, REFLECT)."""
    w = inputs.gem_workload(nx=16, ny=8, nv=16, steps=1)
    f0 = []
    for s in range(2):
        f0.append(inputs.gem_f(w, s))
        w.species[s].f_inf = inputs.gem_f_inf(w, s)
    E, B = inputs.gem_fields(w)
    fg, fo, mg, mo, code = run_both(gpu, orc, w, f0, E, B, w.dt, 31)
    assert code == 0
    for s in range(2):
        assert rel_l2(fg[s], fo[s]) <= TOL1, s
        assert rel_l2(mg[s], mo[s]) <= TOL1, s
        tail_check(fg[s], fo[s], what=f"gem cut one step, species {s}")
        m0 = f0[s].sum()
        assert abs(fg[s].sum() - m0) / m0 <= 1e-13


@pytest.mark.parametrize("nx,ny_band,nv", [(16, 8, 16), (16, 32, 40), (8, 8, 15)])
def test_ghost_fill_band(gpu, orc, nx, ny_band, nv):
    """a0 on a cut of config 4: FLUID sides, 3 ghost rows, seeded fluid state; ghost rows and interior.  15^3: an odd
    velocity block (column-by-column tile loads, one v_z column per thread in the moments).  (16, 32, 40) is
    SURVEY 8(d) config 4's "16x32 x-cut" at the real 40^3 velocity grid: there the ghost fill takes the general vx
    kernel in ghost mode (scale T[15], source cell T[16]) and the 40x40-plane vy+vz kernel."""
    w = inputs.band_workload(nx=nx, ny_band=ny_band, ny_domain=128, nv=nv, g=3)
    f0 = []
    for s in range(2):
        f0.append(inputs.gem_f(w, s))
        w.species[s].f_inf = inputs.gem_f_inf(w, s)
    E, B = inputs.gem_fields(w)
    fluid = [[inputs.band_fluid_state(w, s, side, 0) for side in (0, 1)] for s in range(2)]
    # ghost fill alone
    fg, fo, mg, mo, code = run_both(gpu, orc, w, f0, E, B, w.dt, 8, fluid=fluid)
    assert code == 0
    g = w.nghost_y
    for s in range(2):
        for rows in (slice(0, g), slice(g + w.ny, w.ny_g)):
            assert rel_l2(fg[s][rows], fo[s][rows]) <= TOL1
            assert np.abs(fg[s][rows] - fo[s][rows]).max() <= 1e-12 * w.species[s].f_inf
            tail_check(fg[s][rows], fo[s][rows], what=f"ghost rows, species {s}")
            assert np.abs(fg[s][rows] - f0[s][rows]).max() > 0          # it did something
        assert np.array_equal(fg[s][g:g + w.ny], f0[s][g:g + w.ny])     # interior untouched
    # whole step with ghost rows as Dirichlet data
    fg, fo, mg, mo, code = run_both(gpu, orc, w, f0, E, B, w.dt, 31, fluid=fluid, mark_theta=0.5)
    assert code == 0
    for s in range(2):
        assert rel_l2(fg[s], fo[s]) <= TOL1
        assert rel_l2(mg[s], mo[s]) <= TOL1
        tail_check(fg[s], fo[s], what=f"band step, species {s}")
        # the other direction of the coupling (section 4.1): boundary data for the fluid code at t + dt/2
        for side in (0, 1):
            got, want = run_both.boundary[s][side]
            assert rel_l2(got, want) <= TOL1
            assert np.abs(want[0]).min() > 0


def test_free_streaming_integer_shifts_exact_on_gpu(gpu):
    """T10 on the GPU: integer CFL shifts translate f exactly (no oracle involved)."""
    import torch
    nx, ny, nv = 12, 10, (4, 4, 2)
    sp = inputs.SpeciesSpec("e", -1.0, 1.0, nv, (-4.0, -1.0, -1.0), (4.0, 1.0, 1.0), f_inf=1.0)
    w = inputs.Workload("fs", nx=nx, ny=ny, nghost_y=0, lx=12.0, ly=2.5, x0=0, y0=0, bc_y_lo=0, bc_y_hi=0, dt=2.0,
                        steps=1, species=[sp], fields_yee=0)
    rng = np.random.default_rng(10)
    f0 = rng.random((ny, nx) + nv)
    fg = [dev(f0)]
    ctx = gpu.context_for(w, fg)
    Z = torch.zeros((3, ny, nx), dtype=torch.float64, device="cuda")
    ctx.vlasov_step(2.0, Z, Z, 31)
    ctx.vlasov_check()
    f = fg[0].cpu().numpy()
    vx = sp.centres(0)
    vy = sp.centres(1)
    for a in range(nv[0]):
        for b in range(nv[1]):
            sx = int(round(vx[a] * 2.0 / 1.0))
            sy = int(round(vy[b] * 2.0 / 0.25))
            want = np.roll(f0[:, :, a, b, :], (sy, sx), axis=(0, 1))
            assert np.abs(f[:, :, a, b, :] - want).max() <= 1e-14


def test_uniform_maxwellian_invariant_bitwise_on_gpu(gpu):
    """T11 on the GPU."""
    import torch
    nx, ny, nv = 6, 5, (8, 8, 8)
    sp = inputs.SpeciesSpec("e", -1.0, 1.0, nv, (-6.0,) * 3, (6.0,) * 3, f_inf=1.0)
    c = sp.centres(0)
    g = np.exp(-c ** 2 / 2) / np.sqrt(2 * np.pi)
    M = g[:, None, None] * g[None, :, None] * g[None, None, :]
    f0 = np.ascontiguousarray(np.broadcast_to(M, (ny, nx) + nv))
    sp.f_inf = float(f0.max())
    for bc in (0, 1):
        w = inputs.Workload("um", nx=nx, ny=ny, nghost_y=0, lx=3.0, ly=2.0, x0=0, y0=0, bc_y_lo=bc, bc_y_hi=bc, dt=0.37,
                            steps=1, species=[sp], fields_yee=0)
        fg = [dev(f0)]
        ctx = gpu.context_for(w, fg)
        Z = torch.zeros((3, ny, nx), dtype=torch.float64, device="cuda")
        ctx.vlasov_step(0.37, Z, Z, 31)
        ctx.vlasov_check()
        assert np.array_equal(fg[0].cpu().numpy(), f0)


def _poisson_E(ne_row, nx, dx):
    k = 2 * np.pi * np.fft.fftfreq(nx, d=dx)
    rho_hat = np.fft.fft(1.0 - ne_row)
    Eh = np.zeros(nx, dtype=complex)
    Eh[1:] = rho_hat[1:] / (1j * k[1:])
    return np.fft.ifft(Eh).real


def test_landau_config1_50_steps(gpu, orc):
    """configs[0]: 1 step <= 1e-12, 50 steps <= 1e-10, mass drift <= 1e-13; time-centred Poisson on the host (R11)
    computed by the same harness code from each side's own moments."""
    import torch
    w = inputs.landau_workload(steps=50)
    spec = w.species[0]
    f0 = inputs.landau_f(w)
    sp = osp(orc, spec)
    nx, ny = w.nx, w.ny
    fo = f0.copy()
    fg = [dev(f0)]
    ctx = gpu.context_for(w, fg)
    mom = torch.empty((10, ny, nx), dtype=torch.float64, device="cuda")
    Z = np.zeros((3, ny, nx))
    Zd = dev(Z)
    m0 = f0.sum()
    for n in range(50):
        orc.step(fo, sp, nx, ny, 0, w.lx, w.ly, w.dt, Z, Z, stages=orc.STAGE_X1, want_moments=False)
        Eo = Z.copy()
        Eo[0] = _poisson_E(orc.moments(fo, sp, nx, ny, 0)[0].mean(axis=0), nx, w.dx)[None, :]
        orc.step(fo, sp, nx, ny, 0, w.lx, w.ly, w.dt, Eo, Z, stages=orc.STAGE_V, want_moments=False)
        orc.step(fo, sp, nx, ny, 0, w.lx, w.ly, w.dt, Z, Z, stages=orc.STAGE_X2, want_moments=False)

        ctx.vlasov_step(w.dt, Zd, Zd, gpu.STAGE_X1)
        ctx.vlasov_moments(0, mom)
        Eg = Z.copy()
        Eg[0] = _poisson_E(mom[0].cpu().numpy().mean(axis=0), nx, w.dx)[None, :]
        ctx.vlasov_step(w.dt, dev(Eg), Zd, gpu.STAGE_V)
        ctx.vlasov_step(w.dt, Zd, Zd, gpu.STAGE_X2)
        if n == 0:
            ctx.vlasov_check()
            assert rel_l2(fg[0].cpu().numpy(), fo) <= TOL1
    ctx.vlasov_check()
    out = fg[0].cpu().numpy()
    assert rel_l2(out, fo) <= TOL50
    assert abs(out.sum() - m0) / m0 <= 1e-13


def test_maxwell_and_current(gpu, orc):
    import torch
    rng = np.random.default_rng(5)
    for bc, yee in ((inputs.BC_PERIODIC, 1), (inputs.BC_REFLECT, 1), (inputs.BC_REFLECT, 0)):
        w = random_workload(rng, nx=11, ny=7, nv=(4, 4, 4), bc=bc, nspecies=2, fields_yee=yee)
        f0 = [smooth_random_f(rng, w, s) for s in range(2)]
        fg = [dev(f) for f in f0]
        ctx = gpu.context_for(w, fg)
        J = torch.empty((3, w.ny_g, w.nx), dtype=torch.float64, device="cuda")
        ctx.vlasov_current(J)
        moms = [orc.moments(f0[s], osp(orc, w.species[s]), w.nx, w.ny, 0) for s in range(2)]
        wall = 0 if bc == inputs.BC_PERIODIC else 1
        Jo = orc.current(moms, [s.q for s in w.species], fields_yee=yee, wall=wall)
        assert rel_l2(J.cpu().numpy(), Jo) <= TOL1
        E = rng.standard_normal((3, w.ny_g, w.nx))
        B = rng.standard_normal((3, w.ny_g, w.nx))
        if wall:
            E[0, 0] = 0; E[2, 0] = 0; B[1, 0] = 0
        Eo, Bo = E.copy(), B.copy()
        Bavg_o = orc.maxwell(Eo, Bo, Jo, w.dx, w.dy, w.c, w.mu0, 0.01, 4, wall, want_bavg=True)
        Ed, Bd, Bavg = dev(E), dev(B), torch.empty((3, w.ny_g, w.nx), dtype=torch.float64, device="cuda")
        ctx.vlasov_maxwell(0.01, 4, Ed, Bd, dev(Jo), Bavg)
        ctx.vlasov_check()
        assert rel_l2(Ed.cpu().numpy(), Eo) <= 1e-14
        assert rel_l2(Bd.cpu().numpy(), Bo) <= 1e-14
        assert rel_l2(Bavg.cpu().numpy(), Bavg_o) <= 1e-14
        ctx.close()


@pytest.mark.parametrize("g", [1, 3])
def test_fluid_boundary_data(gpu, orc, g):
    """Section 4.1 (NEXT-2's Vlasov -> fluid half): moments of the g kinetic rows next to either border,
    marked at t, reduced again at t + dt, interpolated linearly in time; two species, both sides, theta inside and at
    the ends of [0, 1]; the call before any mark and on a context without ghost rows is refused."""
    import torch
    rng = np.random.default_rng(12)
    w = random_workload(rng, nx=5, ny=7, nv=(8, 6, 10), g=g, bc=inputs.BC_FLUID, nspecies=2)
    f_t = [smooth_random_f(rng, w, s) for s in range(2)]
    f_t1 = [smooth_random_f(rng, w, s) * rng.uniform(0.5, 1.0) for s in range(2)]
    fg = [dev(f) for f in f_t]
    ctx = gpu.context_for(w, fg)
    out = torch.zeros((10, g, w.nx), dtype=torch.float64, device="cuda")
    with pytest.raises(gpu.VlasovError) as e:
        ctx.vlasov_fluid_boundary(0, 0, 0.5, out)
    assert e.value.code == gpu.EINVAL
    ctx.vlasov_fluid_boundary_mark()
    for s in range(2):
        fg[s].copy_(dev(f_t1[s]))                  # "the Vlasov data has to be advanced before the fluid data"
    ctx.vlasov_touch()
    for s in range(2):
        sp = osp(orc, w.species[s])
        for side in (0, 1):
            for theta in (0.0, 0.3, 0.5, 1.0):
                ctx.vlasov_fluid_boundary(s, side, theta, out)
                assert ctx.check_code() == 0
                want = orc.fluid_boundary(f_t[s], f_t1[s], sp, w.nx, w.ny, g, side, theta)
                assert rel_l2(out.cpu().numpy(), want) <= TOL1, (s, side, theta)
    with pytest.raises(gpu.VlasovError):
        ctx.vlasov_fluid_boundary(2, 0, 0.5, out)
    ctx.close()
    w0 = random_workload(rng, nx=4, ny=4, nv=(4, 4, 4), g=0, bc=inputs.BC_PERIODIC)
    f0 = [dev(smooth_random_f(rng, w0, 0))]
    ctx = gpu.context_for(w0, f0)
    with pytest.raises(gpu.VlasovError) as e:
        ctx.vlasov_fluid_boundary_mark()
    assert e.value.code == gpu.EINVAL
    ctx.close()


def test_error_paths(gpu, orc):
    import torch
    rng = np.random.default_rng(6)
    # ESHIFT: FLUID side with one ghost row and a shift that needs more (R9)
    w = random_workload(rng, nx=4, ny=6, nv=(4, 4, 4), g=1, bc=inputs.BC_FLUID)
    f0 = [smooth_random_f(rng, w, 0)]
    fg = [dev(f0[0])]
    ctx = gpu.context_for(w, fg)
    Z = torch.zeros((3, w.ny_g, w.nx), dtype=torch.float64, device="cuda")
    ctx.vlasov_step(0.05, Z, Z, gpu.STAGE_X1)
    assert ctx.check_code() == gpu.ESHIFT
    assert ctx.check_code() == 0          # cleared
    # EDOMAIN: |t| > 1 makes a Boris denominator non-positive (R13)
    Bbig = torch.zeros((3, w.ny_g, w.nx), dtype=torch.float64, device="cuda")
    Bbig[0] = 100.0
    ctx.vlasov_step(0.05, Z, Bbig, gpu.STAGE_V)
    assert ctx.check_code() == gpu.EDOMAIN
    ctx.close()
    # EINVAL / EALIGN at init
    cfg = gpu.make_config(4, 4, 0, 1, 1.0, 1.0, 0, 0)
    sp = gpu.make_species(w.species)
    with pytest.raises(gpu.VlasovError) as e:
        gpu.Context(cfg, sp, [torch.zeros(4 * 4 * 64 + 2, dtype=torch.float64, device="cuda")[1:-1]])
    assert e.value.code == gpu.EALIGN
    cfg2 = gpu.make_config(0, 4, 0, 1, 1.0, 1.0, 0, 0)
    assert gpu.vlasov_scratch_bytes(cfg2, sp) == 0


def test_full_size_gem128_sampled_window(gpu, orc):
    """Config 3 at full size (128x64x32^3 x 2 species, 4.3 GB of f) in the launch configuration bench.py times: one
    complete step on the GPU, then (i) properties that hold at any size -- relative mass drift <= 1e-13, f >= 0 --
    and (ii) sampled parity: a 16x16 spatial window of the same inputs is advanced by the oracle; the domain of
    dependence of one step is 4 cells per direction (two half sweeps, |sigma| < 1, stencil of 2), so the inner 6x6
    cells of the window must agree with the full run whatever the window's own boundary."""
    import torch
    free, _ = torch.cuda.mem_get_info()
    if free < 9 * 2**30:
        pytest.skip("needs 9 GB of device memory")
    w = inputs.gem_workload(nx=128, ny=64, nv=32, steps=1)
    ix0, iy0, nw, margin = 40, 24, 16, 5
    E, B = inputs.gem_fields(w)
    fg, f0win, mass0 = [], [], []
    for s, sp in enumerate(w.species):
        sp.f_inf = inputs.gem_f_inf(w, s)
        f = torch.empty((w.ny_g, w.nx) + tuple(sp.nv), dtype=torch.float64, device="cuda")
        win = np.empty((nw, nw) + tuple(sp.nv))
        for r in range(w.ny_g):
            row = inputs.gem_f(w, s, rows=[r])[0]
            f[r].copy_(torch.from_numpy(row))
            if iy0 <= r < iy0 + nw:
                win[r - iy0] = row[ix0:ix0 + nw]
        fg.append(f)
        f0win.append(win)
        mass0.append(float(f.sum().item()))
    ctx = gpu.context_for(w, fg)
    ctx.vlasov_timing_enable(True)
    Ed, Bd = dev(E), dev(B)
    ctx.vlasov_step(w.dt, Ed, Bd, gpu.STAGE_ALL)
    assert ctx.check_code() == 0
    kinds = ctx.vlasov_timing_read()
    assert kinds["sweep_xy"][1] == 2 and kinds["sweep_yx"][1] == 2 and kinds["vsweep_yz"][1] == 2   # as bench.py times it
    Ew = np.ascontiguousarray(E[:, iy0:iy0 + nw, ix0:ix0 + nw])
    Bw = np.ascontiguousarray(B[:, iy0:iy0 + nw, ix0:ix0 + nw])
    inner = slice(margin, nw - margin)
    for s, sp in enumerate(w.species):
        drift = abs(float(fg[s].sum().item()) - mass0[s]) / mass0[s]
        assert drift <= 1e-13, (s, drift)
        assert float(fg[s].min().item()) >= 0.0
        fo = f0win[s].copy()
        err, _ = orc.step(fo, osp(orc, sp), nw, nw, 0, nw * w.dx, nw * w.dy, w.dt, Ew, Bw, fields_yee=w.fields_yee,
                          bc_lo=inputs.BC_PERIODIC, bc_hi=inputs.BC_PERIODIC, want_moments=False)
        assert err == 0
        got = fg[s][iy0:iy0 + nw, ix0:ix0 + nw].cpu().numpy()
        assert rel_l2(got[inner, inner], fo[inner, inner]) <= TOL1, s
        assert np.abs(got[inner, inner] - fo[inner, inner]).max() <= 1e-13 * sp.f_inf
        tail_check(got[inner, inner], fo[inner, inner], what=f"gem128 window, species {s}")
        # and the window's own edge does differ (the comparison is not vacuous)
        assert rel_l2(got[0], fo[0]) > 1e-9
    ctx.close()


def _full_size_window(gpu, orc, w, ix0, nw, iy0=None, margin=5, fluid=None, expect=None, need_gb=9):
    """One complete step of workload w at full size on the GPU (as bench.py runs it), then the oracle on the spatial
    window [iy0, iy0 + nw) x [ix0, ix0 + nw) of the same inputs (iy0 None: every row, ghost rows included, with the
    workload's own y boundaries); cells at least `margin` from the window's artificial edges must agree (domain of
    dependence of a step: 4 cells per direction).  Also the properties that hold at any size: mass, f >= 0 up to rounding
    (periodic or wall sides only: ghost fills are not conservative)."""
    import torch
    free, _ = torch.cuda.mem_get_info()
    if free < need_gb * 2**30:
        pytest.skip(f"needs {need_gb} GB of device memory")
    rows = range(w.ny_g) if iy0 is None else range(iy0, iy0 + nw)
    E, B = inputs.gem_fields(w)
    fg, f0win, mass0 = [], [], []
    for s, sp in enumerate(w.species):
        sp.f_inf = inputs.gem_f_inf(w, s)
        f = torch.empty((w.ny_g, w.nx) + tuple(sp.nv), dtype=torch.float64, device="cuda")
        win = np.empty((len(rows), nw) + tuple(sp.nv))
        for r in range(w.ny_g):
            row = inputs.gem_f(w, s, rows=[r])[0]
            f[r].copy_(torch.from_numpy(row))
            if r in rows:
                win[r - rows[0]] = row[ix0:ix0 + nw]
        fg.append(f)
        f0win.append(win)
        mass0.append(float(f.sum().item()))
    ctx = gpu.context_for(w, fg)
    keep = []
    if fluid is not None:
        for s in range(len(w.species)):
            for side in (0, 1):
                keep.append(dev(fluid[s][side]))
                ctx.vlasov_set_boundary(s, side, inputs.BC_FLUID, keep[-1])
    ctx.vlasov_timing_enable(True)
    Ed, Bd = dev(E), dev(B)
    ctx.vlasov_step(w.dt, Ed, Bd, gpu.STAGE_ALL)
    assert ctx.check_code() == 0
    kinds = ctx.vlasov_timing_read()
    for k, n in (expect or {}).items():
        assert kinds[k][1] == n, (k, kinds[k])
    ys = slice(None) if iy0 is None else slice(iy0, iy0 + nw)
    Ew = np.ascontiguousarray(E[:, ys, ix0:ix0 + nw])
    Bw = np.ascontiguousarray(B[:, ys, ix0:ix0 + nw])
    inner_x = slice(margin, nw - margin)
    inner_y = slice(None) if iy0 is None else slice(margin, nw - margin)
    for s, sp in enumerate(w.species):
        if fluid is None:
            drift = abs(float(fg[s].sum().item()) - mass0[s]) / mass0[s]
            assert drift <= 1e-13, (s, drift)
            # eq. (38) forms f + (Phi - Phi): a cell that empties is left with a rounding residue of its neighbours' size
            assert float(fg[s].min().item()) >= -1e-15 * sp.f_inf
        fo = f0win[s].copy()
        if iy0 is None:
            fl = (None, None) if fluid is None else tuple(np.ascontiguousarray(fluid[s][side][:, :, ix0:ix0 + nw]) for side in (0, 1))
            err, _ = orc.step(fo, osp(orc, sp), nw, w.ny, w.nghost_y, nw * w.dx, w.ly, w.dt, Ew, Bw, fields_yee=w.fields_yee,
                              bc_lo=w.bc_y_lo, bc_hi=w.bc_y_hi, fluid_lo=fl[0], fluid_hi=fl[1], want_moments=False)
        else:
            err, _ = orc.step(fo, osp(orc, sp), nw, nw, 0, nw * w.dx, nw * w.dy, w.dt, Ew, Bw, fields_yee=w.fields_yee,
                              bc_lo=inputs.BC_PERIODIC, bc_hi=inputs.BC_PERIODIC, want_moments=False)
        assert err == 0
        got = fg[s][ys, ix0:ix0 + nw].cpu().numpy()
        assert rel_l2(got[inner_y, inner_x], fo[inner_y, inner_x]) <= TOL1, s
        assert np.abs(got[inner_y, inner_x] - fo[inner_y, inner_x]).max() <= 1e-13 * sp.f_inf
        tail_check(got[inner_y, inner_x], fo[inner_y, inner_x], what=f"{w.name} window, species {s}")
        assert rel_l2(got[:, 0], fo[:, 0]) > 1e-9          # the window's own edge does differ: not vacuous
    ctx.close()


@pytest.mark.parametrize("nv", [48, 24, 16])
def test_full_size_velocity_resolution_sweep_sampled_window(gpu, orc, nv):
    """Config 5 (64x64 x nv^3 x 2 species) at full size, as `bench.py --workload nv48 | nv24 | nv16` runs it: persistent
    velocity kernels with many tiles per CTA on 48x48 / 24x24 / 16x16 planes, the compile-time-shape fused stages."""
    w = inputs.gem_workload(nx=64, ny=64, nv=nv, steps=1)
    _full_size_window(gpu, orc, w, ix0=24, nw=16, iy0=24,
                      expect={"sweep_xy": 2, "sweep_yx": 2, "vsweep_yz": 2, "vsweep_x": 2, "sweep_x": 0, "sweep_y": 0},
                      need_gb=14 if nv == 48 else 4)


def test_full_size_band_sampled_window(gpu, orc):
    """Config 4 at full size (256 x 32 band + 3 FLUID ghost rows per side, 40^3, 2 species; 10 GB of f) as
    `bench.py --workload band` runs it: ghost fill, fused stages on the interior, x sweeps of the ghost rows.  The oracle
    advances every row of a 16-column cut with the same fluid state; its inner 6 columns must agree, ghost rows included."""
    w = inputs.band_workload()
    fluid = [[inputs.band_fluid_state(w, s, side, 0) for side in (0, 1)] for s in range(2)]
    _full_size_window(gpu, orc, w, ix0=100, nw=16, iy0=None, fluid=fluid,
                      expect={"sweep_xy": 2, "sweep_yx": 2, "ghost_vsweep_yz": 4, "ghost_sweep_x": 8, "sweep_y": 0}, need_gb=18)


def test_gem_cut_50_cycles(gpu, orc):
    """north_star's long bar on a cut of config 2 (GEM Harris sheet, both species, 50 steps): 50 full cycles of
    section 4.3 (currents -> Maxwell half step -> Vlasov step -> currents -> Maxwell half step) through vlasov_cycle
    against the same cycle composed from the oracle's functions: relative L2 <= 1e-10 on f, fields and moments,
    relative mass drift <= 1e-13 per species."""
    import os
    import sys
    import torch
    sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
    import bench
    w = inputs.gem_workload(nx=16, ny=8, nv=16, steps=50)
    ref = bench.OracleRun(w)                       # sets f_inf of the species, builds f, E, B, initial moments
    fg = [dev(f) for f in ref.f]
    mass0 = [float(f.sum()) for f in ref.f]
    ctx = gpu.context_for(w, fg)
    Ed, Bd = dev(ref.E), dev(ref.B)
    for _ in range(50):
        ctx.vlasov_cycle(w.dt, w.nsub, Ed, Bd)
        ref.cycle()
    assert ctx.check_code() == 0
    assert rel_l2(Ed.cpu().numpy(), ref.E) <= TOL50
    assert rel_l2(Bd.cpu().numpy(), ref.B) <= TOL50
    mom = torch.empty((10, w.ny_g, w.nx), dtype=torch.float64, device="cuda")
    for s in range(2):
        got = fg[s].cpu().numpy()
        assert rel_l2(got, ref.f[s]) <= TOL50, s
        tail_check(got, ref.f[s], tol=1e-8, rel_tol=1e-7, what=f"50 cycles, species {s}")
        ctx.vlasov_moments(s, mom)
        assert rel_l2(mom.cpu().numpy(), ref.mom[s]) <= TOL50, s
        assert abs(float(got.sum()) - mass0[s]) / mass0[s] <= 1e-13, s
        assert np.abs(got - inputs.gem_f(w, s)).max() > 1e-6 * got.max()         # 50 steps did move things
    ctx.close()


def out_of_range_f(rng, w, s):
    """Data OUTSIDE [0, f_inf] (R6: eps is clamped to [0, 1], so negative cells and cells above f_inf take the
    max(0, .) clamps of the limiter): 4 % negative cells down to -0.3, 4 % cells at 1.3 f_inf, the rest rough and
    positive.  The compressive ghost remap produces f > f_inf in practice."""
    f = smooth_random_f(rng, w, s)
    r = rng.random(f.shape)
    f[r < 0.04] = -0.3 * rng.random(int((r < 0.04).sum()))
    f[r > 0.96] = 1.3
    return np.ascontiguousarray(f)


@pytest.mark.parametrize("nv", [(32, 32, 32), (12, 10, 14), (16, 16, 16)])
def test_velocity_step_inputs_outside_0_finf(gpu, orc, nv):
    """a4-a6 with f outside [0, f_inf] (R6 clamps; relu_bits on the CUDA side), multi-cell and
    sub-cell shifts, every walk."""
    rng = np.random.default_rng(31)
    for scale in (0.3, 1.0):
        w = random_workload(rng, nx=3, ny=2, nv=nv, bc=inputs.BC_REFLECT, fields_yee=1)
        f0 = [out_of_range_f(rng, w, 0)]
        E = scale * 2.0 * rng.standard_normal((3, w.ny_g, w.nx))
        B = scale * 2.5 * rng.standard_normal((3, w.ny_g, w.nx))
        fg, fo, mg, mo, code = run_both(gpu, orc, w, f0, E, B, 0.1, 2)
        assert code == 0
        assert fo[0].min() < 0 and fo[0].max() > 1.0
        assert rel_l2(fg[0], fo[0]) <= TOL1
        assert np.abs(fg[0] - fo[0]).max() <= 3e-13
        assert rel_l2(mg[0], mo[0]) <= TOL1


@pytest.mark.parametrize("bc,g", [(inputs.BC_REFLECT, 0), (inputs.BC_FLUID, 2)])
@pytest.mark.parametrize("nx,nv", [(13, (6, 8, 10)), (64, (32, 32, 32))])
@pytest.mark.parametrize("stages", [1, 4])
def test_spatial_stage_inputs_outside_0_finf(gpu, orc, bc, g, nx, nv, stages):
    """a1+a2 / a7+a8 (fused and general kernels) with f outside [0, f_inf]: the batched limiter vote and the clamps."""
    rng = np.random.default_rng(32)
    w = random_workload(rng, nx=nx, ny=5 if nx < 64 else 3, nv=nv, g=g, bc=bc)
    if nx >= 64:
        w.lx = 3.4 * nx / 24
    f0 = [out_of_range_f(rng, w, 0)]
    Z = np.zeros((3, w.ny_g, w.nx))
    for fuse in (1, 0):
        fg, fo, mg, mo, code = run_both(gpu, orc, w, f0, Z, Z, 0.05, stages, fuse=fuse)
        assert code == 0
        assert rel_l2(fg[0], fo[0]) <= TOL1
        assert np.abs(fg[0] - fo[0]).max() <= 3e-13


@pytest.mark.slow
def test_gem64_full_size_50_cycles(gpu, orc):
    """Config 2 at its REAL size (64x32 spatial x 32^3 velocity, electrons and ions, 1.07 GB of f; electron velocity
    shifts up to 2.9 cells): 50 cycles of section 4.3 through vlasov_cycle against oracle.cycle.  north_star's bars:
    relative L2 <= 1e-12 after one cycle and <= 1e-10 after 50 on f, E, B and the moments, relative mass drift
    <= 1e-13 per species; plus the element-wise check that sees the tails."""
    import os
    import sys
    import torch
    sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
    import bench
    w = inputs.gem_workload(nx=64, ny=32, nv=32, steps=50)
    ref = bench.OracleRun(w)
    fg = [dev(f) for f in ref.f]
    mass0 = [float(f.sum()) for f in ref.f]
    ctx = gpu.context_for(w, fg)
    ctx.vlasov_timing_enable(True)
    Ed, Bd = dev(ref.E), dev(ref.B)
    for n in range(50):
        ctx.vlasov_cycle(w.dt, w.nsub, Ed, Bd)
        ref.cycle()
        if n == 0:
            assert ctx.check_code() == 0
            kinds = ctx.vlasov_timing_read()
            assert kinds["sweep_xy"][1] == 2 and kinds["sweep_yx"][1] == 2 and kinds["vsweep_yz"][1] == 2
            ctx.vlasov_timing_enable(False)
            for s in range(2):
                assert rel_l2(fg[s].cpu().numpy(), ref.f[s]) <= TOL1, s
    assert ctx.check_code() == 0
    assert rel_l2(Ed.cpu().numpy(), ref.E) <= TOL50
    assert rel_l2(Bd.cpu().numpy(), ref.B) <= TOL50
    mom = torch.empty((10, w.ny_g, w.nx), dtype=torch.float64, device="cuda")
    for s in range(2):
        got = fg[s].cpu().numpy()
        assert rel_l2(got, ref.f[s]) <= TOL50, s
        tail_check(got, ref.f[s], tol=1e-8, rel_tol=1e-7, what=f"gem64 50 cycles, species {s}")
        ctx.vlasov_moments(s, mom)
        assert rel_l2(mom.cpu().numpy(), ref.mom[s]) <= TOL50, s
        assert abs(float(got.sum()) - mass0[s]) / mass0[s] <= 1e-13, s
        assert float(got.min()) >= 0.0
    ctx.close()


def test_init_and_step_refusals(gpu):
    """Argument checks added for robustness: a REFLECT wall needs a vy grid symmetric about 0 (the image is built by
    mirroring the i_vy index, R19); a ghost fill needs the fluid state of every FLUID side."""
    import torch
    rng = np.random.default_rng(8)
    sp = inputs.SpeciesSpec("e", -1.0, 1.0, (4, 4, 4), (-2.0, -1.0, -2.0), (2.0, 3.0, 2.0), f_inf=1.0)
    w = inputs.Workload("asym", nx=4, ny=4, nghost_y=0, lx=1.0, ly=1.0, x0=0, y0=0, bc_y_lo=inputs.BC_REFLECT,
                        bc_y_hi=inputs.BC_REFLECT, dt=0.1, steps=1, species=[sp], fields_yee=0)
    f = [torch.zeros((4, 4, 4, 4, 4), dtype=torch.float64, device="cuda")]
    with pytest.raises(gpu.VlasovError) as e:
        gpu.context_for(w, f)
    assert e.value.code == gpu.EINVAL
    w.bc_y_lo = w.bc_y_hi = inputs.BC_PERIODIC          # the same grid is fine without a wall
    gpu.context_for(w, f).close()
    w2 = random_workload(rng, nx=4, ny=4, nv=(4, 4, 4), g=2, bc=inputs.BC_FLUID)
    f2 = [dev(smooth_random_f(rng, w2, 0))]
    ctx = gpu.context_for(w2, f2)
    Z = torch.zeros((3, w2.ny_g, w2.nx), dtype=torch.float64, device="cuda")
    with pytest.raises(gpu.VlasovError) as e:
        ctx.vlasov_step(0.01, Z, Z, gpu.STAGE_ALL)
    assert e.value.code == gpu.EINVAL
    ctx.vlasov_step(0.01, Z, Z, gpu.STAGE_ALL & ~gpu.STAGE_GHOST)      # without the ghost stage the caller's rows are used
    assert ctx.check_code() == 0
    ctx.close()


@pytest.mark.parametrize("nv", [(8, 8, 8), (6, 5, 7)])
def test_f_inf_taken_from_the_data_at_init(gpu, orc, nv):
    """f_inf <= 0 asks vlasov_init for max f of the data as it stands (reading R6): the step must then be the
    oracle's with f_inf = max f of each species -- on data that does touch its upper bound (cells at the maximum next
    to empty ones), so a wrong f_inf shows."""
    rng = np.random.default_rng(23)
    w = random_workload(rng, nx=6, ny=5, nv=nv, bc=inputs.BC_REFLECT, nspecies=2, fields_yee=1)
    f0 = [(0.4 + 0.5 * s) * smooth_random_f(rng, w, s) for s in range(2)]
    E = rng.standard_normal((3, w.ny_g, w.nx))
    B = 2.0 * rng.standard_normal((3, w.ny_g, w.nx))
    for s in range(2):
        w.species[s].f_inf = 0.0 if s == 0 else -1.0
    fg = [dev(f) for f in f0]
    ctx = gpu.context_for(w, fg)
    ctx.vlasov_step(0.07, dev(E), dev(B), gpu.STAGE_ALL)
    assert ctx.check_code() == 0
    for s in range(2):
        w.species[s].f_inf = float(f0[s].max())
        assert abs(w.species[s].f_inf - (0.4 + 0.5 * s)) < 1e-15
        fo = f0[s].copy()
        err, _ = orc.step(fo, osp(orc, w.species[s]), w.nx, w.ny, 0, w.lx, w.ly, 0.07, E, B, fields_yee=1, bc_lo=w.bc_y_lo,
                          bc_hi=w.bc_y_hi, want_moments=False)
        assert err == 0
        got = fg[s].cpu().numpy()
        assert rel_l2(got, fo) <= TOL1
        assert np.abs(got - fo).max() <= 2e-13
        # and the bound matters here: the same step with a loose f_inf differs
        w.species[s].f_inf = 10.0
        fl = f0[s].copy()
        orc.step(fl, osp(orc, w.species[s]), w.nx, w.ny, 0, w.lx, w.ly, 0.07, E, B, fields_yee=1, bc_lo=w.bc_y_lo,
                 bc_hi=w.bc_y_hi, want_moments=False)
        assert np.abs(fl - fo).max() > 1e-6
    ctx.close()


@pytest.mark.parametrize("nv", [(32, 32, 32), (16, 16, 16), (24, 24, 24)])
def test_vxv_step_with_moments_fused_into_the_last_velocity_pass(gpu, orc, nv):
    """NEXT-1: the order of the paper's coupled cycle, v/2 - x,y - v/2, with the 10 moments
    of the final f reduced inside the last vy+vz pass (16^3 and 32^3 blocks: no separate moments launch; 24^3 keeps
    the moments kernel).  f and moments against the oracle's VXV step (pinned by T10/T12/T16 under order = 1), and
    against the same step with the fusion switched off."""
    import torch
    rng = np.random.default_rng(17)
    w = random_workload(rng, nx=5, ny=3, nv=nv, bc=inputs.BC_REFLECT, nspecies=2, fields_yee=1, vmax=(4.0, 3.0, 3.5))
    f0 = [smooth_random_f(rng, w, s) for s in range(2)]
    E = rng.standard_normal((3, w.ny_g, w.nx))
    B = 1.5 * rng.standard_normal((3, w.ny_g, w.nx))
    fg, fo, mg, mo, code = run_both(gpu, orc, w, f0, E, B, 0.05, 31, order=1)
    assert code == 0
    k = run_both.kinds
    fused = nv[0] in (16, 32)
    assert k["vsweep_yz"][1] == 4 and k["moments"][1] == (0 if fused else 2), k
    for s in range(2):
        assert rel_l2(fg[s], fo[s]) <= TOL1
        assert np.abs(fg[s] - fo[s]).max() <= 2e-13
        assert rel_l2(mg[s], mo[s]) <= TOL1
        for q in range(10):                       # every moment on its own (the small ones too)
            assert np.abs(mg[s][q] - mo[s][q]).max() <= 1e-12 * np.abs(mo[s][[0, 4, 5, 6]]).max(), (s, q)
    # the same step with the separate moments kernel
    fg2 = [dev(f) for f in f0]
    ctx = gpu.context_for(w, fg2, order=1)
    ctx.vlasov_set_option(gpu.OPT_FUSE_MOMENTS, 0)
    ctx.vlasov_timing_enable(True)
    ctx.vlasov_step(0.05, dev(E), dev(B), 31)
    assert ctx.check_code() == 0
    assert ctx.vlasov_timing_read()["moments"][1] == 2
    m = torch.empty((10, w.ny_g, w.nx), dtype=torch.float64, device="cuda")
    for s in range(2):
        ctx.vlasov_moments(s, m)
        assert np.array_equal(fg2[s].cpu().numpy(), fg[s])
        assert rel_l2(m.cpu().numpy(), mg[s]) <= 1e-14
    ctx.close()
