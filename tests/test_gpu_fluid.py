"""GPU parity of the fluid side of the coupling (vlasov_fluid_step, vlasov_fluid_from_moments, vlasov_fluid_to_boundary;
section 3.2, section 4.1) against oracle/fluid.py, and the closed coupling loop of Fig. 3
(PAPER.md:416): kinetic band <-> two fluid blocks, each feeding the other's ghost rows, on both sides."""
import numpy as np
import pytest

from paper_1406_5445_b200 import inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1406_5445_b200 import binding
    binding.lib()
    return binding


@pytest.fixture(scope="module")
def fl():
    from oracle import fluid
    return fluid


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def rel(a, b):
    return np.linalg.norm(np.ravel(a) - np.ravel(b)) / np.linalg.norm(np.ravel(b))


def rough_state(rng, ns, ny, nx):
    """Positive density and pressure, velocities of the order of the sound speed, rough enough for the weights to act."""
    U = np.zeros((ns, 5, ny + 4, nx))
    for s in range(ns):
        rho = 1.0 + 0.5 * rng.random((ny + 4, nx))
        rho[ny // 2:, : nx // 2] *= 3.0                       # a step
        v = 0.6 * (rng.random((3, ny + 4, nx)) - 0.5)
        p = 0.8 + 0.4 * rng.random((ny + 4, nx))
        U[s, 0] = rho
        U[s, 1:4] = rho[None] * v
        U[s, 4] = 1.5 * p + 0.5 * rho * (v ** 2).sum(0)
    return U


@pytest.mark.parametrize("bc", [0, 1, 2])
@pytest.mark.parametrize("ny,nx", [(7, 9), (16, 32), (2, 3)])
def test_fluid_step_parity(gpu, fl, bc, ny, nx):
    rng = np.random.default_rng(41)
    ns = 2
    q, m = [-1.0, 1.0], [0.04, 1.0]
    U0 = rough_state(rng, ns, ny, nx)
    E = 0.3 * rng.standard_normal((3, ny + 4, nx))
    B = 0.5 * rng.standard_normal((3, ny + 4, nx))
    dx, dy, dt = 0.11, 0.13, 0.004
    blk = gpu.FluidBlock(nx, ny, dx, dy, q, m, bc, bc)
    Ug, Uo = dev(U0), U0.copy()
    for k in range(4):
        gl = gh = None
        if bc == 2:
            gl = rough_state(np.random.default_rng(100 + k), 3 * ns, -2, nx).reshape(3, ns, 5, 2, nx)
            gh = rough_state(np.random.default_rng(200 + k), 3 * ns, -2, nx).reshape(3, ns, 5, 2, nx)
        blk.vlasov_fluid_step(dt, Ug, dev(E), dev(B), None if gl is None else dev(gl), None if gh is None else dev(gh))
        fl.step(Uo, q, m, dt, dx, dy, E, B, bc, bc, gl, gh)
        got = Ug.cpu().numpy()
        assert np.isfinite(got).all()
        assert rel(got[:, :, 2:-2], Uo[:, :, 2:-2]) <= 1e-12, k
        assert np.abs(got[:, :, 2:-2] - Uo[:, :, 2:-2]).max() <= 1e-12 * np.abs(Uo).max(), k
    assert np.abs(Uo[:, :, 2:-2] - U0[:, :, 2:-2]).max() > 1e-3


def test_fluid_step_refusals(gpu):
    import torch
    blk = gpu.FluidBlock(4, 4, 0.1, 0.1, [1.0], [1.0], 2, 2)
    U = torch.ones((1, 5, 8, 4), dtype=torch.float64, device="cuda")
    Z = torch.zeros((3, 8, 4), dtype=torch.float64, device="cuda")
    with pytest.raises(gpu.VlasovError) as e:
        blk.vlasov_fluid_step(0.01, U, Z, Z)          # COUPLED sides without ghost data
    assert e.value.code == gpu.EINVAL
    with pytest.raises(gpu.VlasovError):
        gpu.FluidBlock(4, 4, 0.1, 0.1, [1.0], [1.0], 0, 1).vlasov_fluid_step(0.01, U, Z, Z)     # periodic on one side only


def test_moment_conversions_parity(gpu, fl):
    import torch
    rng = np.random.default_rng(42)
    m = 0.04
    mom = rng.random((10, 3, 5)) + 0.5
    mom[4:7] += 3.0                                   # keeps the pressure positive
    U = torch.empty((5, 3, 5), dtype=torch.float64, device="cuda")
    gpu.vlasov_fluid_from_moments(dev(mom), m, U)
    want = fl.from_moments(mom, m)
    assert rel(U.cpu().numpy(), want) <= 1e-15
    b5 = torch.empty((5, 3, 5), dtype=torch.float64, device="cuda")
    gpu.vlasov_fluid_to_boundary(U, m, b5)
    assert rel(b5.cpu().numpy(), fl.to_boundary5(want, m)) <= 1e-14
    assert (b5[4] > 0).all()


# ---------------------------------------------------------------------------------------------------------------------
# the closed loop of Fig. 3: kinetic band between two fluid blocks
# ---------------------------------------------------------------------------------------------------------------------
class CoupledRun:
    """One side (GPU or oracle) of the coupled run; the two subclasses differ only in who does the arithmetic."""
    NYF = 6

    def __init__(self, w):
        self.w = w
        self.q = [sp.q for sp in w.species]
        self.m = [sp.m for sp in w.species]
        self.E, self.B = inputs.gem_fields(w)
        self.fluid = [inputs.band_fluid_block(w, self.NYF, side) for side in (0, 1)]

    def layers_outward(self, U5_rows, side):
        """[5][3 rows ascending y][nx] of the fluid block next to the band -> ghost layers counted outward."""
        return U5_rows[:, ::-1] if side == 0 else U5_rows


def test_band_between_two_live_fluid_blocks(gpu, fl, orc):
    """Config-4-shaped band (FLUID sides, 3 ghost rows) whose ghost rows are filled from two LIVE five-moment fluid
    blocks, which in turn take their ghost rows from the moments of the band's border rows at t, t + dt, t + dt/2
    (cycle items 3 and 4).  Three coupled steps on the GPU (everything through
    the C ABI) against the same loop composed from the oracles."""
    import torch
    w = inputs.band_workload(nx=8, ny_band=8, ny_domain=128, nv=16, g=3)
    ns, g, nx, nyf = 2, 3, w.nx, CoupledRun.NYF
    f0 = []
    for s in range(ns):
        f0.append(inputs.gem_f(w, s))
        w.species[s].f_inf = inputs.gem_f_inf(w, s)
    base = CoupledRun(w)
    osp = [orc.Species(sp.q, sp.m, sp.nv, sp.vmin, sp.vmax, sp.f_inf) for sp in w.species]
    # ---- oracle side
    fo = [f.copy() for f in f0]
    Uo = [base.fluid[side][0].copy() for side in (0, 1)]
    # ---- GPU side
    fg = [dev(f) for f in f0]
    ctx = gpu.context_for(w, fg)
    Ug = [dev(base.fluid[side][0]) for side in (0, 1)]
    blocks = [gpu.FluidBlock(nx, nyf, w.dx, w.dy, base.q, base.m,
                             gpu.FLUID_BC_WALL if side == 0 else gpu.FLUID_BC_COUPLED,
                             gpu.FLUID_BC_COUPLED if side == 0 else gpu.FLUID_BC_WALL) for side in (0, 1)]
    Ed, Bd = dev(base.E), dev(base.B)
    Ef = [(dev(base.fluid[side][1]), dev(base.fluid[side][2])) for side in (0, 1)]
    thetas = (0.0, 1.0, 0.5)                       # the stage times of the Runge-Kutta step
    for step in range(3):
        # (a) Vlasov ghost rows from the fluid rows next to the band (section 4.2)
        fluid_o = [[None, None] for _ in range(ns)]
        for side in (0, 1):
            rows = slice(2 + nyf - g, 2 + nyf) if side == 0 else slice(2, 2 + g)
            for s in range(ns):
                b5o = base.layers_outward(fl.to_boundary5(Uo[side][s][:, rows], base.m[s]), side)
                fluid_o[s][side] = np.ascontiguousarray(b5o)
                b5g = torch.empty((5, g, nx), dtype=torch.float64, device="cuda")
                gpu.vlasov_fluid_to_boundary(Ug[side][s][:, rows].contiguous(), base.m[s], b5g)
                lay = torch.flip(b5g, dims=[1]).contiguous() if side == 0 else b5g
                ctx.vlasov_set_boundary(s, side, inputs.BC_FLUID, lay)
        # (b) the Vlasov step, fields held fixed
        f_before = [f.copy() for f in fo]
        ctx.vlasov_fluid_boundary_mark()
        ctx.vlasov_step(w.dt, Ed, Bd, gpu.STAGE_ALL)
        assert ctx.check_code() == 0
        for s in range(ns):
            err, _ = orc.step(fo[s], osp[s], nx, w.ny, g, w.lx, w.ly, w.dt, base.E, base.B, fields_yee=w.fields_yee,
                              bc_lo=inputs.BC_FLUID, bc_hi=inputs.BC_FLUID, fluid_lo=fluid_o[s][0], fluid_hi=fluid_o[s][1],
                              want_moments=False)
            assert err == 0
        # (c) fluid ghost rows from the band's border rows at the stage times (section 4.1), then (d) the fluid steps
        for side in (0, 1):
            pick = slice(0, 2) if side == 0 else slice(1, 3)         # the two band rows next to the border, ascending y
            gh_o = np.zeros((3, ns, 5, 2, nx))
            gh_g = torch.zeros((3, ns, 5, 2, nx), dtype=torch.float64, device="cuda")
            mb = torch.empty((10, g, nx), dtype=torch.float64, device="cuda")
            for k, th in enumerate(thetas):
                for s in range(ns):
                    mo = orc.fluid_boundary(f_before[s], fo[s], osp[s], nx, w.ny, g, side, th)
                    gh_o[k, s] = fl.from_moments(mo[:, pick], base.m[s])
                    ctx.vlasov_fluid_boundary(s, side, th, mb)
                    gpu.vlasov_fluid_from_moments(mb[:, pick].contiguous(), base.m[s], gh_g[k, s])
            assert rel(gh_g.cpu().numpy(), gh_o) <= 1e-12
            Eo, Bo = base.fluid[side][1], base.fluid[side][2]
            if side == 0:
                fl.step(Uo[side], base.q, base.m, w.dt, w.dx, w.dy, Eo, Bo, fl.BC_WALL, fl.BC_COUPLED, None, gh_o)
                blocks[side].vlasov_fluid_step(w.dt, Ug[side], Ef[side][0], Ef[side][1], None, gh_g)
            else:
                fl.step(Uo[side], base.q, base.m, w.dt, w.dx, w.dy, Eo, Bo, fl.BC_COUPLED, fl.BC_WALL, gh_o, None)
                blocks[side].vlasov_fluid_step(w.dt, Ug[side], Ef[side][0], Ef[side][1], gh_g, None)
    for s in range(ns):
        assert rel(fg[s].cpu().numpy(), fo[s]) <= 1e-11, s
    for side in (0, 1):
        got = Ug[side].cpu().numpy()[:, :, 2:-2]
        assert rel(got, Uo[side][:, :, 2:-2]) <= 1e-11, side
        assert np.abs(got - base.fluid[side][0][:, :, 2:-2]).max() > 1e-9          # the fluid did move
    ctx.close()
