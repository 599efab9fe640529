"""GPU parity of the 3D3V path: third spatial sweep, 3D Yee gather / current / FDTD,
through the same C ABI (cfg.nz > 1), element by element against the oracle's step3d / maxwell3d / cycle3d (pinned by
tests/test_oracle_3d.py)."""
import numpy as np
import pytest

from paper_1406_5445_b200 import inputs

pytestmark = pytest.mark.gpu
TOL1 = 1e-12


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1406_5445_b200 import binding
    binding.lib()
    return binding


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def rel(a, b):
    return np.linalg.norm(np.ravel(a) - np.ravel(b)) / np.linalg.norm(np.ravel(b))


def workload3d(nx, ny, nz, nv, bc, nspecies=1, fields_yee=1, vmax=(4.0, 3.0, 2.5)):
    sp = []
    for s in range(nspecies):
        sp.append(inputs.SpeciesSpec(f"s{s}", q=-1.0 if s == 0 else 1.0, m=1.0 if s == 0 else 4.0, nv=tuple(nv),
                                     vmin=tuple(-x for x in vmax), vmax=tuple(vmax), f_inf=1.0))
    return inputs.Workload("random3d", nx=nx, ny=ny, nghost_y=0, lx=1.7, ly=0.9, x0=0.0, y0=0.0, bc_y_lo=bc, bc_y_hi=bc,
                           dt=0.05, steps=1, species=sp, c=3.0, mu0=1.0, nsub=1, fields_yee=fields_yee, seed=3, nz=nz, lz=1.1)


def rough_f(rng, w, s):
    sp = w.species[s]
    shape = (w.nz, w.ny, w.nx) + sp.nv
    c = [sp.centres(d) for d in range(3)]
    M = np.exp(-0.5 * ((c[0][:, None, None] / 1.3) ** 2 + (c[1][None, :, None] / 1.1) ** 2 + (c[2][None, None, :] / 0.8) ** 2))
    f = 0.9 * M[None, None, None] * (0.3 + 0.7 * rng.random(shape))
    f[rng.random(shape) < 0.05] = 0.0
    f[rng.random(shape) < 0.02] = 1.0
    return np.ascontiguousarray(f)


def osp(orc, s):
    return orc.Species(s.q, s.m, s.nv, s.vmin, s.vmax, s.f_inf)


@pytest.mark.parametrize("order", [0, 1])
@pytest.mark.parametrize("bc", [inputs.BC_PERIODIC, inputs.BC_REFLECT])
@pytest.mark.parametrize("nx,ny,nz,nv,dt", [(9, 6, 5, (8, 8, 8), 0.07), (16, 5, 3, (16, 16, 16), 0.02), (13, 4, 4, (6, 8, 10), 0.23),
                                            (7, 4, 3, (4, 6, 5), 0.07), (6, 4, 8, (8, 8, 8), 0.02), (5, 3, 16, (4, 4, 8), 0.02),
                                            (5, 3, 4, (4, 6, 8), 0.02)])
def test_full_3d3v_step(gpu, orc, order, bc, nx, ny, nz, nv, dt):
    """x/2 y/2 z/2 - v - z/2 y/2 x/2 (and VXV) for two species with Yee fields.  (16,5,3,16^3): shifts below one cell, the
    fused x,y stage per z slab and the TMA velocity kernels (fused moments under VXV); dt = 0.23: multi-cell shifts in all
    three directions with wrap-around, the general kernels; (4,6,5): an odd nv[2], one cell per thread; nz = 8, 16, 4 with dt = 0.02: the z sweep
    that holds a whole periodic line in registers."""
    import torch
    rng = np.random.default_rng(51)
    w = workload3d(nx, ny, nz, nv, bc, nspecies=2)
    f0 = [rough_f(rng, w, s) for s in range(2)]
    E = rng.standard_normal((3, nz, ny, nx))
    B = 2.0 * rng.standard_normal((3, nz, ny, nx))
    fg = [dev(f) for f in f0]
    ctx = gpu.context_for(w, fg, order=order)
    ctx.vlasov_timing_enable(True)
    ctx.vlasov_step(dt, dev(E), dev(B), gpu.STAGE_ALL)
    assert ctx.check_code() == 0
    kinds = ctx.vlasov_timing_read()
    assert kinds["sweep_z"][1] == (4 if order == 0 else 2)
    if nv[0] == 16:
        assert kinds["sweep_xy"][1] + kinds["sweep_yx"][1] == (4 if order == 0 else 2) and kinds["sweep_y"][1] == 0
    mom = torch.empty((10, nz, ny, nx), dtype=torch.float64, device="cuda")
    for s in range(2):
        fo = f0[s].copy()
        err, mo = orc.step3d(fo, osp(orc, w.species[s]), nx, ny, nz, w.lx, w.ly, w.lz, dt, E, B, fields_yee=1, bc_lo=bc, bc_hi=bc,
                             order=order)
        assert err == 0
        got = fg[s].cpu().numpy()
        assert rel(got, fo) <= TOL1, s
        assert np.abs(got - fo).max() <= 2e-13
        ctx.vlasov_moments(s, mom)
        assert rel(mom.cpu().numpy(), mo) <= TOL1
        m0 = f0[s].sum()
        assert abs(got.sum() - m0) / m0 <= 1e-13
        assert np.abs(got - f0[s]).max() > 0.05
    ctx.close()


def test_3d_free_streaming_integer_shifts_exact_on_gpu(gpu):
    """T10 in 3D on the GPU (no oracle involved): integer CFL shifts in x, y, z translate f exactly."""
    import torch
    nx, ny, nz, nv = 8, 6, 5, (2, 2, 2)
    sp = inputs.SpeciesSpec("e", -1.0, 1.0, nv, (-2.0, -1.0, -4.0), (2.0, 1.0, 4.0), f_inf=1.0)
    w = inputs.Workload("fs3", nx=nx, ny=ny, nghost_y=0, lx=8.0, ly=3.0, x0=0, y0=0, bc_y_lo=0, bc_y_hi=0, dt=2.0, steps=1,
                        species=[sp], fields_yee=0, nz=nz, lz=5.0)
    rng = np.random.default_rng(6)
    f0 = rng.random((nz, ny, nx) + nv)
    fg = [dev(f0)]
    ctx = gpu.context_for(w, fg)
    Z = torch.zeros((3, nz, ny, nx), dtype=torch.float64, device="cuda")
    ctx.vlasov_step(2.0, Z, Z, 31)
    ctx.vlasov_check()
    f = fg[0].cpu().numpy()
    c = [sp.centres(d) for d in range(3)]
    for a in range(2):
        for b in range(2):
            for cc in range(2):
                sx, sy, sz = int(round(c[0][a] * 2.0)), int(round(c[1][b] * 2.0 / 0.5)), int(round(c[2][cc] * 2.0))
                want = np.roll(f0[:, :, :, a, b, cc], (sz, sy, sx), axis=(0, 1, 2))
                assert np.abs(f[:, :, :, a, b, cc] - want).max() <= 1e-14
    ctx.close()


@pytest.mark.parametrize("bc,yee", [(inputs.BC_PERIODIC, 1), (inputs.BC_REFLECT, 1), (inputs.BC_REFLECT, 0)])
def test_3d_maxwell_and_current(gpu, orc, bc, yee):
    import torch
    rng = np.random.default_rng(52)
    w = workload3d(7, 6, 5, (4, 4, 4), bc, nspecies=2, fields_yee=yee)
    f0 = [rough_f(rng, w, s) for s in range(2)]
    fg = [dev(f) for f in f0]
    ctx = gpu.context_for(w, fg)
    wall = 0 if bc == inputs.BC_PERIODIC else 1
    J = torch.empty((3, w.nz, w.ny, w.nx), dtype=torch.float64, device="cuda")
    ctx.vlasov_current(J)
    moms = [orc.moments3d(f0[s], osp(orc, w.species[s]), w.nx, w.ny, w.nz) for s in range(2)]
    Jo = orc.current3d(moms, [s.q for s in w.species], fields_yee=yee, wall=wall)
    assert rel(J.cpu().numpy(), Jo) <= TOL1
    E = rng.standard_normal((3, w.nz, w.ny, w.nx)); B = rng.standard_normal((3, w.nz, w.ny, w.nx))
    if wall:
        E[0, :, 0] = 0; E[2, :, 0] = 0; B[1, :, 0] = 0
    Eo, Bo = E.copy(), B.copy()
    Bao = orc.maxwell3d(Eo, Bo, Jo, w.dx, w.dy, w.lz / w.nz, w.c, w.mu0, 0.01, 4, wall, want_bavg=True)
    Ed, Bd, Ba = dev(E), dev(B), torch.empty((3, w.nz, w.ny, w.nx), dtype=torch.float64, device="cuda")
    ctx.vlasov_maxwell(0.01, 4, Ed, Bd, dev(Jo), Ba)
    ctx.vlasov_check()
    assert rel(Ed.cpu().numpy(), Eo) <= 1e-14 and rel(Bd.cpu().numpy(), Bo) <= 1e-14 and rel(Ba.cpu().numpy(), Bao) <= 1e-14
    ctx.close()


def test_3d_cycles_against_the_oracle(gpu, orc):
    """Ten cycles of section 4.3 on a 3D grid through vlasov_cycle (currents -> Maxwell -> 3D3V step -> currents ->
    Maxwell) against oracle.cycle3d."""
    import torch
    rng = np.random.default_rng(53)
    w = workload3d(8, 6, 4, (8, 8, 8), inputs.BC_REFLECT, nspecies=2)
    f0 = [0.2 * rough_f(rng, w, s) + 0.05 for s in range(2)]
    sps = [osp(orc, s) for s in w.species]
    E = 0.1 * rng.standard_normal((3, w.nz, w.ny, w.nx)); B = 0.5 * rng.standard_normal((3, w.nz, w.ny, w.nx))
    E[0, :, 0] = 0; E[2, :, 0] = 0; B[1, :, 0] = 0
    fo = [f.copy() for f in f0]
    mom = [orc.moments3d(f, sp, w.nx, w.ny, w.nz) for f, sp in zip(fo, sps)]
    Eo, Bo = E.copy(), B.copy()
    fg = [dev(f) for f in f0]
    ctx = gpu.context_for(w, fg)
    Ed, Bd = dev(E), dev(B)
    dt, nsub = 0.02, 2
    for _ in range(10):
        ctx.vlasov_cycle(dt, nsub, Ed, Bd)
        mom = orc.cycle3d(fo, sps, mom, Eo, Bo, w.nx, w.ny, w.nz, w.lx, w.ly, w.lz, dt, nsub, w.c, w.mu0, fields_yee=1,
                          bc_lo=w.bc_y_lo, bc_hi=w.bc_y_hi)
    assert ctx.check_code() == 0
    assert rel(Ed.cpu().numpy(), Eo) <= 1e-11 and rel(Bd.cpu().numpy(), Bo) <= 1e-11
    for s in range(2):
        assert rel(fg[s].cpu().numpy(), fo[s]) <= 1e-11
    ctx.close()


def test_3d_refusals(gpu):
    import torch
    w = workload3d(4, 4, 3, (4, 4, 4), inputs.BC_PERIODIC)
    w.nghost_y = 1
    f = [torch.zeros((3, 6, 4, 4, 4, 4), dtype=torch.float64, device="cuda")]
    with pytest.raises(gpu.VlasovError) as e:
        gpu.context_for(w, f)                       # ghost rows (FLUID sides) are a 2D3V feature
    assert e.value.code == gpu.EINVAL


def test_full_size_gem3d_sampled_window(gpu, orc):
    """The 3D3V bench workload at full size (32x32x8 spatial x 32^3 velocity x 2 species, 4.3 GB of f), as
    `bench.py --workload gem3d` runs it: one complete step on the GPU, then the oracle on a 14x14 window in x, y (all 8
    z slabs: z is periodic) of the same inputs; the inner 4x4 columns must agree (domain of dependence of a step: 4
    cells in x and y).  Mass and positivity at full size."""
    import torch
    free, _ = torch.cuda.mem_get_info()
    if free < 9 * 2**30:
        pytest.skip("needs 9 GB of device memory")
    w = inputs.gem3d_workload(steps=1)
    ix0, iy0, nw, margin = 9, 9, 14, 5
    E, B = inputs.gem3d_fields(w)
    fg, f0win, mass0 = [], [], []
    for s, sp in enumerate(w.species):
        sp.f_inf = inputs.gem_f_inf(w, s)
        f = torch.empty((w.nz, w.ny, w.nx) + tuple(sp.nv), dtype=torch.float64, device="cuda")
        win = np.empty((w.nz, nw, nw) + tuple(sp.nv))
        for k in range(w.nz):
            slab = inputs.gem3d_f(w, s, k)
            f[k].copy_(torch.from_numpy(slab))
            win[k] = slab[iy0:iy0 + nw, ix0:ix0 + nw]
        fg.append(f)
        f0win.append(win)
        mass0.append(float(f.sum().item()))
    ctx = gpu.context_for(w, fg)
    ctx.vlasov_timing_enable(True)
    ctx.vlasov_step(w.dt, dev(E), dev(B), gpu.STAGE_ALL)
    assert ctx.check_code() == 0
    kinds = ctx.vlasov_timing_read()
    assert kinds["sweep_xy"][1] == 2 and kinds["sweep_yx"][1] == 2 and kinds["sweep_z"][1] == 4 and kinds["vsweep_yz"][1] == 2
    Ew = np.ascontiguousarray(E[:, :, iy0:iy0 + nw, ix0:ix0 + nw])
    Bw = np.ascontiguousarray(B[:, :, iy0:iy0 + nw, ix0:ix0 + nw])
    inner = slice(margin, nw - margin)
    for s, sp in enumerate(w.species):
        drift = abs(float(fg[s].sum().item()) - mass0[s]) / mass0[s]
        assert drift <= 1e-13, (s, drift)
        assert float(fg[s].min().item()) >= 0.0
        fo = f0win[s].copy()
        err, _ = orc.step3d(fo, osp(orc, sp), nw, nw, w.nz, nw * w.dx, nw * w.dy, w.lz, w.dt, Ew, Bw, fields_yee=w.fields_yee,
                            bc_lo=inputs.BC_PERIODIC, bc_hi=inputs.BC_PERIODIC, order=0, want_moments=False)
        assert err == 0
        got = fg[s][:, iy0:iy0 + nw, ix0:ix0 + nw].cpu().numpy()
        a, b = got[:, inner, inner], fo[:, inner, inner]
        assert rel(a, b) <= TOL1, s
        assert np.abs(a - b).max() <= 1e-13 * sp.f_inf
        assert rel(got[:, 0], fo[:, 0]) > 1e-9          # the window's own edge does differ: not vacuous
    ctx.close()
