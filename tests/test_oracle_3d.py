"""Pins for the oracle's 3D3V extension ("a generalisation to the full 3-dimensional
case is straightforward"): third spatial sweep, 3D Yee grid (reading R24 = the standard extension of R17).

  D1  nz = 1 reduces every 3D function to its pinned 2D counterpart BIT FOR BIT (step in both orders, gather, current,
      Maxwell with sub-steps and Bavg): ties the 3D code to everything the 2D pins fix;
  D2  the z sweep is the x sweep on data with (x, vx) and (z, vz) exchanged;
  D3  free streaming with integer CFL shifts in x, y and z translates f exactly (T10 in 3D), both orders;
  D4  a vacuum plane wave with all three wave-vector components obeys the 3D Yee dispersion relation; div B stays
      at round-off;
  D5  positions of the six field components: a unit impulse in one component reaches exactly the cell centres around
      its Yee position, with the weights of linear interpolation; likewise the current;
  D6  Langmuir oscillation along z through cycle3d is the velocity-Verlet recurrence (C1 with the drift along z).
Mutants that fail: a z derivative with the wrong sign or missing in one curl component (D4), z wrap missing (D2-D4),
a component gathered from the wrong neighbours (D5), sweep order not a palindrome or the z sweep with dt instead of
dt/2 (D3), J_z not interpolated in x, y (D5, D6).
"""
import numpy as np
import pytest


def _sp(orc, nv, vmin, vmax, q=-1.0, m=1.0, finf=1.0):
    return orc.Species(q, m, nv, vmin, vmax, finf)


@pytest.mark.parametrize("order", [0, 1])
@pytest.mark.parametrize("bc", [0, 1])
def test_D1_nz1_step_is_the_2d_step_bit_for_bit(orc, order, bc):
    rng = np.random.default_rng(3)
    nx, ny, nv = 5, 4, (4, 6, 4)
    sp = _sp(orc, nv, (-2.0, -3.0, -2.0), (2.0, 3.0, 2.0), m=0.5)
    f0 = rng.random((ny, nx) + nv)
    E = rng.standard_normal((3, ny, nx))
    B = rng.standard_normal((3, ny, nx))
    f2 = f0.copy()
    err, m2 = orc.step(f2, sp, nx, ny, 0, 1.3, 0.9, 0.07, E, B, fields_yee=1, bc_lo=bc, bc_hi=bc, order=order)
    f3 = f0.copy()[None].copy()
    err3, m3 = orc.step3d(f3, sp, nx, ny, 1, 1.3, 0.9, 0.4, 0.07, E[:, None].copy(), B[:, None].copy(), fields_yee=1,
                          bc_lo=bc, bc_hi=bc, order=order)
    assert err == 0 and err3 == 0
    assert np.array_equal(f3[0], f2) and np.array_equal(m3[:, 0], m2)
    assert not np.array_equal(f2, f0)


@pytest.mark.parametrize("wall", [0, 1])
def test_D1_nz1_fields_current_and_maxwell_are_the_2d_ones(orc, wall):
    rng = np.random.default_rng(4)
    nx, ny = 6, 5
    E = rng.standard_normal((3, ny, nx)); B = rng.standard_normal((3, ny, nx)); J = rng.standard_normal((3, ny, nx))
    if wall:
        E[0, 0] = E[2, 0] = 0.0; B[1, 0] = 0.0
    for yee in (0, 1):
        for ix, j in ((0, 0), (3, 2), (nx - 1, ny - 1)):
            a = orc.field_at_cell(E, B, yee, wall, ix, j)
            b = orc.field_at_cell3d(E[:, None], B[:, None], yee, wall, ix, j, 0)
            assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])
    moms = [rng.standard_normal((10, ny, nx)) for _ in range(2)]
    for yee in (0, 1):
        J2 = orc.current(moms, [-1.0, 2.0], yee, wall)
        J3 = orc.current3d([m[:, None] for m in moms], [-1.0, 2.0], yee, wall)
        assert np.array_equal(J3[:, 0], J2)
    E2, B2 = E.copy(), B.copy()
    Ba2 = orc.maxwell(E2, B2, J, 0.3, 0.45, 2.0, 1.3, 0.08, 4, wall, want_bavg=True)
    E3, B3 = E[:, None].copy(), B[:, None].copy()
    Ba3 = orc.maxwell3d(E3, B3, J[:, None].copy(), 0.3, 0.45, 0.7, 2.0, 1.3, 0.08, 4, wall, want_bavg=True)
    assert np.array_equal(E3[:, 0], E2) and np.array_equal(B3[:, 0], B2) and np.array_equal(Ba3[:, 0], Ba2)


def test_D2_z_sweep_is_the_x_sweep_on_exchanged_data(orc):
    n, ny, nv = 6, 3, (4, 2, 4)
    sp = _sp(orc, nv, (-2.0, -1.0, -2.0), (2.0, 1.0, 2.0))
    rng = np.random.default_rng(5)
    f = rng.random((n, ny, n) + nv)                                   # [z, y, x, vx, vy, vz]
    ft = np.ascontiguousarray(f.transpose(2, 1, 0, 5, 4, 3))           # exchange (x, vx) and (z, vz)
    fz = f.copy()
    orc.sweep_z(fz, sp, n, ny, n, 0.5, 0.83)                           # shifts up to 1.5 * 0.83 / 0.5 = 2.5 cells
    for k in range(n):                                                 # the 2D x sweep acts slab by slab
        slab = np.ascontiguousarray(ft[k])
        orc.sweep_x(slab, sp, n, ny, 0, 0.5, 0.83)
        ft[k] = slab
    assert np.array_equal(fz, ft.transpose(2, 1, 0, 5, 4, 3))
    assert not np.array_equal(fz, f)


@pytest.mark.parametrize("order", [0, 1])
def test_D3_free_streaming_translates_exactly_in_three_directions(orc, order):
    nx, ny, nz, nv = 8, 6, 5, (2, 2, 2)
    sp = _sp(orc, nv, (-2.0, -1.0, -4.0), (2.0, 1.0, 4.0))             # centres -1, 1 | -0.5, 0.5 | -2, 2
    lx, ly, lz, dt = 8.0, 3.0, 5.0, 2.0                                # dx = 1, dy = 0.5, dz = 1: total shifts +-2, +-2, +-4
    rng = np.random.default_rng(6)
    f0 = rng.random((nz, ny, nx) + nv)
    f = f0.copy()
    Z = np.zeros((3, nz, ny, nx))
    err, _ = orc.step3d(f, sp, nx, ny, nz, lx, ly, lz, dt, Z, Z, order=order)
    assert err == 0
    c = [sp.vmin[d] + (np.arange(2) + 0.5) * (sp.vmax[d] - sp.vmin[d]) / 2 for d in range(3)]
    for a in range(2):
        for b in range(2):
            for cc in range(2):
                sx, sy, sz = (int(round(c[0][a] * dt / 1.0)), int(round(c[1][b] * dt / 0.5)), int(round(c[2][cc] * dt / 1.0)))
                assert sx and sy and sz
                want = np.roll(f0[:, :, :, a, b, cc], (sz, sy, sx), axis=(0, 1, 2))
                assert np.abs(f[:, :, :, a, b, cc] - want).max() <= 1e-14, (a, b, cc)


def test_D4_vacuum_wave_obeys_the_3d_yee_dispersion_and_div_b_stays_zero(orc):
    nx, ny, nz = 8, 6, 5
    dx, dy, dz, c, ddt = 0.5, 0.4, 0.6, 3.0, 0.04
    k = np.array([2 * np.pi * 1 / (nx * dx), 2 * np.pi * 2 / (ny * dy), 2 * np.pi * 1 / (nz * dz)])
    h = np.array([dx, dy, dz])
    K = np.sin(k * h / 2) / h
    # amplitudes with zero DISCRETE divergence: E0 . K = 0
    E0 = np.array([1.0, -0.4, 0.0]); E0[2] = -(E0[0] * K[0] + E0[1] * K[1]) / K[2]
    z, y, x = np.meshgrid(np.arange(nz) * dz, np.arange(ny) * dy, np.arange(nx) * dx, indexing="ij")
    ph = lambda ox, oy, oz: k[0] * (x + ox) + k[1] * (y + oy) + k[2] * (z + oz)
    E = np.stack([E0[0] * np.cos(ph(dx / 2, 0, 0)), E0[1] * np.cos(ph(0, dy / 2, 0)), E0[2] * np.cos(ph(0, 0, dz / 2))])
    B = np.zeros_like(E)
    J = np.zeros_like(E)
    series = {d: [] for d in range(3)}
    modes = [np.cos(ph(dx / 2, 0, 0)), np.cos(ph(0, dy / 2, 0)), np.cos(ph(0, 0, dz / 2))]

    def divb():
        return ((np.roll(B[0], -1, 2) - B[0]) / dx + (np.roll(B[1], -1, 1) - B[1]) / dy + (np.roll(B[2], -1, 0) - B[2]) / dz)

    for _ in range(30):
        orc.maxwell3d(E, B, J, dx, dy, dz, c, 1.0, ddt, 1, 0)
        for d in range(3):
            series[d].append((E[d] * modes[d]).sum())
        assert np.abs(divb()).max() <= 1e-12
    cw = 1.0 - 2.0 * (c * ddt) ** 2 * (K ** 2).sum()
    assert abs(cw) < 1.0
    for d in range(3):
        s = np.array(series[d])
        assert np.abs(s).max() > 1.0
        assert np.abs(s[2:] + s[:-2] - 2 * cw * s[1:-1]).max() <= 1e-11 * np.abs(s).max(), d
    assert np.abs(B).max() > 0.05                      # all three B components take part
    assert min(np.abs(B[d]).max() for d in range(3)) > 1e-3


def test_D5_yee_positions_by_unit_impulses(orc):
    """Reading R24: a unit value of one component at array index (k0, j0, i0) sits at its Yee position; the centres of
    the cells around that position see it with the weights of linear interpolation, every other cell sees nothing."""
    nx, ny, nz = 5, 5, 5
    k0, j0, i0 = 2, 2, 2
    # component -> set of (dk, dj, di) cell offsets (cell = index + offset) that see it, weight
    expect = {
        ("E", 0): ([(dk, dj, 0) for dk in (-1, 0) for dj in (-1, 0)], 0.25),      # Ex(i+1/2, j, k): averaged over y and z
        ("E", 1): ([(dk, 0, di) for dk in (-1, 0) for di in (-1, 0)], 0.25),      # Ey(i, j+1/2, k)
        ("E", 2): ([(0, dj, di) for dj in (-1, 0) for di in (-1, 0)], 0.25),      # Ez(i, j, k+1/2)
        ("B", 0): ([(0, 0, di) for di in (-1, 0)], 0.5),                          # Bx(i, j+1/2, k+1/2)
        ("B", 1): ([(0, dj, 0) for dj in (-1, 0)], 0.5),                          # By(i+1/2, j, k+1/2)
        ("B", 2): ([(dk, 0, 0) for dk in (-1, 0)], 0.5),                          # Bz(i+1/2, j+1/2, k)
    }
    for (which, d), (cells, wgt) in expect.items():
        E = np.zeros((3, nz, ny, nx)); B = np.zeros((3, nz, ny, nx))
        (E if which == "E" else B)[d, k0, j0, i0] = 1.0
        seen = {}
        for kk in range(nz):
            for jj in range(ny):
                for ii in range(nx):
                    Ec, Bc = orc.field_at_cell3d(E, B, 1, 0, ii, jj, kk)
                    v = (Ec if which == "E" else Bc)[d]
                    other = np.abs(np.concatenate([Ec, Bc])).sum() - abs(v)
                    assert other == 0.0
                    if v != 0.0:
                        seen[(kk - k0, jj - j0, ii - i0)] = v
        assert set(seen) == set(cells), (which, d, seen)
        assert all(v == wgt for v in seen.values())
    # the current goes the other way: a unit cell-centre current in cell (k0, j0, i0) reaches the E positions around it
    for d, offs in ((0, [(dk, dj, 0) for dk in (0, 1) for dj in (0, 1)]), (1, [(dk, 0, di) for dk in (0, 1) for di in (0, 1)]),
                    (2, [(0, dj, di) for dj in (0, 1) for di in (0, 1)])):
        m = np.zeros((10, nz, ny, nx)); m[1 + d, k0, j0, i0] = 1.0
        J = orc.current3d([m], [2.0], fields_yee=1, wall=0)
        nzc = {tuple(int(a) - b for a, b in zip(idx, (k0, j0, i0))): J[d][tuple(idx)] for idx in np.argwhere(J[d] != 0)}
        assert set(nzc) == set(offs) and all(v == 0.5 for v in nzc.values()), (d, nzc)
        assert not J[[e for e in range(3) if e != d]].any()


@pytest.mark.parametrize("order", [0, 1])
def test_D6_langmuir_oscillation_along_z_is_the_verlet_recurrence(orc, order):
    nx, ny, nz, nv = 3, 2, 4, (4, 4, 48)
    vmin, vmax = (-8.0,) * 3, (8.0,) * 3
    q, m, c, mu0, dt, nsub = -1.0, 1.0, 2.0, 0.5, 0.1, 2
    sp = orc.Species(q, m, nv, vmin, vmax, 1.0)
    g = []
    for d, u in enumerate((0.0, 0.0, 0.3)):
        cen = vmin[d] + (np.arange(nv[d]) + 0.5) * 16.0 / nv[d]
        g.append(np.exp(-0.5 * (cen - u) ** 2) / np.sqrt(2 * np.pi))
    blk = g[0][:, None, None] * g[1][None, :, None] * g[2][None, None, :]
    f = np.ascontiguousarray(np.broadcast_to(blk, (nz, ny, nx) + nv)).copy()
    E = np.zeros((3, nz, ny, nx)); B = np.zeros((3, nz, ny, nx))
    mom = [orc.moments3d(f, sp, nx, ny, nz)]
    n0 = mom[0][0, 0, 0, 0]
    w2 = c * c * mu0 * q * q * n0 / m
    u, Ez = [mom[0][3, 0, 0, 0] / n0], [0.0]
    for _ in range(30):
        mom = orc.cycle3d([f], [sp], mom, E, B, nx, ny, nz, 1.0, 1.0, 1.0, dt, nsub, c, mu0, fields_yee=1, order=order, limiter=0)
        assert np.ptp(mom[0][3]) <= 1e-13 and np.ptp(E[2]) <= 1e-13 and np.abs(E[:2]).max() <= 1e-13
        u.append(mom[0][3, 0, 0, 0] / n0); Ez.append(E[2, 0, 0, 0])
    u, Ez = np.array(u), np.array(Ez)
    cw = 1.0 - 0.5 * w2 * dt * dt
    assert np.abs(Ez).max() > 0.1
    assert np.abs(u[2:] + u[:-2] - 2 * cw * u[1:-1]).max() <= 1e-12
    assert np.abs(Ez[1:] - Ez[:-1] + 0.5 * dt * c * c * mu0 * q * n0 * (u[1:] + u[:-1])).max() <= 1e-12
