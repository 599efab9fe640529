"""Pins T14 (ghost fill: extrapolation + moment correction, section 4.2, eq. 63) and T15 (Yee/FDTD
Maxwell update, eqs. 9-10, section 3.3) for the oracle, plus the Yee <-> cell-centre interpolation of
PAPER.md:307 (reading R17) and the current of eq. 11."""
import numpy as np
import pytest


def _maxw_block(nv, vmin, vmax, n, V, T):
    g = []
    for d in range(3):
        dv = (vmax[d] - vmin[d]) / nv[d]
        c = vmin[d] + (np.arange(nv[d]) + 0.5) * dv
        g.append(np.exp(-(c - V[d]) ** 2 / (2 * T[d])) / np.sqrt(2 * np.pi * T[d]))
    return n * g[0][:, None, None] * g[1][None, :, None] * g[2][None, None, :]


def _fill_case(orc, nv, block, fluid_of_layer, m=1.0, g=2, nx=2, side=1, limiter=1):
    ny = 2
    sp = orc.Species(1.0, m, (nv,) * 3, (-6.0,) * 3, (6.0,) * 3, 1.0)
    f = np.zeros((ny + 2 * g, nx) + (nv,) * 3)
    f[g:g + ny] = block[None, None]
    if nx > 1:
        f[g:g + ny, 1] *= 1.5                                 # x-dependence: column 1 has 1.5 x the density
    fluid5 = np.zeros((5, g, nx))
    for l in range(g):
        fluid5[:, l, :] = np.asarray(fluid_of_layer(l))[:, None]
    err = orc.ghost_fill(f, sp, nx, ny, g, side, fluid5, limiter)
    return err, f, sp


def test_T14_identity_when_targets_equal_own_moments(orc):
    nv = 16
    blk = _maxw_block((nv,) * 3, (-6.0,) * 3, (6.0,) * 3, 1.3, (0.4, 0.4, 0.4), (1.1, 1.1, 1.1))
    sp = orc.Species(1.0, 2.0, (nv,) * 3, (-6.0,) * 3, (6.0,) * 3, 1.0)
    M = orc.moments_block(blk, sp)
    n, V = M[0], M[1:4] / M[0]
    T = M[4] / M[0] - V[0] ** 2
    for side in (0, 1):
        err, f, _ = _fill_case(orc, nv, blk, lambda l: (n, V[0], V[1], V[2], 2.0 * n * T), m=2.0, side=side)
        assert err == 0
        rows = (1, 0) if side == 0 else (4, 5)           # layer 0 is next to the interior
        for r in rows:
            assert np.abs(f[r, 0] - blk).max() <= 1e-13 * blk.max()
        # column 1 holds 1.5 x the density: the fill scales it back to the fluid density
        assert np.abs(f[rows[0], 1] - blk).max() <= 1e-13 * blk.max()
        other = (4, 5) if side == 0 else (0, 1)
        assert not f[list(other)].any()                  # the other side's ghost rows are untouched


def test_T14_density_exact_and_layers_counted_outward(orc):
    nv = 16
    blk = _maxw_block((nv,) * 3, (-6.0,) * 3, (6.0,) * 3, 1.0, (0.3, -0.1, 0.2), (1.2, 1.0, 0.8))
    sp = orc.Species(1.0, 1.0, (nv,) * 3, (-6.0,) * 3, (6.0,) * 3, 1.0)
    tgt = lambda l: (1.1 + l, -0.2, 0.1, 0.0, (1.1 + l) * 0.9)
    for side, rows in ((0, (2, 1, 0)), (1, (5, 6, 7))):
        err, f, _ = _fill_case(orc, nv, blk, tgt, g=3, side=side)
        assert err == 0
        for l, r in enumerate(rows):
            for ix in range(2):
                M = orc.moments_block(f[r, ix], sp)
                assert abs(M[0] - (1.1 + l)) <= 1e-14 * (1.1 + l), (side, l)


def test_T14_targets_hit_at_second_order_and_maxwellian_maps_to_maxwellian(orc):
    eV, eT, eL = [], [], []
    for nv in (16, 32, 64):
        blk = _maxw_block((nv,) * 3, (-6.0,) * 3, (6.0,) * 3, 1.0, (0.3, 0.3, 0.3), (1.2, 1.2, 1.2))
        err, f, sp = _fill_case(orc, nv, blk, lambda l: (1.1, -0.2, -0.2, -0.2, 1.1 * 0.9), g=1, nx=1)
        assert err == 0
        M = orc.moments_block(f[3, 0], sp)
        V = M[1:4] / M[0]
        T = M[4:7] / M[0] - V ** 2
        eV.append(np.abs(V + 0.2).max())
        eT.append(np.abs(T - 0.9).max())
        want = _maxw_block((nv,) * 3, (-6.0,) * 3, (6.0,) * 3, 1.1, (-0.2,) * 3, (0.9,) * 3)
        eL.append(np.abs(f[3, 0] - want).max() / want.max())
    assert eV[1] < 5e-4 and eV[2] < eV[1] / 3
    assert eT[0] < 4e-2 and eT[1] < 8e-3 and eT[2] < eT[1] / 3
    assert eL[1] < 2e-2 and eL[2] < eL[1] / 3


def test_T14_two_beams_keep_two_maxima(orc):
    nv = 32
    a = _maxw_block((nv,) * 3, (-6.0,) * 3, (6.0,) * 3, 0.5, (-1.8, 0.0, 0.0), (0.35, 1.0, 1.0))
    b = _maxw_block((nv,) * 3, (-6.0,) * 3, (6.0,) * 3, 0.5, (+1.8, 0.0, 0.0), (0.35, 1.0, 1.0))
    err, f, sp = _fill_case(orc, nv, a + b, lambda l: (2.0, 0.5, 0.0, 0.0, 2.0 * 2.5), g=1, nx=1)
    assert err == 0
    line = f[3, 0].sum(axis=(1, 2))
    nmax = sum(1 for k in range(1, nv - 1) if line[k] > line[k - 1] and line[k] >= line[k + 1])
    assert nmax == 2
    M = orc.moments_block(f[3, 0], sp)
    assert abs(M[0] - 2.0) < 1e-14 and abs(M[1] / M[0] - 0.5) < 2e-2


def test_T14_domain_errors(orc):
    nv = 8
    blk = _maxw_block((nv,) * 3, (-6.0,) * 3, (6.0,) * 3, 1.0, (0, 0, 0), (1, 1, 1))
    err, _, _ = _fill_case(orc, nv, blk, lambda l: (1.0, 0, 0, 0, -1.0))
    assert err == orc.ERR_DOMAIN
    err, _, _ = _fill_case(orc, nv, 0 * blk, lambda l: (1.0, 0, 0, 0, 1.0))
    assert err == orc.ERR_DOMAIN


# ---------------------------------------------------------------------------------------------------------
# Maxwell
# ---------------------------------------------------------------------------------------------------------
def _yee_cos_omega_dt(kx, ky, dx, dy, c, ddt):
    s2 = (c * ddt) ** 2 * (np.sin(kx * dx / 2) ** 2 / dx ** 2 + np.sin(ky * dy / 2) ** 2 / dy ** 2)
    return 1.0 - 2.0 * s2               # cos(w dt) from sin^2(w dt/2), the Yee dispersion relation


@pytest.mark.parametrize("mode", ["TM", "TE"])
def test_T15_vacuum_wave_obeys_yee_dispersion_periodic(orc, mode):
    nx, ny = 16, 12
    dx, dy, c, ddt = 0.5, 0.4, 3.0, 0.05
    kx, ky = 2 * np.pi * 2 / (nx * dx), 2 * np.pi * 1 / (ny * dy)
    xi, yj = np.arange(nx) * dx, np.arange(ny) * dy
    E = np.zeros((3, ny, nx))
    B = np.zeros((3, ny, nx))
    J = np.zeros((3, ny, nx))
    if mode == "TM":      # E_z at nodes (i, j)
        E[2] = np.cos(kx * xi[None, :] + ky * yj[:, None])
        obs = lambda: E[2]
        ph = kx * xi[None, :] + ky * yj[:, None]
    else:                 # E_x at (i+1/2, j); observe B_z at (i+1/2, j+1/2)
        E[0] = np.cos(kx * (xi[None, :] + dx / 2) + ky * yj[:, None])
        E[1] = 0.3 * np.sin(kx * xi[None, :] + ky * (yj[:, None] + dy / 2))
        obs = lambda: B[2]
        ph = kx * (xi[None, :] + dx / 2) + ky * (yj[:, None] + dy / 2)
    a, b = [], []
    for _ in range(40):
        orc.maxwell(E, B, J, dx, dy, c, 1.0, ddt, 1, 0)
        a.append((obs() * np.cos(ph)).sum())
        b.append((obs() * np.sin(ph)).sum())
    cw = _yee_cos_omega_dt(kx, ky, dx, dy, c, ddt)
    assert max(np.abs(a).max(), np.abs(b).max()) > 1.0
    for s in (np.array(a), np.array(b)):
        res = s[2:] + s[:-2] - 2 * cw * s[1:-1]
        assert np.abs(res).max() <= 1e-12 * max(np.abs(a).max(), np.abs(b).max())


def test_T15_pec_cavity_mode_and_wall_values(orc):
    nx, nyg = 8, 10
    dx, dy, c, ddt = 0.5, 0.3, 2.0, 0.04
    kx, ky = 2 * np.pi / (nx * dx), np.pi * 2 / (nyg * dy)      # walls at node rows j = 0 and j = nyg
    xi, yj = np.arange(nx) * dx, np.arange(nyg) * dy
    E = np.zeros((3, nyg, nx))
    B = np.zeros((3, nyg, nx))
    J = np.zeros((3, nyg, nx))
    mode = np.cos(kx * xi[None, :]) * np.sin(ky * yj[:, None])
    E[2] = mode
    s = []
    for _ in range(40):
        orc.maxwell(E, B, J, dx, dy, c, 1.0, ddt, 1, 1)
        s.append((E[2] * mode).sum())
        assert not E[0, 0].any() and not E[2, 0].any() and not B[1, 0].any()
    s = np.array(s)
    cw = _yee_cos_omega_dt(kx, ky, dx, dy, c, ddt)
    assert np.abs(s[2:] + s[:-2] - 2 * cw * s[1:-1]).max() <= 1e-12 * np.abs(s).max()


@pytest.mark.parametrize("wall", [0, 1])
def test_T15_div_B_stays_at_roundoff_and_nsub_composes(orc, wall):
    nx, ny = 9, 7
    dx, dy = 0.3, 0.45
    rng = np.random.default_rng(15)
    E = rng.normal(size=(3, ny, nx))
    B = rng.normal(size=(3, ny, nx))
    J = rng.normal(size=(3, ny, nx))
    if wall:
        E[0, 0] = E[2, 0] = 0.0
        B[1, 0] = 0.0

    def div(B):        # at cell centres (i+1/2, j+1/2) from Bx(i, j+1/2), By(i+1/2, j)
        by_up = np.roll(B[1], -1, axis=0)
        if wall:
            by_up[-1] = 0.0
        return (np.roll(B[0], -1, axis=1) - B[0]) / dx + (by_up - B[1]) / dy

    d0 = div(B)
    E1, B1 = E.copy(), B.copy()
    Bavg = orc.maxwell(E1, B1, J, dx, dy, 2.0, 1.3, 0.08, 4, wall, want_bavg=True)
    assert np.abs(div(B1) - d0).max() <= 1e-12
    E2, B2 = E.copy(), B.copy()
    for k in range(4):
        Bprev = B2.copy()
        orc.maxwell(E2, B2, J, dx, dy, 2.0, 1.3, 0.02, 1, wall)
    assert np.abs(E1 - E2).max() <= 1e-14 * np.abs(E1).max() and np.abs(B1 - B2).max() <= 1e-14 * np.abs(B1).max()
    assert np.allclose(Bavg, 0.5 * (Bprev + B2), rtol=0, atol=1e-15)     # B at the E time level


def test_T15_current_enters_ampere_with_minus_mu0_c2(orc):
    nx, ny = 4, 4
    E = np.zeros((3, ny, nx))
    B = np.zeros((3, ny, nx))
    J = np.zeros((3, ny, nx))
    J[1] = 2.0
    orc.maxwell(E, B, J, 1.0, 1.0, 3.0, 0.5, 0.1, 1, 0)
    assert np.allclose(E[1], -0.1 * 9.0 * 0.5 * 2.0, rtol=1e-15) and not E[0].any() and not B.any()


def test_R17_yee_positions_linear_fields_interpolate_exactly(orc):
    nx, nyg, dx, dy = 6, 5, 0.5, 0.25
    xi, yj = np.arange(nx) * dx, np.arange(nyg) * dy
    L = lambda x, y, k: (1.0 + k) + 0.0 * x + (0.7 - 0.1 * k) * y     # linear in y (x is periodic)
    X, Y = np.meshgrid(xi, yj, indexing="xy")
    E = np.stack([L(X + dx / 2, Y, 0), L(X, Y + dy / 2, 1), L(X, Y, 2)])
    B = np.stack([L(X, Y + dy / 2, 3), L(X + dx / 2, Y, 4), L(X + dx / 2, Y + dy / 2, 5)])
    for ix in (0, 3, nx - 1):
        for j in (0, 2, nyg - 2):
            Ec, Bc = orc.field_at_cell(E, B, 1, 0, ix, j)
            xc, yc = (ix + 0.5) * dx, (j + 0.5) * dy
            assert np.allclose(Ec, [L(xc, yc, k) for k in range(3)], rtol=1e-14)
            assert np.allclose(Bc, [L(xc, yc, k) for k in (3, 4, 5)], rtol=1e-14)
    # cell-centred input is passed through
    Ec, Bc = orc.field_at_cell(E, B, 0, 0, 2, 1)
    assert np.array_equal(Ec, E[:, 1, 2]) and np.array_equal(Bc, B[:, 1, 2])
    # x-dependence: E_y, E_z, B_x average over i and i+1 (periodic)
    E2 = np.zeros((3, nyg, nx)); E2[1, :, :] = np.arange(nx)[None, :]
    Ec, _ = orc.field_at_cell(E2, 0 * B, 1, 0, nx - 1, 1)
    assert Ec[1] == 0.5 * ((nx - 1) + 0)


@pytest.mark.parametrize("ix", [0, 2, 5])
def test_R17_yee_gather_at_the_pec_wall_rows(orc, ix):
    """wall = 1 (R17): the walls are the node rows j = 0 and j = nyg; E_x, E_z and B_y vanish there.
    The array holds rows 0 .. nyg-1, so the gather of the TOP row of cells reads "row nyg" as the wall value 0, and
    the gather of the BOTTOM row reads row 0 as stored.  Pin: fields that are linear in y and vanish on the top wall
    are interpolated exactly to the centres of the top row; with the periodic reading (wall = 0) the same call wraps
    to row 0.  Mutants of orc_field_at_cell that fail: "up" left at 1 with a wall (row 0 read as the wall), "up"
    applied to a half-row component (E_y, B_x), jp not wrapped."""
    nx, nyg, dx, dy = 6, 5, 0.5, 0.25
    top = nyg * dy
    xi, yj = np.arange(nx) * dx, np.arange(nyg) * dy
    X, Y = np.meshgrid(xi, yj, indexing="xy")
    W = lambda x, y, k: (1.0 + 0.5 * k) * (top - y)                 # vanishes on the top wall
    F = lambda x, y, k: 2.0 + k + 0.3 * y                           # half-row components: no wall value involved
    E = np.stack([W(X + dx / 2, Y, 0), F(X, Y + dy / 2, 1), W(X, Y, 2)])
    B = np.stack([F(X, Y + dy / 2, 3), W(X + dx / 2, Y, 4), F(X + dx / 2, Y + dy / 2, 5)])
    j = nyg - 1
    xc, yc = (ix + 0.5) * dx, (j + 0.5) * dy
    Ec, Bc = orc.field_at_cell(E, B, 1, 1, ix, j)
    assert np.allclose(Ec, [W(xc, yc, 0), F(xc, yc, 1), W(xc, yc, 2)], rtol=1e-14)
    assert np.allclose(Bc, [F(xc, yc, 3), W(xc, yc, 4), F(xc, yc, 5)], rtol=1e-14)
    # periodic reading of the same arrays: row nyg is row 0, where W = (1 + k/2) top
    Ep, Bp = orc.field_at_cell(E, B, 1, 0, ix, j)
    assert np.isclose(Ep[0], 0.5 * (W(xc, j * dy, 0) + W(xc, 0.0, 0)), rtol=1e-14) and Ep[0] > 2 * Ec[0]
    assert np.isclose(Ep[2], 0.5 * (W(xc, j * dy, 2) + W(xc, 0.0, 2)), rtol=1e-14)
    assert np.isclose(Bp[1], 0.5 * (W(xc, j * dy, 4) + W(xc, 0.0, 4)), rtol=1e-14)
    assert Ep[1] == Ec[1] and Bp[0] == Bc[0] and Bp[2] == Bc[2]
    # bottom row of cells: row 0 is read as stored (the Maxwell solver keeps the wall values at zero there), so
    # fields linear in y interpolate exactly whatever the wall flag
    for wall in (0, 1):
        E0, B0 = orc.field_at_cell(E, B, 1, wall, ix, 0)
        assert np.allclose(E0, [W(xc, dy / 2, 0), F(xc, dy / 2, 1), W(xc, dy / 2, 2)], rtol=1e-14)
        assert np.allclose(B0, [F(xc, dy / 2, 3), W(xc, dy / 2, 4), F(xc, dy / 2, 5)], rtol=1e-14)


def test_eq11_current_on_the_yee_grid_wraps_or_hits_the_wall_at_row_0(orc):
    """eq. 11 on the E positions of R17 at row 0: periodic (wall = 0) averages rows nyg-1 and 0; with a PEC wall the
    tangential components J_x, J_z of the wall row are not used (E_x = E_z = 0 there) and are stored as 0.  J_y sits
    at half rows and is not affected.  Mutants that fail: the wall flag ignored, wrap to the wrong row."""
    nx, nyg = 4, 5
    m1 = np.zeros((10, nyg, nx))
    row = np.arange(nyg, dtype=float)[:, None] + 0 * np.arange(nx)[None, :]
    m1[1] = 1.0 + row; m1[2] = 10.0 + row; m1[3] = 100.0 + 2 * row
    Jp = orc.current([m1], [2.0], fields_yee=1, wall=0)
    assert np.allclose(Jp[0, 0], 2.0 * 0.5 * ((1.0 + nyg - 1) + 1.0)) and np.allclose(Jp[2, 0], 2.0 * 0.5 * ((100.0 + 2 * (nyg - 1)) + 100.0))
    assert np.allclose(Jp[1, 0], 2.0 * 10.0)
    Jw = orc.current([m1], [2.0], fields_yee=1, wall=1)
    assert not Jw[0, 0].any() and not Jw[2, 0].any() and np.allclose(Jw[1, 0], 20.0)
    assert np.array_equal(Jw[:, 1:], Jp[:, 1:])


def test_eq11_current_from_moments(orc):
    nx, nyg = 5, 4
    rng = np.random.default_rng(16)
    me, mi = rng.normal(size=(10, nyg, nx)), rng.normal(size=(10, nyg, nx))
    J = orc.current([me, mi], [-1.0, 2.0], fields_yee=0)
    assert np.allclose(J, -1.0 * me[1:4] + 2.0 * mi[1:4], rtol=1e-15)
    # Yee: cell-centre currents that are linear in y land exactly on the E positions (interior rows)
    yc = (np.arange(nyg) + 0.5)[:, None] + 0 * np.arange(nx)[None, :]
    m1 = np.zeros((10, nyg, nx)); m1[1] = yc; m1[2] = 2 * yc; m1[3] = 3 * yc
    Jy = orc.current([m1], [1.0], fields_yee=1, wall=1)
    assert np.allclose(Jy[0, 1:], yc[1:] - 0.5) and np.allclose(Jy[1], 2 * yc) and np.allclose(Jy[2, 1:], 3 * (yc[1:] - 0.5))
    assert not Jy[0, 0].any() and not Jy[2, 0].any()


@pytest.mark.parametrize("side", [0, 1])
def test_T17_fluid_boundary_rows_moments_and_time_interpolation(orc, side):
    """Section 4.1: the fluid code's boundary data are the moments (eqs. 2-4) of the kinetic rows next
    to the border, linearly interpolated in time.  Pinned against brute-force sums written here (not the oracle's
    moment routine) on data where every row, column and time level is different, so a wrong row, side, moment index
    or weight fails; and against the closed form for drifting Maxwellians whose density changes in time."""
    nv, g, nx, ny = (8, 6, 10), 2, 3, 5
    vmin, vmax = (-5.0, -4.0, -6.0), (5.0, 4.0, 6.0)
    sp = orc.Species(-1.0, 1.0, nv, vmin, vmax, 1.0)
    rng = np.random.default_rng(5)
    f_t = rng.random((ny + 2 * g, nx) + nv)
    f_t1 = rng.random((ny + 2 * g, nx) + nv)
    dv = [(vmax[d] - vmin[d]) / nv[d] for d in range(3)]
    c = [vmin[d] + (np.arange(nv[d]) + 0.5) * dv[d] for d in range(3)]
    V = np.meshgrid(*c, indexing="ij")
    w = dv[0] * dv[1] * dv[2]
    rows = range(g, 2 * g) if side == 0 else range(ny, ny + g)       # ghost-inclusive indices of the g interior rows
    pairs = [(0, 0), (1, 1), (2, 2), (0, 1), (0, 2), (1, 2)]         # M2 order xx yy zz xy xz yz (vlasov.h)
    for theta in (0.0, 0.5, 0.3, 1.0):
        got = orc.fluid_boundary(f_t, f_t1, sp, nx, ny, g, side, theta)
        assert got.shape == (10, g, nx)
        for l, j in enumerate(rows):
            for i in range(nx):
                fb = (1.0 - theta) * f_t[j, i] + theta * f_t1[j, i]      # moments are linear in f
                want = [fb.sum() * w] + [(fb * V[d]).sum() * w for d in range(3)] + \
                       [(fb * V[a] * V[b]).sum() * w for a, b in pairs]
                np.testing.assert_allclose(got[:, l, i], want, rtol=1e-12, atol=1e-10)   # odd moments cancel: sums of terms of size 1e3
    # closed form: Maxwellians, density 1 at t and 3 at t + dt, drift (0.3, -0.2, 0.1), T = 0.5: M0 = 1 + 2 theta,
    # M1 = M0 V, trace M2 = M0 (3 T + V^2) up to the midpoint-rule error (spectrally small for a resolved Gaussian)
    nv2 = (24, 24, 24)
    sp2 = orc.Species(1.0, 1.0, nv2, (-6.0,) * 3, (6.0,) * 3, 1.0)
    Vd, T = (0.3, -0.2, 0.1), (0.5, 0.5, 0.5)
    blk = _maxw_block(nv2, (-6.0,) * 3, (6.0,) * 3, 1.0, Vd, T)
    a = np.zeros((ny + 2 * g, nx) + nv2); b = np.zeros_like(a)
    a[g:g + ny] = blk; b[g:g + ny] = 3.0 * blk
    got = orc.fluid_boundary(a, b, sp2, nx, ny, g, side, 0.25)
    np.testing.assert_allclose(got[0], 1.5, rtol=1e-9)
    for d in range(3):
        np.testing.assert_allclose(got[1 + d], 1.5 * Vd[d], rtol=1e-8)
    np.testing.assert_allclose(got[4] + got[5] + got[6], 1.5 * (1.5 + sum(v * v for v in Vd)), rtol=1e-8)
