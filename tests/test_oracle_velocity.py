"""Pins T8, T9 for the oracle's velocity step (backsubstitution feet, eqs. 25-35, order of
PAPER.md:229) and T13 for its moments (eqs. 2-4).  The Boris push used as the reference here is typed
from eqs. (29)-(32) with numpy cross products, independently of the oracle's foot formulas."""
import numpy as np
import pytest


def boris_forward(vn, qm, dt, E, B):
    """eqs. (26), (28)-(30): v^n -> v^{n+1}."""
    h = qm * dt / 2 * E
    t = qm * dt / 2 * B
    s = 2 * t / (1 + t @ t)
    vm = vn + h
    vprime = vm + np.cross(vm, t)
    vp = vm + np.cross(vprime, s)
    return vp + h


def boris_backward(vnp1, qm, dt, E, B):
    """eqs. (26), (28), (31), (32): v^{n+1} -> v^n."""
    h = qm * dt / 2 * E
    t = qm * dt / 2 * B
    s = 2 * t / (1 + t @ t)
    vp = vnp1 - h
    vt = vp - np.cross(vp, t)
    vm = vp - np.cross(vt, s)
    return vm - h


def test_reference_boris_is_self_consistent():
    rng = np.random.default_rng(0)
    for _ in range(20):
        E, B, v = rng.normal(size=3), rng.normal(size=3), rng.normal(size=3)
        w = boris_forward(v, -1.3, 0.2, E, B)
        assert np.abs(boris_backward(w, -1.3, 0.2, E, B) - v).max() < 1e-14
        # the implicit midpoint rule eq. (25)
        lhs = (w - v) / 0.2
        rhs = -1.3 * (E + np.cross((w + v) / 2, B))
        assert np.abs(lhs - rhs).max() < 1e-13
        # |v| conserved without E
        w0 = boris_forward(v, -1.3, 0.2, 0 * E, B)
        assert abs(np.linalg.norm(w0) - np.linalg.norm(v)) < 1e-14


def test_T8_feet_cascade_reproduces_backward_boris(orc):
    """eq. 33 -> eq. 34 -> eq. 35 evaluated through the oracle's foot routine, with the +/- bookkeeping
    of PAPER.md:210-229, gives the full backward Boris map component by component."""
    rng = np.random.default_rng(1)
    for _ in range(50):
        E, B = rng.normal(size=3), 0.6 * rng.normal(size=3)
        q, m, dt = rng.choice([-1.0, 1.0]), rng.uniform(0.04, 2.0), rng.uniform(0.01, 0.5)
        t, s, h, err = orc.boris_coeffs(E, B, q, m, dt)
        if err:
            continue
        assert np.allclose(t, q / m * dt / 2 * B, rtol=1e-15) and np.allclose(h, q / m * dt / 2 * E, rtol=1e-15)
        assert np.allclose(s, 2 * t / (1 + t @ t), rtol=1e-15)
        vnp1 = rng.normal(size=3) * 3
        ref = boris_backward(vnp1, q / m, dt, E, B)
        vz_n = orc.vfoot(2, vnp1[2], vnp1[0], vnp1[1], t, s, h)
        vy_n = orc.vfoot(1, vnp1[1], vnp1[0], vz_n, t, s, h)
        vx_n = orc.vfoot(0, vnp1[0], vy_n, vz_n, t, s, h)
        assert np.abs(np.array([vx_n, vy_n, vz_n]) - ref).max() < 2e-13
        assert np.abs(orc.boris_back(vnp1, t, s, h) - ref).max() < 1e-13


def test_T8_special_cases(orc):
    # B = 0: every foot is v - (q/m) E dt (uniform shift)
    E = np.array([0.3, -0.2, 0.5])
    t, s, h, err = orc.boris_coeffs(E, np.zeros(3), -1.0, 2.0, 0.4)
    assert err == 0
    for d in range(3):
        assert abs(orc.vfoot(d, 1.25, 0.7, -0.3, t, s, h) - (1.25 - (-0.5) * E[d] * 0.4)) < 1e-15
    # E = 0: |v^-| = |v^+|
    B = np.array([0.4, -0.7, 1.0])
    t, s, h, err = orc.boris_coeffs(np.zeros(3), B, 1.0, 1.0, 0.3)
    v = np.array([1.1, -2.0, 0.7])
    assert abs(np.linalg.norm(orc.boris_back(v, t, s, h)) - np.linalg.norm(v)) < 1e-15
    # R13: |t| ~ 1 makes a denominator of eqs. (34)/(35) non-positive
    _, _, _, err = orc.boris_coeffs(np.zeros(3), np.array([0.0, 3.0, 0.0]), 1.0, 1.0, 1.0)
    assert err == orc.ERR_DOMAIN


def _block_case(orc, nv, limiter, reverse=False):
    sp = orc.Species(-1.0, 1.0, (nv,) * 3, (-6.0,) * 3, (6.0,) * 3, 1.0)
    dt = 0.4
    E = np.array([0.3, -0.2, 0.5])
    B = np.array([0.4, -0.7, 1.0])
    c = sp.vmin[0] + (np.arange(nv) + 0.5) * (12.0 / nv)
    VX, VY, VZ = np.meshgrid(c, c, c, indexing="ij")
    u0 = np.array([1.2, -0.5, 0.3])

    def f0(vx, vy, vz):
        return np.exp(-((vx - u0[0]) ** 2 + (vy - u0[1]) ** 2 + (vz - u0[2]) ** 2) / (2 * 0.8 ** 2))

    fb = np.ascontiguousarray(f0(VX, VY, VZ))
    mass0 = fb.sum()
    t, s, h, err = orc.boris_coeffs(E, B, sp.q, sp.m, dt)
    assert err == 0
    orc.vsweeps_block(fb, sp, t, s, h, limiter=limiter, order_reversed=reverse)
    # exact solution of the discretised characteristics: f(v, t+dt) = f0(BorisBack(v))
    hh = -1.0 * dt / 2 * E
    tt = -1.0 * dt / 2 * B
    ss = 2 * tt / (1 + tt @ tt)
    V = np.stack([VX, VY, VZ], -1) - hh
    Vt = V - np.cross(V, tt)
    Vm = V - np.cross(Vt, ss) - hh
    ref = f0(Vm[..., 0], Vm[..., 1], Vm[..., 2])
    return np.abs(fb - ref).max(), abs(fb.sum() - mass0) / mass0


def test_T9_three_sweeps_converge_to_f_of_boris_back_at_third_order(orc):
    e16, m16 = _block_case(orc, 16, 0)
    e32, m32 = _block_case(orc, 32, 0)
    e64, m64 = _block_case(orc, 64, 0)
    assert max(m16, m32, m64) < 1e-14
    assert e16 < 0.08 and e32 < 0.012 and e64 < 0.0011
    assert np.log2(e32 / e64) > 2.7          # approaching third order
    # negative control: sweeps in the reversed order do not converge
    r32, _ = _block_case(orc, 32, 0, reverse=True)
    r64, _ = _block_case(orc, 64, 0, reverse=True)
    assert r32 > 0.2 and r64 > 0.2


def test_T9_limited_scheme_converges_too(orc):
    e16, _ = _block_case(orc, 16, 1)
    e64, m = _block_case(orc, 64, 1)
    assert e64 < 0.02 and e64 < e16 / 4 and m < 1e-14


def test_T13_moments_closed_form_and_brute_force(orc):
    nv = (32, 32, 32)
    sp = orc.Species(1.0, 1.0, nv, (-6.0, -6.0, -6.0), (6.0, 6.0, 6.0), 1.0)
    c = [sp.vmin[d] + (np.arange(nv[d]) + 0.5) * 12.0 / nv[d] for d in range(3)]
    n0, u, T = 1.7, np.array([0.3, -0.2, 0.5]), 0.9
    g = [np.exp(-(c[d] - u[d]) ** 2 / (2 * T)) / np.sqrt(2 * np.pi * T) for d in range(3)]
    fb = n0 * g[0][:, None, None] * g[1][None, :, None] * g[2][None, None, :]
    M = orc.moments_block(fb, sp)
    assert abs(M[0] / n0 - 1) < 1e-7
    for d in range(3):
        assert abs(M[1 + d] / M[0] - u[d]) < 1e-7
        assert abs(M[4 + d] / M[0] - u[d] ** 2 - T) < 1e-6
    assert abs(M[7] / M[0] - u[0] * u[1]) < 1e-7 and abs(M[8] / M[0] - u[0] * u[2]) < 1e-7
    assert abs(M[9] / M[0] - u[1] * u[2]) < 1e-7
    # brute force with numpy on an anisotropic, asymmetric small grid (catches swapped axes / indices)
    nv2 = (3, 4, 5)
    sp2 = orc.Species(1.0, 1.0, nv2, (-1.0, -2.0, 0.5), (2.0, 1.0, 3.0), 1.0)
    rng = np.random.default_rng(4)
    fb2 = rng.random(nv2)
    c2 = [sp2.vmin[d] + (np.arange(nv2[d]) + 0.5) * (sp2.vmax[d] - sp2.vmin[d]) / nv2[d] for d in range(3)]
    dv3 = np.prod([(sp2.vmax[d] - sp2.vmin[d]) / nv2[d] for d in range(3)])
    VX, VY, VZ = np.meshgrid(*c2, indexing="ij")
    want = [fb2.sum(), (VX * fb2).sum(), (VY * fb2).sum(), (VZ * fb2).sum(), (VX * VX * fb2).sum(),
            (VY * VY * fb2).sum(), (VZ * VZ * fb2).sum(), (VX * VY * fb2).sum(), (VX * VZ * fb2).sum(),
            (VY * VZ * fb2).sum()]
    got = orc.moments_block(fb2, sp2)
    assert np.allclose(got, np.array(want) * dv3, rtol=1e-13, atol=0)
