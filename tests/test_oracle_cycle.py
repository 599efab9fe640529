"""Pins for the oracle's time-stepping cycle of section 4.3 (oracle.cycle; Fig. 2): the order
currents -> fields half a step -> complete Vlasov step with the new E and with B interpolated to the E time level
 -> currents -> fields another half step.  Neither pin re-types the composition: each compares the
cycle with something the mathematics fixes.

  C1  cold-plasma (Langmuir) oscillation of a spatially uniform drifting plasma: the cycle is then exactly the
      velocity-Verlet recurrence of a harmonic oscillator, whose frequency is known in closed form,
      cos(omega_num dt) = 1 - omega_pe^2 dt^2 / 2.
      Mutants of oracle.cycle that fail it: second current update dropped (J of the old moments reused), a field half
      step taking dt instead of dt/2, the Vlasov step run with the OLD E, the current with the wrong sign or without
      q_s, the Maxwell half steps dropped.
  C2  test particles in a vacuum plane wave: with a vanishing charge the fields follow the discrete (Yee) plane wave,
      known in closed form at every time level, and the Vlasov step of the cycle must equal oracle.step with E at
      t + dt/2 and B AVERAGED to that time (the closed form of the average is cos(omega ddt/2) times the wave).
      Mutants that fail it: the un-averaged B handed to the Vlasov step (negative control below), E and Bavg of the
      wrong half step, the second half step dropped or doubled (E, B after the cycle are checked too).
"""
import numpy as np
import pytest


def _drifting_maxwellian(nv, vmin, vmax, u):
    g = []
    for d in range(3):
        dv = (vmax[d] - vmin[d]) / nv[d]
        c = vmin[d] + (np.arange(nv[d]) + 0.5) * dv
        g.append(np.exp(-0.5 * (c - u[d]) ** 2) / np.sqrt(2 * np.pi))
    return g[0][:, None, None] * g[1][None, :, None] * g[2][None, None, :]


@pytest.mark.parametrize("order", [0, 1])
@pytest.mark.parametrize("fields_yee", [0, 1])
def test_C1_langmuir_oscillation_is_the_verlet_recurrence(orc, fields_yee, order):
    nx, ny, nv = 4, 2, (48, 4, 4)
    vmin, vmax = (-8.0,) * 3, (8.0,) * 3
    q, m, c, mu0, dt, nsub = -1.0, 1.0, 2.0, 0.5, 0.1, 2
    sp = orc.Species(q, m, nv, vmin, vmax, 1.0)
    blk = _drifting_maxwellian(nv, vmin, vmax, (0.3, 0.0, 0.0))
    f = np.ascontiguousarray(np.broadcast_to(blk, (ny, nx) + nv)).copy()
    E = np.zeros((3, ny, nx))
    B = np.zeros((3, ny, nx))
    mom = [orc.moments(f, sp, nx, ny, 0)]
    n0 = mom[0][0, 0, 0]
    w2 = c * c * mu0 * q * q * n0 / m              # omega_pe^2 of the DISCRETE density
    u, Ex = [mom[0][1, 0, 0] / n0], [0.0]
    for _ in range(40):
        # unlimited scheme: the first velocity moment of a compactly supported f moves exactly by the shift
        mom = orc.cycle([f], [sp], mom, E, B, nx, ny, 0, 1.0, 1.0, dt, nsub, c, mu0, fields_yee=fields_yee,
                        order=order, limiter=0)
        assert np.ptp(mom[0][1]) <= 1e-13 and np.ptp(E[0]) <= 1e-13       # stays uniform
        assert abs(mom[0][0, 0, 0] - n0) <= 1e-13
        u.append(mom[0][1, 0, 0] / n0)
        Ex.append(E[0, 0, 0])
    u, Ex = np.array(u), np.array(Ex)
    cw = 1.0 - 0.5 * w2 * dt * dt
    assert np.abs(u).max() > 0.29 and np.abs(Ex).max() > 0.15             # it oscillates: omega_pe dt = 0.06, 40 steps
    assert u.min() < -0.2                                                 # ... through more than half a period
    assert np.abs(u[2:] + u[:-2] - 2 * cw * u[1:-1]).max() <= 1e-12
    assert np.abs(Ex[2:] + Ex[:-2] - 2 * cw * Ex[1:-1]).max() <= 1e-12
    # and the phase relation of the two: E' = E - (dt/2) c^2 mu0 q n (u + u')
    assert np.abs(Ex[1:] - Ex[:-1] + 0.5 * dt * c * c * mu0 * q * n0 * (u[1:] + u[:-1])).max() <= 1e-12


def _yee_wave(nx, nyg, dx, c, ddt, mode_n):
    """Discrete plane wave along x of the 2D Yee scheme (TM: E_z at nodes, B_y at (i+1/2, j)), as closed forms of
    time: E_z(x_i, t) = cos(k x_i - w t), B_y(x_i + dx/2, t) = b cos(k (x_i + dx/2) - w t), with w from the Yee
    dispersion relation sin(w ddt/2) = (c ddt/dx) sin(k dx/2) and b from Faraday's law."""
    k = 2 * np.pi * mode_n / (nx * dx)
    w = 2.0 / ddt * np.arcsin(c * ddt / dx * np.sin(k * dx / 2))
    b = -ddt * np.sin(k * dx / 2) / (dx * np.sin(w * ddt / 2))
    xi = np.arange(nx) * dx

    def Ez(t):
        return np.broadcast_to(np.cos(k * xi - w * t), (nyg, nx)).copy()

    def By(t, amp=1.0):
        return np.broadcast_to(amp * b * np.cos(k * (xi + dx / 2) - w * t), (nyg, nx)).copy()

    return w, Ez, By


def test_C2_test_particles_in_a_vacuum_wave_see_E_and_averaged_B_at_mid_step(orc):
    nx, ny, nv = 8, 2, (12, 6, 12)
    dx, c, dt, nsub = 0.5, 1.0, 0.4, 1
    ddt = dt / 2 / nsub
    lx, ly = nx * dx, 1.0
    vmin, vmax = (-5.0,) * 3, (5.0,) * 3
    # vanishing charge, q/m = -1.5: the plasma does not act back on the fields (J ~ 1e-14)
    sp = orc.Species(-1.5e-14, 1e-14, nv, vmin, vmax, 1.0)
    rng = np.random.default_rng(21)
    blk = _drifting_maxwellian(nv, vmin, vmax, (0.8, 0.0, -0.4))
    f0 = np.ascontiguousarray(blk[None, None] * (0.5 + 0.5 * rng.random((ny, nx, 1, 1, 1))))
    w, Ez, By = _yee_wave(nx, ny, dx, c, ddt, 1)
    amp = 1.2
    E = np.zeros((3, ny, nx)); B = np.zeros((3, ny, nx))
    E[2] = amp * Ez(0.0)
    B[1] = amp * By(ddt / 2)                       # B is half a sub-step ahead of E (8(c)-5)
    f = f0.copy()
    mom = [orc.moments(f, sp, nx, ny, 0)]
    mom = orc.cycle([f], [sp], mom, E, B, nx, ny, 0, lx, ly, dt, nsub, c, 1.0, fields_yee=1)
    # fields after the cycle: the wave at t = dt (E) and t = dt + ddt/2 (B)
    assert np.abs(E[2] - amp * Ez(dt)).max() <= 1e-13 and np.abs(B[1] - amp * By(dt + ddt / 2)).max() <= 1e-13
    assert np.abs(E[:2]).max() <= 1e-13 and np.abs(B[0]).max() + np.abs(B[2]).max() <= 1e-13
    # the Vlasov step saw E at t + dt/2 and B averaged to that time: (B(t - ddt/2) + B(t + ddt/2)) / 2 = cos(w ddt/2) B(t)
    Eh = np.zeros((3, ny, nx)); Bh = np.zeros((3, ny, nx))
    Eh[2] = amp * Ez(dt / 2)
    Bh[1] = amp * np.cos(w * ddt / 2) * By(dt / 2)
    want = f0.copy()
    err, mw = orc.step(want, sp, nx, ny, 0, lx, ly, dt, Eh, Bh, fields_yee=1)
    assert err == 0
    assert np.abs(f - want).max() <= 1e-13 * want.max()
    assert np.abs(mom[0] - mw).max() <= 1e-12 * np.abs(mw).max()
    # negative controls, from the closed forms alone: the un-averaged B (half a sub-step late), or the fields of time t
    for Eb, Bb in ((Eh[2], amp * By(dt / 2 + ddt / 2)), (amp * Ez(0.0), Bh[1])):
        Em = np.zeros((3, ny, nx)); Bm = np.zeros((3, ny, nx))
        Em[2] = Eb; Bm[1] = Bb
        wrong = f0.copy()
        orc.step(wrong, sp, nx, ny, 0, lx, ly, dt, Em, Bm, fields_yee=1, want_moments=False)
        assert np.abs(f - wrong).max() >= 1e-4 * want.max()
