"""ORACLE -- TEST INFRASTRUCTURE ONLY: the five-moment fluid step of the coupled scheme (numpy, fp64, plain loops
over stages; no blocking, no fusion).

PAPER.md:301 (section 3.2): "For the discretization in space, we use the CWENO scheme [18], an easy to implement third
order finite-volume scheme.  The third order strong-stability-preserving Runge-Kutta scheme by Shu and Osher [19] is
employed for the time integration."  Equations: the moment equations (5)-(7) PAPER.md:50-54 with the closure (8)
PAPER.md:61 (P = p 1, p = (2/3) E - (1/3) u^2 / rho, div Q = 0), i.e. the Euler equations with gamma = 5/3 per species
plus the Lorentz source (q/m)(rho E + u x B), (q/m) u . E.  Here u is the MOMENTUM density (eq. 3).

The paper gives no more than the two names, so the details are reading R23 of DESIGN.md:
  * state per species and cell: U = (rho, u_x, u_y, u_z, E) -- cell averages on a 2D grid [ny_g][nx], x periodic,
    ny_g = ny + 4: two ghost rows per y side (the stencil of one stage reaches two cells);
  * reconstruction: the third-order compact central WENO of Levy, Puppo, Russo as used by Kurganov and Levy's
    semi-discrete scheme, dimension by dimension, component by component on the conserved variables: in every cell
    the convex combination of the two one-sided linear polynomials and the central parabola that completes them to
    the optimal quadratic, constants 1/4, 1/2, 1/4, weights c_k / (eps + IS_k)^2, eps = 1e-6;
  * flux through a face: the central-upwind (local Lax-Friedrichs) flux of the semi-discrete scheme,
    H = (F(U+) + F(U-))/2 - a/2 (U+ - U-), a = the larger of |v_n| + c_s of the two states, evaluated at the face
    centre (third order in 1D and for linear problems, second order for nonlinear 2D ones: "easy to implement");
  * sources: evaluated from the stage's cell averages with E, B at the cell centres, held fixed over the step;
  * time: Shu-Osher SSP-RK3, U1 = U + dt L(U); U2 = 3/4 U + 1/4 (U1 + dt L(U1)); U' = 1/3 U + 2/3 (U2 + dt L(U2)),
    whose stages sit at t, t + dt and t + dt/2: ghost rows of a COUPLED side are given at these three times
    ("needs boundary conditions at times t, t + dt/2 and t + dt");
  * y sides: PERIODIC, WALL (mirror image, u_y odd) or COUPLED (ghost rows are data: section 4.1).

It shares nothing with paper_1406_5445_b200/.  Pins: tests/test_oracle_fluid.py (third order on a smooth wave in x and in
y, conservation to round-off, Sod's shock tube against the exact Riemann solution and without new extrema, cyclotron
rotation and E.u work of the source at third order in dt, stage times of the boundary data).
"""
import numpy as np

GAMMA = 5.0 / 3.0            # eq. (8): p = (2/3)(E - u^2 / (2 rho))
EPS = 1e-6
BC_PERIODIC, BC_WALL, BC_COUPLED = 0, 1, 2
G = 2                        # ghost rows per y side


def pressure(U):
    """eq. (8) PAPER.md:61.  U: [5, ...] = rho, u (momentum density), E."""
    return (2.0 / 3.0) * U[4] - (1.0 / 3.0) * (U[1] ** 2 + U[2] ** 2 + U[3] ** 2) / U[0]


def from_moments(mom10, m):
    """eqs. (2)-(4) PAPER.md:39-46 from the raw velocity moments M0, M1, M2 (order of vlasov.h):
    rho = m M0, u = m M1, E = (m/2)(M2xx + M2yy + M2zz)."""
    mom10 = np.asarray(mom10)
    return np.stack([m * mom10[0], m * mom10[1], m * mom10[2], m * mom10[3], 0.5 * m * (mom10[4] + mom10[5] + mom10[6])])


def to_boundary5(U, m):
    """What the ghost fill of the Vlasov side takes (vlasov_set_boundary): n, bulk velocity, scalar pressure."""
    U = np.asarray(U)
    return np.stack([U[0] / m, U[1] / U[0], U[2] / U[0], U[3] / U[0], pressure(U)])


def cweno3_faces(u, axis):
    """Point values of the CWENO3 reconstruction of the cell averages u at the lower (W) and upper (E) face of every
    cell along `axis` (periodic indexing: the caller has filled ghost cells where the axis is not periodic)."""
    um = np.roll(u, 1, axis)
    up = np.roll(u, -1, axis)
    dl = u - um                      # slope of the left linear polynomial (times dx)
    dr = up - u
    d2 = up - 2.0 * u + um
    dc = up - um
    is_l = dl * dl
    is_r = dr * dr
    is_c = (13.0 / 3.0) * d2 * d2 + 0.25 * dc * dc
    a_l = 0.25 / (EPS + is_l) ** 2
    a_r = 0.25 / (EPS + is_r) ** 2
    a_c = 0.5 / (EPS + is_c) ** 2
    s = a_l + a_r + a_c
    w_l, w_r, w_c = a_l / s, a_r / s, a_c / s
    # values of the three polynomials at x_j +- dx/2 (P_C = 2 P_opt - (P_L + P_R)/2, P_opt the conservative parabola)
    pe = w_l * (u + 0.5 * dl) + w_r * (u + 0.5 * dr) + w_c * (u + d2 / 6.0 + 0.25 * dc)
    pw = w_l * (u - 0.5 * dl) + w_r * (u - 0.5 * dr) + w_c * (u + d2 / 6.0 - 0.25 * dc)
    return pw, pe


def flux(U, d):
    """Flux of eqs. (5)-(7) with the closure (8) along direction d (0: x, 1: y)."""
    rho = U[0]
    vn = U[1 + d] / rho
    p = pressure(U)
    F = np.empty_like(U)
    F[0] = U[1 + d]
    F[1] = U[1] * vn
    F[2] = U[2] * vn
    F[3] = U[3] * vn
    F[1 + d] = F[1 + d] + p
    F[4] = (U[4] + p) * vn
    return F


def max_speed(U, d):
    rho = U[0]
    return np.abs(U[1 + d] / rho) + np.sqrt(GAMMA * pressure(U) / rho)


def rhs(U, E, B, qm, dx, dy):
    """L(U) for one species on the ghost-inclusive array U[5][ny_g][nx] (valid on the interior rows)."""
    L = np.zeros_like(U)
    for d, h in ((0, dx), (1, dy)):
        axis = 2 if d == 0 else 1
        W = np.empty_like(U)
        Ef = np.empty_like(U)
        for k in range(5):
            W[k], Ef[k] = cweno3_faces(U[k], axis - 1)
        # face j+1/2 between cell j (its E value: "minus" state) and cell j+1 (its W value: "plus" state)
        Um = Ef
        Up = np.roll(W, -1, axis)
        a = np.maximum(max_speed(Um, d), max_speed(Up, d))
        H = 0.5 * (flux(Up, d) + flux(Um, d)) - 0.5 * a[None] * (Up - Um)
        L -= (H - np.roll(H, 1, axis)) / h
    # Lorentz source, eqs. (6), (7): (q/m)(rho E + u x B), (q/m) u . E
    rho, ux, uy, uz = U[0], U[1], U[2], U[3]
    L[1] += qm * (rho * E[0] + (uy * B[2] - uz * B[1]))
    L[2] += qm * (rho * E[1] + (uz * B[0] - ux * B[2]))
    L[3] += qm * (rho * E[2] + (ux * B[1] - uy * B[0]))
    L[4] += qm * (ux * E[0] + uy * E[1] + uz * E[2])
    return L


def fill_ghost(U, bc_lo, bc_hi, ghost_lo=None, ghost_hi=None):
    """Ghost rows of U[5][ny+4][nx] (in place).  COUPLED: ghost_* [5][2][nx] in ascending y."""
    ny = U.shape[1] - 2 * G
    if bc_lo == BC_PERIODIC:
        U[:, :G] = U[:, ny:ny + G]
    elif bc_lo == BC_WALL:
        U[:, :G] = U[:, 2 * G - 1:G - 1:-1]
        U[2, :G] *= -1.0
    else:
        U[:, :G] = ghost_lo
    if bc_hi == BC_PERIODIC:
        U[:, ny + G:] = U[:, G:2 * G]
    elif bc_hi == BC_WALL:
        U[:, ny + G:] = U[:, ny + G - 1:ny - 1:-1]
        U[2, ny + G:] *= -1.0
    else:
        U[:, ny + G:] = ghost_hi


def step(U, q, m, dt, dx, dy, E, B, bc_lo=BC_PERIODIC, bc_hi=BC_PERIODIC, ghost_lo=None, ghost_hi=None):
    """One SSP-RK3 step of every species.  U: [ns][5][ny+4][nx] (updated in place, ghost rows are scratch);
    E, B: [3][ny+4][nx] at the cell centres; ghost_lo / ghost_hi: None or [3][ns][5][2][nx], the ghost rows of a
    COUPLED side at the stage times t, t + dt, t + dt/2 (in THIS order: the order of the stages)."""
    ns = U.shape[0]
    ny = U.shape[2] - 2 * G
    inner = slice(G, G + ny)
    for s in range(ns):
        qm = q[s] / m[s]

        def Lop(V, stage):
            gl = None if ghost_lo is None else ghost_lo[stage][s]
            gh = None if ghost_hi is None else ghost_hi[stage][s]
            fill_ghost(V, bc_lo, bc_hi, gl, gh)
            return rhs(V, E, B, qm, dx, dy)

        U0 = U[s].copy()
        U1 = U0.copy()
        U1[:, inner] = U0[:, inner] + dt * Lop(U0, 0)[:, inner]
        U2 = U0.copy()
        U2[:, inner] = 0.75 * U0[:, inner] + 0.25 * (U1[:, inner] + dt * Lop(U1, 1)[:, inner])
        Un = U0.copy()
        Un[:, inner] = (1.0 / 3.0) * U0[:, inner] + (2.0 / 3.0) * (U2[:, inner] + dt * Lop(U2, 2)[:, inner])
        U[s] = Un
    return U
