"""Pins T1-T7 for the oracle's core routine (1D PFC remap, eqs. 38-47).

None of these re-type the oracle's flux formula: they check it against integer translation, mirror
symmetry, polynomial exactness, an independent exact-rational integration of the reconstruction
(eq. 17 + eq. 40/45, built here with sympy/fractions), conservation and the positivity claim.
"""
import os
from fractions import Fraction

import numpy as np
import pytest
import sympy as sp

GOLD = os.path.join(os.path.dirname(__file__), "golden")


from pfc_exact import _newton_F, _recon_limited, _x, exact_remap_periodic


def test_T4_reconstruction_is_derivative_of_eq40_and_has_cell_mean():
    fhat, (fm, f0, fp, ep, em) = _recon_limited()
    dF = sp.diff(_newton_F(fm, f0, fp), _x)
    assert sp.simplify(fhat.subs({ep: 1, em: 1}) - dF) == 0          # eq. (41) with the corrected sign
    mean = sp.integrate(fhat, (_x, sp.Rational(-1, 2), sp.Rational(1, 2)))
    assert sp.simplify(mean - f0) == 0                                   # any eps keeps the cell average
    # border value quoted in DESIGN.md erratum A-1
    assert sp.simplify(dF.subs(_x, sp.Rational(1, 2)) - (-fm + 5 * f0 + 2 * fp) / 6) == 0


def test_T1_integer_shifts_translate_exactly(orc):
    rng = np.random.default_rng(1)
    f = rng.random(16)
    for n in (0, 1, 3, -2, -7, 16, 35, -40):
        out = orc.remap1d(f, float(n), "periodic", 1.0, 1)
        assert np.abs(out - np.roll(f, n)).max() <= 2e-15 * max(1, abs(n)), n


def test_T2_mirror_symmetry(orc):
    rng = np.random.default_rng(2)
    f = rng.random(16)
    for s in (0.3, 1.7, 2.25, 0.999, 5.5):
        a = orc.remap1d(f[::-1].copy(), -s, "periodic", 1.0, 1)
        b = orc.remap1d(f, s, "periodic", 1.0, 1)[::-1]
        assert np.abs(a - b).max() <= 4e-16 * max(1.0, s), s


def test_T3_unlimited_scheme_exact_on_quadratics(orc):
    n = 24
    c0, c1, c2 = 0.7, -0.3, 0.05
    edges = np.arange(n + 1) - 0.5

    def avg(lo, hi):
        P = lambda x: c0 * x + c1 * x ** 2 / 2 + c2 * x ** 3 / 3
        return (P(hi) - P(lo)) / (hi - lo)

    f = avg(edges[:-1], edges[1:])
    for s in (0.37, -0.81, 2.6, -1.2):
        out = orc.remap1d(f, s, "periodic", 10.0, 0)
        expect = avg(edges[:-1] - s, edges[1:] - s)
        inner = slice(6, n - 6)         # away from the periodic seam, where the data is not a quadratic
        assert np.abs(out[inner] - expect[inner]).max() <= 1e-14, s


@pytest.mark.parametrize("limiter", [0, 1])
def test_T4_T7_against_exact_integration_of_the_reconstruction(orc, limiter):
    rng = np.random.default_rng(3 + limiter)
    finf = Fraction(1)
    for trial in range(6):
        n = 9
        f = [Fraction(int(v), 1000) for v in rng.integers(0, 1000, n)]
        if trial == 0:
            f = [Fraction(v).limit_denominator(1000) for v in (0, 0, 0.1, 1.0, 0.9, 0.2, 0, 0, 0)]
        for s in (Fraction(1, 4), Fraction(-3, 5), Fraction(3, 2), Fraction(-23, 10), Fraction(0), Fraction(-1), Fraction(29, 8)):
            sig = [s] * (n + 1)
            ex = exact_remap_periodic(f, sig, finf, limiter)
            got = orc.remap1d(np.array([float(v) for v in f]), float(s), "periodic", 1.0, limiter)
            assert np.abs(got - np.array([float(v) for v in ex])).max() <= 5e-15, (trial, s)


def test_T4_nonuniform_shifts_against_exact_integration(orc):
    rng = np.random.default_rng(9)
    n = 10
    f = [Fraction(int(v), 997) for v in rng.integers(0, 997, n)]
    # per-face shifts that change sign and exceed one cell; face n wraps onto face 0
    sig = [Fraction(int(v), 16) for v in rng.integers(-40, 40, n)]
    sig.append(sig[0])
    for limiter in (0, 1):
        ex = exact_remap_periodic(f, sig, Fraction(1), limiter)
        got = orc.remap1d(np.array([float(v) for v in f]), np.array([float(v) for v in sig]), "periodic", 1.0, limiter)
        assert np.abs(got - np.array([float(v) for v in ex])).max() <= 5e-15


def test_T7_worked_example_golden(orc):
    """tests/golden/pfc_worked_example.txt: 8-cell example (B-2); the paper prints no worked
    example, the stored values come from exact rational integration (make_pfc_worked_example.py)."""
    rows = [l.split() for l in open(os.path.join(GOLD, "pfc_worked_example.txt")) if l.strip() and not l.startswith("#")]
    f = np.array([float(v) for v in rows[0][1:]])
    assert rows[0][0] == "f"
    for r in rows[1:]:
        s = float(r[0])
        want = np.array([float(v) for v in r[1:]])
        got = orc.remap1d(f, s, "periodic", 1.0, 1)
        assert np.abs(got - want).max() <= 3e-16, s


def test_T5_mass_conservation_any_per_face_shift(orc):
    rng = np.random.default_rng(5)
    for bc in ("periodic", "zero"):
        for trial in range(20):
            n = int(rng.integers(5, 40))
            f = rng.random(n)
            sig = rng.uniform(-3.5, 3.5, n + 1)
            if bc == "periodic":
                sig[n] = sig[0]
            out = orc.remap1d(f, sig, bc, 1.0, int(trial % 2))
            assert abs(out.sum() - f.sum()) <= 1e-14 * f.sum(), (bc, trial)


def test_T5_zero_bc_outer_faces_carry_no_flux(orc):
    f = np.array([1.0, 2.0, 3.0, 4.0])
    sig = np.array([5.0, 0.0, 0.0, 0.0, -5.0])      # outer shifts must be ignored (R7)
    out = orc.remap1d(f, sig, "zero", 10.0, 1)
    assert np.array_equal(out, f)


def test_T6_positivity_and_maximum_for_uniform_shifts(orc):
    rng = np.random.default_rng(6)
    for trial in range(200):
        n = int(rng.integers(6, 30))
        f = rng.random(n)
        if trial % 3 == 0:
            f[rng.random(n) < 0.4] = 0.0
        if trial % 5 == 0:
            f[rng.random(n) < 0.3] = 1.0
        s = float(rng.uniform(-3, 3))
        out = orc.remap1d(f, s, "periodic", 1.0, 1)
        assert out.min() >= -1e-15 and out.max() <= 1.0 + 1e-15, (trial, s)


def test_R6_limiter_edge_cases(orc):
    # equal neighbours: no 0/0, value preserved; data outside [0, f_inf]: eps clamps to 0 -> donor-cell
    f = np.array([0.5, 0.5, 0.5, 0.5, 0.5])
    assert np.array_equal(orc.remap1d(f, 0.3, "periodic", 1.0, 1), f)
    g = np.array([0.0, -0.2, 0.0, 1.3, 0.0, 0.0])
    out = orc.remap1d(g, 0.5, "periodic", 1.0, 1)
    assert np.all(np.isfinite(out)) and abs(out.sum() - g.sum()) < 1e-15


def test_R8_foot_on_a_face_is_continuous(orc):
    rng = np.random.default_rng(8)
    f = rng.random(12)
    for s in (1.0, -2.0, 3.0):
        a = orc.remap1d(f, np.nextafter(s, -10.0), "periodic", 1.0, 1)
        b = orc.remap1d(f, np.nextafter(s, 10.0), "periodic", 1.0, 1)
        assert np.abs(a - b).max() <= 4e-15
