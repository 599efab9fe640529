"""Exact-rational evaluation of eq. (17) with the PFC reconstruction (eqs. 40, 43-45; sign of R4).

Test-side brute force, independent of oracle/ and of the CUDA path.
"""
import math
from fractions import Fraction

import sympy as sp

# ------------------------------------------------------------------------------------------------
# independent reference: eq. (17) evaluated exactly -- integrate the piecewise reconstruction
# (derivative of eq. 40's Newton interpolant, limited as in eq. 45 with the sign of reading R4)
# between the feet of the two faces of every cell.  Rational arithmetic, periodic line, dx = 1.
# ------------------------------------------------------------------------------------------------
_x = sp.symbols("x")


def _newton_F(fm, f0, fp):
    """eq. (40) for cell i = 0 with dx = 1: borders at -3/2, -1/2, 1/2, 3/2, F(-3/2) = 0."""
    xm32, xm12, xp12 = sp.Rational(-3, 2), sp.Rational(-1, 2), sp.Rational(1, 2)
    return (fm * (_x - xm32) + (f0 - fm) / 2 * (_x - xm32) * (_x - xm12)
            + (fp - 2 * f0 + fm) / 6 * (_x - xm32) * (_x - xm12) * (_x - xp12))


def _recon_limited():
    """eq. (45) with R4's corrected sign, cell centre x_i = 0, dx = 1; symbols fm, f0, fp, ep, em."""
    fm, f0, fp, ep, em = sp.symbols("fm f0 fp ep em")
    a = 2 * _x * (_x + sp.Rational(3, 2)) + (_x + sp.Rational(1, 2)) * (_x - sp.Rational(1, 2))
    b = 2 * _x * (_x - sp.Rational(3, 2)) + (_x + sp.Rational(1, 2)) * (_x - sp.Rational(1, 2))
    fhat = f0 + ep * (fp - f0) / 6 * a - em * (f0 - fm) / 6 * b
    return fhat, (fm, f0, fp, ep, em)


_FH, _SYMS = _recon_limited()
_PRIM = sp.integrate(_FH, _x)          # antiderivative in the cell-local coordinate
_PRIM_FN = sp.lambdify((_x,) + _SYMS, _PRIM, "math")


def _prim_exact(xl, fm, f0, fp, ep, em):
    return _PRIM.subs({_x: xl, _SYMS[0]: fm, _SYMS[1]: f0, _SYMS[2]: fp, _SYMS[3]: ep, _SYMS[4]: em})


def _eps_exact(fm, f0, fp, finf, limiter):
    """eqs. (43)/(44), reading R6, in exact arithmetic."""
    if not limiter:
        return Fraction(1), Fraction(1)
    one = Fraction(1)
    dp, dm = fp - f0, f0 - fm
    ep = one if dp == 0 else (min(one, 2 * f0 / dp) if dp > 0 else min(one, -2 * (finf - f0) / dp))
    em = one if dm == 0 else (min(one, 2 * (finf - f0) / dm) if dm > 0 else min(one, -2 * f0 / dm))
    clamp = lambda e: max(Fraction(0), min(one, e))
    return clamp(ep), clamp(em)


def _primitive_at(f, X, finf, limiter):
    """Exact primitive of the piecewise reconstruction at position X (cell k spans [k-1/2, k+1/2]),
    periodic line of n cells, counted from -1/2."""
    n = len(f)
    k = math.floor(X + Fraction(1, 2))
    total = sum(f) * (k // n) + sum(f[: k % n])
    j = k % n
    fm, f0, fp = f[(j - 1) % n], f[j], f[(j + 1) % n]
    ep, em = _eps_exact(fm, f0, fp, finf, limiter)
    xl = X - k
    part = _prim_exact(sp.Rational(xl.numerator, xl.denominator), *[sp.Rational(v.numerator, v.denominator) for v in (fm, f0, fp, ep, em)]) \
        - _prim_exact(sp.Rational(-1, 2), *[sp.Rational(v.numerator, v.denominator) for v in (fm, f0, fp, ep, em)])
    return total + Fraction(int(part.p), int(part.q))


def exact_remap_periodic(f, sigma_faces, finf, limiter):
    """eq. (17): new average of cell i = primitive(foot of face i+1/2) - primitive(foot of face i-1/2)."""
    n = len(f)
    out = []
    for i in range(n):
        Xl = Fraction(i) - Fraction(1, 2) - sigma_faces[i]
        Xr = Fraction(i) + Fraction(1, 2) - sigma_faces[i + 1]
        out.append(_primitive_at(f, Xr, finf, limiter) - _primitive_at(f, Xl, finf, limiter))
    return out


