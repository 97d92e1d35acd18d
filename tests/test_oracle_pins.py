"""Pins for the CPU oracle (SURVEY 8(c) P1..P14 + VJP): `-m "not gpu"`.

Each test checks ``oracle/`` against something OTHER than itself: closed forms (golden text
fixtures), the theta/phi definition (Eq. 2 + Eq. 4), symbolic differentiation of the definition
(sympy), a library routine (scipy), exact quadrature, and invariants that a dropped term, a wrong
sign or index, or a transposed operand would break.  No CUDA anywhere in this file.

``P:n`` = line n of PAPER.md (arXiv 2302.08381).
"""
import math
from pathlib import Path

import numpy as np
import pytest

LD = np.longdouble
EPS_LD = float(np.finfo(LD).eps)  # 1.08e-19
GOLDEN = Path(__file__).parent / "golden"


def k_of(l, m):
    return l * (l + 1) + m


def row_scale(l, r=1.0, solid=False, order=0):
    """S_d of DESIGN.md: the 2-norm of the l-row, times (max(l,1)/r)^order."""
    rho = r ** l if solid else 1.0
    return math.sqrt((2 * l + 1) / (4 * math.pi)) * rho * (max(l, 1) / r) ** order


def random_points(n, seed, scale=1.0):
    rng = np.random.default_rng(seed)
    return rng.standard_normal((n, 3)) * scale


# --------------------------------------------------------------------------------------------
# P1  closed-form low-l polynomials (values, ordering, signs, normalisation)
# --------------------------------------------------------------------------------------------
def _read_closed_forms():
    rows = []
    for line in (GOLDEN / "low_l_closed_forms.txt").read_text().splitlines():
        if not line.strip() or line.startswith("#"):
            continue
        l, m, pref, poly = [t.strip() for t in line.split(";")]
        rows.append((int(l), int(m), pref, poly))
    return rows


def test_P1_low_l_closed_forms(oracle):
    rows = _read_closed_forms()
    assert len(rows) == 16
    pts = np.array([[0.5, -0.25, 0.75], [1.5, 2.0, -0.5], [0.0, 0.0, 1.25], [-0.375, 0.0, 0.0],
                    [0.0, -3.0, 0.0], [-1.0, 1.0, 1.0], [0.125, 0.25, -4.0]])
    solid, _, _ = oracle.compute(pts, 3, normalized=False)
    unit, _, _ = oracle.compute(pts, 3, normalized=True)
    env = {"sqrt": math.sqrt, "pi": math.pi}
    for i, (x, y, z) in enumerate(pts):
        r = math.sqrt(x * x + y * y + z * z)
        for l, m, pref, poly in rows:
            want = eval(pref, env) * eval(poly, dict(env, x=x, y=y, z=z))
            k = k_of(l, m)
            assert abs(float(solid[i, k]) - want) <= 4e-15 * max(1.0, r ** l), (l, m, i)
            assert abs(float(unit[i, k]) - want / r ** l) <= 4e-15, (l, m, i)


def test_P1_l1_is_yzx_over_r(oracle):
    """north_star: "l=1 proportional to (y,z,x)/r"."""
    pts = random_points(50, 1)
    sph, _, _ = oracle.compute(pts, 1, normalized=True)
    r = np.linalg.norm(pts, axis=1)
    c = math.sqrt(3 / (4 * math.pi))
    want = c * pts[:, [1, 2, 0]] / r[:, None]
    assert np.max(np.abs(sph[:, 1:4].astype(float) - want)) < 1e-15


# --------------------------------------------------------------------------------------------
# P2  the theta/phi route: Eq. 2 + Eq. 3 + Eq. 4, away from the poles
# --------------------------------------------------------------------------------------------
def _sph_theta_phi(xyz, l_max):
    """Real Y_l^m by the traditional route the paper describes at P:43-49 (long double)."""
    xyz = np.asarray(xyz, LD)
    x, y, z = xyz[:, 0], xyz[:, 1], xyz[:, 2]
    r = np.sqrt(x * x + y * y + z * z)
    t = z / r                                   # cos(theta)
    st = np.sqrt((1 - t) * (1 + t))             # sin(theta)
    phi = np.arctan2(y, x)
    n = xyz.shape[0]
    P = {(0, 0): np.ones(n, LD)}
    for l in range(1, l_max + 1):               # Eq. 4
        P[(l, l)] = -(2 * l - 1) * st * P[(l - 1, l - 1)]
        P[(l, l - 1)] = (2 * l - 1) * t * P[(l - 1, l - 1)]
        for m in range(0, l - 1):
            P[(l, m)] = ((2 * l - 1) * t * P[(l - 1, m)] - (l + m - 1) * P[(l - 2, m)]) / (l - m)
    out = np.zeros((n, (l_max + 1) ** 2), LD)
    pi = LD("3.14159265358979323846264338327950288")
    for l in range(l_max + 1):
        for m in range(0, l + 1):
            # Eq. 3 with exact integer factorials
            ratio = LD(math.factorial(l - m)) / LD(math.factorial(l + m))
            F = (-1) ** m * np.sqrt(LD(2 * l + 1) / (2 * pi) * ratio)
            if m == 0:
                out[:, k_of(l, 0)] = F * P[(l, 0)] / np.sqrt(LD(2))
            else:
                out[:, k_of(l, m)] = F * P[(l, m)] * np.cos(m * phi)
                out[:, k_of(l, -m)] = F * P[(l, m)] * np.sin(m * phi)
    return out


def test_P2_theta_phi_route(oracle):
    l_max = 12
    pts = random_points(400, 2)
    pts = pts[np.hypot(pts[:, 0], pts[:, 1]) > 0.05 * np.linalg.norm(pts, axis=1)]  # off the poles
    got, _, _ = oracle.compute(pts, l_max, normalized=True)
    want = _sph_theta_phi(pts, l_max)
    # trig of m*phi in long double: ~m*eps; far below any plausible formula slip
    assert float(np.max(np.abs(got - want))) < 1e-15
    # solid = r^l * normalised
    solid, _, _ = oracle.compute(pts, l_max, normalized=False)
    r = np.linalg.norm(pts.astype(LD), axis=1)
    for l in range(l_max + 1):
        sl = slice(l * l, (l + 1) ** 2)
        err = np.abs(solid[:, sl] - want[:, sl] * (r ** l)[:, None]) / (r ** l)[:, None]
        assert float(err.max()) < 1e-15, l


# --------------------------------------------------------------------------------------------
# P12  library special case: scipy's complex harmonics (Condon-Shortley) mapped per reading S2
# --------------------------------------------------------------------------------------------
def test_P12_scipy_sph_harm(oracle):
    sp = pytest.importorskip("scipy.special")
    if not hasattr(sp, "sph_harm_y"):
        pytest.skip("scipy too old for sph_harm_y")
    l_max = 10
    pts = random_points(200, 12)
    got, _, _ = oracle.compute(pts, l_max, normalized=True)
    got = got.astype(np.float64)
    r = np.linalg.norm(pts, axis=1)
    theta = np.arccos(pts[:, 2] / r)
    phi = np.arctan2(pts[:, 1], pts[:, 0])
    for l in range(l_max + 1):
        for m in range(0, l + 1):
            Y = sp.sph_harm_y(l, m, theta, phi)
            if m == 0:
                np.testing.assert_allclose(got[:, k_of(l, 0)], Y.real, atol=2e-13)
            else:
                sgn = math.sqrt(2) * (-1) ** m
                np.testing.assert_allclose(got[:, k_of(l, m)], sgn * Y.real, atol=2e-13)
                np.testing.assert_allclose(got[:, k_of(l, -m)], sgn * Y.imag, atol=2e-13)


# --------------------------------------------------------------------------------------------
# P14  brute force on tiny inputs: symbolic expansion + symbolic differentiation of the definition
# --------------------------------------------------------------------------------------------
def _sympy_solid_harmonics(l_max):
    """r^l Y_l^m as polynomials in x,y,z from Eq. 2/3 and the Rodrigues form of P_l^m
    (with Condon-Shortley sign, as Eq. 4's P_l^l = -(2l-1) sqrt(1-t^2) P_{l-1}^{l-1} implies)."""
    import sympy as sp

    x, y, z, t = sp.symbols("x y z t", real=True)
    r2 = x * x + y * y + z * z
    out = {}
    for l in range(l_max + 1):
        Pl = sp.legendre(l, t)
        for m in range(0, l + 1):
            dP = sp.diff(Pl, t, m)                      # d^m P_l / dt^m, degree l-m, parity l-m
            poly = sp.Poly(sp.expand(dP), t) if dP != 0 else None
            # r^(l-m) * dP(z/r): every term t^j r^(l-m) -> z^j r^(l-m-j), l-m-j even
            Qlm = 0
            if poly is not None:
                for (j,), coef in poly.terms():
                    assert (l - m - j) % 2 == 0
                    Qlm += coef * z ** j * r2 ** ((l - m - j) // 2)
            Qlm = (-1) ** m * Qlm                       # Condon-Shortley sign of P_l^m
            F = (-1) ** m * sp.sqrt(sp.Rational(2 * l + 1, 2) / sp.pi
                                    * sp.Rational(math.factorial(l - m), math.factorial(l + m)))
            w = sp.expand((x + sp.I * y) ** m)          # r_xy^m e^{i m phi}
            cm, sm = sp.re(w), sp.im(w)
            if m == 0:
                out[(l, 0)] = sp.expand(F * Qlm / sp.sqrt(2))
            else:
                out[(l, m)] = sp.expand(F * Qlm * cm)
                out[(l, -m)] = sp.expand(F * Qlm * sm)
    return (x, y, z), out


def _to_ld(expr, subs):
    import sympy as sp

    return LD(str(sp.N(expr.subs(subs), 30)))


@pytest.mark.parametrize("normalized", [False, True])
def test_P14_symbolic_brute_force(oracle, normalized):
    import sympy as sp

    l_max = 4
    (x, y, z), Y = _sympy_solid_harmonics(l_max)
    r = sp.sqrt(x * x + y * y + z * z)
    # dyadic rationals: exact in binary, so oracle and sympy see the same numbers
    pts = [(sp.Rational(1, 2), sp.Rational(-1, 4), sp.Rational(3, 4)),
           (sp.Rational(3, 2), sp.Integer(2), sp.Rational(-1, 2)),
           (sp.Integer(0), sp.Integer(0), sp.Rational(5, 4)),          # on +z
           (sp.Integer(0), sp.Integer(0), sp.Rational(-3, 4)),         # on -z
           (sp.Rational(-3, 8), sp.Integer(0), sp.Integer(0)),
           (sp.Rational(1, 1024), sp.Rational(-1, 2048), sp.Rational(1, 4096))]  # near the origin
    xyz = np.array([[float(a) for a in p] for p in pts])
    sph, dsph, ddsph = oracle.compute(xyz, l_max, normalized, gradients=True, hessians=True)
    var = (x, y, z)
    for (l, m), f in Y.items():
        if normalized:
            f = f / r ** l
        g = [sp.diff(f, v) for v in var]
        H = [[sp.diff(gi, v) for v in var] for gi in g]
        k = k_of(l, m)
        for i, p in enumerate(pts):
            subs = dict(zip(var, p))
            rr = float(np.linalg.norm(xyz[i]))
            rho = 1.0 if normalized else rr ** l
            tol = 64 * EPS_LD
            S0 = row_scale(l) * rho
            assert abs(sph[i, k] - _to_ld(f, subs)) <= tol * S0, (l, m, i)
            for a in range(3):
                S1 = S0 * max(l, 1) / rr
                assert abs(dsph[i, a, k] - _to_ld(g[a], subs)) <= tol * S1, (l, m, i, a)
                for b in range(3):
                    S2 = S1 * max(l, 1) / rr
                    assert abs(ddsph[i, a, b, k] - _to_ld(H[a][b], subs)) <= tol * S2, (l, m, i, a, b)


def test_P14_symbolic_values_l6(oracle):
    """Same brute force, values + gradients only, up to the paper's hard-coded limit l=6."""
    import sympy as sp

    l_max = 6
    (x, y, z), Y = _sympy_solid_harmonics(l_max)
    pts = [(sp.Rational(1, 2), sp.Rational(-1, 4), sp.Rational(3, 4)),
           (sp.Rational(-5, 4), sp.Rational(7, 8), sp.Rational(1, 16)),
           (sp.Integer(0), sp.Integer(0), sp.Integer(-1))]
    xyz = np.array([[float(a) for a in p] for p in pts])
    sph, dsph, _ = oracle.compute(xyz, l_max, False, gradients=True)
    for (l, m), f in Y.items():
        k = k_of(l, m)
        for i, p in enumerate(pts):
            subs = dict(zip((x, y, z), p))
            rr = float(np.linalg.norm(xyz[i]))
            S0 = row_scale(l) * rr ** l
            assert abs(sph[i, k] - _to_ld(f, subs)) <= 64 * EPS_LD * S0
            for a, v in enumerate((x, y, z)):
                assert abs(dsph[i, a, k] - _to_ld(sp.diff(f, v), subs)) <= 64 * EPS_LD * S0 * l / rr + 1e-30


# --------------------------------------------------------------------------------------------
# P3  addition theorem,  P8  gradient sum rule,  P9  parity
# --------------------------------------------------------------------------------------------
@pytest.mark.parametrize("l_max", [8, 32])
def test_P3_addition_theorem_and_P8_gradient_sum(oracle, l_max):
    pts = random_points(300, 3, scale=1.3)
    pts_ld = pts.astype(LD)
    r2 = (pts_ld ** 2).sum(axis=1)
    pi = LD("3.14159265358979323846264338327950288")
    solid, dsolid, _ = oracle.compute(pts, l_max, False, gradients=True)
    unit, dunit, _ = oracle.compute(pts, l_max, True, gradients=True)
    for l in range(l_max + 1):
        sl = slice(l * l, (l + 1) ** 2)
        c = LD(2 * l + 1) / (4 * pi)
        # sum_m (r^l Y)^2 = r^(2l) (2l+1)/4pi   (north_star; use the r^(2l) form for solid output)
        s = (solid[:, sl] ** 2).sum(axis=1)
        assert float(np.max(np.abs(s / (c * r2 ** l) - 1))) < 200 * EPS_LD * (l + 1)
        s = (unit[:, sl] ** 2).sum(axis=1)
        assert float(np.max(np.abs(s / c - 1))) < 200 * EPS_LD * (l + 1)
        if l == 0:
            assert float(np.max(np.abs(dsolid[:, :, 0]))) == 0.0
            continue
        # sum_m |grad r^l Y|^2 = l (2l+1)^2 r^(2l-2) / 4pi ;  normalised: l(l+1)(2l+1)/(4 pi r^2)
        g = (dsolid[:, :, sl] ** 2).sum(axis=(1, 2))
        want = l * LD(2 * l + 1) ** 2 * r2 ** (l - 1) / (4 * pi)
        assert float(np.max(np.abs(g / want - 1))) < 400 * EPS_LD * (l + 1)
        g = (dunit[:, :, sl] ** 2).sum(axis=(1, 2))
        want = l * (l + 1) * LD(2 * l + 1) / (4 * pi * r2)
        assert float(np.max(np.abs(g / want - 1))) < 400 * EPS_LD * (l + 1)


def test_P9_parity(oracle):
    l_max = 9
    pts = random_points(100, 9)
    a, da, _ = oracle.compute(pts, l_max, True, gradients=True)
    b, db, _ = oracle.compute(-pts, l_max, True, gradients=True)
    for l in range(l_max + 1):
        sl = slice(l * l, (l + 1) ** 2)
        assert np.array_equal(b[:, sl], (-1) ** l * a[:, sl])
        assert np.array_equal(db[:, :, sl], (-1) ** (l + 1) * da[:, :, sl])


# --------------------------------------------------------------------------------------------
# P4  rotation: per-l norms invariant; z-rotation mixes (m, -m) by angle m*alpha
# --------------------------------------------------------------------------------------------
def _random_rotation(rng):
    q, _ = np.linalg.qr(rng.standard_normal((3, 3)))
    if np.linalg.det(q) < 0:
        q[:, 0] = -q[:, 0]
    return q


def test_P4_rotation_invariance_of_row_norms(oracle):
    l_max = 16
    rng = np.random.default_rng(4)
    pts = rng.standard_normal((64, 3))
    a, _, _ = oracle.compute(pts, l_max, True)
    for _ in range(3):
        R = _random_rotation(rng)
        b, _, _ = oracle.compute(pts @ R.T, l_max, True)
        for l in range(l_max + 1):
            sl = slice(l * l, (l + 1) ** 2)
            na = (a[:, sl] ** 2).sum(axis=1)
            nb = (b[:, sl] ** 2).sum(axis=1)
            # R is orthogonal only to f64 rounding, and norms are stationary in direction
            assert float(np.max(np.abs(na - nb))) < 1e-15


def test_P4_z_rotation_law(oracle):
    """Rotating the point by alpha about z: Y_l^m -> cos(m a) Y_l^m - sin(m a) Y_l^-m,
    Y_l^-m -> sin(m a) Y_l^m + cos(m a) Y_l^-m  (SURVEY pin P4)."""
    l_max = 10
    alpha = 0.7371
    ca, sa = math.cos(alpha), math.sin(alpha)
    pts = random_points(64, 44)
    rot = pts.copy()
    rot[:, 0] = ca * pts[:, 0] - sa * pts[:, 1]
    rot[:, 1] = sa * pts[:, 0] + ca * pts[:, 1]
    a, _, _ = oracle.compute(pts, l_max, True)
    b, _, _ = oracle.compute(rot, l_max, True)
    a = a.astype(float)
    b = b.astype(float)
    for l in range(l_max + 1):
        assert np.allclose(b[:, k_of(l, 0)], a[:, k_of(l, 0)], atol=1e-13)
        for m in range(1, l + 1):
            cm, sm = math.cos(m * alpha), math.sin(m * alpha)
            yc, ys = a[:, k_of(l, m)], a[:, k_of(l, -m)]
            assert np.allclose(b[:, k_of(l, m)], cm * yc - sm * ys, atol=1e-13), (l, m)
            assert np.allclose(b[:, k_of(l, -m)], sm * yc + cm * ys, atol=1e-13), (l, m)


# --------------------------------------------------------------------------------------------
# P5  closed forms on the z axis (where Eq. 4 has poles)
# --------------------------------------------------------------------------------------------
def _read_pole_rows():
    rows = {}
    for line in (GOLDEN / "pole_closed_forms.txt").read_text().splitlines():
        if not line.strip() or line.startswith("#"):
            continue
        sigma, l, y0, tang, dz = [t.strip() for t in line.split(";")]
        rows[(int(sigma), int(l))] = (LD(y0), LD(tang), LD(dz))
    return rows


def test_P5_pole_closed_forms(oracle):
    """Values and gradients ON the z axis against the stored closed forms (tests/golden/pole_closed_forms.txt,
    written by make_pole_closed_forms.py from the formulas in its header, 25 digits)."""
    rows = _read_pole_rows()
    l_max = 12
    assert len(rows) == 2 * (l_max + 1)
    for sigma in (+1, -1):
        pts = np.array([[0.0, 0.0, float(sigma)]])
        for normalized in (False, True):
            sph, dsph, ddsph = oracle.compute(pts, l_max, normalized, True, True)
            assert np.all(np.isfinite(sph)) and np.all(np.isfinite(dsph)) and np.all(np.isfinite(ddsph))
            for l in range(l_max + 1):
                y0, tang, dz = rows[(sigma, l)]
                for m in range(-l, l + 1):
                    k = k_of(l, m)
                    want = y0 if m == 0 else LD(0)
                    assert abs(sph[0, k] - want) < 64 * EPS_LD * (1 + abs(want))
                    gx = tang if m == 1 else LD(0)
                    gy = tang if m == -1 else LD(0)
                    gz = dz if (m == 0 and not normalized) else LD(0)   # the radial derivative survives only for solid
                    for a, g in enumerate((gx, gy, gz)):
                        assert abs(dsph[0, a, k] - g) < 64 * EPS_LD * (1 + l * l) * (1 + abs(g)), (sigma, normalized, l, m, a)


# --------------------------------------------------------------------------------------------
# P6  harmonicity,  P7  Euler homogeneity
# --------------------------------------------------------------------------------------------
@pytest.mark.parametrize("l_max", [6, 32])
def test_P6_harmonicity_and_P7_euler(oracle, l_max):
    pts = random_points(120, 6, scale=1.1)
    pts = np.concatenate([pts, [[0, 0, 1.5], [0, 0, -0.5], [1e-5, -2e-5, 3e-5]]])
    x = pts.astype(LD)
    r2 = (x ** 2).sum(axis=1)
    r = np.sqrt(r2)
    ys, gs, hs = oracle.compute(pts, l_max, False, True, True)
    yn, gn, hn = oracle.compute(pts, l_max, True, True, True)
    tol = 2000 * EPS_LD
    for l in range(l_max + 1):
        sl = slice(l * l, (l + 1) ** 2)
        lam = max(l, 1)
        S0s = (row_scale(l) * r ** l)[:, None]
        S0n = row_scale(l)
        # P6: solid harmonics are harmonic; normalised: tr H = -l(l+1) Y / r^2
        tr = hs[:, 0, 0, sl] + hs[:, 1, 1, sl] + hs[:, 2, 2, sl]
        assert float(np.max(np.abs(tr) / (S0s * lam ** 2 / r2[:, None]))) < tol
        tr = hn[:, 0, 0, sl] + hn[:, 1, 1, sl] + hn[:, 2, 2, sl]
        res = tr + l * (l + 1) * yn[:, sl] / r2[:, None]
        assert float(np.max(np.abs(res) / (S0n * lam ** 2 / r2[:, None]))) < tol
        # P7: x.grad = l Y (solid), 0 (normalised);  H x = (l-1) grad (solid), -grad (normalised)
        xg = np.einsum("na,nak->nk", x, gs[:, :, sl])
        assert float(np.max(np.abs(xg - l * ys[:, sl]) / (S0s * lam))) < tol
        xg = np.einsum("na,nak->nk", x, gn[:, :, sl])
        assert float(np.max(np.abs(xg) / (S0n * lam))) < tol
        hx = np.einsum("nb,nabk->nak", x, hs[:, :, :, sl])
        assert float(np.max(np.abs(hx - (l - 1) * gs[:, :, sl]) / (S0s * lam ** 2 / r[:, None])[:, None, :])) < tol
        hx = np.einsum("nb,nabk->nak", x, hn[:, :, :, sl])
        assert float(np.max(np.abs(hx + gn[:, :, sl]) / (S0n * lam ** 2 / r[:, None, None]))) < tol
        # S4: both triangles of the Hessian are stored; equal exactly for the solid harmonics and
        # to rounding for the plain chain rule (its sums run in a different order for (a,b), (b,a))
        for a in range(3):
            for b in range(a):
                assert np.array_equal(hs[:, a, b, sl], hs[:, b, a, sl])
                d = np.abs(hn[:, a, b, sl] - hn[:, b, a, sl])
                assert float(np.max(d / (S0n * lam ** 2 / r2[:, None]))) < 64 * EPS_LD


# --------------------------------------------------------------------------------------------
# P10  finite differences (named in north_star)
# --------------------------------------------------------------------------------------------
@pytest.mark.parametrize("normalized", [False, True])
def test_P10_finite_differences(oracle, normalized):
    l_max = 20
    pts = random_points(24, 10)
    pts = np.concatenate([pts, [[0, 0, 1.0], [0, 0, -2.0]]])  # including the poles
    r = np.linalg.norm(pts, axis=1)
    _, g, H = oracle.compute(pts, l_max, normalized, True, True)
    # inputs must be exactly representable in f64 (the oracle widens doubles): use dyadic steps
    h = 2.0 ** -22
    for a in range(3):
        e = np.zeros(3)
        e[a] = h
        # 4th-order central differences: truncation ~ (l h / r)^4 / 30
        yp1, gp1, _ = oracle.compute(pts + e, l_max, normalized, True)
        ym1, gm1, _ = oracle.compute(pts - e, l_max, normalized, True)
        yp2, gp2, _ = oracle.compute(pts + 2 * e, l_max, normalized, True)
        ym2, gm2, _ = oracle.compute(pts - 2 * e, l_max, normalized, True)
        # the perturbed points must differ from pts by exactly +-h, +-2h
        assert np.all((pts + e) - pts == e) and np.all((pts + 2 * e) - pts == 2 * e)
        fd_g = (8 * (yp1 - ym1) - (yp2 - ym2)) / (12 * LD(h))
        fd_H = (8 * (gp1 - gm1) - (gp2 - gm2)) / (12 * LD(h))
        for l in range(l_max + 1):
            sl = slice(l * l, (l + 1) ** 2)
            lam = max(l, 1)
            rho = (r ** l if not normalized else np.ones_like(r))
            S1 = (row_scale(l) * rho * lam / r)[:, None]
            assert float(np.max(np.abs(fd_g[:, sl] - g[:, a, sl]) / S1)) < 1e-11, (a, l)
            S2 = (row_scale(l) * rho * (lam / r) ** 2)[:, None, None]
            assert float(np.max(np.abs(fd_H[:, :, sl] - H[:, :, a, sl]) / S2)) < 1e-11, (a, l)


# --------------------------------------------------------------------------------------------
# P11  orthonormality by exact quadrature
# --------------------------------------------------------------------------------------------
def test_P11_orthonormality_quadrature(oracle):
    l_max = 10
    nodes, weights = np.polynomial.legendre.leggauss(l_max + 1)       # exact to degree 2 l_max + 1
    nphi = 2 * l_max + 2
    phis = 2 * np.pi * np.arange(nphi) / nphi
    T, PH = np.meshgrid(nodes, phis, indexing="ij")
    W = np.repeat(weights[:, None], nphi, axis=1) * (2 * np.pi / nphi)
    st = np.sqrt(1 - T ** 2)
    pts = np.stack([st * np.cos(PH), st * np.sin(PH), T], axis=-1).reshape(-1, 3)
    Y, _, _ = oracle.compute(pts, l_max, True)
    Y = Y.astype(float)
    gram = Y.T @ (Y * W.reshape(-1, 1))
    assert np.max(np.abs(gram - np.eye(gram.shape[0]))) < 5e-14


# --------------------------------------------------------------------------------------------
# P13  other recurrences the paper prints (Eq. 8 sign-corrected, B20, B23, Eq. 11 corrected, C2)
# --------------------------------------------------------------------------------------------
def test_P13_alternative_Q_recurrences(oracle):
    l_max = 14
    tri = lambda l, m: l * (l + 1) // 2 + m
    rng = np.random.default_rng(13)
    for _ in range(5):
        x, y, z = rng.standard_normal(3)
        r2 = LD(x) ** 2 + LD(y) ** 2 + LD(z) ** 2
        rxy2 = LD(x) ** 2 + LD(y) ** 2
        Q = oracle.Q_triangle(z, r2, l_max)
        for l in range(l_max + 1):
            scale = max(abs(float(Q[tri(l, m)])) for m in range(l + 1))
            for m in range(l + 1):
                q = Q[tri(l, m)]
                # Eq. 8 with the leading minus (reading E1), Q_l^{l+1} = Q_l^{l+2} = 0
                if m <= l - 1:
                    q1 = Q[tri(l, m + 1)]
                    q2 = Q[tri(l, m + 2)] if m + 2 <= l else LD(0)
                    rhs = -(2 * (m + 1) * LD(z) * q1 + rxy2 * q2) / ((l + m + 1) * (l - m))
                    assert abs(float(q - rhs)) <= 1e-16 * scale * (1 + float(r2)), (l, m)
                # B20: Q_l^m = -(2l-1) Q_{l-1}^{m-1} + r^2 Q_{l-2}^m
                if m >= 1 and l >= 1:
                    a = Q[tri(l - 1, m - 1)]
                    b = Q[tri(l - 2, m)] if (l >= 2 and m <= l - 2) else LD(0)
                    assert abs(float(q - (-(2 * l - 1) * a + r2 * b))) <= 1e-16 * scale * (1 + float(r2)), (l, m)
                # B23 shifted: Q_l^{m-1} = (-z Q_l^m + r^2 Q_{l-1}^m) / (l+1-m)
                if m >= 1:
                    b = Q[tri(l - 1, m)] if m <= l - 1 else LD(0)
                    lhs = Q[tri(l, m - 1)]
                    rhs = (-LD(z) * q + r2 * b) / (l + 1 - m)
                    assert abs(float(lhs - rhs)) <= 1e-16 * scale * (1 + float(r2)), (l, m)


def test_P13_eq11_derivative_shortcuts(oracle):
    """Eq. 11 with the indices corrected (reading E2), and App. C's folded relation (E4)."""
    l_max = 9
    pts = random_points(40, 130)
    Y, dY, _ = oracle.compute(pts, l_max, False, gradients=True)
    F = oracle.F_table(l_max)
    tri = lambda l, m: l * (l + 1) // 2 + m
    for l in range(1, l_max + 1):
        for m in range(-l, l + 1):
            am = abs(m)
            got = dY[:, 2, k_of(l, m)]
            if am <= l - 1:
                want = F[tri(l, am)] / F[tri(l - 1, am)] * (l + am) * Y[:, k_of(l - 1, m)]
                # E4: the same ratio in closed form, sqrt((2l+1)/(2l-1)) sqrt(l^2 - m^2)
                closed = math.sqrt((2 * l + 1) / (2 * l - 1)) * math.sqrt(l * l - am * am)
                assert abs(float(F[tri(l, am)] / F[tri(l - 1, am)] * (l + am)) - closed) < 1e-13 * closed
            else:
                want = np.zeros_like(got)
            scale = np.max(np.abs(got)) + 1e-300
            assert float(np.max(np.abs(got - want))) <= 1e-16 * scale + 1e-300, (l, m)
        if l >= 2:
            got = dY[:, 0, k_of(l, l)]
            want = -l * (2 * l - 1) * F[tri(l, l)] / F[tri(l - 1, l - 1)] * Y[:, k_of(l - 1, l - 1)]
            assert float(np.max(np.abs(got - want))) <= 1e-16 * float(np.max(np.abs(got))), l


def test_F_table_matches_eq3(oracle):
    """Eq. C1 iteration == Eq. 3 with exact integer factorials."""
    import sympy as sp

    l_max = 32
    F = oracle.F_table(l_max)
    for l in (0, 1, 2, 5, 16, 29, 32):
        for m in range(l + 1):
            want = (-1) ** m * sp.sqrt(sp.Rational(2 * l + 1, 2) / sp.pi
                                       * sp.Rational(math.factorial(l - m), math.factorial(l + m)))
            want = LD(str(sp.N(want, 30)))
            assert abs(F[l * (l + 1) // 2 + m] / want - 1) < 100 * EPS_LD, (l, m)


# --------------------------------------------------------------------------------------------
# double build == long double build to f64 rounding (the timed CPU baseline computes the same thing)
# --------------------------------------------------------------------------------------------
def test_double_build_agrees_with_long_double(oracle):
    l_max = 8
    pts = random_points(500, 77)
    for normalized in (False, True):
        a = oracle.compute(pts, l_max, normalized, True, True, kind="ld")
        b = oracle.compute(pts, l_max, normalized, True, True, kind="f64")
        r = np.linalg.norm(pts, axis=1)
        for d, (x, y) in enumerate(zip(a, b)):
            for l in range(l_max + 1):
                sl = slice(l * l, (l + 1) ** 2)
                rho = np.ones_like(r) if normalized else r ** l
                S = row_scale(l) * rho * (max(l, 1) / r) ** d
                S = S.reshape((-1,) + (1,) * (x.ndim - 1))
                assert float(np.max(np.abs(x[..., sl] - y[..., sl]) / S)) < 2e-14


# --------------------------------------------------------------------------------------------
# VJP
# --------------------------------------------------------------------------------------------
def test_vjp_against_einsum_and_closed_forms(oracle):
    l_max = 7
    L = (l_max + 1) ** 2
    rng = np.random.default_rng(5)
    pts = rng.standard_normal((200, 3))
    w = rng.standard_normal((200, L))
    Ys, dYs, _ = oracle.compute(pts, l_max, False, gradients=True)
    Yn, dYn, _ = oracle.compute(pts, l_max, True, gradients=True)
    # library contraction
    got = oracle.vjp(dYn, w.astype(LD), l_max)
    want = np.einsum("nak,nk->na", dYn, w.astype(LD))
    assert float(np.max(np.abs(got - want))) < 1e-17 * L
    # operand order / transposition: a one-hot upstream gradient picks out one column of dsph
    onehot = np.zeros((200, L), LD)
    onehot[:, 11] = 1
    assert np.array_equal(oracle.vjp(dYn, onehot, l_max), dYn[:, :, 11])
    # closed form 1: grad_sph = sph on the unit sphere -> (1/2) grad sum_k Y_k^2 = 0 (addition theorem)
    z = oracle.vjp(dYn, Yn, l_max)
    assert float(np.max(np.abs(z))) < 1e-15
    # closed form 2 (solid): (1/2) grad sum_l r^(2l)(2l+1)/4pi = sum_l l(2l+1)/(4pi) r^(2l-2) x
    g = oracle.vjp(dYs, Ys, l_max)
    x = pts.astype(LD)
    r2 = (x ** 2).sum(axis=1)
    pi = LD("3.14159265358979323846264338327950288")
    fac = sum(l * LD(2 * l + 1) / (4 * pi) * r2 ** (l - 1) for l in range(1, l_max + 1))
    want = fac[:, None] * x
    assert float(np.max(np.abs(g - want) / np.abs(want).max(axis=1, keepdims=True))) < 1e-15
    # Euler: x . vjp(solid dsph, w) = sum_k l_k w_k Y_k
    g = oracle.vjp(dYs, w.astype(LD), l_max)
    lk = np.concatenate([[l] * (2 * l + 1) for l in range(l_max + 1)]).astype(LD)
    lhs = (x * g).sum(axis=1)
    rhs = (lk * w.astype(LD) * Ys).sum(axis=1)
    assert float(np.max(np.abs(lhs - rhs) / (np.abs(rhs) + 1))) < 1e-15


@pytest.mark.parametrize("normalized", [False, True])
def test_vjp_recompute_is_gradient_of_weighted_sum(oracle, normalized):
    """N1 pin: vjp_recompute(x, w) is the Cartesian gradient of the scalar f(x) = sum_k w_k Y_k(x);
    checked against 4th-order central differences of f built from the oracle's VALUES only
    (the gradients under test never enter the reference), poles included."""
    l_max = 12
    L = (l_max + 1) ** 2
    pts = random_points(40, 11)
    pts = np.concatenate([pts, [[0, 0, 1.5], [0, 0, -0.75]]])
    rng = np.random.default_rng(12)
    w = rng.standard_normal((len(pts), L)).astype(LD)
    got = oracle.vjp_recompute(pts, w, l_max, normalized)
    assert got.shape == (len(pts), 3) and got.dtype == LD
    h = 2.0 ** -22
    f = lambda x: (oracle.compute(x, l_max, normalized)[0] * w).sum(axis=1)
    r = np.linalg.norm(pts, axis=1)
    # scale of one term of the sum: |w| * row scale * l / r (times r^l for solid harmonics)
    scale = np.zeros(len(pts), LD)
    for l in range(l_max + 1):
        rho = r ** l if not normalized else np.ones_like(r)
        scale += row_scale(l) * rho * max(l, 1) / r * np.abs(w[:, l * l:(l + 1) ** 2]).max(axis=1)
    for a in range(3):
        e = np.zeros(3)
        e[a] = h
        fd = (8 * (f(pts + e) - f(pts - e)) - (f(pts + 2 * e) - f(pts - 2 * e))) / (12 * LD(h))
        assert float(np.max(np.abs(fd - got[:, a]) / scale)) < 1e-11, a
    # and it is exactly the two-step route
    _, d, _ = oracle.compute(pts, l_max, normalized, gradients=True)
    assert np.array_equal(got, oracle.vjp(d, w, l_max))


@pytest.mark.parametrize("normalized", [False, True])
def test_vjp2_is_the_backward_of_the_backward(oracle, normalized):
    """N4 pin (double backward): with f(x, w) = sum_a v_a * vjp_recompute(x, w)[a],
    vjp2's out_xyz is the Cartesian gradient of f in x -- checked against 4th-order central
    differences of oracle.vjp_recompute (the Hessians under test never enter the reference) --
    and out_w is its gradient in w, which by linearity in w is f evaluated at one-hot w."""
    l_max = 10
    L = (l_max + 1) ** 2
    pts = random_points(30, 21)
    pts = np.concatenate([pts, [[0, 0, 1.25], [0, 0, -0.5]]])
    rng = np.random.default_rng(22)
    w = rng.standard_normal((len(pts), L)).astype(LD)
    v = rng.standard_normal((len(pts), 3)).astype(LD)
    out_xyz, out_w = oracle.vjp2(pts, w, v, l_max, normalized)
    assert out_xyz.shape == (len(pts), 3) and out_w.shape == (len(pts), L) and out_xyz.dtype == LD
    f = lambda x: (oracle.vjp_recompute(x, w, l_max, normalized) * v).sum(axis=1)
    h = 2.0 ** -22
    r = np.linalg.norm(pts, axis=1)
    scale = np.zeros(len(pts), LD)
    for l in range(l_max + 1):
        rho = r ** l if not normalized else np.ones_like(r)
        scale += row_scale(l) * rho * (max(l, 1) / r) ** 2 * np.abs(w[:, l * l:(l + 1) ** 2]).max(axis=1)
    scale *= np.abs(v).max(axis=1)
    for b in range(3):
        e = np.zeros(3)
        e[b] = h
        fd = (8 * (f(pts + e) - f(pts - e)) - (f(pts + 2 * e) - f(pts - 2 * e))) / (12 * LD(h))
        assert float(np.max(np.abs(fd - out_xyz[:, b]) / scale)) < 1e-10, b
    for k in (0, 1, 3, 17, L - 1):
        onehot = np.zeros((len(pts), L), LD)
        onehot[:, k] = 1
        fk = (oracle.vjp_recompute(pts, onehot, l_max, normalized) * v).sum(axis=1)
        assert np.max(np.abs(fk - out_w[:, k])) <= 8 * EPS_LD * np.max(np.abs(fk) + 1)
    # symmetric Hessians: swapping the roles of v's axis and the output axis gives the same contraction
    _, _, H = oracle.compute(pts, l_max, normalized, True, True)
    alt = np.einsum("nbak,na,nk->nb", H, v, w)
    assert float(np.max(np.abs(alt - out_xyz) / scale[:, None])) < 1e-15


def test_conventions_closed_forms_and_row_norms(oracle):
    """N4 pin (conventions): with the e3nn axes the l = 1 row is proportional to (x, y, z) in
    that order; 'integral' rows have norm^2 (2l+1)/4pi, 'component' 2l+1, 'norm' 1 on the unit
    sphere; gradients against finite differences of the converted values; the standard axes with
    the integral scale are `compute` itself."""
    l_max = 9
    pts = random_points(25, 31)
    r = np.sqrt((pts.astype(LD) ** 2).sum(axis=1))
    u = pts.astype(LD) / r[:, None]
    want_norm2 = {oracle.SCALE_INTEGRAL: lambda l: (2 * l + 1) / (16 * np.arctan(LD(1))), oracle.SCALE_COMPONENT: lambda l: LD(2 * l + 1),
                  oracle.SCALE_NORM: lambda l: LD(1)}
    for scale, norm2 in want_norm2.items():
        y, g, H = oracle.compute_convention(pts, l_max, True, oracle.AXES_E3NN, scale, True, True)
        c1 = np.sqrt(norm2(1))                       # |Y_1|^2 = norm2 and Y_1 = c1 * (x, y, z)/r
        assert np.max(np.abs(y[:, 1:4] - c1 * u)) < 8 * EPS_LD * float(c1)
        for l in range(l_max + 1):
            n2 = (y[:, l * l:(l + 1) ** 2] ** 2).sum(axis=1)
            assert np.max(np.abs(n2 / norm2(l) - 1)) < 64 * (l + 1) * EPS_LD
        h = 2.0 ** -22
        val = lambda x: oracle.compute_convention(x, l_max, True, oracle.AXES_E3NN, scale, True)
        for a in range(3):
            e = np.zeros(3)
            e[a] = h
            (yp1, gp1, _), (ym1, gm1, _), (yp2, gp2, _), (ym2, gm2, _) = (val(pts + e), val(pts - e), val(pts + 2 * e),
                                                                            val(pts - 2 * e))
            fd_g = (8 * (yp1 - ym1) - (yp2 - ym2)) / (12 * LD(h))
            fd_H = (8 * (gp1 - gm1) - (gp2 - gm2)) / (12 * LD(h))
            for l in range(l_max + 1):
                sl = slice(l * l, (l + 1) ** 2)
                S = np.sqrt(norm2(l))
                assert float(np.max(np.abs(fd_g[:, sl] - g[:, a, sl]) / (S * max(l, 1) / r)[:, None])) < 1e-11
                assert float(np.max(np.abs(fd_H[:, :, sl] - H[:, :, a, sl]) / (S * (max(l, 1) / r) ** 2)[:, None, None])) < 1e-11
    # solid harmonics, e3nn axes: l = 1 row is c1 * (x, y, z) itself
    y, _, _ = oracle.compute_convention(pts, 2, False, oracle.AXES_E3NN, oracle.SCALE_COMPONENT)
    assert np.max(np.abs(y[:, 1:4] - np.sqrt(LD(3)) * pts.astype(LD))) < 16 * EPS_LD * 4
    # the paper's own convention is untouched
    a = oracle.compute_convention(pts, l_max, True, oracle.AXES_STANDARD, oracle.SCALE_INTEGRAL, True, True)
    b = oracle.compute(pts, l_max, True, True, True)
    assert all(np.array_equal(x, z) for x, z in zip(a, b))


def test_expand_eq1(oracle):
    """N2 pins for the density expansion of Eq. 1: one-point segments, brute force, order
    independence, parity of antipodal pairs, rotation invariance of the power spectrum."""
    l_max, n_rad = 6, 3
    L = (l_max + 1) ** 2
    rng = np.random.default_rng(21)
    pts = rng.standard_normal((37, 3))
    rad = rng.standard_normal((37, n_rad, l_max + 1))
    Y = oracle.compute(pts, l_max, True)[0]
    l_of = np.concatenate([[l] * (2 * l + 1) for l in range(l_max + 1)])
    # (1) one point per segment: c = R_nl Y_lm, nothing summed
    c1 = oracle.expand(pts, rad, np.arange(38), l_max)
    assert c1.shape == (37, n_rad, L)
    for k in (0, 5, 36):
        for n in range(n_rad):
            assert np.array_equal(c1[k, n], rad[k, n].astype(LD)[l_of] * Y[k])
    # (2) brute force with python scalars over ragged segments, one of them empty
    seg = np.array([0, 4, 4, 20, 37])
    c = oracle.expand(pts, rad, seg, l_max)
    assert np.all(c[1] == 0)
    for s_, n, lm in ((0, 0, 0), (2, 1, 17), (3, 2, L - 1), (2, 0, 30)):
        want = LD(0)
        for k in range(seg[s_], seg[s_ + 1]):
            want += LD(rad[k, n, l_of[lm]]) * Y[k, lm]
        assert abs(c[s_, n, lm] - want) <= 1e-17 * 37
    # (3) the sum does not depend on the order of the points (to rounding)
    perm = rng.permutation(37)
    cp = oracle.expand(pts[perm], rad[perm], np.array([0, 37]), l_max)
    ca = oracle.expand(pts, rad, np.array([0, 37]), l_max)
    assert float(np.max(np.abs(cp - ca))) < 1e-16 * 37
    # (4) antipodal pair with equal radial values: odd l cancel, even l double (P9: Y(-x) = (-1)^l Y(x))
    pair = np.stack([pts[3], -pts[3]])
    c2 = oracle.expand(pair, np.stack([rad[3], rad[3]]), np.array([0, 2]), l_max)[0]
    odd = (l_of % 2) == 1
    assert float(np.max(np.abs(c2[:, odd]))) < 1e-17
    assert float(np.max(np.abs(c2[:, ~odd] - 2 * c1[3][:, ~odd]))) < 1e-17
    # (5) rotating every point leaves the power spectrum p_nl = sum_m c_nlm^2 unchanged (P4)
    Rm = _random_rotation(rng)
    cr = oracle.expand(pts @ Rm.T, rad, np.array([0, 37]), l_max)[0]
    for l in range(l_max + 1):
        sl = slice(l * l, (l + 1) ** 2)
        p0 = (ca[0][:, sl] ** 2).sum(axis=1)
        p1 = (cr[:, sl] ** 2).sum(axis=1)
        assert float(np.max(np.abs(p0 - p1) / (np.abs(p0) + 1e-30))) < 1e-13, l


# --------------------------------------------------------------------------------------------
# edge cases of the oracle's interface
# --------------------------------------------------------------------------------------------
def test_edge_cases(oracle):
    # n = 0
    s, d, h = oracle.compute(np.zeros((0, 3)), 3, True, True, True)
    assert s.shape == (0, 16) and d.shape == (0, 3, 16) and h.shape == (0, 3, 3, 16)
    # l_max = 0
    s, d, _ = oracle.compute(random_points(5, 0), 0, True, True)
    assert np.allclose(s.astype(float), 1 / (2 * math.sqrt(math.pi))) and np.all(d == 0)
    # solid harmonics at the origin are well defined: Y_0^0 = 1/(2 sqrt(pi)), the rest 0
    s, d, _ = oracle.compute(np.zeros((1, 3)), 4, False, True)
    assert abs(float(s[0, 0]) - 1 / (2 * math.sqrt(math.pi))) < 1e-16 and np.all(s[0, 1:] == 0)
    # normalised at the origin is undefined: NaN for that point only (reading S5)
    s, _, _ = oracle.compute(np.array([[0, 0, 0], [1, 0, 0]], float), 2, True)
    assert np.all(np.isnan(s[0, 1:].astype(float))) and np.all(np.isfinite(s[1].astype(float)))
    # f32 inputs are widened exactly
    p32 = random_points(10, 8).astype(np.float32)
    a, _, _ = oracle.compute(p32, 5, True)
    b, _, _ = oracle.compute(p32.astype(np.float64), 5, True)
    assert np.array_equal(a, b)
