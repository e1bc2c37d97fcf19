"""Pins of the CPU oracle against things OTHER than itself (CPU only, -m "not gpu").

Each test names what it pins and the passage it comes from.  PAPER.md is
/root/reference/PAPER.md; "reading 8c-N" is SURVEY.md sec. 8(c) row N (restated in
DESIGN.md sec. 3).  The paper prints neither the potentials nor a worked example,
so the pins are: the Poisson integral that DEFINES alpha from kappa (eq. 2), an
independent arbitrary-precision evaluation of a different closed form
(complex-log, Appendix A.5), textbook special cases, and invariants.
"""
import math
import os

import mpmath as mp
import numpy as np
import pytest
from scipy import integrate

import lens_inputs as li
import oracle

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "appendix_b.txt")


# ----------------------------------------------------------------------------- helpers
def eps_of(ehat):
    return ehat / (1.0 + math.sqrt(1.0 - ehat * ehat))


def kappa_piemd_def(X, Y, x, y, ehat, theta, r, b0):
    """Reading 8c-1: kappa = b0 / (2 sqrt(r^2 + rho^2)), rho^2 = x'^2/(1+eps)^2 + y'^2/(1-eps)^2."""
    e = eps_of(ehat)
    c, s = math.cos(theta), math.sin(theta)
    dx, dy = X - x, Y - y
    xp, yp = c * dx + s * dy, -s * dx + c * dy
    rho2 = xp * xp / (1 + e) ** 2 + yp * yp / (1 - e) ** 2
    return 0.5 * b0 / math.sqrt(r * r + rho2)


def kappa_dpie_def(X, Y, x, y, ehat, theta, rc, rt, b0):
    return rt / (rt - rc) * (kappa_piemd_def(X, Y, x, y, ehat, theta, rc, b0)
                             - kappa_piemd_def(X, Y, x, y, ehat, theta, rt, b0))


def read_golden():
    lenses, pts, eps, single, pair = [], [], [], None, None
    for line in open(GOLDEN):
        line = line.split("#")[0].split()
        if not line:
            continue
        tag, v = line[0], [float(t) for t in line[1:]]
        if tag == "lens":
            lenses.append(v)
        elif tag == "eps":
            eps.append(v)
        elif tag == "point":
            pts.append(v)
        elif tag == "single0":
            single = v
        elif tag == "pair01":
            pair = v
    L = li.make_lenses(len(lenses))
    for k, v in enumerate(lenses):
        L[k] = (int(v[0]), 0, *v[1:])
    return L, pts, eps, single, pair


def rel(a, b):
    return abs(a - b) / max(abs(b), 1e-300)


# ----------------------------------------------------------------------------- Appendix B
def test_appendix_b_golden():
    """Whole pipeline, all conventions at once: SURVEY Appendix B, 1e-14 relative."""
    L, pts, eps, single, pair = read_golden()
    for eh, e in eps:
        assert rel(oracle.eps_from_ehat(eh), e) < 1e-15
    names = ("ax", "ay", "a11", "a12", "a22", "kappa", "gamma1", "gamma2")
    for row in pts:
        X, Y = row[0], row[1]
        r = oracle.point(L, X, Y)
        for n, g in zip(names, row[2:10]):
            assert rel(r[n], g) < 1e-14, (X, Y, n, r[n], g)
        assert rel(1.0 / r["mu"], row[10]) < 3e-14, (X, Y, "invmu")
        # mu itself: conditioned (reading 8c-13): C = ((1-k)^2 + g^2) |mu|
        Cn = ((1 - row[7]) ** 2 + row[8] ** 2 + row[9] ** 2) * abs(row[11])
        assert rel(r["mu"], row[11]) < 1e-14 * max(1.0, Cn)
    d = oracle.lens_deriv(L[:1], single[0], single[1])
    for n, g in zip(("ax", "ay", "a11", "a12", "a22"), single[2:]):
        assert rel(d[n], g) < 1e-14
    r = oracle.point(L[:2], pair[0], pair[1])
    assert rel(r["ax"], pair[2]) < 1e-14 and rel(r["ay"], pair[3]) < 1e-14


# independent arbitrary-precision evaluation: complex-log form (Appendix A.5; Kassiola-Kovner style)
def _mp_piemd_I(xp, yp, eps, r):
    o = 1 - eps ** 2
    q = (1 - eps) / (1 + eps)
    se = 2 * mp.sqrt(eps)
    w = mp.sqrt(r ** 2 + xp ** 2 / (1 + eps) ** 2 + yp ** 2 / (1 - eps) ** 2)
    z = (q * xp + 1j * (se * w - yp / q)) / (xp + 1j * (se * r - yp))
    return -1j * o / se * mp.log(z)


def _mp_alpha(rec, X, Y):
    t = int(rec["type"])
    x, y, eh, th, rc, rt, b0 = (mp.mpf(float(rec[k])) for k in ("x", "y", "ellipticity", "theta", "rcore", "rcut", "b0"))
    dx, dy = X - x, Y - y
    if t == li.SIS:
        R = mp.sqrt(dx ** 2 + dy ** 2)
        return b0 * dx / R, b0 * dy / R
    eps = eh / (1 + mp.sqrt(1 - eh ** 2))
    c, s = mp.cos(th), mp.sin(th)
    xp, yp = c * dx + s * dy, -s * dx + c * dy
    if t == li.NSIE:
        I = b0 * _mp_piemd_I(xp, yp, eps, rc)
    else:
        I = b0 * rt / (rt - rc) * (_mp_piemd_I(xp, yp, eps, rc) - _mp_piemd_I(xp, yp, eps, rt))
    jx, jy = mp.re(I), mp.im(I)
    return c * jx - s * jy, s * jx + c * jy


def _mp_sum_alpha(L, X, Y):
    ax = ay = mp.mpf(0)
    for rec in L:
        a, b = _mp_alpha(rec, X, Y)
        ax += a
        ay += b
    return ax, ay


def test_appendix_b_mpmath():
    """Golden values AND the oracle vs a 40-digit complex-log evaluation; Hessian by
    40-digit numerical differentiation of that alpha (independent of A.1's h_ij)."""
    L, pts, *_ = read_golden()
    with mp.workdps(40):
        for row in pts:
            X, Y = mp.mpf(row[0]), mp.mpf(row[1])
            ax, ay = _mp_sum_alpha(L, X, Y)
            a11 = mp.diff(lambda u: _mp_sum_alpha(L, u, Y)[0], X)
            a12 = mp.diff(lambda v: _mp_sum_alpha(L, X, v)[0], Y)
            a21 = mp.diff(lambda u: _mp_sum_alpha(L, u, Y)[1], X)
            a22 = mp.diff(lambda v: _mp_sum_alpha(L, X, v)[1], Y)
            assert abs(a12 - a21) < mp.mpf(10) ** -25  # a potential flow: curl-free
            o = oracle.point(L, row[0], row[1])
            for n, ref, gold in (("ax", ax, row[2]), ("ay", ay, row[3]), ("a11", a11, row[4]),
                                 ("a12", a12, row[5]), ("a22", a22, row[6])):
                assert rel(gold, float(ref)) < 2e-16 * 4, (n, "golden")
                assert rel(o[n], float(ref)) < 1e-14, (n, "oracle")


# ----------------------------------------------------------------------------- definition of alpha
@pytest.mark.parametrize("P", [(1.5, 0.8), (-2.0, 3.0)])
def test_poisson_integral_defines_alpha(P):
    """alpha = grad psi with psi the log-kernel integral of kappa (PAPER.md:43 eq. 2, :53):
    alpha(t) = -(1/pi) int_0^2pi int_0^inf kappa(t + r n) n dr dphi.  Pins the PIEMD/dPIE
    deflection formula, the kappa normalisation, the e-hat -> eps map and the angle convention."""
    par = (0.4, -0.3, 0.5, 0.7, 0.3, 7.0, 2.0)  # x y ehat theta rc rt b0 (rotated, elliptical)
    L = li.lens(li.DPIE, *par)
    dist = math.hypot(P[0] - par[0], P[1] - par[1])

    def inner(phi, comp):
        n = (math.cos(phi), math.sin(phi))
        f = lambda r: kappa_dpie_def(P[0] + r * n[0], P[1] + r * n[1], *par) * n[comp]
        q = lambda a, b: integrate.quad(f, a, b, epsabs=1e-13, epsrel=1e-13, limit=200)[0]
        return q(0, dist) + q(dist, 3 * dist + 50) + q(3 * dist + 50, np.inf)

    phi0 = math.atan2(par[1] - P[1], par[0] - P[0])
    got = [-integrate.quad(inner, phi0, phi0 + 2 * math.pi, args=(c,), epsabs=1e-12, epsrel=1e-12, limit=400)[0]
           / math.pi for c in (0, 1)]
    o = oracle.point(L, *P)
    assert abs(got[0] - o["ax"]) < 1e-10 and abs(got[1] - o["ay"]) < 1e-10


def test_trace_of_hessian_is_twice_kappa_definition():
    """kappa = (a11 + a22)/2 (eq. 7; reading 8c-5) against the profile DEFINITION."""
    rng = np.random.default_rng(11)
    for _ in range(200):
        par = (rng.uniform(-3, 3), rng.uniform(-3, 3), rng.uniform(0, 0.9), rng.uniform(0, math.pi),
               rng.uniform(0.05, 1.0), rng.uniform(2.0, 30.0), rng.uniform(0.1, 5))
        X, Y = rng.uniform(-10, 10, 2)
        d = oracle.point(li.lens(li.DPIE, *par), X, Y)
        assert rel(d["kappa"], kappa_dpie_def(X, Y, *par)) < 1e-13
        n = oracle.point(li.lens(li.NSIE, *par), X, Y)
        assert rel(n["kappa"], kappa_piemd_def(X, Y, par[0], par[1], par[2], par[3], par[4], par[6])) < 1e-13


def test_hessian_matches_finite_differences_and_is_symmetric():
    """Hessian = derivative of the oracle's own gradient (central FD), a12 from both routes."""
    c = li.config(2)  # mixed dPIE / NSIE / SIS
    L = c.lenses
    rng = np.random.default_rng(5)
    checked = 0
    while checked < 40:
        X, Y = rng.uniform(-90, 90, 2)
        # stay >= 5 rcore (and >= 0.5") from any centre so FD truncation is small
        if np.min(np.hypot(L["x"] - X, L["y"] - Y)) < 0.5:
            continue
        h = 1e-5
        f = lambda x, y: oracle.point(L, x, y)
        d = f(X, Y)
        a11 = (f(X + h, Y)["ax"] - f(X - h, Y)["ax"]) / (2 * h)
        a12a = (f(X, Y + h)["ax"] - f(X, Y - h)["ax"]) / (2 * h)
        a12b = (f(X + h, Y)["ay"] - f(X - h, Y)["ay"]) / (2 * h)
        a22 = (f(X, Y + h)["ay"] - f(X, Y - h)["ay"]) / (2 * h)
        scale = max(abs(d["a11"]), abs(d["a12"]), abs(d["a22"]))
        for got, ref in ((a11, d["a11"]), (a12a, d["a12"]), (a12b, d["a12"]), (a22, d["a22"])):
            assert abs(got - ref) < 2e-7 * scale + 1e-9
        checked += 1


# ----------------------------------------------------------------------------- closed forms
def test_circular_dpie_closed_form_and_printed_value():
    """north_star pin: e = 0 -> alpha = b0 rt/(rt-rc) [(sqrt(rc^2+R^2)-rc) - (sqrt(rt^2+R^2)-rt)]/R radially.
    Printed value (SURVEY 8c pins table): b0=2, rc=0.5, rt=10, R=3 -> |alpha| = 1.4744384254305682."""
    L = li.lens(li.DPIE, 0.0, 0.0, 0.0, 0.3, 0.5, 10.0, 2.0)
    for phi in np.linspace(0, 2 * math.pi, 13):
        d = oracle.point(L, 3 * math.cos(phi), 3 * math.sin(phi))
        assert rel(math.hypot(d["ax"], d["ay"]), 1.4744384254305682) < 2e-15
        assert abs(d["ax"] * math.sin(phi) - d["ay"] * math.cos(phi)) < 1e-15  # radial
    rng = np.random.default_rng(3)
    for _ in range(100):
        rc, rt, b0 = rng.uniform(0.01, 2), rng.uniform(3, 100), rng.uniform(0.1, 30)
        x, y = rng.uniform(-5, 5, 2)
        X, Y = rng.uniform(-20, 20, 2)
        R = math.hypot(X - x, Y - y)
        ref = b0 * rt / (rt - rc) * ((math.sqrt(rc * rc + R * R) - rc) - (math.sqrt(rt * rt + R * R) - rt)) / R
        d = oracle.point(li.lens(li.DPIE, x, y, 0.0, rng.uniform(0, 3), rc, rt, b0), X, Y)
        assert rel(d["ax"], ref * (X - x) / R) < 1e-13 and rel(d["ay"], ref * (Y - y) / R) < 1e-13


def test_sis_constant_deflection_and_kappa():
    """north_star pin: |alpha| = b0 at every R > 0; kappa = b0/(2R); zero at the centre (reading 8c-11)."""
    L = li.lens(li.SIS, 1.0, -2.0, 0.3, 1.0, 0.7, 9.0, 0.8)  # e, theta, rcore, rcut ignored
    rng = np.random.default_rng(0)
    for _ in range(100):
        X, Y = rng.uniform(-50, 50, 2)
        R = math.hypot(X - 1.0, Y + 2.0)
        d = oracle.point(L, X, Y)
        assert rel(math.hypot(d["ax"], d["ay"]), 0.8) < 1e-15
        assert rel(d["kappa"], 0.8 / (2 * R)) < 1e-14
        # SIS shear magnitude equals kappa
        assert rel(math.hypot(d["gamma1"], d["gamma2"]), d["kappa"]) < 1e-13
    d = oracle.point(L, 1.0, -2.0)
    assert all(d[k] == 0.0 for k in ("ax", "ay", "a11", "a12", "a22")) and d["mu"] == 1.0


def test_small_ellipticity_is_smooth():
    """Appendix A.2: e = 0 is the smooth limit; the elliptical result differs by O(eps)."""
    base = (0.3, 0.2, 0.0, 0.9, 0.2, 15.0, 1.5)
    d0 = oracle.point(li.lens(li.DPIE, *base), 2.0, -1.0)
    for eh in (1e-14, 1e-10, 1e-6):
        par = list(base)
        par[2] = eh
        d = oracle.point(li.lens(li.DPIE, *par), 2.0, -1.0)
        for n in ("ax", "ay", "a11", "a12", "a22"):
            assert abs(d[n] - d0[n]) < 3 * eh * max(abs(d0[n]), 1.0) + 1e-15


# ----------------------------------------------------------------------------- invariants
def test_linearity_under_superposition():
    """eq. 10 and sec. 2.4 (:112): eval(L1 u L2) = eval(L1) + eval(L2)."""
    c = li.config(2, scale=64)
    L = c.lenses
    g = c.grid
    cut = 211
    full = oracle.grid(L, g.x0, g.y0, g.dx, g.nx, g.ny, planes=("ax", "ay", "a11", "a12", "a22"))
    p1 = oracle.grid(L[:cut], g.x0, g.y0, g.dx, g.nx, g.ny, planes=("ax", "ay", "a11", "a12", "a22"))
    p2 = oracle.grid(L[cut:], g.x0, g.y0, g.dx, g.nx, g.ny, planes=("ax", "ay", "a11", "a12", "a22"))
    for n in full:
        assert np.max(np.abs(full[n] - (p1[n] + p2[n]))) < 1e-14 * np.max(np.abs(full[n]))


def test_epilogue_identities():
    """eq. 4-5, eq. 7-9 (:105-110) as read in 8c-5..7."""
    rng = np.random.default_rng(2)
    for _ in range(200):
        a11, a12, a22 = rng.uniform(-3, 3, 3)
        e = oracle.epilogue(a11, a12, a22)
        assert e["kappa"] == 0.5 * (a11 + a22)
        assert e["gamma1"] == 0.5 * (a11 - a22) and e["gamma2"] == a12
        Ainv = np.array([[1 - a11, -a12], [-a12, 1 - a22]])
        assert rel(1.0 / e["mu"], np.linalg.det(Ainv)) < 1e-12 + 1e-15 * abs(e["mu"])
        g = math.hypot(e["gamma1"], e["gamma2"])
        ev = np.sort(np.linalg.eigvalsh(Ainv))
        assert np.allclose(ev, sorted([1 - e["kappa"] - g, 1 - e["kappa"] + g]), rtol=0, atol=1e-14)
        # eq. 9 with the MINUS sign (reading 8c-7)
        assert rel(e["mu"] * ((1 - e["kappa"]) ** 2 - g * g), 1.0) < 1e-9 * max(1.0, abs(e["mu"]))
    assert oracle.epilogue(1.0, 0.0, 1.0)["mu"] == math.inf  # det = 0 exactly
    assert oracle.epilogue(0.0, 0.0, 0.0)["mu"] == 1.0


def test_rotation_covariance():
    """Rotating the lens angle by D and the pixel about the lens centre by D rotates alpha by R(D),
    H by R H R^T, leaves kappa, mu (reading 8c-3)."""
    rng = np.random.default_rng(9)
    for t in (li.DPIE, li.NSIE):
        for _ in range(50):
            x, y = rng.uniform(-5, 5, 2)
            eh, th, rc, rt, b0 = rng.uniform(0, 0.8), rng.uniform(0, 3), rng.uniform(0.05, 1), rng.uniform(3, 40), 1.3
            X, Y = rng.uniform(-20, 20, 2)
            D = rng.uniform(-3, 3)
            cD, sD = math.cos(D), math.sin(D)
            Xr = x + cD * (X - x) - sD * (Y - y)
            Yr = y + sD * (X - x) + cD * (Y - y)
            a = oracle.point(li.lens(t, x, y, eh, th, rc, rt, b0), X, Y)
            b = oracle.point(li.lens(t, x, y, eh, th + D, rc, rt, b0), Xr, Yr)
            tol = 2e-14
            assert abs(b["ax"] - (cD * a["ax"] - sD * a["ay"])) < tol * b0
            assert abs(b["ay"] - (sD * a["ax"] + cD * a["ay"])) < tol * b0
            R = np.array([[cD, -sD], [sD, cD]])
            Ha = np.array([[a["a11"], a["a12"]], [a["a12"], a["a22"]]])
            Hb = np.array([[b["a11"], b["a12"]], [b["a12"], b["a22"]]])
            assert np.max(np.abs(Hb - R @ Ha @ R.T)) < tol * max(1.0, np.max(np.abs(Ha)))
            assert abs(a["kappa"] - b["kappa"]) < tol * max(1.0, abs(a["kappa"]))


def test_major_axis_direction():
    """theta is the MAJOR axis (reading 8c-3): kappa falls off more slowly along it."""
    L = li.lens(li.NSIE, 0, 0, 0.5, 0.4, 0.1, 0, 1.0)
    along = oracle.point(L, 3 * math.cos(0.4), 3 * math.sin(0.4))["kappa"]
    across = oracle.point(L, -3 * math.sin(0.4), 3 * math.cos(0.4))["kappa"]
    e = eps_of(0.5)
    assert rel(along / across, (1 + e) / (1 - e)) < 1e-2  # rho ratio for R >> rc
    assert along > across


def test_limits_between_types():
    """dPIE(rt -> inf) -> NSIE; NSIE(rc -> 0, e = 0) -> SIS; far field |alpha| R -> (1-eps^2) b0 rt."""
    rng = np.random.default_rng(4)
    for _ in range(30):
        x, y, eh, th, rc, b0 = rng.uniform(-2, 2), rng.uniform(-2, 2), rng.uniform(0, 0.7), rng.uniform(0, 3), \
            rng.uniform(0.05, 1), rng.uniform(0.2, 3)
        X, Y = rng.uniform(-10, 10, 2)
        a = oracle.point(li.lens(li.DPIE, x, y, eh, th, rc, 1e12, b0), X, Y)
        b = oracle.point(li.lens(li.NSIE, x, y, eh, th, rc, 0.0, b0), X, Y)
        # the hessian is exact to 1e-10; the deflection of an NSIE is defined up to the
        # (divergent) constant the cut removes: J(rt) -> ~ direction-independent only in H
        for n in ("a11", "a12", "a22"):
            assert abs(a[n] - b[n]) < 1e-10 * max(1.0, abs(b[n]))
        s1 = oracle.point(li.lens(li.NSIE, x, y, 0.0, th, 1e-9, 0.0, b0), X, Y)
        s2 = oracle.point(li.lens(li.SIS, x, y, 0.0, 0.0, 0.0, 0.0, b0), X, Y)
        for n in ("ax", "ay", "a11", "a12", "a22"):
            assert abs(s1[n] - s2[n]) < 1e-8 * max(1.0, abs(s2[n]))
    eh, rt, b0 = 0.5, 7.0, 2.0
    e = eps_of(eh)
    for phi in (0.0, 0.7, 1.9, 4.0):
        Rr = 1e7
        d = oracle.point(li.lens(li.DPIE, 0, 0, eh, 0.3, 0.2, rt, b0), Rr * math.cos(phi), Rr * math.sin(phi))
        # finite total mass M = pi (1-eps^2) b0 rt  (minus the core: rt/(rt-rc) (rt - rc) = rt)
        assert rel(math.hypot(d["ax"], d["ay"]) * Rr, (1 - e * e) * b0 * rt) < 1e-6


def test_dpie_to_nsie_deflection_difference_is_curl_and_divergence_free():
    """(the part of the previous limit the Hessian test cannot see) dPIE(rt=1e9) - NSIE deflection
    varies by < 1e-7 relative across a 20" field: the cut only removes a near-constant."""
    par = (0.3, -0.4, 0.4, 1.1, 0.2)
    vals = []
    for X, Y in [(-10, -10), (10, -10), (10, 10), (-10, 10), (0, 0)]:
        a = oracle.point(li.lens(li.DPIE, *par, 1e9, 1.0), X, Y)
        b = oracle.point(li.lens(li.NSIE, *par, 0.0, 1.0), X, Y)
        vals.append((a["ax"] - b["ax"], a["ay"] - b["ay"]))
    vals = np.array(vals)
    assert np.max(np.abs(vals - vals[0])) < 1e-7


def test_r20_oracle_vs_40_digits_at_extreme_ellipticity():
    """Reading R20 (tests/parity.py::conditioned_rel), pinned: as e-hat -> 1 the closed form loses
    digits in ANY double-precision evaluation (one rounding of the atanh argument moves the result by 2^-53/q^2), so
    the north-star 1e-11 cannot be asked of GPU-vs-oracle beyond some ellipticity -- the oracle itself is no longer
    that close to the true value.  Measured here on the three-lens model and grid of
    tests/test_gpu_parity.py::test_ellipticity_range against the 40-digit complex-log form, under the same
    per-element rule the parity tests use (max(rel |ref|, rel/1e-11 * 1e-13 max|ref|)):
      e-hat = 0.9992 (q = 0.02): the oracle's alpha is INSIDE the plain 1e-11 rule (worst 0.40 of it);
      e-hat = 0.9999 (q = 0.007): OUTSIDE the plain rule (worst 4.7 x) and inside conditioned_rel (worst 0.66).
    Pixels: all of rows 36-56 (the band through the lens centres, where the worst cases sit) and every 7th elsewhere."""
    from parity import FLOOR, REL, conditioned_rel

    old = mp.mp.dps
    mp.mp.dps = 40
    try:
        g = li.Grid(x0=-15.0, y0=-15.0, dx=0.31, nx=97, ny=97)
        pix = [(j, i) for j in range(g.ny) for i in range(g.nx) if 36 <= j <= 56 or (i % 7 == 0 and j % 7 == 0)]
        worst = {}
        for ehat in (0.9992, 0.9999):
            L = li.make_lenses(3)
            L[0] = (li.DPIE, 0, 0.3, -0.2, ehat, 0.7, 0.08, 30.0, 1.7)
            L[1] = (li.NSIE, 0, -4.0, 2.0, ehat, 2.4, 0.3, 0.0, 0.6)
            L[2] = (li.DPIE, 0, 5.0, 5.0, ehat, 1.1, 2.0, 900.0, 9.0)
            ref = oracle.grid(L, g.x0, g.y0, g.dx, g.nx, g.ny, planes=("ax", "ay"))
            d = np.zeros((2, len(pix)))
            t = np.zeros((2, len(pix)))
            for k, (j, i) in enumerate(pix):
                X, Y = mp.mpf(float(g.x0 + i * g.dx)), mp.mpf(float(g.y0 + j * g.dx))  # the pixel as the oracle forms it
                tx, ty = _mp_sum_alpha(L, X, Y)
                d[0, k], d[1, k] = float(mp.mpf(float(ref["ax"][j, i])) - tx), float(mp.mpf(float(ref["ay"][j, i])) - ty)
                t[0, k], t[1, k] = float(tx), float(ty)
            for rel in (REL, conditioned_rel(ehat)):
                allowed = np.maximum(rel * np.abs(t), rel / REL * FLOOR * np.max(np.abs(t), axis=1, keepdims=True))
                worst[ehat, rel] = float(np.max(np.abs(d) / allowed))
    finally:
        mp.mp.dps = old
    assert conditioned_rel(0.9992) == REL  # the plain rule is what the parity tests apply up to here
    assert worst[0.9992, REL] <= 0.5, worst
    c = conditioned_rel(0.9999)
    assert 7.0e-11 < c < 7.2e-11
    assert worst[0.9999, REL] > 3.0, worst        # the plain rule is not reachable in double precision here
    assert worst[0.9999, c] <= 0.8, worst         # the conditioned one is, with room for the GPU's own roundings


# ----------------------------------------------------------------------------- brute force, tiny grid
def test_bruteforce_tiny_grid_complex_log():
    """north_star pin: brute-force agreement on a tiny grid -- config 0's lenses on a coarse grid,
    deflection from the 30-digit complex-log form, Hessian by 30-digit differentiation at a few pixels."""
    c = li.config(0, scale=8)  # 8 x 8 pixels, 10 dPIE lenses
    g = c.grid
    o = oracle.grid(c.lenses, g.x0, g.y0, g.dx, g.nx, g.ny)
    with mp.workdps(30):
        for j in range(g.ny):
            for i in range(g.nx):
                X, Y = mp.mpf(g.x0 + i * g.dx), mp.mpf(g.y0 + j * g.dx)
                ax, ay = _mp_sum_alpha(c.lenses, X, Y)
                assert abs(float(ax) - o["ax"][j, i]) < 1e-13 * max(1, abs(float(ax)))
                assert abs(float(ay) - o["ay"][j, i]) < 1e-13 * max(1, abs(float(ay)))
        for (i, j) in [(0, 0), (3, 5), (7, 2)]:
            X, Y = mp.mpf(g.x0 + i * g.dx), mp.mpf(g.y0 + j * g.dx)
            a11 = mp.diff(lambda u: _mp_sum_alpha(c.lenses, u, Y)[0], X)
            a12 = mp.diff(lambda v: _mp_sum_alpha(c.lenses, X, v)[0], Y)
            a22 = mp.diff(lambda v: _mp_sum_alpha(c.lenses, X, v)[1], Y)
            k, g1 = (a11 + a22) / 2, (a11 - a22) / 2
            mu = 1 / ((1 - k) ** 2 - g1 ** 2 - a12 ** 2)
            for n, ref in (("a11", a11), ("a12", a12), ("a22", a22), ("kappa", k), ("gamma1", g1),
                           ("gamma2", a12), ("mu", mu)):
                assert abs(float(ref) - o[n][j, i]) < 1e-12 * max(1.0, abs(float(ref))), n


# ----------------------------------------------------------------------------- grid plumbing
def test_grid_indexing_rows_and_threads():
    """Pixel (i, j) at (x0 + i dx, y0 + j dx), index j*nx + i (reading 8c-10); row slabs on
    threads give the one-thread result bit for bit; unrequested rows stay untouched."""
    c = li.config(0)
    g = li.Grid(x0=-3.0, y0=2.0, dx=0.25, nx=7, ny=5)
    full = oracle.grid(c.lenses, g.x0, g.y0, g.dx, g.nx, g.ny)
    for (i, j) in [(0, 0), (6, 0), (0, 4), (3, 2)]:
        p = oracle.point(c.lenses, g.x0 + i * g.dx, g.y0 + j * g.dx)
        for n in oracle.PLANES:
            assert full[n][j, i] == p[n]
    thr = oracle.grid(c.lenses, g.x0, g.y0, g.dx, g.nx, g.ny, threads=3)
    for n in oracle.PLANES:
        assert np.array_equal(full[n], thr[n])
    part = oracle.grid(c.lenses, g.x0, g.y0, g.dx, g.nx, g.ny, rows=(1, 3), planes=("ax",))
    assert np.array_equal(part["ax"][1:3], full["ax"][1:3]) and np.all(np.isnan(part["ax"][[0, 3, 4]]))
    xs, ys = np.meshgrid(g.xs(), g.ys())
    pts = oracle.points(c.lenses, xs, ys)
    for n in oracle.PLANES:
        assert np.array_equal(pts[n], full[n])


def test_empty_model():
    """nlens = 0: alpha = 0, Hessian = 0, kappa = gamma = 0, mu = 1."""
    o = oracle.grid(li.make_lenses(0), 0.0, 0.0, 1.0, 3, 2)
    for n in oracle.PLANES:
        assert np.all(o[n] == (1.0 if n == "mu" else 0.0))
