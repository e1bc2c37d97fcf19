"""Pins of the oracle's chi^2 (NEXT row f3; PAPER.md:76-81 eq. 6, :192-194; readings R23) -- CPU only."""
import numpy as np

import lens_inputs as li
import oracle

NONE = li.make_lenses(0)


def test_no_lens_single_constraints_chi2_is_exactly_zero():
    g = li.Grid(x0=-4.0, y0=-4.0, dx=0.5, nx=17, ny=17)
    rng = np.random.default_rng(0)
    pts = rng.uniform(-3.9, 3.9, (6, 2))
    c = li.make_constraints((k, pts[k, 0], pts[k, 1], 0.3) for k in range(6))
    r = oracle.chi2(NONE, g.x0, g.y0, g.dx, g.nx, g.ny, c, 6)
    assert r["chi2"] == 0.0 and r["nimages"] == 6
    assert np.allclose(r["sources"], pts, atol=1e-15) and np.allclose(r["predicted"], pts, atol=1e-14)


def test_no_lens_two_constraints_on_one_source_closed_form():
    """alpha = 0: the source is the midpoint m, its only image is m, so chi2 = sum |c_j - m|^2 / sigma_j^2."""
    g = li.Grid(x0=-4.0, y0=-4.0, dx=0.5, nx=17, ny=17)
    c = li.make_constraints([(0, 1.1, 0.3, 0.5), (0, -0.7, 1.9, 0.25), (1, 2.2, -2.3, 1.0)])
    r = oracle.chi2(NONE, g.x0, g.y0, g.dx, g.nx, g.ny, c, 2)
    m = np.array([0.2, 1.1])
    want = ((1.1 - m[0]) ** 2 + (0.3 - m[1]) ** 2) / 0.25 + ((-0.7 - m[0]) ** 2 + (1.9 - m[1]) ** 2) / 0.0625
    assert abs(r["chi2"] - want) < 1e-13 * want
    assert np.allclose(r["sources"], [m, [2.2, -2.3]], atol=1e-15)
    assert np.allclose(r["predicted"], [m, m, [2.2, -2.3]], atol=1e-14)


def test_sis_true_images_give_chi2_of_fourth_order_in_dx():
    """SIS, source at distance s < b0 on a ray: the two images are at b0 + s and -(b0 - s).  With the exact images as
    constraints the source is recovered and the predicted images differ from the constraints only by the
    linear-interpolation error O(dx^2): chi2 = O(dx^4).  The ORDER is pinned: chi2 averaged over 12 source positions
    (radius and angle drawn once, seeded -- the images then fall at different places inside their cells, which is what
    makes a single position fluctuate around the asymptotic law) is fitted against dx over three grids, each twice
    as fine as the last; the fitted exponent must be >= 3.5 (4 asymptotically)."""
    b0 = 2.0
    L = li.lens(li.SIS, 0.0, 0.0, 0, 0, 0, 0, b0)
    rng = np.random.default_rng(7)
    cases = [(rng.uniform(0.3, 1.2), rng.uniform(0.0, 2.0 * np.pi)) for _ in range(12)]
    dxs, means = [], []
    for n in (121, 241, 481):
        g = li.centred_grid(6.0, n)
        vals = []
        for s, phi in cases:
            u = np.array([np.cos(phi), np.sin(phi)])
            c = li.make_constraints([(0, *((b0 + s) * u), 0.1), (0, *(-(b0 - s) * u), 0.1)])
            r = oracle.chi2(L, g.x0, g.y0, g.dx, g.nx, g.ny, c, 1)
            assert np.allclose(r["sources"][0], s * u, atol=1e-14)
            assert np.all(np.hypot(*(r["predicted"] - np.column_stack([c["x"], c["y"]])).T) < g.dx ** 2)
            vals.append(r["chi2"])
        dxs.append(g.dx)
        means.append(np.mean(vals))
    assert means[0] < 1e-3
    order = np.polyfit(np.log(dxs), np.log(means), 1)[0]
    assert order >= 3.5, (order, means)


def test_wrong_model_costs_more_and_missing_image_is_infinite():
    b0, s, phi = 2.0, 0.7, 0.4
    u = np.array([np.cos(phi), np.sin(phi)])
    c = li.make_constraints([(0, *((b0 + s) * u), 0.1), (0, *(-(b0 - s) * u), 0.1)])
    g = li.centred_grid(6.0, 121)
    good = oracle.chi2(li.lens(li.SIS, 0.0, 0.0, 0, 0, 0, 0, b0), g.x0, g.y0, g.dx, g.nx, g.ny, c, 1)["chi2"]
    bad = oracle.chi2(li.lens(li.SIS, 0.1, 0.0, 0, 0, 0, 0, 1.1 * b0), g.x0, g.y0, g.dx, g.nx, g.ny, c, 1)["chi2"]
    assert bad > 100 * good
    far = li.make_constraints([(0, 50.0, 50.0, 0.1)])  # its source (and image) lie outside the grid
    assert oracle.chi2(NONE, g.x0, g.y0, g.dx, g.nx, g.ny, far, 1)["chi2"] == np.inf
    # a source without constraints is ignored
    r = oracle.chi2(NONE, g.x0, g.y0, g.dx, g.nx, g.ny, li.make_constraints([(1, 0.3, 0.2, 1.0)]), 3)
    assert r["chi2"] == 0.0 and r["nimages"] == 1 and np.isnan(r["sources"][0]).all()
