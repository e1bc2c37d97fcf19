"""Pins of the oracle's source-plane map and brute-force delensing (NEXT row f1; PAPER.md:39 eq. 1, :87-91, :194;
readings R22) against what the lens equation fixes -- CPU only."""
import numpy as np

import lens_inputs as li
import oracle


def _alpha(L, g):
    m = oracle.grid(L, g.x0, g.y0, g.dx, g.nx, g.ny, planes=("ax", "ay"))
    return m["ax"], m["ay"]


def test_no_lens_every_source_is_its_own_single_image():
    g = li.Grid(x0=-4.0, y0=-3.0, dx=0.5, nx=17, ny=13)
    z = np.zeros((g.ny, g.nx))
    rng = np.random.default_rng(0)
    src = np.column_stack([rng.uniform(-3.9, 3.9, 50), rng.uniform(-2.9, 2.9, 50)])
    src = np.vstack([src, [[100.0, 0.0]]])  # outside the grid: no image
    im, found = oracle.delens(z, z, g.x0, g.y0, g.dx, src)
    assert found == 50 and sorted(im["source"]) == list(range(50))
    for r in im:
        assert abs(r["x"] - src[r["source"], 0]) < 1e-14 and abs(r["y"] - src[r["source"], 1]) < 1e-14
        i, j = int((r["x"] - g.x0) // g.dx), int((r["y"] - g.y0) // g.dx)
        assert r["triangle"] // 2 == j * (g.nx - 1) + i  # the cell that holds the source
        fx, fy = (r["x"] - g.x0) / g.dx - i, (r["y"] - g.y0) / g.dx - j
        assert r["triangle"] % 2 == (1 if fx + fy > 1.0 else 0)  # cut along V10-V01


def test_source_plane_of_an_sis_is_radial_shrink_by_b0():
    """SIS: alpha = b0 R-hat, so beta = (R - b0) R-hat: |beta| = |R - b0| at every pixel."""
    g = li.Grid(x0=-5.25, y0=-5.25, dx=0.5, nx=22, ny=22)
    L = li.lens(li.SIS, 0.0, 0.0, 0, 0, 0, 0, 1.7)
    ax, ay = _alpha(L, g)
    bx, by = oracle.source_plane(ax, ay, g.x0, g.y0, g.dx)
    X, Y = np.meshgrid(g.xs(), g.ys())
    R = np.hypot(X, Y)
    assert np.allclose(np.hypot(bx, by), np.abs(R - 1.7), rtol=1e-13, atol=1e-14)
    assert np.allclose(bx * Y, by * X, atol=1e-12)  # beta stays on the ray through the centre


def test_images_solve_the_lens_equation_to_second_order_in_dx_and_come_in_odd_numbers():
    """Non-singular lens (NSIE + dPIE): each found image theta satisfies theta - alpha(theta) = beta up to the
    linear-interpolation error O(dx^2 |H'|), which must shrink ~4x when dx halves; a smooth lens gives an odd
    number of images of every source (odd-number theorem) as long as the grid covers them all."""
    L = li.make_lenses(2)
    L[0] = (li.NSIE, 0, 0.2, -0.1, 0.3, 0.5, 1.0, 0.0, 4.0)
    L[1] = (li.DPIE, 0, 3.0, 2.0, 0.2, 1.0, 1.0, 15.0, 1.2)
    src = np.array([[0.3, 0.1], [-0.5, 0.4], [2.0, 1.5], [6.0, -5.0], [0.05, -0.02]])
    worst = []
    for n in (161, 321):
        g = li.centred_grid(12.0, n)
        ax, ay = _alpha(L, g)
        im, found = oracle.delens(ax, ay, g.x0, g.y0, g.dx, src)
        assert found == len(im)
        counts = np.bincount(im["source"], minlength=len(src))
        assert np.all(counts % 2 == 1), counts
        assert counts.max() >= 3  # some source is multiply imaged
        res = []
        for r in im:
            p = oracle.point(L, r["x"], r["y"])
            res.append(np.hypot(r["x"] - p["ax"] - src[r["source"], 0], r["y"] - p["ay"] - src[r["source"], 1]))
        worst.append(max(res))
    assert worst[0] < 0.05 and worst[1] < worst[0] / 2.5, worst


def test_sis_two_images_at_known_radii():
    """SIS, source at distance s < b0 from the centre: images on the source's ray at R = b0 + s and, on the
    opposite side, R = b0 - s (plus whatever the cells touching the singular centre produce, excluded here)."""
    b0, s = 2.0, 0.7
    g = li.centred_grid(6.0, 241)
    L = li.lens(li.SIS, 0.0, 0.0, 0, 0, 0, 0, b0)
    ax, ay = _alpha(L, g)
    phi = 0.4
    im, _ = oracle.delens(ax, ay, g.x0, g.y0, g.dx, [[s * np.cos(phi), s * np.sin(phi)]])
    far = im[np.hypot(im["x"], im["y"]) > 3 * g.dx]
    assert len(far) == 2
    r = np.sort(np.hypot(far["x"], far["y"]))
    assert abs(r[0] - (b0 - s)) < g.dx ** 2 and abs(r[1] - (b0 + s)) < g.dx ** 2
    ang = np.arctan2(far["y"], far["x"])
    assert np.allclose(np.sort(np.mod(ang - phi, 2 * np.pi)), [0.0, np.pi], atol=5e-3) or \
        np.allclose(np.sort(np.mod(ang - phi + 1e-3, 2 * np.pi)), [1e-3, np.pi + 1e-3], atol=5e-3)


def test_max_images_truncates_but_counts_everything():
    g = li.Grid(x0=0.0, y0=0.0, dx=1.0, nx=9, ny=9)
    z = np.zeros((g.ny, g.nx))
    src = np.column_stack([np.linspace(0.3, 7.3, 8), np.full(8, 0.4)])
    im, found = oracle.delens(z, z, g.x0, g.y0, g.dx, src, max_images=3)
    assert found == 8 and len(im) == 3
