"""Pins of the oracle's source-plane map and brute-force delensing (NEXT row f1; PAPER.md:39 eq. 1, :87-91, :194;
readings R22) against what the lens equation fixes -- CPU only."""
import os

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
    linear-interpolation error O(dx^2 |H'|).  The ORDER is pinned: the mean residual over the images of 16 sources
    (their in-cell positions differ, which averages the position-in-cell factor out) is fitted against dx over three
    grids, each twice as fine as the last; the fitted exponent must be >= 1.8 (2 asymptotically).  A smooth lens
    gives an odd number of images of every source (odd-number theorem) as long as the grid covers them all."""
    L = li.make_lenses(2)
    L[0] = (li.NSIE, 0, 0.2, -0.1, 0.3, 0.5, 1.0, 0.0, 4.0)
    L[1] = (li.DPIE, 0, 3.0, 2.0, 0.2, 1.0, 1.0, 15.0, 1.2)
    rng = np.random.default_rng(3)
    src = np.vstack([[[0.3, 0.1], [-0.5, 0.4], [2.0, 1.5], [6.0, -5.0], [0.05, -0.02]], rng.uniform(-3.0, 3.0, (11, 2))])
    dxs, mean_res = [], []
    for n in (321, 641, 1281):
        g = li.centred_grid(12.0, n)
        m = oracle.grid(L, g.x0, g.y0, g.dx, g.nx, g.ny, planes=("ax", "ay"), threads=os.cpu_count() or 1)
        im, found = oracle.delens(m["ax"], m["ay"], g.x0, g.y0, g.dx, src)
        assert found == len(im)
        counts = np.bincount(im["source"], minlength=len(src))
        assert np.all(counts % 2 == 1), counts
        assert counts.max() >= 3  # some source is multiply imaged
        res = []
        for r in im:
            p = oracle.point(L, r["x"], r["y"])
            res.append(np.hypot(r["x"] - p["ax"] - src[r["source"], 0], r["y"] - p["ay"] - src[r["source"], 1]))
        assert max(res) < 0.3 * g.dx ** 2 * 4.0  # |H'| <~ b0 / rcore^2 = 4 here
        dxs.append(g.dx)
        mean_res.append(np.mean(res))
    order = np.polyfit(np.log(dxs), np.log(mean_res), 1)[0]
    assert order >= 1.8, (order, mean_res)


def test_closed_triangle_rule_on_shared_edges_and_vertices():
    """R22: the triangles are CLOSED -- with no lens, a source exactly on an edge shared by two triangles is reported
    by both, a source exactly on an interior grid vertex by the six triangles that meet there (the cut runs along
    V10-V01, so a vertex touches 1 + 2 + 1 + 2 triangles of its four cells), a source on the outer boundary edge by
    one, and a source on a grid corner by the triangles of the one cell that has it.  Every reported image is the
    source position itself."""
    g = li.Grid(x0=-2.0, y0=-1.0, dx=0.5, nx=9, ny=7)  # dyadic: the coordinates below are exact
    z = np.zeros((g.ny, g.nx))

    def tri(src):
        im, found = oracle.delens(z, z, g.x0, g.y0, g.dx, [src])
        assert found == len(im)
        assert np.all(im["x"] == src[0]) and np.all(im["y"] == src[1])
        return sorted(int(t) for t in im["triangle"])

    ncx = g.nx - 1
    cell = lambda i, j: 2 * (j * ncx + i)
    # strictly inside triangle 0 / triangle 1 of cell (3, 2)
    assert tri((-0.4, 0.1)) == [cell(3, 2)]
    assert tri((-0.1, 0.4)) == [cell(3, 2) + 1]
    # on the diagonal V10-V01 of cell (3, 2): both triangles of that cell
    assert tri((-0.25, 0.25)) == [cell(3, 2), cell(3, 2) + 1]
    # on the vertical edge x = -0.5 between cells (2, 2) and (3, 2), away from the vertices
    assert tri((-0.5, 0.125)) == sorted([cell(2, 2) + 1, cell(3, 2)])
    # on the horizontal edge y = 0 between cells (3, 1) and (3, 2)
    assert tri((-0.375, 0.0)) == sorted([cell(3, 1) + 1, cell(3, 2)])
    # exactly on the interior vertex (i, j) = (3, 2) at (-0.5, 0): six triangles
    got = tri((-0.5, 0.0))
    want = sorted([cell(2, 1) + 1, cell(3, 1), cell(3, 1) + 1, cell(2, 2), cell(2, 2) + 1, cell(3, 2)])
    assert got == want and len(got) == 6
    # on the outer boundary (left edge, between vertices): one triangle; on the corner V00 of the grid: one;
    # on the opposite corner of the grid (V11 of the last cell): one
    assert tri((-2.0, 0.125)) == [cell(0, 2)]
    assert tri((-2.0, -1.0)) == [cell(0, 0)]
    assert tri((2.0, 2.0)) == [cell(ncx - 1, g.ny - 2) + 1]
    # one ulp outside the grid: nothing (the bounding box of R22 decides, not the rounded barycentric test)
    assert tri((np.nextafter(2.0, 3.0), 2.0)) == [] and tri((-2.0, np.nextafter(-1.0, -2.0))) == []


def test_bounding_box_clause_decides_where_the_rounded_barycentric_test_cannot():
    """R22's box clause, seen on its own.  No lens, coarse grid x in {-3, 1, 5}: the source
    (1 + 1 ulp, 0) lies in cell 1 and, by the plain definition of a closed triangle, NOT in triangle 0 of cell 0,
    whose vertices all have x <= 1.  In floating point S - A = 4 + 2.2e-16 rounds to B - A = 4 exactly, so the
    barycentric test alone gives u = 1, v = 0 and accepts it: without the box there are two images (triangles 0
    and 2), with it one (triangle 2).  (On the finer grid of the test above S - A is exactly representable and u > 1
    rejects the point either way -- that case does not see the clause; this one does.)  Mirrored on a y edge."""
    one_up = np.nextafter(1.0, 2.0)
    z = np.zeros((2, 3))
    im, found = oracle.delens(z, z, -3.0, 0.0, 4.0, [[one_up, 0.0]])
    assert found == 1 and [int(t) for t in im["triangle"]] == [2]
    assert im["x"][0] == one_up and im["y"][0] == 0.0
    z = np.zeros((3, 2))
    im, found = oracle.delens(z, z, 0.0, -3.0, 4.0, [[0.0, one_up]])  # cells stacked in y; cell (0, 1) = triangles 2, 3
    assert found == 1 and [int(t) for t in im["triangle"]] == [2]
    assert im["x"][0] == 0.0 and im["y"][0] == one_up


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
