"""NEXT row f1 on the GPU: lh_source_plane and lh_delens_grid vs the oracle (-m gpu), through the C ABI.

Index work is compared exactly: with the SAME deflection planes on both sides the decision arithmetic is the
same IEEE operations in the same order (no FMA contraction on either side), so the (source, triangle) sets and the
image positions must be bit-identical.  With each side's own deflection (1e-13 apart) a source within rounding of a
triangle edge may legitimately switch triangles, so that test matches images by position instead."""
import numpy as np
import pytest

import lens_inputs as li
import oracle
import paper_2004_06352_b200 as lh

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


def _gpu_delens(ax, ay, g, src, max_images=1 << 16):
    dax = torch.as_tensor(ax, device="cuda").contiguous()
    day = torch.as_tensor(ay, device="cuda").contiguous()
    images = torch.zeros(32 * max(max_images, 1), dtype=torch.uint8, device="cuda")
    count = torch.full((1,), -7, dtype=torch.int64, device="cuda")
    lh.lh_delens_grid(dax, day, g, src, images, max_images, count)
    torch.cuda.synchronize()
    found = int(count.item())
    rec = images.cpu().numpy().view(lh.LH_IMAGE_DTYPE)[: min(found, max_images)]
    return rec, found


def _sorted(rec):
    return np.sort(rec, order=["source", "triangle"])


def _sources(rng, n, half):
    return np.column_stack([rng.uniform(-half, half, n), rng.uniform(-half, half, n)])


def test_source_plane_bit_exact():
    c = li.config(1, scale=8)
    g = c.grid
    ref = oracle.grid(c.lenses, g.x0, g.y0, g.dx, g.nx, g.ny, planes=("ax", "ay"))
    bx, by = oracle.source_plane(ref["ax"], ref["ay"], g.x0, g.y0, g.dx)
    dax, day = torch.as_tensor(ref["ax"], device="cuda"), torch.as_tensor(ref["ay"], device="cuda")
    dbx, dby = torch.full_like(dax, float("nan")), torch.full_like(dax, float("nan"))
    lh.lh_source_plane(dax, day, g, dbx, dby)
    assert np.array_equal(dbx.cpu().numpy(), bx) and np.array_equal(dby.cpu().numpy(), by)
    only = torch.full_like(dax, float("nan"))
    lh.lh_source_plane(dax, day, g, None, only)  # one plane, and in place
    lh.lh_source_plane(dax, day, g, dax, None)
    assert np.array_equal(only.cpu().numpy(), by) and np.array_equal(dax.cpu().numpy(), bx)


@pytest.mark.parametrize("idx,scale,ns", [(1, 4, 80), (2, 16, 300), (3, 16, 1500)])
def test_delens_same_deflection_bit_exact(idx, scale, ns):
    """cluster configs on coarser grids (ragged sizes via a crop), 80-1500 sources (> one launch of 1024)."""
    c = li.config(idx, scale=scale)
    g0 = c.grid
    g = li.Grid(x0=g0.x0, y0=g0.y0, dx=g0.dx, nx=g0.nx - 3, ny=g0.ny - 1)
    ref = oracle.grid(c.lenses, g.x0, g.y0, g.dx, g.nx, g.ny, planes=("ax", "ay"), threads=8)
    src = _sources(np.random.default_rng(idx), ns, 0.35 * g0.nx * g0.dx / 2)
    want, nwant = oracle.delens(ref["ax"], ref["ay"], g.x0, g.y0, g.dx, src)
    got, ngot = _gpu_delens(ref["ax"], ref["ay"], g, src)
    assert ngot == nwant and nwant > ns  # multiple images exist
    a, b = _sorted(got), _sorted(want)
    assert np.array_equal(a["source"], b["source"]) and np.array_equal(a["triangle"], b["triangle"])
    assert np.array_equal(a["x"], b["x"]) and np.array_equal(a["y"], b["y"])
    assert np.all(a["_pad"] == 0)


def test_bounding_box_clause_cases_agree_with_the_definition():
    """The sources of tests/test_delens_cpu.py::test_bounding_box_clause_...: one ulp beyond a shared vertex, where
    the rounded barycentric test alone would report a second image.  Expected values are the definition's (a closed
    triangle lies in the box of its vertices), stated here as literals; the oracle must say the same."""
    one_up = np.nextafter(1.0, 2.0)
    for g, src, tri in ((li.Grid(x0=-3.0, y0=0.0, dx=4.0, nx=3, ny=2), [[one_up, 0.0]], 2),
                        (li.Grid(x0=0.0, y0=-3.0, dx=4.0, nx=2, ny=3), [[0.0, one_up]], 2)):
        z = np.zeros((g.ny, g.nx))
        got, ngot = _gpu_delens(z, z, g, np.asarray(src))
        want, nwant = oracle.delens(z, z, g.x0, g.y0, g.dx, src)
        assert ngot == nwant == 1
        assert int(got["triangle"][0]) == int(want["triangle"][0]) == tri
        assert got["x"][0] == src[0][0] and got["y"][0] == src[0][1]


def test_delens_whole_pipeline_own_deflection():
    """gradient on the GPU -> delens on the GPU, against gradient + delens in the oracle."""
    c = li.config(1, scale=4)
    g = c.grid
    ax = torch.empty((g.ny, g.nx), dtype=torch.float64, device="cuda")
    ay = torch.empty_like(ax)
    lh.lh_grid_gradient(c.lenses, g, ax, ay)
    src = _sources(np.random.default_rng(9), 80, 30.0)
    got, ngot = _gpu_delens(ax, ay, g, src)
    ref = oracle.grid(c.lenses, g.x0, g.y0, g.dx, g.nx, g.ny, planes=("ax", "ay"), threads=8)
    want, nwant = oracle.delens(ref["ax"], ref["ay"], g.x0, g.y0, g.dx, src)
    assert abs(ngot - nwant) <= 2  # a source within rounding of an edge may be seen by one or two triangles
    a, b = _sorted(got), _sorted(want)
    same = (len(a) == len(b)) and np.array_equal(a["source"], b["source"]) and np.array_equal(a["triangle"], b["triangle"])
    if same:
        assert np.allclose(a["x"], b["x"], rtol=0, atol=1e-9) and np.allclose(a["y"], b["y"], rtol=0, atol=1e-9)
    else:  # every oracle image has a GPU image of the same source within 1e-9 arcsec, and vice versa
        for p, q in ((a, b), (b, a)):
            for r in p:
                m = q[q["source"] == r["source"]]
                assert np.min(np.hypot(m["x"] - r["x"], m["y"] - r["y"])) < 1e-9


def test_delens_edge_cases():
    g = li.Grid(x0=0.0, y0=0.0, dx=1.0, nx=9, ny=9)
    z = np.zeros((g.ny, g.nx))
    src = np.column_stack([np.linspace(0.3, 7.3, 8), np.full(8, 0.4)])
    got, found = _gpu_delens(z, z, g, src, max_images=3)      # truncation: count keeps counting
    assert found == 8 and len(got) == 3
    got, found = _gpu_delens(z, z, g, np.zeros((0, 2)))        # no sources
    assert found == 0
    got, found = _gpu_delens(z, z, g, [[2.0, 2.0]])            # on a vertex: six closed triangles share it
    want, nwant = oracle.delens(z, z, g.x0, g.y0, g.dx, [[2.0, 2.0]])
    assert found == nwant == 6 and np.array_equal(_sorted(got)["triangle"], _sorted(want)["triangle"])
    one = li.Grid(x0=0.0, y0=0.0, dx=1.0, nx=1, ny=5)          # no cells at all
    got, found = _gpu_delens(np.zeros((5, 1)), np.zeros((5, 1)), one, [[0.0, 1.0]])
    assert found == 0
    with pytest.raises(lh.LhError):
        _gpu_delens(z, z, g, [[float("nan"), 0.0]])
