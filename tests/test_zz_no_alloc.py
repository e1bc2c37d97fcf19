"""lh_grid_eval_noalloc against the allocating path it stands in for (include/lh.h; csrc/lh_noalloc.cu).

Some users of the library cannot let it call cudaMalloc: their device memory belongs to a caching allocator or to a
scheduler's fixed partition, or the call sits in a loop that may not stall on the device-wide synchronisation of
cudaMalloc / cudaFree.  For them the `carry` scratch of a chunked lens list (more than 160 lenses) and the
reduction tables live in `static __device__` arrays inside liblh.so, and the call is limited to
LH_NOALLOC_MAX_PIXELS pixels.  The arithmetic is the same kernel, so the planes must agree with lh_grid_eval_rows
(which takes its scratch from cudaMalloc) within the parity tolerance of tests/parity.py -- on two calls in a row,
because all calls share the one scratch array and the second sees what the first left in it.

The file name sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not hide the
parity tests.  The test needs nothing from the tests before it and passes alone in a fresh process too."""
import numpy as np
import pytest

import lens_inputs as li
import paper_2004_06352_b200 as lh
from parity import check_planes

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


def dev_planes(names, shape):
    return {n: torch.full(shape, float("nan"), dtype=torch.float64, device="cuda") for n in names}


def both_paths(lenses, g, j0, nrows, names):
    """The slab through the static-scratch entry point and through lh_grid_eval_rows; host copies of both."""
    new = dev_planes(names, (nrows, g.nx))
    old = dev_planes(names, (nrows, g.nx))
    lh.lh_grid_eval_noalloc(lenses, g, j0, nrows, **new)
    lh.lh_grid_eval_rows(lenses, g, j0, nrows, **old)
    torch.cuda.synchronize()
    return {n: new[n].cpu().numpy() for n in names}, {n: old[n].cpu().numpy() for n in names}


def test_static_scratch_matches_the_allocating_path_on_two_calls_in_a_row():
    lh.lh_set_stream(None)
    # call 1: 500 mixed dPIE / NSIE / SIS lenses = 4 launches chained through the scratch, all nine planes,
    # a slab in the middle of a grid that is neither dyadic nor a whole number of tiles
    c1 = li.config(2, scale=16)
    g1 = li.Grid(x0=c1.grid.x0 + 0.1, y0=c1.grid.y0 + 0.3, dx=c1.grid.dx * 1.1, nx=c1.grid.nx + 5, ny=c1.grid.ny + 3)
    got, ref = both_paths(c1.lenses, g1, 7, g1.ny - 9, li.ALL_PLANES)
    assert all(np.isfinite(got[n]).all() for n in ("ax", "ay", "kappa"))
    w1 = check_planes(got, ref, "no-alloc call 1")
    # call 2, straight after, on the scratch call 1 left behind: another model (1000 dPIE = 7 launches), another
    # grid shape with MORE pixels per row and fewer rows, so every scratch element it reads holds call 1's sums
    # unless this call wrote it first
    c2 = li.config(3, scale=16)
    g2 = li.Grid(x0=c2.grid.x0, y0=c2.grid.y0, dx=c2.grid.dx, nx=c2.grid.nx + 77, ny=61)
    got, ref = both_paths(c2.lenses, g2, 0, g2.ny, ("ax", "ay", "kappa", "gamma1", "gamma2", "mu"))
    w2 = check_planes(got, ref, "no-alloc call 2")
    # and once more call 1's job: the result does not depend on what ran in between
    got, ref = both_paths(c1.lenses, g1, 7, g1.ny - 9, ("ax", "kappa", "gamma1", "gamma2", "mu"))
    w3 = check_planes(got, ref, "no-alloc call 3")
    print(f"no-alloc vs allocating path, worst |d|/allowed: {max(w1.values()):.3g}, {max(w2.values()):.3g}, "
          f"{max(w3.values()):.3g}")


def test_short_lens_list_and_empty_list():
    """At most 160 lenses: one launch, the scratch is not used at all; no lens: zeros and mu = 1."""
    lh.lh_set_stream(None)
    c = li.config(0)
    got, ref = both_paths(c.lenses, c.grid, 0, c.grid.ny, li.ALL_PLANES)
    check_planes(got, ref, "no-alloc, 10 lenses")
    got, ref = both_paths(c.lenses[:0], c.grid, 3, 5, ("ax", "mu"))
    assert np.array_equal(got["ax"], np.zeros((5, c.grid.nx))) and np.array_equal(got["mu"], np.ones((5, c.grid.nx)))


def test_sizes_beyond_the_reservation_are_refused_and_nothing_is_written():
    c = li.config(3, scale=16)
    nx = 2048
    nrows = lh.LH_NOALLOC_MAX_PIXELS // nx + 1  # one row too many
    g = li.Grid(x0=-1.0, y0=-1.0, dx=0.01, nx=nx, ny=nrows)
    out = dev_planes(("ax",), (nrows, nx))
    with pytest.raises(lh.LhError) as e:
        lh.lh_grid_eval_noalloc(c.lenses, g, 0, nrows, **out)
    assert e.value.code == lh.LH_EINVAL and "LH_NOALLOC_MAX_PIXELS" in str(e.value)
    torch.cuda.synchronize()
    assert bool(torch.isnan(out["ax"]).all())
    # exactly at the limit it runs, all five scratch planes in use to their last element
    nrows -= 1
    g = li.Grid(x0=-1.0, y0=-1.0, dx=0.01, nx=nx, ny=nrows)
    few = c.lenses[:170]  # two launches through the scratch; keeps the full-size slab cheap
    got, ref = both_paths(few, g, 0, nrows, ("ax", "kappa"))
    check_planes(got, ref, "no-alloc at LH_NOALLOC_MAX_PIXELS")
    # too many lenses for the fixed host table
    many = np.tile(c.lenses, 5)[: lh.LH_NOALLOC_MAX_LENSES + 1]
    small = dev_planes(("ax",), (4, 8))
    with pytest.raises(lh.LhError) as e:
        lh.lh_grid_eval_noalloc(many, li.Grid(x0=0.0, y0=0.0, dx=1.0, nx=8, ny=4), 0, 4, **small)
    assert e.value.code == lh.LH_EINVAL and "LH_NOALLOC_MAX_LENSES" in str(e.value)
    assert bool(torch.isnan(small["ax"]).all())
