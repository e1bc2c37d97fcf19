"""CUDA path vs CPU oracle, element by element, through the C ABI (-m gpu).

Small/medium cases compare whole maps; BASELINE.json's full-size configs are run in the
launch configuration bench.py times and compared on seeded samples of pixels the oracle
evaluates one by one.  Tolerances: tests/parity.py (north_star: 1e-11 relative, floor
1e-13 x max|plane|; mu conditioned, reading 8c-13).
"""
import os

import numpy as np
import pytest

import lens_inputs as li
import oracle
import paper_2004_06352_b200 as lh
from parity import check_planes, conditioned_rel, plain_violation, stats_violation

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
NTHREADS = max(1, min(16, os.cpu_count() or 1))


def dev_planes(names, shape):
    return {n: torch.full(shape, float("nan"), dtype=torch.float64, device="cuda") for n in names}


def run_gpu(lenses, grid, names, nmodel=1, nlens=None):
    nlens = len(lenses) // nmodel if nlens is None else nlens
    shape = (nmodel, grid.ny, grid.nx) if nmodel > 1 else (grid.ny, grid.nx)
    out = dev_planes(names, shape)
    if nmodel == 1:
        lh.lh_grid_eval(lenses, grid, **out)
    else:
        lh.lh_grid_eval_batch(lenses, nmodel, nlens, grid, **out)
    torch.cuda.synchronize()
    return {n: v.cpu().numpy() for n, v in out.items()}


def ref_grid(lenses, grid, names):
    need = set(names)
    if "mu" in need:
        need |= {"kappa", "gamma1", "gamma2"}
    return oracle.grid(lenses, grid.x0, grid.y0, grid.dx, grid.nx, grid.ny, planes=tuple(sorted(need)),
                       threads=NTHREADS)


def ref_samples(lenses, grid, ii, jj, names):
    need = set(names)
    if "mu" in need:
        need |= {"kappa", "gamma1", "gamma2"}
    return oracle.points(lenses, grid.x0 + ii * grid.dx, grid.y0 + jj * grid.dx, planes=tuple(sorted(need)))


# ------------------------------------------------------------------ BASELINE.json configs, whole maps
def test_cfg0_all_nine_planes_and_the_four_calls():
    c = li.config(0)
    g = c.grid
    ref = ref_grid(c.lenses, g, li.ALL_PLANES)
    got = run_gpu(c.lenses, g, li.ALL_PLANES)
    check_planes(got, ref, "cfg0 lh_grid_eval")
    # the four named calls give bit-identical planes to lh_grid_eval's matching kernel variant
    o = dev_planes(li.ALL_PLANES, (g.ny, g.nx))
    lh.lh_grid_gradient(c.lenses, g, o["ax"], o["ay"])
    lh.lh_grid_hessian(c.lenses, g, o["a11"], o["a12"], o["a22"])
    lh.lh_lens_maps(c.lenses, g, o["kappa"], o["gamma1"], o["gamma2"], o["mu"])
    torch.cuda.synchronize()
    check_planes({n: v.cpu().numpy() for n, v in o.items()}, ref, "cfg0 four calls")


@pytest.mark.parametrize("idx,scale", [(1, 4), (2, 8), (3, 16)])
def test_cfg_scaled_whole_map(idx, scale):
    """configs 1-3 on a coarser grid of the same extent (same lenses): several tiles, every class."""
    c = li.config(idx, scale=scale)
    ref = ref_grid(c.lenses, c.grid, c.outputs)
    got = run_gpu(c.lenses, c.grid, c.outputs)
    check_planes(got, ref, c.name)


def test_cfg4_scaled_batch_whole_maps():
    c = li.config(4, scale=16)  # 64 models x 300 lenses on 64 x 64
    got = run_gpu(c.lenses, c.grid, c.outputs, nmodel=c.nmodel, nlens=c.nlens)
    for m in range(c.nmodel):
        ref = ref_grid(c.lenses[m * c.nlens:(m + 1) * c.nlens], c.grid, c.outputs)
        check_planes({n: got[n][m] for n in got}, ref, f"{c.name} model {m}")


# ------------------------------------------------------------------ full size, bench launch configuration, sampled
@pytest.mark.parametrize("idx", [1, 2, 3])
def test_cfg_full_size_sampled(idx):
    c = li.config(idx)
    got = run_gpu(c.lenses, c.grid, c.outputs)
    ii, jj = li.random_points(100 + idx, c.grid, 3000)
    # always include the corners and the last row/column (ragged-tail logic at full size)
    ii = np.concatenate([ii, [0, c.grid.nx - 1, 0, c.grid.nx - 1]])
    jj = np.concatenate([jj, [0, 0, c.grid.ny - 1, c.grid.ny - 1]])
    ref = ref_samples(c.lenses, c.grid, ii, jj, c.outputs)
    check_planes({n: got[n][jj, ii] for n in got}, ref, c.name + " sampled")
    for n in got:
        assert np.isfinite(got[n]).all() or n == "mu"
        assert not np.isnan(got[n]).any()


def test_cfg4_full_size_batch_sampled():
    c = li.config(4)
    out = dev_planes(c.outputs, (c.nmodel, c.grid.ny, c.grid.nx))
    lh.lh_grid_gradient_batch(c.lenses, c.nmodel, c.nlens, c.grid, out["ax"], out["ay"])
    torch.cuda.synchronize()
    ii, jj = li.random_points(104, c.grid, 400)
    it, jt = torch.as_tensor(ii, device="cuda"), torch.as_tensor(jj, device="cuda")
    for m in range(c.nmodel):
        ref = ref_samples(c.lenses[m * c.nlens:(m + 1) * c.nlens], c.grid, ii, jj, c.outputs)
        check_planes({n: out[n][m][jt, it].cpu().numpy() for n in out}, ref, f"{c.name} model {m} sampled")
    assert not torch.isnan(out["ax"]).any() and not torch.isnan(out["ay"]).any()


# ------------------------------------------------------------------ tiling edge cases
@pytest.mark.parametrize("nx,ny", [(1, 1), (1, 9), (9, 1), (63, 3), (64, 4), (65, 5), (67, 7), (129, 2), (200, 13)])
def test_ragged_grids(nx, ny):
    c = li.config(2)
    L = c.lenses[:130]  # dPIE + NSIE + SIS in one launch
    g = li.Grid(x0=-20.3, y0=11.7, dx=0.37, nx=nx, ny=ny)
    ref = ref_grid(L, g, li.ALL_PLANES)
    got = run_gpu(L, g, li.ALL_PLANES)
    check_planes(got, ref, f"ragged {nx}x{ny}")


@pytest.mark.parametrize("nlens", [0, 1, 63, 159, 160, 161, 320, 321, 481])
def test_lens_counts_around_launch_capacity(nlens):
    """A launch carries at most 160 records in its kernel parameters (lh_kernels.h); more lenses are evaluated by
    consecutive launches that hand the accumulators on through the carry buffer."""
    c = li.config(3)
    L = c.lenses[:nlens]
    g = li.Grid(x0=-30.0, y0=-30.0, dx=0.9, nx=70, ny=9)
    ref = ref_grid(L, g, li.ALL_PLANES)
    got = run_gpu(L, g, li.ALL_PLANES)
    check_planes(got, ref, f"nlens={nlens}")
    if nlens == 0:
        for n in got:
            assert np.all(got[n] == (1.0 if n == "mu" else 0.0))


def test_many_small_models_share_launches():
    """Models with few lenses share one launch (blockIdx.y); 50 x 7 records need three launches of <= 22 models."""
    c = li.config(2)
    rng = np.random.default_rng(5)
    nmodel, nlens = 50, 7
    L = c.lenses[rng.integers(0, len(c.lenses), nmodel * nlens)]  # dPIE / NSIE / SIS mix differs per model
    g = li.Grid(x0=-40.0, y0=-25.0, dx=0.77, nx=131, ny=5)
    n0 = lh.lh_launch_count()
    got = run_gpu(L, g, li.ALL_PLANES, nmodel=nmodel, nlens=nlens)
    assert lh.lh_launch_count() - n0 == 3
    for m in range(nmodel):
        ref = ref_grid(L[m * nlens:(m + 1) * nlens], g, li.ALL_PLANES)
        check_planes({n: got[n][m] for n in got}, ref, f"small model {m}")


def test_batch_of_empty_models():
    g = li.Grid(x0=0.0, y0=0.0, dx=1.0, nx=33, ny=3)
    got = run_gpu(li.make_lenses(0), g, li.ALL_PLANES, nmodel=200, nlens=0)
    for n in got:
        assert got[n].shape == (200, 3, 33) and np.all(got[n] == (1.0 if n == "mu" else 0.0))


def test_chunked_model_with_every_class():
    """> 160 lenses with dPIE, NSIE, SIS and extreme-ellipticity lenses: class boundaries fall inside and on
    the edges of the lens chunks; also as a batch of two such models (chunks run model by model)."""
    c = li.config(2)
    L = c.lenses[:330].copy()
    L["ellipticity"][[5, 170, 171, 329]] = 0.9995  # CLS_EXTREME (sorted last by the packer)
    g = li.Grid(x0=-60.0, y0=-60.0, dx=1.3, nx=93, ny=21)
    rel = conditioned_rel(0.9995)
    check_planes(run_gpu(L, g, li.ALL_PLANES), ref_grid(L, g, li.ALL_PLANES), "chunked, all classes", rel=rel)
    L2 = np.concatenate([L, L[::-1]])
    got = run_gpu(L2, g, ("ax", "kappa", "mu"), nmodel=2, nlens=330)
    for m in range(2):
        ref = ref_grid(L2[m * 330:(m + 1) * 330], g, ("ax", "kappa", "mu"))
        check_planes({n: got[n][m] for n in got}, ref, f"chunked batch model {m}", rel=rel)


def test_extreme_length_scales_stay_inside_the_shared_reciprocal_range():
    """rcp4 takes the reciprocal of a product of two squared and two cubed scaled lengths (include/lh.h: lengths
    between ~1e-20 and ~1e+17 of the unit in use):
    micro-arcsec and 1e12-arcsec units must still give oracle-grade results."""
    for scale in (1e-9, 1e12):
        L = li.make_lenses(2)
        L[0] = (li.DPIE, 0, 0.3 * scale, -0.2 * scale, 0.4, 0.7, 0.08 * scale, 30.0 * scale, 1.7 * scale)
        L[1] = (li.DPIE, 0, -4.0 * scale, 2.0 * scale, 0.0, 0.0, 0.5 * scale, 9.0 * scale, 0.6 * scale)
        g = li.Grid(x0=-15.0 * scale, y0=-15.0 * scale, dx=0.61 * scale, nx=49, ny=49)
        got = run_gpu(L, g, li.ALL_PLANES)
        check_planes(got, ref_grid(L, g, li.ALL_PLANES), f"scale {scale}")
        assert all(np.isfinite(v).all() for v in got.values())


def test_mixed_types_any_order():
    """The library sorts by class; the sum must equal the oracle's index-order sum within tolerance."""
    c = li.config(2)
    rng = np.random.default_rng(77)
    L = c.lenses[rng.permutation(len(c.lenses))[:200]]
    g = li.Grid(x0=-50.0, y0=-50.0, dx=1.01, nx=99, ny=33)
    check_planes(run_gpu(L, g, li.ALL_PLANES), ref_grid(L, g, li.ALL_PLANES), "mixed order")
    for t in (li.NSIE, li.SIS):  # single-class models
        Lt = c.lenses[c.lenses["type"] == t]
        check_planes(run_gpu(Lt, g, li.ALL_PLANES), ref_grid(Lt, g, li.ALL_PLANES), f"only type {t}")


# ------------------------------------------------------------------ degenerate cases of the method
@pytest.mark.parametrize("ehat", [0.0, 1e-14, 1e-12, 1e-9, 1e-6, 1e-3, 0.3, 0.9, 0.99, 0.9999])
def test_ellipticity_range(ehat):
    L = li.make_lenses(3)
    L[0] = (li.DPIE, 0, 0.3, -0.2, ehat, 0.7, 0.08, 30.0, 1.7)
    L[1] = (li.NSIE, 0, -4.0, 2.0, ehat, 2.4, 0.3, 0.0, 0.6)
    L[2] = (li.DPIE, 0, 5.0, 5.0, ehat, 1.1, 2.0, 900.0, 9.0)
    g = li.Grid(x0=-15.0, y0=-15.0, dx=0.31, nx=97, ny=97)
    # 1e-11 for e-hat <= 0.9992; conditioned by 1/q^2 beyond (parity.conditioned_rel, R20)
    check_planes(run_gpu(L, g, li.ALL_PLANES), ref_grid(L, g, li.ALL_PLANES), f"ehat={ehat}", rel=conditioned_rel(ehat))


def test_pixel_on_and_next_to_centres():
    g = li.Grid(x0=-1.0, y0=-1.0, dx=0.25, nx=9, ny=9)  # pixel (4,4) is exactly (0,0)
    L = li.make_lenses(4)
    L[0] = (li.SIS, 0, 0.0, 0.0, 0, 0, 0, 0, 0.7)              # exactly on a pixel: zero contribution
    L[1] = (li.DPIE, 0, 0.25 + 1e-9, 0.5, 0.4, 0.3, 0.01, 8.0, 1.0)  # rcore << dx, pixel 1e-9" from centre
    L[2] = (li.NSIE, 0, -0.5, -0.25, 0.2, 1.0, 0.02, 0.0, 0.4)  # exactly on a pixel
    L[3] = (li.DPIE, 0, 0.75, -0.75, 0.0, 0.0, 0.05, 3.0, 0.0)  # b0 = 0
    got = run_gpu(L, g, li.ALL_PLANES)
    ref = ref_grid(L, g, li.ALL_PLANES)
    check_planes(got, ref, "centres")
    assert not any(np.isnan(v).any() for v in got.values())
    only_sis = run_gpu(L[:1], g, li.ALL_PLANES)
    assert only_sis["ax"][4, 4] == 0.0 and only_sis["kappa"][4, 4] == 0.0 and only_sis["mu"][4, 4] == 1.0


def test_far_field_and_large_scales():
    """|x| up to 1e4 arcsec and rcut = 1e6: no overflow/cancellation surprises in the merged forms."""
    L = li.make_lenses(2)
    L[0] = (li.DPIE, 0, 10.0, -20.0, 0.5, 0.4, 0.5, 1e6, 30.0)
    L[1] = (li.DPIE, 0, -3.0, 4.0, 0.6, 2.0, 1e-3, 2e-3, 1.0)  # rcut barely above rcore scale
    g = li.Grid(x0=-1e4, y0=-1e4, dx=157.3, nx=128, ny=128)
    check_planes(run_gpu(L, g, li.ALL_PLANES), ref_grid(L, g, li.ALL_PLANES), "far field")


# ------------------------------------------------------------------ arbitrary points
@pytest.mark.parametrize("npts", [1, 5, 127, 128, 129, 1000])
def test_points_eval_matches_oracle_points(npts):
    c = li.config(2)  # 500 mixed lenses: four lens chunks
    rng = np.random.default_rng(npts)
    xs, ys = rng.uniform(-90, 90, npts), rng.uniform(-90, 90, npts)
    dx_, dy_ = torch.as_tensor(xs, device="cuda"), torch.as_tensor(ys, device="cuda")
    out = dev_planes(li.ALL_PLANES, (npts,))
    lh.lh_points_eval(c.lenses, dx_, dy_, **out)
    torch.cuda.synchronize()
    ref = oracle.points(c.lenses, xs, ys, planes=li.ALL_PLANES)
    check_planes({n: v.cpu().numpy() for n, v in out.items()}, ref, f"{npts} points")


def test_points_on_the_grid_equal_the_grid_call_bitwise():
    c = li.config(1, scale=16)
    g = c.grid
    full = run_gpu(c.lenses, g, ("ax", "ay"))
    X, Y = np.meshgrid(g.xs(), g.ys())
    out = dev_planes(("ax", "ay"), (g.npix,))
    lh.lh_points_eval(c.lenses, torch.as_tensor(X.ravel(), device="cuda"), torch.as_tensor(Y.ravel(), device="cuda"), **out)
    torch.cuda.synchronize()
    for n in full:
        assert np.array_equal(out[n].cpu().numpy().reshape(g.ny, g.nx), full[n])


# ------------------------------------------------------------------ multi-GPU primitive: row slabs
@pytest.mark.parametrize("world", [2, 3, 8])
def test_row_slabs_reassemble_the_full_map_bitwise(world):
    """Every rank evaluates lens_inputs.row_slab(rank) with lh_grid_eval_rows; stacked, the slabs are bit-identical
    to the single-device map (same pixel coordinates, same arithmetic) -- including a model with lens chunks."""
    c = li.config(2, scale=16)  # 128 x 128, 500 mixed lenses (4 lens chunks through the carry buffer)
    g = li.Grid(x0=c.grid.x0 + 0.1, y0=c.grid.y0 + 0.3, dx=c.grid.dx * 1.1, nx=c.grid.nx, ny=c.grid.ny)  # not dyadic
    full = run_gpu(c.lenses, g, ("ax", "kappa", "mu"))
    parts = {n: [] for n in full}
    for rank in range(world):
        j0, nrows = li.row_slab(g, rank, world)
        out = dev_planes(tuple(full), (nrows, g.nx))
        lh.lh_grid_eval_rows(c.lenses, g, j0, nrows, **out)
        torch.cuda.synchronize()
        host = {n: np.full((nrows, g.nx), np.nan) for n in full}
        lh.lh_grid_eval_rows_host(c.lenses, g, j0, nrows, **host)  # the same slab into HOST planes: same bits
        for n in full:
            parts[n].append(out[n].cpu().numpy())
            assert np.array_equal(host[n], parts[n][-1], equal_nan=True)
    for n in full:
        assert np.array_equal(np.concatenate(parts[n]), full[n], equal_nan=True)
    with pytest.raises(lh.LhError):
        lh.lh_grid_eval_rows(c.lenses, g, g.ny - 1, 2, ax=dev_planes(("ax",), (2, g.nx))["ax"])


# ------------------------------------------------------------------ f4: batches that share most of their lenses
def test_shared_lens_batch_cfg4_scaled():
    """cfg 4 keeps the 298 galaxies fixed and perturbs the 2 halos: shared = galaxies (two lens chunks, evaluated
    once), varying = 2 halos per model.  Must match the oracle on every model's full 300-lens list."""
    c = li.config(4, scale=16)
    g = c.grid
    L = c.lenses.reshape(c.nmodel, c.nlens)
    shared, varying = L[0, 2:].copy(), np.ascontiguousarray(L[:, :2]).reshape(-1)
    assert all(np.array_equal(L[m, 2:], shared) for m in range(c.nmodel))
    names = ("ax", "ay", "kappa", "gamma1", "mu")
    out = dev_planes(names, (c.nmodel, g.ny, g.nx))
    n0 = lh.lh_launch_count()
    lh.lh_grid_eval_batch_shared(shared, varying, c.nmodel, 2, g, **out)
    torch.cuda.synchronize()
    assert lh.lh_launch_count() - n0 == 2 + 1  # 298 shared lenses in two chunks + 64 x 2 varying in one launch
    for m in range(0, c.nmodel, 7):
        ref = ref_grid(c.lenses[m * c.nlens:(m + 1) * c.nlens], g, names)
        check_planes({n: out[n][m].cpu().numpy() for n in names}, ref, f"shared batch model {m}")


def test_shared_lens_batch_edge_cases():
    c = li.config(2)
    g = li.Grid(x0=-30.0, y0=-20.0, dx=0.9, nx=67, ny=9)
    shared = c.lenses[:40]  # dPIE + NSIE + SIS
    # nvar = 0: every model is the shared list
    out = dev_planes(("ax", "kappa"), (3, g.ny, g.nx))
    lh.lh_grid_eval_batch_shared(shared, li.make_lenses(0), 3, 0, g, **out)
    ref = ref_grid(shared, g, ("ax", "kappa"))
    for m in range(3):
        check_planes({n: out[n][m].cpu().numpy() for n in out}, ref, "nvar=0")
    # nshared = 0: plain batch, bitwise
    var = c.lenses[40:52]
    a = dev_planes(("ay", "mu"), (3, g.ny, g.nx))
    b = dev_planes(("ay", "mu"), (3, g.ny, g.nx))
    lh.lh_grid_eval_batch_shared(li.make_lenses(0), var, 3, 4, g, **a)
    lh.lh_grid_eval_batch(var, 3, 4, g, **b)
    torch.cuda.synchronize()
    assert all(torch.equal(a[n], b[n]) for n in a)
    # too many varying lenses beside a shared list, bad lens in the shared list: nothing written
    o = dev_planes(("ax",), (1, g.ny, g.nx))
    with pytest.raises(lh.LhError):
        lh.lh_grid_eval_batch_shared(shared, c.lenses[:161], 1, 161, g, **o)
    bad = shared.copy()
    bad["rcore"][0] = -1.0
    with pytest.raises(lh.LhError):
        lh.lh_grid_eval_batch_shared(bad, var, 3, 4, g, **dev_planes(("ax",), (3, g.ny, g.nx)))
    assert torch.isnan(o["ax"]).all()


# ------------------------------------------------------------------ f2: map statistics over a batch
def _stats_gpu(c, names, var_names):
    g = c.grid
    mean = dev_planes(names, (g.ny, g.nx))
    var = dev_planes(var_names, (g.ny, g.nx))
    lh.lh_grid_stats_batch(c.lenses, c.nmodel, c.nlens, g, mean, var)
    torch.cuda.synchronize()
    return {n: v.cpu().numpy() for n, v in mean.items()}, {n: v.cpu().numpy() for n, v in var.items()}


def test_stats_cfg4_scaled_whole_maps():
    """64 models x 300 lenses (two lens chunks per model) on 64 x 64: mean and variance of ax, ay, kappa, gamma1."""
    c = li.config(4, scale=16)
    names = ("ax", "ay", "kappa", "gamma1")
    g = c.grid
    mean, var = _stats_gpu(c, names, names)
    rmean, rvar = oracle.stats(c.lenses, c.nmodel, c.nlens, g.x0, g.y0, g.dx, g.nx, g.ny, planes=names, threads=NTHREADS)
    for n in names:
        vm, vv = stats_violation(mean[n], var[n], rmean[n], rvar[n], c.nmodel)
        assert vm <= 1.0 and vv <= 1.0, (n, vm, vv)
        assert (var[n] >= 0).all()


def test_stats_small_models_mean_only_and_single_model():
    c = li.config(2)
    rng = np.random.default_rng(11)
    nmodel, nlens = 9, 12
    L = c.lenses[rng.integers(0, len(c.lenses), nmodel * nlens)]
    g = li.Grid(x0=-30.0, y0=-20.0, dx=0.9, nx=67, ny=9)
    names = ("ax", "a11", "a12", "a22", "kappa", "gamma2")
    mean = dev_planes(names, (g.ny, g.nx))
    var = dev_planes(("kappa",), (g.ny, g.nx))
    n0 = lh.lh_launch_count()
    lh.lh_grid_stats_batch(L, nmodel, nlens, g, mean, var)
    torch.cuda.synchronize()
    assert lh.lh_launch_count() - n0 == nmodel  # statistics mode: one launch chain per model
    rmean, rvar = oracle.stats(L, nmodel, nlens, g.x0, g.y0, g.dx, g.nx, g.ny, planes=names)
    for n in names:
        vm, _ = stats_violation(mean[n].cpu().numpy(), rvar[n], rmean[n], rvar[n], nmodel)
        assert vm <= 1.0, (n, vm)
    _, vv = stats_violation(rmean["kappa"], var["kappa"].cpu().numpy(), rmean["kappa"], rvar["kappa"], nmodel)
    assert vv <= 1.0
    # one model: mean is the map itself (bitwise), variance exactly zero
    one = dev_planes(("ax", "kappa"), (g.ny, g.nx))
    onev = dev_planes(("ax", "kappa"), (g.ny, g.nx))
    lh.lh_grid_stats_batch(L[:nlens], 1, nlens, g, one, onev)
    ref = run_gpu(L[:nlens], g, ("ax", "kappa"))
    for n in ref:
        assert np.array_equal(one[n].cpu().numpy(), ref[n]) and (onev[n] == 0).all()


def test_stats_argument_errors():
    c = li.config(0)
    g = c.grid
    k = dev_planes(("kappa",), (g.ny, g.nx))
    with pytest.raises(lh.LhError):
        lh.lh_grid_stats_batch(c.lenses, 1, c.nlens, g, {}, k)           # variance without its mean
    with pytest.raises(lh.LhError):
        lh.lh_grid_stats_batch(c.lenses, 1, c.nlens, g, k, k)            # shared buffer
    with pytest.raises(lh.LhError):
        lh.lh_grid_stats_batch(c.lenses, 1, c.nlens, g, {}, None)        # nothing requested
    assert torch.isnan(k["kappa"]).all()


# ------------------------------------------------------------------ ABI behaviour on the device
def test_unrequested_planes_are_never_touched():
    c = li.config(0)
    g = c.grid
    for req in (("ax", "ay"), ("kappa", "mu"), ("a12",), ("ay", "gamma1")):
        out = dev_planes(li.ALL_PLANES, (g.ny, g.nx))
        lh.lh_grid_eval(c.lenses, g, **{n: out[n] for n in req})
        torch.cuda.synchronize()
        for n in li.ALL_PLANES:
            if n in req:
                assert not torch.isnan(out[n]).any()
            else:
                assert torch.isnan(out[n]).all()


@pytest.mark.parametrize("which", ["cfg0", "chunked"])
def test_every_subset_of_the_nine_planes(which):
    """"every nullable-output combination of lh_grid_eval" -- all 511 non-empty subsets of the nine
    planes.  The requested planes match the oracle, the others keep their NaN fill.  cfg 0 (10 lenses, one launch)
    and a 500-lens mixed model (four launches through the carry buffer: the subset also decides which accumulators
    are parked between launches)."""
    c = li.config(0) if which == "cfg0" else li.config(2, scale=32)
    g = c.grid
    ref = ref_grid(c.lenses, g, li.ALL_PLANES)
    buf = torch.empty((9, g.ny, g.nx), dtype=torch.float64, device="cuda")
    worst = 0.0
    for mask in range(1, 512):
        req = [n for k, n in enumerate(li.ALL_PLANES) if mask >> k & 1]
        buf.fill_(float("nan"))
        lh.lh_grid_eval(c.lenses, g, **{n: buf[li.ALL_PLANES.index(n)] for n in req})
        torch.cuda.synchronize()
        host = buf.cpu().numpy()
        for k, n in enumerate(li.ALL_PLANES):
            if n not in req:
                assert np.isnan(host[k]).all(), (req, n)
        w = check_planes({n: host[li.ALL_PLANES.index(n)] for n in req}, ref, f"{which} subset {req}")
        worst = max(worst, max(w.values()))
    assert worst <= 1.0


def test_guard_bands_not_overwritten():
    c = li.config(0)
    g = li.Grid(x0=-10.0, y0=-10.0, dx=0.3, nx=67, ny=5)
    pad = 64
    buf = torch.full((2, g.npix + 2 * pad), 7.25, dtype=torch.float64, device="cuda")
    ax, ay = buf[0, pad:pad + g.npix], buf[1, pad:pad + g.npix]
    lh.lh_grid_gradient(c.lenses, g, ax, ay)
    torch.cuda.synchronize()
    assert (buf[:, :pad] == 7.25).all() and (buf[:, pad + g.npix:] == 7.25).all()
    # odd plane offset: 8-byte but not 16-byte aligned outputs are legal
    ax2, ay2 = buf[0, pad + 1:pad + 1 + g.npix - 1], buf[1, pad + 1:pad + 1 + g.npix - 1]
    g2 = li.Grid(x0=g.x0, y0=g.y0, dx=g.dx, nx=g.npix - 1, ny=1)
    lh.lh_grid_gradient(c.lenses, g2, ax2, ay2)
    torch.cuda.synchronize()
    ref = ref_grid(c.lenses, g2, ("ax", "ay"))
    check_planes({"ax": ax2.cpu().numpy().reshape(1, -1), "ay": ay2.cpu().numpy().reshape(1, -1)}, ref, "odd offset")


def test_batch_of_one_equals_single_call_bitwise():
    c = li.config(1, scale=8)
    a = run_gpu(c.lenses, c.grid, ("ax", "ay"))
    out = dev_planes(("ax", "ay"), (1, c.grid.ny, c.grid.nx))
    lh.lh_grid_gradient_batch(c.lenses, 1, c.nlens, c.grid, out["ax"], out["ay"])
    torch.cuda.synchronize()
    assert np.array_equal(a["ax"], out["ax"][0].cpu().numpy()) and np.array_equal(a["ay"], out["ay"][0].cpu().numpy())


def test_errors_write_nothing():
    c = li.config(0)
    g = c.grid
    out = dev_planes(("ax", "ay"), (g.ny, g.nx))
    before = lh.lh_launch_count()
    bad = c.lenses.copy()
    bad["ellipticity"][3] = 1.0
    with pytest.raises(lh.LhError) as e:
        lh.lh_grid_gradient(bad, g, out["ax"], out["ay"])
    assert e.value.code == lh.LH_EINVAL and "lens 3" in str(e.value)
    cpu = torch.zeros(g.npix, dtype=torch.float64)
    with pytest.raises(lh.LhError):
        lh.lh_grid_gradient(c.lenses, g, cpu, out["ay"])  # host tensor is not device memory
    torch.cuda.synchronize()
    assert torch.isnan(out["ax"]).all() and torch.isnan(out["ay"]).all()
    assert lh.lh_launch_count() == before
    lh.lh_grid_gradient(c.lenses, g, out["ax"], out["ay"])  # and the library still works afterwards
    torch.cuda.synchronize()
    assert not torch.isnan(out["ax"]).any()


def test_two_streams_do_not_interfere():
    c1, c3 = li.config(1, scale=4), li.config(3, scale=16)
    r1, r3 = ref_grid(c1.lenses, c1.grid, ("ax", "ay")), ref_grid(c3.lenses, c3.grid, ("ax", "ay"))
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    o1 = [dev_planes(("ax", "ay"), (c1.grid.ny, c1.grid.nx)) for _ in range(4)]
    o3 = [dev_planes(("ax", "ay"), (c3.grid.ny, c3.grid.nx)) for _ in range(4)]
    torch.cuda.synchronize()
    try:
        for k in range(4):
            lh.lh_set_stream(s1)
            lh.lh_grid_gradient(c1.lenses, c1.grid, o1[k]["ax"], o1[k]["ay"])
            lh.lh_set_stream(s2)
            lh.lh_grid_gradient(c3.lenses, c3.grid, o3[k]["ax"], o3[k]["ay"])
    finally:
        lh.lh_set_stream(None)
    torch.cuda.synchronize()
    for k in range(4):
        check_planes({n: v.cpu().numpy() for n, v in o1[k].items()}, r1, "stream 1")
        check_planes({n: v.cpu().numpy() for n, v in o3[k].items()}, r3, "stream 2")


def test_host_entry_point_matches_device_entry_point():
    c = li.config(2, scale=16)
    g = c.grid
    dev = run_gpu(c.lenses, g, li.ALL_PLANES)
    host = {n: np.full((g.ny, g.nx), np.nan) for n in ("ax", "kappa", "mu")}
    lh.lh_grid_eval_host(c.lenses, 1, c.nlens, g, **host)
    for n in host:
        assert np.array_equal(host[n], dev[n])


def test_host_entry_point_pipelined_pieces_are_bitwise_the_device_result():
    """Large jobs are cut into row slabs (one map) or model groups (batch) whose device-to-host copies overlap the
    next piece's computation (lh_api.cu): same bits as the device entry point, ragged slab sizes included."""
    c = li.config(1)  # 100 dPIE
    g = li.Grid(x0=c.grid.x0, y0=c.grid.y0, dx=c.grid.dx, nx=1024, ny=1001)  # 16 MB of results -> 3 slabs, ragged
    dev = run_gpu(c.lenses, g, ("ax", "ay"))
    host = {n: np.full((g.ny, g.nx), np.nan) for n in ("ax", "ay")}
    lh.lh_grid_eval_host(c.lenses, 1, c.nlens, g, **host)
    for n in host:
        assert np.array_equal(host[n], dev[n])
    # a model with lens chunks (carry buffer addressed per slab) and the Hessian planes
    c3 = li.config(3, scale=4)  # 1024 x 1024, 1000 dPIE
    dev = run_gpu(c3.lenses, c3.grid, ("ay", "kappa", "mu"))
    host = {n: np.full((c3.grid.ny, c3.grid.nx), np.nan) for n in ("ay", "kappa", "mu")}
    lh.lh_grid_eval_host(c3.lenses, 1, c3.nlens, c3.grid, **host)
    for n in host:
        assert np.array_equal(host[n], dev[n], equal_nan=True)
    # a batch: 64 models x 300 lenses on 256 x 256 (64 MB of results -> 8 groups of models)
    c4 = li.config(4, scale=4)
    dev = run_gpu(c4.lenses, c4.grid, ("ax", "ay"), nmodel=c4.nmodel, nlens=c4.nlens)
    host = {n: np.full((c4.nmodel, c4.grid.ny, c4.grid.nx), np.nan) for n in ("ax", "ay")}
    lh.lh_grid_eval_host(c4.lenses, c4.nmodel, c4.nlens, c4.grid, **host)
    for n in host:
        assert np.array_equal(host[n], dev[n])


def test_fp64_probe_runs():
    flops, secs = lh.lh_fp64_peak_probe(2048)
    assert secs > 0 and 1e12 < flops < 1e14


def test_host_entry_point_validates_every_model_before_writing_anything():
    """A bad lens in the LAST model of a batch large enough to be pipelined in pieces (>= 8 MB of results): LH_EINVAL,
    and not one element of the caller's host planes written (include/lh.h: nothing enqueued, nothing written)."""
    c = li.config(4, scale=4)  # 64 models x 300 lenses on 256 x 256: 64 MB of results, 8 pieces
    bad = c.lenses.copy()
    bad["rcore"][-1] = -1.0
    host = {n: np.full((c.nmodel, c.grid.ny, c.grid.nx), np.nan) for n in ("ax", "ay")}
    n0 = lh.lh_launch_count()
    with pytest.raises(lh.LhError) as e:
        lh.lh_grid_eval_host(bad, c.nmodel, c.nlens, c.grid, **host)
    assert e.value.code == lh.LH_EINVAL and "model 63" in str(e.value)
    assert lh.lh_launch_count() == n0
    assert all(np.isnan(v).all() for v in host.values())


def test_binding_refuses_undersized_or_misplaced_tensors():
    """The C ABI only sees addresses: the binding checks element counts (and the device) before the call."""
    c = li.config(0)
    g = c.grid
    small = torch.empty(g.npix - 1, dtype=torch.float64, device="cuda")
    ok = torch.empty(g.npix, dtype=torch.float64, device="cuda")
    with pytest.raises(ValueError):
        lh.lh_grid_gradient(c.lenses, g, small, ok)
    with pytest.raises(ValueError):
        lh.lh_grid_eval(c.lenses, g, kappa=small)
    with pytest.raises(ValueError):
        lh.lh_grid_gradient_batch(np.concatenate([c.lenses, c.lenses]), 2, c.nlens, g, ok, ok)  # needs 2 * npix
    with pytest.raises(ValueError):
        lh.lh_grid_eval_rows(c.lenses, g, 0, 3, ax=torch.empty(3 * g.nx - 1, dtype=torch.float64, device="cuda"))
    with pytest.raises(ValueError):
        lh.lh_grid_eval_host(c.lenses, 1, c.nlens, g, ax=np.empty(g.npix - 1))
    with pytest.raises(TypeError):
        lh.lh_grid_eval_host(c.lenses, 1, c.nlens, g, ax=ok)  # a device tensor where a host plane is expected


# ------------------------------------------------------------------ multi-GPU: two devices, bench arm
@pytest.mark.skipif(torch.cuda.device_count() < 2, reason="needs two CUDA devices")
def test_two_devices_row_slabs_assemble_the_single_device_map_bitwise():
    """Rank r's slab on device r (lh_grid_eval_rows, current device switched per call), copied into the owner's
    planes over the peer link: bit-identical to the map one device computes alone."""
    c = li.config(3, scale=8)  # 512 x 512, 1000 dPIE: lens chunks through the per-device carry buffers
    g = c.grid
    names = ("ax", "kappa", "mu")
    torch.cuda.set_device(0)
    full = dev_planes(names, (g.ny, g.nx))
    lh.lh_grid_eval(c.lenses, g, **full)
    torch.cuda.synchronize()
    asm = dev_planes(names, (g.ny, g.nx))
    for rank in range(2):
        j0, nrows = li.row_slab(g, rank, 2)
        torch.cuda.set_device(rank)
        lh.lh_set_stream(None)
        out = {n: torch.full((nrows, g.nx), float("nan"), dtype=torch.float64, device=f"cuda:{rank}") for n in names}
        lh.lh_grid_eval_rows(c.lenses, g, j0, nrows, **out)
        torch.cuda.synchronize()
        for n in names:
            asm[n][j0:j0 + nrows].copy_(out[n])  # device-to-device (peer) copy into the owner's plane
    torch.cuda.set_device(0)
    torch.cuda.synchronize()
    for n in names:
        assert torch.equal(asm[n].view(torch.int64), full[n].view(torch.int64))


@pytest.mark.parametrize("assemble", ["peer", "gather"])
def test_bench_strong_scaling_arm_two_ranks_over_gloo(assemble):
    """`bench.py --gpus 2` as the driver launches it (torchrun, one process per rank), with the process group on gloo
    so that two ranks can share this one GPU: the default N > 1 arm shards the ROWS of one map, the
    assembled map equals the single-device map bit for bit, and the line carries the contract's keys.  `peer`: rank 1
    maps rank 0's planes through CUDA IPC and its kernel stores its rows straight into them (on several GPUs the
    same stores cross NVLink); `gather`: one gather after the computation."""
    import json
    import socket
    import subprocess
    import sys

    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    env = dict(os.environ, LH_BENCH_BACKEND="gloo")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", str(port), os.path.join(root, "bench.py"), "--gpus", "2", "--steps", "3",
           "--warmup", "3", "--config", "1", "--no-cpu-baseline", "--assemble", assemble]
    r = subprocess.run(cmd, env=env, cwd=root, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, r.stdout[-2000:]
    d = json.loads(lines[0])
    assert d["n_gpus"] == 2 and d["scaling"] == "strong"
    assert d["gpu_launches"] == 6 and d["gpu_launches_rank0"] == 3  # one launch per rank and step
    assert d["assemble"]["mode"] == assemble
    assert d["assemble"]["bitwise_check"] is True and d["assemble"]["bytes"] == 2 * 1024 * 1024 * 8
    assert d["parity_last_step"]["ok"] and d["e2e"]["same_bits_as_device_planes"] is True
    assert d["config"]["evals_per_step"] == 1024 * 1024 * 100
    assert abs(d["value"] - d["config"]["evals_per_step"] / (d["ms_per_step"] * 1e-3)) < 1e-6 * d["value"]


@pytest.mark.parametrize("assemble", ["peer", "gather"])
def test_bench_by_model_split_of_the_batch_two_ranks_over_gloo(assemble):
    """SURVEY sec. 8(e) split (ii), "for the batch path, models per GPU", through the product and the bench:
    `bench.py --config 4 --gpus 2` (two ranks on this one GPU, process group on gloo) gives rank r the models
    lens_inputs.model_slab(64, r, 2) of the ONE batch via lh_grid_gradient_batch; the assembled [64][ny][nx] planes
    on rank 0 equal its own single-device batch bit for bit; `value` counts the batch once."""
    import json
    import socket
    import subprocess
    import sys

    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    env = dict(os.environ, LH_BENCH_BACKEND="gloo")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", str(port), os.path.join(root, "bench.py"), "--gpus", "2", "--steps", "3",
           "--warmup", "3", "--config", "4", "--no-cpu-baseline", "--assemble", assemble]
    r = subprocess.run(cmd, env=env, cwd=root, capture_output=True, text=True, timeout=900)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, r.stdout[-2000:]
    d = json.loads(lines[0])
    assert d["n_gpus"] == 2 and d["scaling"] == "strong" and "model_slab" in d["config"]["parallelism"]
    # 300 lenses = 2 launches per model; 32 models per rank and step
    assert d["gpu_launches"] == 3 * 64 * 2 and d["gpu_launches_rank0"] == 3 * 32 * 2
    assert d["assemble"]["mode"] == assemble
    assert d["assemble"]["bitwise_check"] is True and d["assemble"]["bytes"] == 2 * 64 * 1024 * 1024 * 8
    assert d["parity_last_step"]["ok"] and d["e2e"]["same_bits_as_device_planes"] is True
    assert d["config"]["evals_per_step"] == 64 * 1024 * 1024 * 300
    assert abs(d["value"] - d["config"]["evals_per_step"] / (d["ms_per_step"] * 1e-3)) < 1e-6 * d["value"]


def test_ipc_export_open_roundtrip_in_another_process():
    """lh_ipc_export / lh_ipc_open / lh_ipc_close: a child process maps a tensor of this process (which sits INSIDE a
    larger allocation of torch's caching allocator, at a non-zero offset), lets lh_grid_eval_rows write two rows of
    a map into it through the mapped address, and this process finds exactly those rows written."""
    import subprocess
    import sys

    c = li.config(1, scale=8)
    g = c.grid
    pad = torch.empty(12345, dtype=torch.float64, device="cuda")  # pushes the next tensor off the segment start
    buf = torch.full((g.ny, g.nx), float("nan"), dtype=torch.float64, device="cuda")
    handle, offset = lh.lh_ipc_export(buf)
    torch.cuda.synchronize()
    child = f"""
import sys, numpy as np
sys.path.insert(0, {os.path.dirname(os.path.dirname(os.path.abspath(__file__)))!r})
import torch, lens_inputs as li, paper_2004_06352_b200 as lh
torch.cuda.set_device(0)
c = li.config(1, scale=8); g = c.grid
p = lh.lh_ipc_open(bytes.fromhex({handle.hex()!r}), {offset})
lh.lh_grid_eval_rows(c.lenses, g, 5, 2, ax=p + 5 * g.nx * 8)
torch.cuda.synchronize()
lh.lh_ipc_close(p)
try:
    lh.lh_ipc_close(p)
except lh.LhError:
    print("second close refused")
"""
    r = subprocess.run([sys.executable, "-c", child], capture_output=True, text=True, timeout=300)
    assert r.returncode == 0 and "second close refused" in r.stdout, r.stderr[-2000:]
    torch.cuda.synchronize()
    ref = run_gpu(c.lenses, g, ("ax",))["ax"]
    got = buf.cpu().numpy()
    assert np.array_equal(got[5:7], ref[5:7]) and np.isnan(got[:5]).all() and np.isnan(got[7:]).all()
    del pad
