"""Child process of tests/test_gpu_bounds.py: runs with LH_LIBRARY = the CHECKING build of the library
(-DLH_BOUNDS_CHECK, paper_2004_06352_b200/liblh_check.so), in which every global-memory access of the
superposition kernel is compared with the address ranges the launch may touch.  The caller's buffers are
registered here EXACTLY (no slack); the library adds its own carry / statistics / table buffers exactly as large
as each job needs them.  Prints one JSON line: violations per case, parity per case, and the negative control."""
import ctypes as C
import json
import os
import sys

import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
for p in (ROOT, os.path.join(ROOT, "tests")):
    if p not in sys.path:
        sys.path.insert(0, p)

import lens_inputs as li  # noqa: E402
import oracle  # noqa: E402
import paper_2004_06352_b200 as lh  # noqa: E402
from parity import check_planes, stats_violation  # noqa: E402

lib = C.CDLL(lh.library_path())
# The checking library is git-ignored and may have travelled with the tree from another build: refuse to vouch for
# the kernel with a library that was compiled from other sources than the ones in this tree.
from paper_2004_06352_b200 import _build  # noqa: E402

lib.lh_source_hash.restype = C.c_char_p
if lib.lh_source_hash().decode() != _build.source_hash():
    sys.exit(f"{lh.library_path()} was built from other sources (hash {lib.lh_source_hash().decode()[:16]}..., tree "
             f"{_build.source_hash()[:16]}...): rebuild it with __graft_entry__.build()")
lib.lh_debug_bounds_add.argtypes = [C.c_void_p, C.c_ulonglong]
lib.lh_debug_violations.restype = C.c_longlong


def allow(*tensors):
    lib.lh_debug_bounds_reset()
    for t in tensors:
        assert lib.lh_debug_bounds_add(t.data_ptr(), t.numel() * t.element_size()) == 0


def planes(names, shape):
    return {n: torch.full(shape, float("nan"), dtype=torch.float64, device="cuda") for n in names}


def ref(L, g, names):
    need = set(names) | ({"kappa", "gamma1", "gamma2"} if "mu" in names else set())
    return oracle.grid(L, g.x0, g.y0, g.dx, g.nx, g.ny, planes=tuple(sorted(need)), threads=os.cpu_count() or 1)


def host(d):
    torch.cuda.synchronize()
    return {n: v.cpu().numpy() for n, v in d.items()}


report = {"library": os.path.basename(lh.library_path()), "cases": {}}


def case(name, fn):
    worst = fn()
    report["cases"][name] = {"violations": int(lib.lh_debug_violations()), "worst_parity_ratio": float(worst)}


torch.cuda.set_device(0)
c2, c3 = li.config(2), li.config(3)


def ragged():
    w = 0.0
    for nx, ny in [(1, 1), (9, 1), (65, 5), (129, 2), (200, 13)]:
        g = li.Grid(x0=-20.3, y0=11.7, dx=0.37, nx=nx, ny=ny)
        o = planes(li.ALL_PLANES, (ny, nx))
        allow(*o.values())
        lh.lh_grid_eval(c2.lenses[:130], g, **o)
        w = max(w, max(check_planes(host(o), ref(c2.lenses[:130], g, li.ALL_PLANES), "ragged").values()))
    return w


def chunked():
    w = 0.0
    for nlens in (161, 481, 1000):
        g = li.Grid(x0=-30.0, y0=-30.0, dx=0.9, nx=70, ny=9)
        o = planes(li.ALL_PLANES, (g.ny, g.nx))
        allow(*o.values())
        lh.lh_grid_eval(c3.lenses[:nlens], g, **o)
        w = max(w, max(check_planes(host(o), ref(c3.lenses[:nlens], g, li.ALL_PLANES), "chunked").values()))
    return w


def row_halves():
    # one chunked model on a grid large enough for the two-chain split of its rows (lh_kernels.cu `halves`): ragged
    # width, odd height, so that the half boundary and the last tile row are both exercised
    g = li.Grid(x0=-90.0, y0=-91.0, dx=0.18, nx=1000, ny=1023)
    names = ("ax", "kappa", "mu")
    o = planes(names, (g.ny, g.nx))
    allow(*o.values())
    lh.lh_grid_eval(c3.lenses[:161], g, **o)
    return max(check_planes(host(o), ref(c3.lenses[:161], g, names), "row halves").values())


def slabs():
    c = li.config(2, scale=16)
    g = li.Grid(x0=c.grid.x0 + 0.1, y0=c.grid.y0 + 0.3, dx=c.grid.dx * 1.1, nx=c.grid.nx, ny=c.grid.ny)
    full = ref(c.lenses, g, ("ax", "kappa", "mu"))
    w = 0.0
    for rank in range(3):
        j0, nrows = li.row_slab(g, rank, 3)
        o = planes(("ax", "kappa", "mu"), (nrows, g.nx))
        allow(*o.values())
        lh.lh_grid_eval_rows(c.lenses, g, j0, nrows, **o)
        got = host(o)
        w = max(w, max(check_planes(got, {n: v[j0:j0 + nrows] for n, v in full.items()}, "slab").values()))
        hp = {n: np.full((nrows, g.nx), np.nan) for n in ("ax", "kappa", "mu")}
        allow()  # host entry point: only the library's own device planes are touched
        lh.lh_grid_eval_rows_host(c.lenses, g, j0, nrows, **hp)
        assert all(np.array_equal(hp[n], got[n], equal_nan=True) for n in hp)
    return w


def batches():
    w = 0.0
    rng = np.random.default_rng(5)
    nmodel, nlens = 50, 7  # models share launches (blockIdx.y)
    L = c2.lenses[rng.integers(0, len(c2.lenses), nmodel * nlens)]
    g = li.Grid(x0=-40.0, y0=-25.0, dx=0.77, nx=131, ny=5)
    o = planes(("ax", "a12", "mu"), (nmodel, g.ny, g.nx))
    allow(*o.values())
    lh.lh_grid_eval_batch(L, nmodel, nlens, g, **o)
    got = host(o)
    for m in (0, 21, 49):
        w = max(w, max(check_planes({n: got[n][m] for n in got}, ref(L[m * nlens:(m + 1) * nlens], g, tuple(got)), "batch").values()))
    c4 = li.config(4, scale=16)  # chunked models: two launch chains, two carry buffers
    o = planes(c4.outputs, (c4.nmodel, c4.grid.ny, c4.grid.nx))
    allow(*o.values())
    lh.lh_grid_gradient_batch(c4.lenses, c4.nmodel, c4.nlens, c4.grid, o["ax"], o["ay"])
    got = host(o)
    for m in (0, 1, 62, 63):
        w = max(w, max(check_planes({n: got[n][m] for n in got}, ref(c4.lenses[m * 300:(m + 1) * 300], c4.grid, c4.outputs), "cfg4").values()))
    hp = {n: np.full((c4.nmodel, c4.grid.ny, c4.grid.nx), np.nan) for n in c4.outputs}
    allow()
    lh.lh_grid_eval_host(c4.lenses, c4.nmodel, c4.nlens, c4.grid, **hp)
    assert all(np.array_equal(hp[n], got[n]) for n in hp)
    return w


def stats_and_shared():
    c4 = li.config(4, scale=16)
    g = c4.grid
    names = ("ax", "kappa", "gamma1")
    mean, var = planes(names, (g.ny, g.nx)), planes(names, (g.ny, g.nx))
    allow(*mean.values(), *var.values())
    lh.lh_grid_stats_batch(c4.lenses, c4.nmodel, c4.nlens, g, mean, var)
    rm, rv = oracle.stats(c4.lenses, c4.nmodel, c4.nlens, g.x0, g.y0, g.dx, g.nx, g.ny, planes=names, threads=os.cpu_count() or 1)
    hm, hv = host(mean), host(var)
    w = 0.0
    for n in names:
        w = max(w, *stats_violation(hm[n], hv[n], rm[n], rv[n], c4.nmodel))
    L = c4.lenses.reshape(c4.nmodel, c4.nlens)
    o = planes(("ax", "ay"), (c4.nmodel, g.ny, g.nx))
    allow(*o.values())
    lh.lh_grid_eval_batch_shared(L[0, 2:].copy(), np.ascontiguousarray(L[:, :2]).reshape(-1), c4.nmodel, 2, g, **o)
    got = host(o)
    w = max(w, max(check_planes({n: got[n][17] for n in got}, ref(c4.lenses[17 * 300:18 * 300], g, ("ax", "ay")), "shared").values()))
    return w


def points():
    rng = np.random.default_rng(127)
    xs, ys = rng.uniform(-90, 90, 127), rng.uniform(-90, 90, 127)
    dx_, dy_ = torch.as_tensor(xs, device="cuda"), torch.as_tensor(ys, device="cuda")
    o = planes(li.ALL_PLANES, (127,))
    allow(dx_, dy_, *o.values())
    lh.lh_points_eval(c2.lenses, dx_, dy_, **o)
    return max(check_planes(host(o), oracle.points(c2.lenses, xs, ys, planes=li.ALL_PLANES), "points").values())


for name, fn in (("ragged grids, all planes", ragged), ("lens chunks through the carry buffer", chunked),
                 ("one chunked model, row halves on two chains", row_halves),
                 ("row slabs of a chunked model, device and host planes", slabs),
                 ("batches: shared launches, two launch chains, host entry", batches),
                 ("statistics (two chains + merge) and shared-lens batch", stats_and_shared), ("arbitrary points", points)):
    case(name, fn)

# negative control: the checker must SEE an access outside the registered ranges -- allow one element less than the
# plane holds; the store that covers the last pixel (a double2: the last TWO pixels) must be refused -- counted and
# skipped, so those two elements keep their NaN and everything before them is written
c0 = li.config(0)
o = planes(("ax",), (c0.grid.ny, c0.grid.nx))
lib.lh_debug_bounds_reset()
lib.lh_debug_bounds_add(o["ax"].data_ptr(), (o["ax"].numel() - 1) * 8)
lh.lh_grid_eval(c0.lenses, c0.grid, **o)
v = int(lib.lh_debug_violations())
a = host(o)["ax"].ravel()
report["negative_control"] = {"violations": v, "last_element_untouched": bool(np.isnan(a[-1])),
                              "all_others_written": bool(not np.isnan(a[:-2]).any())}
print("BOUNDS_REPORT " + json.dumps(report))
