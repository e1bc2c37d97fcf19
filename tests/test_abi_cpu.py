"""CPU-only checks of the boundary: liblh.so loads, exports every symbol include/lh.h
declares, and the host logic (step a1: validation, class sorting, per-lens constants;
argument checks that fail before any CUDA work) behaves.  No compute calls here."""
import ctypes
import math
import os
import re

import numpy as np
import pytest

import lens_inputs as li
import paper_2004_06352_b200 as lh

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions(headers=("lh.h", "lh_diag.h")):
    """every function the headers declare; the lh_debug_* calls exist in the checking build only"""
    names = set()
    for h in headers:
        src = open(os.path.join(ROOT, "include", h)).read()
        src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
        src = re.sub(r"#ifdef LH_BOUNDS_CHECK.*?#endif", "", src, flags=re.S)
        names |= set(re.findall(r"\b(lh_[a-z0-9_]+)\s*\(", src))
    return sorted(names)


def test_boundary_header_holds_the_method_only():
    """include/lh.h is the boundary of SURVEY.md sec. 8(b) and its documented extensions; probes and test hooks are
    declared in include/lh_diag.h."""
    method, diag = set(declared_functions(("lh.h",))), set(declared_functions(("lh_diag.h",)))
    assert diag == {"lh_launch_count", "lh_fp64_peak_probe", "lh_math_host_eval", "lh_source_hash"}
    assert not method & diag and not any("debug" in n or "probe" in n for n in method)


def test_library_was_built_from_this_tree():
    lh._build.build()
    assert lh.lh_source_hash() == lh._build.source_hash()


def test_library_exports_every_declared_symbol():
    lh._build.build()
    lib = ctypes.CDLL(lh.library_path())
    names = declared_functions()
    assert {"lh_grid_gradient", "lh_grid_hessian", "lh_lens_maps", "lh_grid_gradient_batch", "lh_grid_eval",
            "lh_grid_eval_batch", "lh_grid_eval_host", "lh_set_stream", "lh_last_error"} <= set(names)
    for n in names:
        assert hasattr(lib, n), f"{n} declared in lh.h but not exported"
    assert lh.lh_version().endswith("sm_100a")


def test_binding_has_the_same_names():
    for n in declared_functions():
        assert callable(getattr(lh, n)), n


def test_struct_layouts_match_header():
    assert li.LENS_DTYPE.itemsize == 64
    assert ctypes.sizeof(lh.lh_grid) == 32 and ctypes.sizeof(lh.lh_outputs) == 72
    offs = {n: li.LENS_DTYPE.fields[n][1] for n in li.LENS_DTYPE.names}
    assert offs == {"type": 0, "_pad": 4, "x": 8, "y": 16, "ellipticity": 24, "theta": 32, "rcore": 40,
                    "rcut": 48, "b0": 56}


def test_pack_sorts_by_class_and_is_stable():
    c = li.config(2)
    table, begin = lh.lh_pack_model(c.lenses)
    assert list(begin) == [0, 402, 451, 500, 500]  # dPIE | NSIE | SIS | extreme-ellipticity
    for cls, t in ((0, li.DPIE), (1, li.NSIE), (2, li.SIS)):
        src = c.lenses[c.lenses["type"] == t]
        sl = table[begin[cls]:begin[cls + 1]]
        assert np.array_equal(sl[:, 0], src["x"]) and np.array_equal(sl[:, 1], src["y"])  # index order kept


def test_pack_routes_extreme_ellipticity_to_its_own_class():
    """eps > 0.85 (e-hat > 0.98694, axis ratio < 0.081) leaves the fast dPIE / NSIE classes (lh_pack.h)."""
    L = li.make_lenses(5)
    L[0] = (li.DPIE, 0, 0.0, 0.0, 0.986, 0.1, 0.1, 10.0, 1.0)    # eps = 0.8451: fast
    L[1] = (li.DPIE, 0, 1.0, 0.0, 0.988, 0.1, 0.1, 10.0, 1.0)    # eps = 0.8558: extreme
    L[2] = (li.NSIE, 0, 2.0, 0.0, 0.99999, 0.1, 0.1, 0.0, 1.0)   # extreme, no cut
    L[3] = (li.SIS, 0, 3.0, 0.0, 0.99999, 0.0, 0.0, 0.0, 1.0)    # SIS ignores ellipticity
    L[4] = (li.NSIE, 0, 4.0, 0.0, 0.5, 0.1, 0.1, 0.0, 1.0)
    t, begin = lh.lh_pack_model(L)
    assert list(begin) == [0, 1, 2, 3, 5]
    assert list(t[:, 0]) == [0.0, 4.0, 3.0, 1.0, 2.0]
    assert t[3, 17] == 100.0 and t[4, 17] == 0.0 and t[4, 7] == 0.0  # rt^2; 0 marks "no cut term" in the extreme class
    e = 0.988
    assert t[3, 21] == e / (1 + math.sqrt(1 - e * e))  # eps slot


def test_pack_constants():
    """Per-lens constants (lh_pack.h): recomputed here from their definitions."""
    L = li.lens(li.DPIE, 1.5, -2.0, 0.6, 0.3, 0.25, 40.0, 3.0)
    t, _ = lh.lh_pack_model(L)
    k = t[0]
    eps = 1.0 / 3.0  # e-hat 0.6 <-> eps 1/3 (reading R2)
    o, p, m = 1 - eps ** 2, (1 + eps) ** 2, (1 - eps) ** 2
    T = 3.0 * 40.0 / (40.0 - 0.25)
    sg = 2 * math.sqrt(eps)
    kk = o / sg  # the lens frame is carried scaled by k = o / (2 sqrt eps)
    G, TF = T * kk, T * kk * p / sg ** 2
    want = [1.5, -2.0, math.cos(0.3), math.sin(0.3), kk * kk / p, kk * kk / m, kk * kk * 0.25 ** 2, kk * kk * 40.0 ** 2,
            p / sg * 0.25, p / sg * 40.0, m / sg * 0.25, m / sg * 40.0, math.cos(0.3) * G, math.sin(0.3) * G, G, TF,
            0.25 ** 2, 40.0 ** 2, -4 * eps * math.cos(0.6) * TF, -2 * eps * math.sin(0.6) * TF,
            kk * kk * (40.0 ** 2 - 0.25 ** 2), eps, sg, T]
    assert np.allclose(k, want, rtol=1e-15, atol=0)
    # circular lens: 2 sqrt(eps) is never below 2^-40 (the scaled frame then takes the eps -> 0 limit exactly)
    k0 = lh.lh_pack_model(li.lens(li.DPIE, 0.0, 0.0, 0.0, 0.0, 0.25, 40.0, 3.0))[0][0]
    assert k0[22] == 2.0 ** -40 and k0[14] == T * 2.0 ** 40 and k0[13] == 0.0 and k0[18] == 0.0 and k0[19] == 0.0
    assert k0[4] == 2.0 ** 80 and k0[8] == 0.25 * 2.0 ** 40
    # SIS: only the centre and b0 are used
    ks = lh.lh_pack_model(li.lens(li.SIS, 2.0, 3.0, 0.0, 0.0, 0.0, 0.0, 0.7))[0][0]
    assert ks[0] == 2.0 and ks[1] == 3.0 and ks[14] == 0.7


@pytest.mark.parametrize("field,value,ok", [
    ("type", 7, False), ("ellipticity", 1.0, False), ("ellipticity", -0.1, False), ("ellipticity", 0.0, True),
    ("rcore", 0.0, False), ("rcut", 0.05, False), ("b0", float("nan"), False), ("x", float("inf"), False),
    ("theta", float("nan"), False), ("b0", 0.0, True), ("b0", -1.0, False),
])
def test_pack_validation(field, value, ok):
    L = li.lens(li.DPIE, 0.0, 0.0, 0.3, 0.1, 0.1, 10.0, 1.0)
    L[field][0] = value
    if ok:
        lh.lh_pack_model(L, validate_only=True)
    else:
        with pytest.raises(lh.LhError) as e:
            lh.lh_pack_model(L, validate_only=True)
        assert e.value.code == lh.LH_EINVAL and "lens 0" in str(e.value)


def test_sis_and_nsie_ignore_unused_fields():
    lh.lh_pack_model(li.lens(li.SIS, 0, 0, float("nan"), float("nan"), -1.0, float("nan"), 1.0), validate_only=True)
    lh.lh_pack_model(li.lens(li.NSIE, 0, 0, 0.2, 0.0, 0.1, float("nan"), 1.0), validate_only=True)
    with pytest.raises(lh.LhError):
        lh.lh_pack_model(li.lens(li.NSIE, 0, 0, 0.2, 0.0, 0.0, 1.0, 1.0), validate_only=True)


def test_argument_errors_before_any_cuda_work():
    c = li.config(0)
    g = c.grid
    bad_grids = [li.Grid(g.x0, g.y0, 0.0, 8, 8), li.Grid(g.x0, g.y0, g.dx, 0, 8), li.Grid(g.x0, g.y0, g.dx, 8, -1),
                 li.Grid(float("nan"), g.y0, g.dx, 8, 8), li.Grid(g.x0, g.y0, -1.0, 8, 8),
                 li.Grid(g.x0, g.y0, g.dx, 2 ** 20, 2 ** 20)]
    for bg in bad_grids:
        with pytest.raises(lh.LhError) as e:
            lh.lh_grid_gradient(c.lenses, bg, 256, 512)
        assert e.value.code == lh.LH_EINVAL
    with pytest.raises(lh.LhError) as e:  # NULL output
        lh.lh_grid_gradient(c.lenses, g, None, 512)
    assert e.value.code == lh.LH_EINVAL
    with pytest.raises(lh.LhError) as e:  # nothing requested
        lh.lh_grid_eval(c.lenses, g)
    assert e.value.code == lh.LH_EINVAL
    with pytest.raises(lh.LhError) as e:  # misaligned
        lh.lh_grid_gradient(c.lenses, g, 260, 512)
    assert "aligned" in str(e.value)
    with pytest.raises(lh.LhError) as e:  # host address is not device memory
        buf = np.zeros(g.npix)
        lh.lh_grid_gradient(c.lenses, g, buf.ctypes.data, buf.ctypes.data)
    assert e.value.code == lh.LH_EINVAL
    with pytest.raises(lh.LhError):
        lh.lh_grid_gradient_batch(c.lenses[:0], 0, 10, g, 256, 512)
    assert lh.lh_launch_count() == 0


def test_missing_library_fails_loudly(monkeypatch, tmp_path):
    """No CPU fallback: without liblh.so the binding raises."""
    monkeypatch.setattr(lh, "_lib", None)
    monkeypatch.setattr(lh._build, "LIB", str(tmp_path / "nope.so"))
    with pytest.raises(ImportError):
        lh.lh_version()


def test_binding_checks_host_plane_sizes_before_the_call():
    """lh_grid_eval_host writes nmodel*ny*nx doubles into each HOST plane; the C ABI cannot know the size of the
    caller's array, the binding can: too small a plane is refused before anything is called (no GPU needed)."""
    c = li.config(0)
    g = c.grid
    with pytest.raises(ValueError):
        lh.lh_grid_eval_host(c.lenses, 1, c.nlens, g, ax=np.empty(g.npix - 1))
    with pytest.raises(ValueError):
        lh.lh_grid_eval_host(np.concatenate([c.lenses, c.lenses]), 2, c.nlens, g, ax=np.empty(g.npix))
    with pytest.raises(TypeError):
        lh.lh_grid_eval_host(c.lenses, 1, c.nlens, g, ax=np.empty(g.npix, dtype=np.float32))


def test_row_slab_and_ipc_argument_errors_before_any_cuda_work():
    """lh_grid_eval_rows / lh_grid_eval_rows_host: a slab outside the grid; the IPC wrappers: NULL / unknown pointers."""
    c = li.config(0)
    g = c.grid
    for j0, nrows in ((-1, 2), (0, 0), (g.ny - 1, 2), (g.ny, 1)):
        with pytest.raises(lh.LhError) as e:
            lh.lh_grid_eval_rows(c.lenses, g, j0, nrows, ax=256)
        assert e.value.code == lh.LH_EINVAL and "slab" in str(e.value)
        with pytest.raises(lh.LhError) as e:
            lh.lh_grid_eval_rows_host(c.lenses, g, j0, nrows, ax=np.empty(max(nrows, 1) * g.nx))
        assert e.value.code == lh.LH_EINVAL and "slab" in str(e.value)
    with pytest.raises(lh.LhError) as e:  # a bad lens is reported before anything else happens
        bad = c.lenses.copy()
        bad["rcut"][2] = 0.0
        lh.lh_grid_eval_rows_host(bad, g, 0, 4, ax=np.empty(4 * g.nx))
    assert e.value.code == lh.LH_EINVAL and "lens 2" in str(e.value)
    with pytest.raises(lh.LhError) as e:
        lh.lh_ipc_export(0)
    assert e.value.code == lh.LH_EINVAL
    buf = np.zeros(16)
    with pytest.raises(lh.LhError) as e:  # host memory cannot be exported
        lh.lh_ipc_export(buf.ctypes.data)
    assert e.value.code == lh.LH_EINVAL
    with pytest.raises(lh.LhError) as e:
        lh.lh_ipc_close(12345 * 8)
    assert e.value.code == lh.LH_EINVAL
    assert lh.lh_launch_count() == 0
