"""ctypes binding of the CPU oracle (oracle/lens_oracle.c) -- TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
reference legs may import this.  It never imports the CUDA package
(paper_2004_06352_b200) and the CUDA package never imports it.

`grid()` can fan disjoint row ranges of the single-threaded C routine out over
host threads (ctypes drops the GIL); the arithmetic per pixel is unchanged, so
the result is identical to the one-thread run bit for bit.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from concurrent.futures import ThreadPoolExecutor

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lens_oracle.c")
_LIB = os.path.join(_HERE, "liblens_oracle.so")

PLANES = ("ax", "ay", "a11", "a12", "a22", "kappa", "gamma1", "gamma2", "mu")

# numpy view of the oracle's own 64-byte record `orc_lens`
ORC_LENS_DTYPE = np.dtype(
    [("type", "<i4"), ("pad_", "<i4"), ("x", "<f8"), ("y", "<f8"), ("ellipticity", "<f8"), ("theta", "<f8"),
     ("rcore", "<f8"), ("rcut", "<f8"), ("b0", "<f8")]
)


class _Deriv(C.Structure):
    _fields_ = [(n, C.c_double) for n in ("ax", "ay", "a11", "a12", "a22")]


class _Planes(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in PLANES]


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (no FMA contraction). Returns the .so path."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fPIC", "-shared", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.orc_eps_from_ehat.restype = C.c_double
        L.orc_eps_from_ehat.argtypes = [C.c_double]
        L.orc_lens_deriv.restype = None
        L.orc_lens_deriv.argtypes = [C.c_void_p, C.c_double, C.c_double, C.POINTER(_Deriv)]
        L.orc_point.restype = None
        L.orc_point.argtypes = [C.c_void_p, C.c_int, C.c_double, C.c_double, C.POINTER(_Deriv)]
        L.orc_epilogue.restype = None
        L.orc_epilogue.argtypes = [C.c_double] * 3 + [C.POINTER(C.c_double)] * 4
        L.orc_points.restype = None
        L.orc_points.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_size_t, C.POINTER(_Planes)]
        L.orc_grid_rows.restype = None
        L.orc_grid_rows.argtypes = [C.c_void_p, C.c_int, C.c_double, C.c_double, C.c_double, C.c_int, C.c_int,
                                    C.c_int, C.c_int, C.POINTER(_Planes)]
        _lib = L
    return _lib


def _as_lenses(lenses) -> np.ndarray:
    a = np.ascontiguousarray(lenses)
    if a.dtype.itemsize != 64:
        raise ValueError("lens records must be 64 bytes")
    return a.view(ORC_LENS_DTYPE).reshape(-1)


def eps_from_ehat(ehat: float) -> float:
    return lib().orc_eps_from_ehat(float(ehat))


def lens_deriv(one_lens, X: float, Y: float) -> dict:
    """(ax, ay, a11, a12, a22) of a single potential at one point."""
    a = _as_lenses(one_lens)
    d = _Deriv()
    lib().orc_lens_deriv(a.ctypes.data, float(X), float(Y), C.byref(d))
    return {n: getattr(d, n) for n in ("ax", "ay", "a11", "a12", "a22")}


def point(lenses, X: float, Y: float) -> dict:
    """Superposed (ax, ay, a11, a12, a22) + epilogue at one point."""
    a = _as_lenses(lenses)
    d = _Deriv()
    lib().orc_point(a.ctypes.data, len(a), float(X), float(Y), C.byref(d))
    out = {n: getattr(d, n) for n in ("ax", "ay", "a11", "a12", "a22")}
    out.update(epilogue(d.a11, d.a12, d.a22))
    return out


def epilogue(a11: float, a12: float, a22: float) -> dict:
    k, g1, g2, mu = (C.c_double() for _ in range(4))
    lib().orc_epilogue(a11, a12, a22, C.byref(k), C.byref(g1), C.byref(g2), C.byref(mu))
    return {"kappa": k.value, "gamma1": g1.value, "gamma2": g2.value, "mu": mu.value}


def points(lenses, xs, ys, planes=PLANES) -> dict:
    """All requested planes at arbitrary points (xs[k], ys[k])."""
    a = _as_lenses(lenses)
    xs = np.ascontiguousarray(xs, dtype=np.float64)
    ys = np.ascontiguousarray(ys, dtype=np.float64)
    assert xs.shape == ys.shape
    out = {n: np.empty(xs.size, dtype=np.float64) for n in planes}
    P = _Planes(**{n: out[n].ctypes.data for n in planes})
    lib().orc_points(a.ctypes.data, len(a), xs.ctypes.data, ys.ctypes.data, xs.size, C.byref(P))
    return {n: v.reshape(xs.shape) for n, v in out.items()}


def grid(lenses, x0: float, y0: float, dx: float, nx: int, ny: int, planes=PLANES, threads: int = 1,
         rows=None) -> dict:
    """Requested planes on the regular grid, each [ny, nx].  `rows=(j0, j1)` limits
    the rows written (the rest of each plane stays NaN)."""
    a = _as_lenses(lenses)
    out = {n: np.full((ny, nx), np.nan, dtype=np.float64) for n in planes}
    P = _Planes(**{n: out[n].ctypes.data for n in planes})
    j0, j1 = (0, ny) if rows is None else rows
    L = lib()

    def run(r):
        L.orc_grid_rows(a.ctypes.data, len(a), x0, y0, dx, nx, ny, r[0], r[1], C.byref(P))

    threads = max(1, min(int(threads), j1 - j0))
    if threads == 1:
        run((j0, j1))
    else:
        cuts = np.linspace(j0, j1, threads * 4 + 1).astype(int)
        jobs = [(int(cuts[k]), int(cuts[k + 1])) for k in range(len(cuts) - 1) if cuts[k + 1] > cuts[k]]
        with ThreadPoolExecutor(threads) as ex:
            list(ex.map(run, jobs))
    return out


def stats(lenses, nmodel: int, nlens: int, x0: float, y0: float, dx: float, nx: int, ny: int, planes=PLANES,
          threads: int = 1) -> tuple:
    """Per-pixel mean and variance of each plane over the `nmodel` lens models of a batch (PAPER.md:101, :114:
    "map variances" over the tested parameter combinations).  The paper gives no formula; reading R21
    (DESIGN.md): POPULATION variance.  Plain two-pass definition, in the order written:
        mean = (1/M) sum_m P_m ;   var = (1/M) sum_m (P_m - mean)^2
    with every P_m produced by grid() above.  Returns (mean, var), dicts name -> [ny, nx]."""
    a = _as_lenses(lenses)
    assert len(a) == nmodel * nlens and nmodel >= 1
    maps = [grid(a[m * nlens:(m + 1) * nlens], x0, y0, dx, nx, ny, planes=planes, threads=threads)
            for m in range(nmodel)]
    mean, var = {}, {}
    with np.errstate(invalid="ignore", over="ignore"):
        for n in planes:
            s = np.zeros((ny, nx), dtype=np.float64)
            for m in range(nmodel):
                s = s + maps[m][n]
            mean[n] = s / nmodel
            q = np.zeros((ny, nx), dtype=np.float64)
            for m in range(nmodel):
                d = maps[m][n] - mean[n]
                q = q + d * d
            var[n] = q / nmodel
    return mean, var


# ---------------------------------------------------------------- NEXT row f1: source plane, delensing
ORC_IMAGE_DTYPE = np.dtype([("source", "<i4"), ("pad_", "<i4"), ("triangle", "<i8"), ("x", "<f8"), ("y", "<f8")])


def source_plane(ax, ay, x0: float, y0: float, dx: float):
    """beta = theta - alpha on the grid (eq. 1): returns (bx, by), each [ny, nx]."""
    ax = np.ascontiguousarray(ax, dtype=np.float64)
    ay = np.ascontiguousarray(ay, dtype=np.float64)
    ny, nx = ax.shape
    bx, by = np.empty_like(ax), np.empty_like(ay)
    L = lib()
    L.orc_source_plane.restype = None
    L.orc_source_plane.argtypes = [C.c_void_p, C.c_void_p, C.c_double, C.c_double, C.c_double, C.c_int, C.c_int,
                                   C.c_void_p, C.c_void_p]
    L.orc_source_plane(ax.ctypes.data, ay.ctypes.data, x0, y0, dx, nx, ny, bx.ctypes.data, by.ctypes.data)
    return bx, by


def delens(ax, ay, x0: float, y0: float, dx: float, sources, max_images: int = 1 << 20):
    """Brute-force image search (readings R22): returns (images[ORC_IMAGE_DTYPE], found)."""
    ax = np.ascontiguousarray(ax, dtype=np.float64)
    ay = np.ascontiguousarray(ay, dtype=np.float64)
    ny, nx = ax.shape
    src = np.ascontiguousarray(sources, dtype=np.float64).reshape(-1, 2)
    images = np.zeros(max_images, dtype=ORC_IMAGE_DTYPE)
    L = lib()
    L.orc_delens.restype = C.c_longlong
    L.orc_delens.argtypes = [C.c_void_p, C.c_void_p, C.c_double, C.c_double, C.c_double, C.c_int, C.c_int, C.c_void_p,
                             C.c_int, C.c_void_p, C.c_longlong]
    found = L.orc_delens(ax.ctypes.data, ay.ctypes.data, x0, y0, dx, nx, ny, src.ctypes.data, len(src),
                         images.ctypes.data, max_images)
    return images[: min(found, max_images)], int(found)


# ---------------------------------------------------------------- NEXT row f3: chi^2 of image constraints
ORC_CONSTRAINT_DTYPE = np.dtype([("source", "<i4"), ("pad_", "<i4"), ("x", "<f8"), ("y", "<f8"), ("sigma", "<f8")])


def chi2(lenses, x0: float, y0: float, dx: float, nx: int, ny: int, constraints, nsources: int) -> dict:
    """PAPER.md:76-81 eq. 6 through the four stages of sec. 4.2 (readings R23): returns chi2, sources [N, 2],
    predicted [K, 2] (the back-and-forth lensed constraint x_k), nimages."""
    a = _as_lenses(lenses)
    c = np.ascontiguousarray(constraints)
    assert c.dtype.itemsize == 32
    K = len(c)
    src = np.empty((max(nsources, 1), 2), dtype=np.float64)
    pred = np.empty((max(K, 1), 2), dtype=np.float64)
    nim = C.c_longlong(0)
    L = lib()
    L.orc_chi2.restype = C.c_double
    L.orc_chi2.argtypes = [C.c_void_p, C.c_int, C.c_double, C.c_double, C.c_double, C.c_int, C.c_int, C.c_void_p, C.c_int,
                           C.c_int, C.c_void_p, C.c_void_p, C.POINTER(C.c_longlong)]
    v = L.orc_chi2(a.ctypes.data, len(a), x0, y0, dx, nx, ny, c.ctypes.data, K, nsources, src.ctypes.data,
                   pred.ctypes.data, C.byref(nim))
    return {"chi2": float(v), "sources": src[:nsources], "predicted": pred[:K], "nimages": int(nim.value)}
