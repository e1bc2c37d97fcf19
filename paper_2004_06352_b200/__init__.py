"""paper_2004_06352_b200 -- thin Python binding of liblh.so (include/lh.h).

Argument marshalling only: every step of the hot path runs in the CUDA kernels
behind the C ABI.  PyTorch is used by callers for device memory and streams; this
module needs nothing but ctypes + numpy and fails loudly when the CUDA library is
missing -- there is no CPU fallback (and it never imports `oracle`).

Names mirror the C ABI one to one:
    lh_grid_gradient, lh_grid_hessian, lh_lens_maps, lh_grid_gradient_batch,
    lh_grid_eval, lh_grid_eval_batch, lh_grid_eval_host, lh_grid_eval_rows_host, lh_grid_eval_noalloc, lh_grid_stats_batch, lh_pack_model, lh_set_stream,
    lh_ipc_export, lh_ipc_open, lh_ipc_close, lh_last_error, lh_launch_count, lh_fp64_peak_probe, lh_math_host_eval,
    lh_version, lh_source_hash (the diagnostics are declared in include/lh_diag.h)
Outputs may be torch CUDA tensors (float64, contiguous), anything with a
`data_ptr()`, or raw integer device addresses.
"""
from __future__ import annotations

import ctypes as C
import os
import sys

import numpy as np

from . import _build

LH_OK, LH_EINVAL, LH_ECUDA = 0, -1, -2
LH_DPIE, LH_NSIE, LH_SIS = 0, 1, 2
PLANES = ("ax", "ay", "a11", "a12", "a22", "kappa", "gamma1", "gamma2", "mu")


class LhError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"liblh error {code}: {msg}")
        self.code = code


class lh_grid(C.Structure):
    _fields_ = [("x0", C.c_double), ("y0", C.c_double), ("dx", C.c_double), ("nx", C.c_int32), ("ny", C.c_int32)]


class lh_outputs(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in PLANES]


_lib = None


def library_path() -> str:
    return os.environ.get("LH_LIBRARY", _build.LIB)


def _load():
    global _lib
    if _lib is None:
        path = os.environ.get("LH_LIBRARY", _build.LIB)  # LH_LIBRARY: another build of the same library
        if not os.path.exists(path):
            raise ImportError(
                f"{path} is missing: build it with `python -m paper_2004_06352_b200._build` "
                "(or __graft_entry__.build()). There is no CPU fallback."
            )
        L = C.CDLL(path)
        vp, ci, dp = C.c_void_p, C.c_int, C.c_void_p
        gp = C.POINTER(lh_grid)
        op = C.POINTER(lh_outputs)
        L.lh_grid_gradient.argtypes = [vp, ci, gp, dp, dp]
        L.lh_grid_hessian.argtypes = [vp, ci, gp, dp, dp, dp]
        L.lh_lens_maps.argtypes = [vp, ci, gp, dp, dp, dp, dp]
        L.lh_grid_gradient_batch.argtypes = [vp, ci, ci, gp, dp, dp]
        L.lh_grid_eval.argtypes = [vp, ci, gp, op]
        L.lh_grid_eval_batch.argtypes = [vp, ci, ci, gp, op]
        L.lh_grid_eval_host.argtypes = [vp, ci, ci, gp, op]
        L.lh_grid_eval_rows_host.argtypes = [vp, ci, gp, ci, ci, op]
        L.lh_grid_eval_rows_host.restype = ci
        L.lh_grid_stats_batch.argtypes = [vp, ci, ci, gp, op, op]
        L.lh_grid_stats_batch.restype = ci
        L.lh_chi2.argtypes = [vp, ci, gp, vp, ci, ci, dp, dp, dp, vp]
        L.lh_chi2.restype = ci
        L.lh_points_eval.argtypes = [vp, ci, dp, dp, C.c_longlong, op]
        L.lh_points_eval.restype = ci
        L.lh_grid_eval_rows.argtypes = [vp, ci, gp, ci, ci, op]
        L.lh_grid_eval_rows.restype = ci
        L.lh_grid_eval_noalloc.argtypes = [vp, ci, gp, ci, ci, op]
        L.lh_grid_eval_noalloc.restype = ci
        L.lh_grid_eval_batch_shared.argtypes = [vp, ci, vp, ci, ci, gp, op]
        L.lh_grid_eval_batch_shared.restype = ci
        L.lh_source_plane.argtypes = [dp, dp, gp, dp, dp]
        L.lh_source_plane.restype = ci
        L.lh_delens_grid.argtypes = [dp, dp, gp, vp, ci, vp, C.c_longlong, vp]
        L.lh_delens_grid.restype = ci
        L.lh_set_stream.argtypes = [vp]
        L.lh_ipc_export.argtypes = [vp, vp, C.POINTER(C.c_ulonglong)]
        L.lh_ipc_export.restype = ci
        L.lh_ipc_open.argtypes = [vp, C.c_ulonglong, C.POINTER(vp)]
        L.lh_ipc_open.restype = ci
        L.lh_ipc_close.argtypes = [vp]
        L.lh_ipc_close.restype = ci
        L.lh_pack_model.argtypes = [vp, ci, vp, vp]
        L.lh_pack_model.restype = ci
        L.lh_last_error.restype = C.c_char_p
        L.lh_launch_count.restype = C.c_longlong
        L.lh_fp64_peak_probe.argtypes = [ci, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.lh_math_host_eval.argtypes = [ci, vp, vp, C.c_size_t, vp]
        L.lh_math_host_eval.restype = ci
        L.lh_version.restype = C.c_char_p
        L.lh_source_hash.restype = C.c_char_p
        for f in ("lh_grid_gradient", "lh_grid_hessian", "lh_lens_maps", "lh_grid_gradient_batch", "lh_grid_eval",
                  "lh_grid_eval_batch", "lh_grid_eval_host", "lh_set_stream", "lh_fp64_peak_probe"):
            getattr(L, f).restype = ci
        _lib = L
    return _lib


# ---------------------------------------------------------------- marshalling helpers
def _lenses_ptr(lenses):
    """numpy array of 64-byte lh_lens records (any dtype of itemsize 64), host memory."""
    a = np.ascontiguousarray(lenses)
    if a.dtype.itemsize != 64:
        raise TypeError("lenses must be an array of 64-byte lh_lens records")
    return a, a.ctypes.data, a.size


def _grid(g) -> lh_grid:
    if isinstance(g, lh_grid):
        return g
    return lh_grid(float(g.x0), float(g.y0), float(g.dx), int(g.nx), int(g.ny))


def _dev_ptr(t, count=None):
    """Device address of an output / input buffer.  `count`: the number of float64 elements the call will write
    (or read) there; a tensor that is smaller, or lives on another device than the current one, is refused HERE --
    the C ABI only sees an address and cannot tell (it would be an out-of-bounds write on the device)."""
    if t is None:
        return None
    if isinstance(t, int):
        return t
    if hasattr(t, "data_ptr"):
        if hasattr(t, "is_contiguous") and not t.is_contiguous():
            raise TypeError("output tensors must be contiguous")
        if hasattr(t, "dtype") and "float64" not in str(t.dtype):
            raise TypeError("output tensors must be float64")
        if count is not None and hasattr(t, "numel") and int(t.numel()) < count:
            raise ValueError(f"tensor of {int(t.numel())} elements where the call needs {count}")
        if getattr(t, "is_cuda", False):
            torch = sys.modules.get("torch")
            if torch is not None and t.device.index is not None and t.device.index != torch.cuda.current_device():
                raise ValueError(f"tensor on cuda:{t.device.index} but the current device is cuda:{torch.cuda.current_device()}")
        return t.data_ptr()
    raise TypeError(f"cannot take a device pointer from {type(t)}")


def _check(rc: int):
    if rc != LH_OK:
        raise LhError(rc, _load().lh_last_error().decode())


def _outputs(planes: dict, to_ptr, count=None) -> lh_outputs:
    bad = set(planes) - set(PLANES)
    if bad:
        raise KeyError(f"unknown planes {sorted(bad)}")
    return lh_outputs(**{n: to_ptr(planes.get(n), count) for n in PLANES})


def _npix(grid, nmodel=1) -> int:
    return int(grid.nx) * int(grid.ny) * int(nmodel)


# ---------------------------------------------------------------- the C ABI, name for name
def lh_grid_gradient(lenses, grid, out_ax, out_ay):
    a, p, n = _lenses_ptr(lenses)
    k = _npix(grid)
    _check(_load().lh_grid_gradient(p, n, C.byref(_grid(grid)), _dev_ptr(out_ax, k), _dev_ptr(out_ay, k)))


def lh_grid_hessian(lenses, grid, a11, a12, a22):
    a, p, n = _lenses_ptr(lenses)
    k = _npix(grid)
    _check(_load().lh_grid_hessian(p, n, C.byref(_grid(grid)), _dev_ptr(a11, k), _dev_ptr(a12, k), _dev_ptr(a22, k)))


def lh_lens_maps(lenses, grid, kappa, gamma1, gamma2, mu):
    a, p, n = _lenses_ptr(lenses)
    k = _npix(grid)
    _check(_load().lh_lens_maps(p, n, C.byref(_grid(grid)), _dev_ptr(kappa, k), _dev_ptr(gamma1, k), _dev_ptr(gamma2, k),
                                _dev_ptr(mu, k)))


def lh_grid_gradient_batch(lenses, nmodel, nlens, grid, out_ax, out_ay):
    a, p, n = _lenses_ptr(lenses)
    if n != nmodel * nlens:
        raise ValueError("len(lenses) != nmodel*nlens")
    k = _npix(grid, nmodel)
    _check(_load().lh_grid_gradient_batch(p, nmodel, nlens, C.byref(_grid(grid)), _dev_ptr(out_ax, k), _dev_ptr(out_ay, k)))


def lh_grid_eval(lenses, grid, **planes):
    """planes: any of ax, ay, a11, a12, a22, kappa, gamma1, gamma2, mu = device tensor."""
    a, p, n = _lenses_ptr(lenses)
    o = _outputs(planes, _dev_ptr, _npix(grid))
    _check(_load().lh_grid_eval(p, n, C.byref(_grid(grid)), C.byref(o)))


def lh_chi2(lenses, grid, constraints, nsources: int, chi2, predicted=None, sources=None, nimages=None):
    """constraints: host array of 32-byte lh_constraint records (lens_inputs.CONSTRAINT_DTYPE); chi2: device float64[1];
    predicted [K, 2], sources [nsources, 2]: device float64 or None; nimages: device int64[1] or None."""
    a, p, n = _lenses_ptr(lenses)
    c = np.ascontiguousarray(constraints)
    if c.dtype.itemsize != 32:
        raise TypeError("constraints must be an array of 32-byte lh_constraint records")
    _check(_load().lh_chi2(p, n, C.byref(_grid(grid)), c.ctypes.data, c.size, int(nsources), _dev_ptr(chi2, 1),
                           _dev_ptr(predicted, 2 * c.size), _dev_ptr(sources, 2 * int(nsources)),
                           None if nimages is None else nimages.data_ptr()))


def lh_points_eval(lenses, xs, ys, **planes):
    """xs, ys: device float64 tensors of equal length; planes: device tensors of that length."""
    a, p, n = _lenses_ptr(lenses)
    npts = int(xs.numel()) if hasattr(xs, "numel") else None
    if npts is None or npts != int(ys.numel()):
        raise ValueError("xs and ys must be device tensors of equal length")
    o = _outputs(planes, _dev_ptr, npts)
    _check(_load().lh_points_eval(p, n, _dev_ptr(xs, npts), _dev_ptr(ys, npts), npts, C.byref(o)))


def lh_grid_eval_rows(lenses, grid, j0: int, nrows: int, **planes):
    """Rows [j0, j0+nrows) of the grid into planes of shape [nrows, nx] (the multi-GPU row-slab primitive)."""
    a, p, n = _lenses_ptr(lenses)
    o = _outputs(planes, _dev_ptr, int(nrows) * int(grid.nx))
    _check(_load().lh_grid_eval_rows(p, n, C.byref(_grid(grid)), int(j0), int(nrows), C.byref(o)))


LH_NOALLOC_MAX_PIXELS, LH_NOALLOC_MAX_LENSES = 1 << 20, 4096


def lh_grid_eval_noalloc(lenses, grid, j0: int, nrows: int, **planes):
    """lh_grid_eval_rows for programs that must not let a library allocate device memory (a caching allocator owns
    the GPU, a loop that may not stall on cudaMalloc, "reserve everything at start-up" rules): the scratch is a fixed
    40 MiB array inside liblh.so.  At most LH_NOALLOC_MAX_PIXELS pixels per call and LH_NOALLOC_MAX_LENSES lenses,
    else LhError(LH_EINVAL).  Make the first call on each device during set-up; keep all calls of a device on one
    stream (they share the scratch).  Planes of shape [nrows, nx]; see include/lh.h."""
    a, p, n = _lenses_ptr(lenses)
    o = _outputs(planes, _dev_ptr, int(nrows) * int(grid.nx))
    _check(_load().lh_grid_eval_noalloc(p, n, C.byref(_grid(grid)), int(j0), int(nrows), C.byref(o)))


def lh_grid_eval_batch(lenses, nmodel, nlens, grid, **planes):
    a, p, n = _lenses_ptr(lenses)
    if n != nmodel * nlens:
        raise ValueError("len(lenses) != nmodel*nlens")
    o = _outputs(planes, _dev_ptr, _npix(grid, nmodel))
    _check(_load().lh_grid_eval_batch(p, nmodel, nlens, C.byref(_grid(grid)), C.byref(o)))


def lh_grid_eval_batch_shared(shared, varying, nmodel, nvar, grid, **planes):
    """model m = shared + varying[m*nvar:(m+1)*nvar]; planes [nmodel, ny, nx]; the shared lenses are evaluated once."""
    sa, sp, sn = _lenses_ptr(shared)
    va, vpn, vn = _lenses_ptr(varying)
    if vn != nmodel * nvar:
        raise ValueError("len(varying) != nmodel*nvar")
    o = _outputs(planes, _dev_ptr, _npix(grid, nmodel))
    _check(_load().lh_grid_eval_batch_shared(sp, sn, vpn, nmodel, nvar, C.byref(_grid(grid)), C.byref(o)))


def lh_grid_stats_batch(lenses, nmodel, nlens, grid, mean: dict, var: dict | None = None):
    """mean / var: dicts plane name -> device tensor [ny, nx]; per-pixel mean and population variance over models."""
    a, p, n = _lenses_ptr(lenses)
    if n != nmodel * nlens:
        raise ValueError("len(lenses) != nmodel*nlens")
    om = _outputs(mean, _dev_ptr, _npix(grid))
    ov = _outputs(var, _dev_ptr, _npix(grid)) if var else None
    _check(_load().lh_grid_stats_batch(p, nmodel, nlens, C.byref(_grid(grid)), C.byref(om),
                                       C.byref(ov) if ov is not None else None))


LH_IMAGE_DTYPE = np.dtype([("source", "<i4"), ("_pad", "<i4"), ("triangle", "<i8"), ("x", "<f8"), ("y", "<f8")])


def lh_source_plane(ax, ay, grid, bx=None, by=None):
    """beta = theta - alpha on the grid; device planes [ny, nx]."""
    k = _npix(grid)
    _check(_load().lh_source_plane(_dev_ptr(ax, k), _dev_ptr(ay, k), C.byref(_grid(grid)), _dev_ptr(bx, k), _dev_ptr(by, k)))


def lh_delens_grid(ax, ay, grid, sources, images, max_images: int, count):
    """sources: host float64 [ns, 2]; images: device buffer of >= max_images 32-byte lh_image records (e.g. a
    torch uint8 tensor of 32*max_images bytes, view it with LH_IMAGE_DTYPE on the host); count: device int64[1]."""
    src = np.ascontiguousarray(sources, dtype=np.float64).reshape(-1, 2)

    def raw(t, nbytes):  # any device buffer: only the address is taken, the size in bytes is checked
        if t is None or isinstance(t, int):
            return t
        if hasattr(t, "numel") and hasattr(t, "element_size") and int(t.numel()) * int(t.element_size()) < nbytes:
            raise ValueError(f"buffer of {int(t.numel()) * int(t.element_size())} bytes where the call needs {nbytes}")
        return t.data_ptr()

    _check(_load().lh_delens_grid(_dev_ptr(ax, _npix(grid)), _dev_ptr(ay, _npix(grid)), C.byref(_grid(grid)), src.ctypes.data, len(src),
                                  raw(images, 32 * int(max_images)), int(max_images), raw(count, 8)))


def _host_ptr(v, count):
    """Address of a HOST plane of at least `count` float64 elements (numpy array or torch CPU tensor, pinned or not)."""
    if v is None:
        return None
    if isinstance(v, np.ndarray):
        if v.dtype != np.float64 or not v.flags.c_contiguous:
            raise TypeError("host planes must be C-contiguous float64")
        if v.size < count:
            raise ValueError(f"host plane of {v.size} elements where the call needs {count}")
        return v.ctypes.data
    if hasattr(v, "data_ptr"):  # e.g. a pinned torch CPU tensor
        if getattr(v, "is_cuda", False):
            raise TypeError("the *_host entry points take HOST planes")
        if "float64" not in str(v.dtype) or not v.is_contiguous():
            raise TypeError("host planes must be contiguous float64")
        if int(v.numel()) < count:
            raise ValueError(f"host plane of {int(v.numel())} elements where the call needs {count}")
        return v.data_ptr()
    raise TypeError(f"cannot take a host pointer from {type(v)}")


def lh_grid_eval_host(lenses, nmodel, nlens, grid, **host_planes):
    """host_planes: numpy float64 C-contiguous arrays of nmodel*ny*nx elements (HOST memory,
    pinned or not); the copies back and a stream synchronise happen inside the call."""
    a, p, n = _lenses_ptr(lenses)
    if n != nmodel * nlens:
        raise ValueError("len(lenses) != nmodel*nlens")
    o = _outputs(host_planes, _host_ptr, _npix(grid, nmodel))
    _check(_load().lh_grid_eval_host(p, nmodel, nlens, C.byref(_grid(grid)), C.byref(o)))


def lh_grid_eval_rows_host(lenses, grid, j0: int, nrows: int, **host_planes):
    """Rows [j0, j0+nrows) of one map into HOST planes of nrows*nx elements (numpy or pinned torch CPU tensors)."""
    a, p, n = _lenses_ptr(lenses)
    o = _outputs(host_planes, _host_ptr, int(nrows) * int(grid.nx))
    _check(_load().lh_grid_eval_rows_host(p, n, C.byref(_grid(grid)), int(j0), int(nrows), C.byref(o)))


LH_PACK_DOUBLES, LH_PACK_CLASSES = 24, 4


def lh_pack_model(lenses, validate_only: bool = False):
    """Step a1 on the host: returns (table[n, LH_PACK_DOUBLES], class_begin[LH_PACK_CLASSES+1])."""
    a, p, n = _lenses_ptr(lenses)
    begin = np.zeros(LH_PACK_CLASSES + 1, dtype=np.int32)
    if validate_only:
        _check(_load().lh_pack_model(p, n, None, begin.ctypes.data))
        return None, begin
    raw = np.zeros(n * LH_PACK_DOUBLES + 2, dtype=np.float64)
    off = (16 - raw.ctypes.data % 16) % 16 // 8
    table = raw[off: off + n * LH_PACK_DOUBLES]
    _check(_load().lh_pack_model(p, n, table.ctypes.data, begin.ctypes.data))
    return table.reshape(n, LH_PACK_DOUBLES), begin


def lh_ipc_export(t):
    """(handle bytes, offset) of a device tensor / address of this process, for lh_ipc_open in another process."""
    h = (C.c_ubyte * 64)()
    off = C.c_ulonglong(0)
    p = t if isinstance(t, int) else t.data_ptr()
    _check(_load().lh_ipc_export(p, h, C.byref(off)))
    return bytes(h), int(off.value)


def lh_ipc_open(handle: bytes, offset: int) -> int:
    """Device address, in THIS process, of the buffer another process exported (peer access over NVLink when it
    lives on another GPU).  Pass it (plus a byte offset) as an output plane; close it with lh_ipc_close."""
    h = (C.c_ubyte * 64).from_buffer_copy(handle)
    out = C.c_void_p()
    _check(_load().lh_ipc_open(h, int(offset), C.byref(out)))
    return int(out.value)


def lh_ipc_close(ptr: int) -> None:
    _check(_load().lh_ipc_close(int(ptr)))


def lh_set_stream(stream) -> None:
    """stream: None (legacy default), an int handle, or a torch.cuda.Stream."""
    h = 0 if stream is None else (stream if isinstance(stream, int) else stream.cuda_stream)
    _check(_load().lh_set_stream(h))


def lh_last_error() -> str:
    return _load().lh_last_error().decode()


def lh_launch_count() -> int:
    return int(_load().lh_launch_count())


def lh_fp64_peak_probe(iters: int = 4096):
    f, s = C.c_double(), C.c_double()
    _check(_load().lh_fp64_peak_probe(int(iters), C.byref(f), C.byref(s)))
    return f.value, s.value


def lh_math_host_eval(fn: int, a, b=None):
    """HOST evaluation of the kernel's FP64 primitives (include/lh.h); numpy in, numpy out."""
    a = np.ascontiguousarray(a, dtype=np.float64)
    bb = None if b is None else np.ascontiguousarray(np.broadcast_to(b, a.shape), dtype=np.float64)
    out = np.empty_like(a)
    _check(_load().lh_math_host_eval(int(fn), a.ctypes.data, None if bb is None else bb.ctypes.data, a.size,
                                     out.ctypes.data))
    return out


def lh_version() -> str:
    return _load().lh_version().decode()


def lh_source_hash() -> str:
    """SHA-256 of the sources the loaded library was compiled from (include/lh_diag.h); compare with
    _build.source_hash() to tell a stale prebuilt library from a current one."""
    return _load().lh_source_hash().decode()
