"""CPU oracle for the X-engine -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Thin ctypes/numpy marshalling around ``xengine_oracle.c`` (the plain triple loop of
PAPER.md:54-57, Sec. 2, Eq. 2).  Only ``tests/``, ``__graft_entry__.smoke()`` and
``bench.py``'s ``cpu_baseline`` / ``--impl reference`` leg may import this package; the
product (``paper_1305_5639_b200``) never does, and this package never imports the product.

Layouts:
  x   [T, C, N, P, 2]  int8 (ci8) or float16 (cf16), last axis = (re, im)
  V   [n_sel, B, P, P, 2]  int64 / float64, B = N(N+1)/2, b(i,j) = i(i+1)/2 + j, j <= i,
      axis 2 = polarisation p of the conjugated station i, axis 3 = polarisation q of j.
"""
import ctypes
import numpy as np

_lib = None


def _load():
    global _lib
    if _lib is None:
        from .build import build as _build_lib
        lib = ctypes.CDLL(_build_lib())
        i32, vp = ctypes.c_int, ctypes.c_void_p
        lib.xo_baseline_index.restype = ctypes.c_longlong
        lib.xo_baseline_index.argtypes = [i32, i32]
        lib.xo_max_threads.restype = i32
        lib.xo_set_threads.argtypes = [i32]
        lib.xo_half_to_double.restype = ctypes.c_double
        lib.xo_half_to_double.argtypes = [ctypes.c_uint16]
        for name in ("xo_xengine_ci8", "xo_xengine_cf16"):
            f = getattr(lib, name)
            f.restype = i32
            f.argtypes = [vp, vp, i32, i32, i32, i32, vp, i32, i32]
        for name in ("xo_xengine_cross_ci8", "xo_xengine_cross_cf16"):
            f = getattr(lib, name)
            f.restype = i32
            f.argtypes = [vp, vp, vp, i32, i32, i32, i32, i32, vp, i32, i32]
        for name in ("xo_pair_ci8", "xo_pair_cf16"):
            f = getattr(lib, name)
            f.restype = None
            f.argtypes = [vp, i32, i32, i32, i32, i32, i32, i32, i32, i32, vp]
        _lib = lib
    return _lib


def baseline_index(i: int, j: int) -> int:
    """b(i,j) = i(i+1)/2 + j for j <= i (row-major lower triangle, reading R7)."""
    return int(_load().xo_baseline_index(int(i), int(j)))


def n_baselines(n_station: int) -> int:
    return n_station * (n_station + 1) // 2


def max_threads() -> int:
    return int(_load().xo_max_threads())


def set_threads(n: int) -> None:
    _load().xo_set_threads(int(n))


def half_to_double(bits: int) -> float:
    return float(_load().xo_half_to_double(int(bits) & 0xFFFF))


def _check_x(x):
    x = np.ascontiguousarray(x)
    if x.ndim != 5 or x.shape[-1] != 2:
        raise ValueError("x must be [T, C, N, P, 2]")
    if x.dtype == np.int8:
        return x, "ci8"
    if x.dtype == np.float16:
        return x, "cf16"
    raise TypeError("x must be int8 or float16, got %s" % x.dtype)


def xengine(x, chans=None, accumulate_into=None):
    """Eq. 2 for every selected channel -> packed triangle V (int64 for ci8, float64 for cf16).

    ``accumulate_into``: a previous V of the same shape; the new sums are ADDED to it in place
    (integration across calls) and it is returned.
    """
    x, kind = _check_x(x)
    T, C, N, P, _ = x.shape
    if chans is None:
        sel, n_sel, sel_ptr = None, C, None
    else:
        sel = np.ascontiguousarray(chans, dtype=np.int32)
        n_sel, sel_ptr = int(sel.size), sel.ctypes.data
    odt = np.int64 if kind == "ci8" else np.float64
    shape = (n_sel, n_baselines(N), P, P, 2)
    if accumulate_into is None:
        out, acc = np.empty(shape, dtype=odt), 0
    else:
        out, acc = accumulate_into, 1
        if out.shape != shape or out.dtype != odt or not out.flags.c_contiguous:
            raise ValueError("accumulate_into has the wrong shape/dtype/layout")
    fn = _load().xo_xengine_ci8 if kind == "ci8" else _load().xo_xengine_cf16
    rc = fn(x.ctypes.data, out.ctypes.data, N, P, C, T, sel_ptr, n_sel, acc)
    if rc != 0:
        raise RuntimeError("oracle failed with code %d" % rc)
    return out


def visibility(x, c, i, p, j, q):
    """One visibility V_ij^{pq}[c] as a Python complex (exact ints for ci8), straight from Eq. 2."""
    x, kind = _check_x(x)
    T, C, N, P, _ = x.shape
    if kind == "ci8":
        v = (ctypes.c_int64 * 2)()
        _load().xo_pair_ci8(x.ctypes.data, N, P, C, T, c, i, p, j, q, v)
        return int(v[0]), int(v[1])
    v = (ctypes.c_double * 2)()
    _load().xo_pair_cf16(x.ctypes.data, N, P, C, T, c, i, p, j, q, v)
    return float(v[0]), float(v[1])


def xengine_cross(xa, xb, chans=None, accumulate_into=None):
    """Rectangular cross-only X-engine (Sec. 4): V[n_sel, Na, Nb, P, P, 2] with
    V[c, i, j, p, q] = sum_t conj(xa[t, c, i, p]) * xb[t, c, j, q]; no triangle, no autocorrelations."""
    xa, kind = _check_x(xa)
    xb, kind_b = _check_x(xb)
    T, C, Na, P, _ = xa.shape
    Tb, Cb, Nb, Pb, _ = xb.shape
    if kind != kind_b or (T, C, P) != (Tb, Cb, Pb):
        raise ValueError("the two groups must share dtype, T, C and P")
    if chans is None:
        n_sel, sel_ptr = C, None
    else:
        sel = np.ascontiguousarray(chans, dtype=np.int32)
        n_sel, sel_ptr = int(sel.size), sel.ctypes.data
    odt = np.int64 if kind == "ci8" else np.float64
    shape = (n_sel, Na, Nb, P, P, 2)
    if accumulate_into is None:
        out, acc = np.empty(shape, dtype=odt), 0
    else:
        out, acc = accumulate_into, 1
        if out.shape != shape or out.dtype != odt or not out.flags.c_contiguous:
            raise ValueError("accumulate_into has the wrong shape/dtype/layout")
    fn = _load().xo_xengine_cross_ci8 if kind == "ci8" else _load().xo_xengine_cross_cf16
    rc = fn(xa.ctypes.data, xb.ctypes.data, out.ctypes.data, Na, Nb, P, C, T, sel_ptr, n_sel, acc)
    if rc != 0:
        raise RuntimeError("oracle failed with code %d" % rc)
    return out
