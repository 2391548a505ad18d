"""Thin ctypes binding of libcorr.so (include/corr.h): argument marshalling only.

Every step of the X-engine (Eq. 2) runs inside the library's CUDA kernels.  torch is
used by callers for device memory and streams; this module only extracts ``data_ptr()`` and the raw
``cudaStream_t``.  There is NO CPU fallback: if the library is missing or the device is not a B200,
the calls raise.
"""
import ctypes
import os

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libcorr.so")

CORR_CI8, CORR_CF16 = 0, 1
CORR_OK, CORR_EINVAL, CORR_EUNSUPPORTED, CORR_ENOMEM, CORR_ECUDA, CORR_EOVERFLOW = 0, -1, -2, -3, -4, -5
KERNELS = {"auto": 0, "single": 1, "pair": 2, "simt": 3}      # CORR_KERNEL_*
KERNEL_NAMES = {v: k for k, v in KERNELS.items()}
DTYPES = {"ci8": CORR_CI8, "cf16": CORR_CF16}

# name -> (restype, argtypes): every symbol include/corr.h declares
_vp, _i, _sz, _ll, _cp = ctypes.c_void_p, ctypes.c_int, ctypes.c_size_t, ctypes.c_longlong, ctypes.c_char_p
SYMBOLS = {
    "corr_create": (_vp, [_i, _i, _i, _i, _i]),
    "corr_create_window": (_vp, [_i, _i, _i, _i, _i, _i, _i]),
    "corr_xengine": (_i, [_vp, _vp, _vp, _i, _vp]),
    "corr_xengine_host": (_i, [_vp, _vp, _vp, _i]),
    "corr_create_cross": (_vp, [_i, _i, _i, _i, _i, _i]),
    "corr_xengine_cross": (_i, [_vp, _vp, _vp, _vp, _i, _vp]),
    "corr_input_bytes_b": (_sz, [_vp]),
    "corr_fengine": (_i, [_vp, _vp, _i, _ll, _vp]),
    "corr_fengine_simt": (_i, [_vp, _vp, _i, _ll, _vp]),
    "corr_fengine_uses_tensor_cores": (_i, [_i, _vp]),
    "corr_fengine_ci8": (_i, [_vp, _vp, _i, _ll, ctypes.c_float, _vp]),
    "corr_xengine_dumps": (_i, [_vp, _vp, _vp, _i, _vp]),
    "corr_destroy": (None, [_vp]),
    "corr_input_bytes": (_sz, [_vp]),
    "corr_output_bytes": (_sz, [_vp]),
    "corr_baseline_index": (_ll, [_i, _i]),
    "corr_last_error": (_cp, [_vp]),
    "corr_set_kernel": (_i, [_vp, _i]),
    "corr_get_kernel": (_i, [_vp]),
    "corr_uses_tensor_cores": (_i, [_vp]),
    "corr_corner_turn": (_i, [_vp, _vp, _vp, _vp]),
    "corr_corner_turn_planes": (_i, [_vp, _vp, _vp, _i, _vp]),
    "corr_workspace_bytes": (_sz, [_vp]),
    "corr_workspace_time": (_i, [_vp]),
    "corr_tile_schedule": (_i, [_i, _i, _i, _i, ctypes.POINTER(_i), _i]),
    "corr_last_launch_count": (_i, [_vp]),
    "corr_xengine_static": (_i, [_i, _i, _i, _i, _i, _vp, _vp, _i, _vp]),
    "corr_static_scratch_bytes": (_sz, []),
}

_lib = None


class CorrError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("libcorr error %d: %s" % (code, msg))
        self.code = code


def lib():
    """Load libcorr.so (building it in-tree if the sources are newer).  Raises if unavailable."""
    global _lib
    if _lib is None:
        from .build import build
        build()                       # no-op when libcorr.so is newer than its sources
        L = ctypes.CDLL(LIB_PATH)
        for name, (res, args) in SYMBOLS.items():
            f = getattr(L, name)      # AttributeError if the library does not export it
            f.restype, f.argtypes = res, args
        _lib = L
    return _lib


def baseline_index(i, j):
    return int(lib().corr_baseline_index(int(i), int(j)))


def tile_schedule(n_station, n_pol, dtype="ci8", kernel="single"):
    """Per-channel triangular tile schedule as a list of (row0, col0, ncols); host logic only."""
    L = lib()
    feed = KERNELS[kernel]
    n = L.corr_tile_schedule(n_station, n_pol, DTYPES[dtype], feed, None, 0)
    if n < 0:
        raise CorrError(n, "corr_tile_schedule")
    buf = (_i * (3 * n))()
    L.corr_tile_schedule(n_station, n_pol, DTYPES[dtype], feed, buf, n)
    return [(buf[3 * k], buf[3 * k + 1], buf[3 * k + 2]) for k in range(n)]


def _stream_ptr(stream):
    if stream is None:
        import torch
        stream = torch.cuda.current_stream()
    return ctypes.c_void_p(getattr(stream, "cuda_stream", stream))


def fengine(samples, out=None, stream=None, scale=None, simt=False):
    """corr_fengine: int8 real samples [n_stream, n_spectra * 256] (CUDA) -> complex fp16 [n_spectra, 128, n_stream, 2];
    with ``scale`` (corr_fengine_ci8): requantised complex int8 codes clip(rint(S * scale), +-127) of the same shape.
    ``simt=True`` forces the CUDA-core kernel (corr_fengine_simt)."""
    import torch
    if scale is not None:
        return _fengine_ci8(samples, float(scale), out, stream)
    if samples.dtype != torch.int8 or samples.dim() != 2 or samples.shape[1] % 256 or not samples.is_contiguous() \
            or samples.device.type != "cuda":
        raise ValueError("samples must be a contiguous CUDA int8 tensor [n_stream, n_spectra * 256]")
    n_stream, n_spec = samples.shape[0], samples.shape[1] // 256
    if out is None:
        out = torch.empty((n_spec, 128, n_stream, 2), dtype=torch.float16, device=samples.device)
    if out.dtype != torch.float16 or tuple(out.shape) != (n_spec, 128, n_stream, 2) or not out.is_contiguous():
        raise ValueError("out must be a contiguous float16 tensor [n_spectra, 128, n_stream, 2]")
    L = lib()
    fn = L.corr_fengine_simt if simt else L.corr_fengine
    rc = fn(samples.data_ptr(), out.data_ptr(), n_stream, n_spec, _stream_ptr(stream))
    if rc != CORR_OK:
        raise CorrError(rc, L.corr_last_error(None).decode())
    return out


def fengine_uses_tensor_cores(n_stream, out=None):
    """Which kernel corr_fengine launches for this stream count (and output alignment)."""
    return bool(lib().corr_fengine_uses_tensor_cores(int(n_stream), None if out is None else out.data_ptr()))


def _fengine_ci8(samples, scale, out, stream):
    import torch
    if samples.dtype != torch.int8 or samples.dim() != 2 or samples.shape[1] % 256 or not samples.is_contiguous() \
            or samples.device.type != "cuda":
        raise ValueError("samples must be a contiguous CUDA int8 tensor [n_stream, n_spectra * 256]")
    n_stream, n_spec = samples.shape[0], samples.shape[1] // 256
    if out is None:
        out = torch.empty((n_spec, 128, n_stream, 2), dtype=torch.int8, device=samples.device)
    if out.dtype != torch.int8 or tuple(out.shape) != (n_spec, 128, n_stream, 2) or not out.is_contiguous():
        raise ValueError("out must be a contiguous int8 tensor [n_spectra, 128, n_stream, 2]")
    L = lib()
    rc = L.corr_fengine_ci8(samples.data_ptr(), out.data_ptr(), n_stream, n_spec, scale, _stream_ptr(stream))
    if rc != CORR_OK:
        raise CorrError(rc, L.corr_last_error(None).decode())
    return out


STATIC_MAX_STREAMS = 8192       # CORR_STATIC_MAX_STREAMS


def xengine_static(x, out=None, accumulate=False, stream=None, dtype=None):
    """corr_xengine_static: the X-engine for callers that may not allocate device memory.

    Same result as ``Correlator(...).xengine(x, out, accumulate)`` on the pair kernel, but with no handle and no
    cudaMalloc anywhere in the library: the kernel's tile table and tile-feed counter sit in a 16.5 KB array built into
    libcorr.so.  It exists for users such as a real-time capture process that gave all GPU memory to its ring buffers at
    start-up, or a plug-in whose host forbids driver allocations after initialisation.  Limits: ``N * P <= 8192`` and a
    16-byte multiple per channel row.  All calls on a GPU share that one array, so calls that may overlap on the GPU
    (different streams with no event between them) corrupt each other; calls on one stream are safe back to back.

    ``x``: CUDA ``[T, C, N, P, 2]`` int8 (ci8) or float16 (cf16).  ``out``: the caller's ``[C, B, P, P, 2]`` int32 /
    float32 tensor.  (``out=None`` lets torch allocate one for convenience; a caller that really cannot allocate passes
    its own.)  The first call on a device does a one-time host-side set-up; make it before any stream capture.
    """
    import torch
    if dtype is None:
        dtype = "ci8" if x.dtype == torch.int8 else "cf16"
    want_in = torch.int8 if dtype == "ci8" else torch.float16
    want_out = torch.int32 if dtype == "ci8" else torch.float32
    if x.dtype != want_in or x.dim() != 5 or x.shape[4] != 2 or not x.is_contiguous() or x.device.type != "cuda":
        raise ValueError("input must be a contiguous CUDA %s tensor [T, C, N, P, 2]" % want_in)
    T, C, N, P, _ = (int(v) for v in x.shape)
    shape = (C, N * (N + 1) // 2, P, P, 2)
    if out is None:
        if accumulate:
            raise ValueError("accumulate=True needs the running `out`")
        out = torch.empty(shape, dtype=want_out, device=x.device)
    if out.dtype != want_out or tuple(out.shape) != shape or not out.is_contiguous() or out.device.type != "cuda":
        raise ValueError("output must be a contiguous CUDA %s tensor of shape %s" % (want_out, shape))
    L = lib()
    rc = L.corr_xengine_static(N, P, C, T, DTYPES[dtype], x.data_ptr(), out.data_ptr(), int(bool(accumulate)), _stream_ptr(stream))
    if rc != CORR_OK:
        raise CorrError(rc, L.corr_last_error(None).decode())
    return out


class Correlator:
    """corr_create / corr_xengine / corr_destroy with torch tensors as the device buffers."""

    def __init__(self, n_station, n_pol, n_chan, n_time, dtype="ci8", window=None):
        """``window=(chan0, n_chan_window)``: corr_create_window -- the handle integrates only those channels of the
        whole-band ``[T, n_chan, N, P, 2]`` input into their slabs of the whole-band output, in place."""
        self._L = lib()
        self.N, self.P, self.C, self.T, self.dtype = n_station, n_pol, n_chan, n_time, dtype
        self.window = None if window is None else (int(window[0]), int(window[1]))
        if window is None:
            self._h = self._L.corr_create(n_station, n_pol, n_chan, n_time, DTYPES[dtype])
        else:
            self._h = self._L.corr_create_window(n_station, n_pol, n_chan, self.window[0], self.window[1], n_time, DTYPES[dtype])
        if not self._h:
            msg = self._L.corr_last_error(None).decode()
            raise CorrError(CORR_EINVAL if "invalid" in msg or "too large" in msg else CORR_EUNSUPPORTED, msg)
        self.n_baseline = n_station * (n_station + 1) // 2

    # ---- sizes / introspection -------------------------------------------------------------
    @property
    def input_bytes(self):
        return int(self._L.corr_input_bytes(self._h))

    @property
    def output_bytes(self):
        return int(self._L.corr_output_bytes(self._h))

    @property
    def workspace_bytes(self):
        return int(self._L.corr_workspace_bytes(self._h))

    @property
    def workspace_time(self):
        return int(self._L.corr_workspace_time(self._h))

    @property
    def uses_tensor_cores(self):
        return bool(self._L.corr_uses_tensor_cores(self._h))

    @property
    def last_launch_count(self):
        return int(self._L.corr_last_launch_count(self._h))

    @property
    def kernel(self):
        """Name of the kernel corr_xengine will launch: single / pair / simt."""
        return KERNEL_NAMES[int(self._L.corr_get_kernel(self._h))]

    def set_kernel(self, kernel):
        self._check(self._L.corr_set_kernel(self._h, KERNELS[kernel]))

    def _check(self, rc):
        if rc != CORR_OK:
            raise CorrError(rc, self._L.corr_last_error(self._h).decode())

    # ---- buffers ---------------------------------------------------------------------------
    def input_shape(self):
        return (self.T, self.C, self.N, self.P, 2)

    def output_shape(self):
        return (self.C, self.n_baseline, self.P, self.P, 2)

    def empty_output(self, device="cuda"):
        import torch
        return torch.empty(self.output_shape(), device=device,
                           dtype=torch.int32 if self.dtype == "ci8" else torch.float32)

    def _check_in(self, x, device_type):
        import torch
        want = torch.int8 if self.dtype == "ci8" else torch.float16
        if x.dtype != want or tuple(x.shape) != self.input_shape() or not x.is_contiguous():
            raise ValueError("input must be a contiguous %s tensor of shape %s" % (want, self.input_shape()))
        if x.device.type != device_type:
            raise ValueError("input must live on %s" % device_type)

    def _check_out(self, out, device_type):
        import torch
        want = torch.int32 if self.dtype == "ci8" else torch.float32
        if out.dtype != want or tuple(out.shape) != self.output_shape() or not out.is_contiguous():
            raise ValueError("output must be a contiguous %s tensor of shape %s" % (want, self.output_shape()))
        if out.device.type != device_type:
            raise ValueError("output must live on %s" % device_type)

    # ---- the calls -------------------------------------------------------------------------
    def xengine(self, x, out=None, accumulate=False, stream=None):
        """corr_xengine on device tensors; asynchronous on ``stream`` (default: torch's current)."""
        self._check_in(x, "cuda")
        if out is None:
            if accumulate or self.window is not None:
                raise ValueError("accumulate=True and window plans need the caller's `out`")
            out = self.empty_output(x.device)
        self._check_out(out, "cuda")
        self._check(self._L.corr_xengine(self._h, x.data_ptr(), out.data_ptr(), int(bool(accumulate)),
                                         _stream_ptr(stream)))
        return out

    def xengine_dumps(self, x, n_dump, out=None, stream=None):
        """corr_xengine_dumps: n_dump separate integrations of n_time / n_dump samples in one launch ->
        [n_dump, C, B, P, P, 2]."""
        import torch
        self._check_in(x, "cuda")
        shape = (int(n_dump),) + tuple(self.output_shape())
        if out is None:
            out = torch.empty(shape, device=x.device, dtype=torch.int32 if self.dtype == "ci8" else torch.float32)
        if tuple(out.shape) != shape or not out.is_contiguous() or out.device.type != "cuda":
            raise ValueError("out must be a contiguous CUDA tensor of shape %s" % (shape,))
        self._check(self._L.corr_xengine_dumps(self._h, x.data_ptr(), out.data_ptr(), int(n_dump), _stream_ptr(stream)))
        return out

    def xengine_host(self, x_host, out_host, accumulate=False):
        """corr_xengine_host: HOST tensors in and out (blocking; copies inside the library)."""
        self._check_in(x_host, "cpu")
        if out_host is not None:
            self._check_out(out_host, "cpu")
        self._check(self._L.corr_xengine_host(self._h, x_host.data_ptr(),
                                              None if out_host is None else out_host.data_ptr(),
                                              int(bool(accumulate))))
        return out_host

    def corner_turn(self, x, ws=None, stream=None, planes=2):
        """corr_corner_turn_planes: returns the uint8 workspace holding the plane ws (and ws_rot when planes == 2)."""
        import torch
        self._check_in(x, "cuda")
        if ws is None:
            ws = torch.empty((self.workspace_bytes * planes // 2,), dtype=torch.uint8, device=x.device)
        self._check(self._L.corr_corner_turn_planes(self._h, x.data_ptr(), ws.data_ptr(), int(planes), _stream_ptr(stream)))
        return ws

    def close(self):
        if getattr(self, "_h", None):
            self._L.corr_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()


class CrossCorrelator(Correlator):
    """corr_create_cross / corr_xengine_cross: rectangular cross-only X-engine of two station groups."""

    def __init__(self, n_station_a, n_station_b, n_pol, n_chan, n_time, dtype="ci8"):
        self._L = lib()
        self.N, self.Nb, self.P, self.C, self.T, self.dtype = n_station_a, n_station_b, n_pol, n_chan, n_time, dtype
        self._h = self._L.corr_create_cross(n_station_a, n_station_b, n_pol, n_chan, n_time, DTYPES[dtype])
        if not self._h:
            msg = self._L.corr_last_error(None).decode()
            raise CorrError(CORR_EINVAL if "invalid" in msg or "too large" in msg else CORR_EUNSUPPORTED, msg)
        self.n_baseline = n_station_a * n_station_b

    @property
    def input_bytes_b(self):
        return int(self._L.corr_input_bytes_b(self._h))

    def input_shape_b(self):
        return (self.T, self.C, self.Nb, self.P, 2)

    def output_shape(self):
        return (self.C, self.N, self.Nb, self.P, self.P, 2)

    def xengine_cross(self, xa, xb, out=None, accumulate=False, stream=None):
        import torch
        self._check_in(xa, "cuda")
        want = torch.int8 if self.dtype == "ci8" else torch.float16
        if xb.dtype != want or tuple(xb.shape) != self.input_shape_b() or not xb.is_contiguous() or xb.device.type != "cuda":
            raise ValueError("group B must be a contiguous CUDA %s tensor of shape %s" % (want, self.input_shape_b()))
        if out is None:
            if accumulate:
                raise ValueError("accumulate=True needs the running `out`")
            out = self.empty_output(xa.device)
        self._check_out(out, "cuda")
        self._check(self._L.corr_xengine_cross(self._h, xa.data_ptr(), xb.data_ptr(), out.data_ptr(),
                                               int(bool(accumulate)), _stream_ptr(stream)))
        return out
