"""Thin Python binding of the C ABI (include/me_b200.h): argument marshalling only.

Same names as the C entry points (me_create -> MatrixElement(...), me_compute -> .compute(...), ...).
torch is used for device memory and streams, nothing else; every step of the hot path runs in the
CUDA kernels of libme_b200.so.  There is no CPU path: if the library or a CUDA device is missing,
construction raises.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libme_b200.so")
PRECISIONS = {"fp64": 0, "fp32": 1, "mixed": 2}
PROCESSES = ("ee_mumu", "gg_tt", "gg_ttg", "gg_ttgg", "gg_ttggg", "gux_taptamux", "gux_taptamgux", "gux_taptamggux")

EXPORTS = ("me_create", "me_destroy", "me_last_error", "me_info", "me_helicity_table", "me_color_table",
           "me_color_matrix", "me_filter_helicities", "me_get_good_helicities", "me_set_good_helicities",
           "me_compute", "me_reserve", "me_compute_noalloc", "me_compute_multichannel", "me_channel_table", "me_compute_host", "me_generate", "me_launch_info", "me_launch_stats", "me_fma_peak", "me_mma_peak")


class MEError(RuntimeError):
    pass


class me_params(ctypes.Structure):
    _fields_ = [(k, ctypes.c_double) for k in ("mt", "wt", "mz", "wz", "aewm1", "gf")]


_lib = None


def load_library(path: str = LIB_PATH):
    """dlopen libme_b200.so and declare the prototypes.  Raises if it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(path):
        raise MEError(f"{path} not found: run `python -m paper_2503_21935_b200.build` (there is no fallback path)")
    L = ctypes.CDLL(path)
    vp, i64, ip = ctypes.c_void_p, ctypes.c_int64, ctypes.POINTER(ctypes.c_int)
    L.me_create.argtypes = [ctypes.POINTER(vp), ctypes.c_char_p, ctypes.c_int, ctypes.POINTER(me_params), ctypes.c_int]
    L.me_destroy.argtypes = [vp]
    L.me_last_error.argtypes = [vp]
    L.me_last_error.restype = ctypes.c_char_p
    L.me_info.argtypes = [vp, ip, ip, ip, ip, ip]
    L.me_helicity_table.argtypes = [vp, vp]
    L.me_color_table.argtypes = [vp, vp]
    L.me_color_matrix.argtypes = [vp, vp]
    L.me_filter_helicities.argtypes = [vp, vp, vp, i64, vp]
    L.me_get_good_helicities.argtypes = [vp, ip, vp]
    L.me_set_good_helicities.argtypes = [vp, vp]
    L.me_reserve.argtypes = [vp, i64]
    L.me_compute.argtypes = [vp, vp, vp, vp, vp, i64, vp, vp, vp, vp]
    L.me_compute_noalloc.argtypes = [ctypes.POINTER(me_params), vp, vp, vp, vp, vp, i64, vp, vp, vp, vp, ctypes.c_char_p, ctypes.c_int]
    L.me_compute_multichannel.argtypes = [vp, vp, vp, vp, vp, vp, i64, vp, vp, vp, vp, vp, vp]
    L.me_channel_table.argtypes = [vp, ctypes.c_char_p, ctypes.c_int]
    L.me_compute_host.argtypes = [vp, vp, vp, vp, vp, i64, vp, vp, vp]
    L.me_generate.argtypes = [vp, ctypes.c_uint64, i64, i64, ctypes.c_double, ctypes.c_double, vp, vp, vp, vp, vp, vp]
    L.me_launch_info.argtypes = [vp, ip, ip, ip, ip]
    L.me_launch_stats.argtypes = [vp, ip, ctypes.POINTER(ctypes.c_int64), ctypes.POINTER(ctypes.c_int64)]
    L.me_fma_peak.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.POINTER(ctypes.c_double)]
    L.me_mma_peak.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.POINTER(ctypes.c_double)]
    for n in EXPORTS:
        if n != "me_last_error":
            getattr(L, n).restype = ctypes.c_int
    _lib = L
    return L


def _ptr(t, dtype=None, device=None):
    """Device pointer of a contiguous CUDA tensor (or None); with `device`, the tensor must live on that ordinal."""
    if t is None:
        return None
    if not t.is_cuda or not t.is_contiguous():
        raise MEError("expected a contiguous CUDA tensor")
    if device is not None and t.device.index != device:
        raise MEError(f"tensor on cuda:{t.device.index}, but this handle was created for cuda:{device}")
    if dtype is not None and t.dtype != dtype:
        raise MEError(f"expected dtype {dtype}, got {t.dtype}")
    return ctypes.c_void_p(t.data_ptr())


def _hptr(a):
    return None if a is None else ctypes.c_void_p(a.ctypes.data)


class MatrixElement:
    """One handle of the C library: a (process, precision, parameters, device) tuple."""

    def __init__(self, process: str, precision: str = "fp64", params: dict | None = None, device: int = 0):
        self._L = load_library()
        self._h = ctypes.c_void_p()
        p = None
        if params is not None:
            d = dict(mt=173.0, wt=1.4915, mz=91.188, wz=2.441, aewm1=132.507, gf=1.16639e-5)
            d.update(params)
            p = me_params(**d)
        rc = self._L.me_create(ctypes.byref(self._h), process.encode(), PRECISIONS[precision],
                               ctypes.byref(p) if p is not None else None, device)
        if rc != 0:
            msg = self._L.me_last_error(None)
            self._h = ctypes.c_void_p()
            raise MEError(f"me_create failed ({rc}): {msg.decode() if msg else ''}")
        self.process, self.precision, self.device = process, precision, device
        v = [ctypes.c_int() for _ in range(5)]
        self._check(self._L.me_info(self._h, *[ctypes.byref(x) for x in v]))
        self.npar, self.ncomb, self.ncol, self.ndiag, self.denom = (x.value for x in v)
        self.ngluon = {"ee_mumu": 0, "gux_taptamux": 1, "gux_taptamgux": 2, "gux_taptamggux": 3}.get(process, self.npar - 2)

    def _check(self, rc):
        if rc != 0:
            msg = self._L.me_last_error(self._h)
            raise MEError(f"error {rc}: {msg.decode() if msg else ''}")

    def _same_device(self, stream):
        if getattr(stream, "device", None) is not None and stream.device.index != self.device:
            raise MEError(f"stream on cuda:{stream.device.index}, but this handle was created for cuda:{self.device}")

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            self._L.me_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- tables
    def helicity_table(self) -> np.ndarray:
        out = np.zeros((self.ncomb, self.npar), dtype=np.int8)
        self._check(self._L.me_helicity_table(self._h, _hptr(out)))
        return out

    def color_table(self) -> np.ndarray:
        out = np.zeros((self.ncol, self.ngluon), dtype=np.int8)
        self._check(self._L.me_color_table(self._h, _hptr(out) if self.ngluon else None))
        return out

    def color_matrix(self) -> np.ndarray:
        out = np.zeros((self.ncol, self.ncol), dtype=np.float64)
        self._check(self._L.me_color_matrix(self._h, _hptr(out)))
        return out

    # ---- helicity filter
    def filter_helicities(self, momenta, gs=None, stream=None):
        import torch
        nevt = momenta.shape[0]
        s = stream if stream is not None else torch.cuda.current_stream(momenta.device)
        self._same_device(s)
        self._check(self._L.me_filter_helicities(self._h, _ptr(momenta, torch.float64, self.device), _ptr(gs, torch.float64, self.device), nevt,
                                                 ctypes.c_void_p(s.cuda_stream)))
        return self.get_good_helicities()

    def get_good_helicities(self) -> np.ndarray:
        n = ctypes.c_int()
        mask = np.zeros(self.ncomb, dtype=np.uint8)
        self._check(self._L.me_get_good_helicities(self._h, ctypes.byref(n), _hptr(mask)))
        return mask

    def set_good_helicities(self, mask):
        m = np.ascontiguousarray(mask, dtype=np.uint8)
        if m.shape != (self.ncomb,):
            raise MEError("mask must have ncomb entries")
        self._check(self._L.me_set_good_helicities(self._h, _hptr(m)))

    def reserve(self, max_events_per_call: int):
        """me_reserve: size the pipeline scratch (gg_ttgg / gg_ttggg) for calls of up to that many events."""
        self._check(self._L.me_reserve(self._h, int(max_events_per_call)))

    # ---- hot path
    def compute(self, momenta, gs=None, rndhel=None, rndcol=None, out=None, selhel=None, selcol=None, stream=None):
        """Enqueue ME (and optional selections) on `stream` (default: torch's current stream).

        momenta: cuda float64 [nevt, npar, 4]; gs: cuda float64 [nevt]; rndhel/rndcol: cuda float64 [nevt].
        Returns (me, selhel, selcol) tensors (selections None unless their random numbers are given).
        """
        import torch
        nevt = momenta.shape[0]
        if tuple(momenta.shape[1:]) != (self.npar, 4):
            raise MEError(f"momenta must be [nevt, {self.npar}, 4]")
        dev = momenta.device
        if out is None:
            out = torch.empty(nevt, dtype=torch.float64, device=dev)
        if rndhel is not None and selhel is None:
            selhel = torch.empty(nevt, dtype=torch.int32, device=dev)
        if rndcol is not None and selcol is None:
            selcol = torch.empty(nevt, dtype=torch.int32, device=dev)
        s = stream if stream is not None else torch.cuda.current_stream(dev)
        f64, d = torch.float64, self.device
        self._same_device(s)
        self._check(self._L.me_compute(self._h, _ptr(momenta, f64, d), _ptr(gs, f64, d), _ptr(rndhel, f64, d), _ptr(rndcol, f64, d),
                                       nevt, _ptr(out, f64, d), _ptr(selhel, torch.int32, d), _ptr(selcol, torch.int32, d),
                                       ctypes.c_void_p(s.cuda_stream)))
        return out, selhel, selcol

    def compute_multichannel(self, momenta, gs, channel, rndhel=None, rndcol=None, stream=None):
        """me_compute_multichannel: returns (me, selhel, selcol, num, den); channel: cuda int32 [nevt]."""
        import torch
        nevt = momenta.shape[0]
        dev, d = momenta.device, self.device
        f64 = torch.float64
        out, num, den = (torch.empty(nevt, dtype=f64, device=dev) for _ in range(3))
        selhel = torch.empty(nevt, dtype=torch.int32, device=dev) if rndhel is not None else None
        selcol = torch.empty(nevt, dtype=torch.int32, device=dev) if rndcol is not None else None
        s = stream if stream is not None else torch.cuda.current_stream(dev)
        self._same_device(s)
        self._check(self._L.me_compute_multichannel(
            self._h, _ptr(momenta, f64, d), _ptr(gs, f64, d), _ptr(rndhel, f64, d), _ptr(rndcol, f64, d),
            _ptr(channel, torch.int32, d), nevt, _ptr(out, f64, d), _ptr(selhel, torch.int32, d), _ptr(selcol, torch.int32, d),
            _ptr(num, f64, d), _ptr(den, f64, d), ctypes.c_void_p(s.cuda_stream)))
        return out, selhel, selcol, num, den

    def channel_table(self) -> list:
        n = self._L.me_channel_table(self._h, None, 0)
        if n < 0:
            self._check(n)
        buf = ctypes.create_string_buffer(n)
        self._check(min(0, self._L.me_channel_table(self._h, buf, n)))
        return buf.value.decode().split("\n")[:-1]

    def compute_host(self, momenta, gs=None, rndhel=None, rndcol=None, out=None, selhel=None, selcol=None):
        """Host buffers in, host buffers out (numpy arrays or pinned CPU tensors viewed as numpy); synchronous."""
        mom = _as_np(momenta, np.float64)
        nevt = mom.shape[0]
        gs, rndhel, rndcol = _as_np(gs, np.float64), _as_np(rndhel, np.float64), _as_np(rndcol, np.float64)
        out = np.empty(nevt, dtype=np.float64) if out is None else _as_np(out, np.float64)
        if rndhel is not None and selhel is None:
            selhel = np.empty(nevt, dtype=np.int32)
        if rndcol is not None and selcol is None:
            selcol = np.empty(nevt, dtype=np.int32)
        selhel, selcol = _as_np(selhel, np.int32), _as_np(selcol, np.int32)
        self._check(self._L.me_compute_host(self._h, _hptr(mom), _hptr(gs), _hptr(rndhel), _hptr(rndcol), nevt,
                                            _hptr(out), _hptr(selhel), _hptr(selcol)))
        return out, selhel, selcol

    def generate(self, nevt, seed=1, start=0, sqrts=1500.0, alphas=0.0, device=None, want_weight=False, stream=None):
        """Seeded RAMBO inputs made on the device (me_generate): returns (momenta, gs, rndhel, rndcol[, weight])
        as cuda float64 tensors for events start..start+nevt-1 of the stream; alphas <= 0 draws alpha_s ~ U[0.10, 0.13]."""
        import torch
        dev = torch.device("cuda", self.device) if device is None else device
        f64 = torch.float64
        mom = torch.empty((nevt, self.npar, 4), dtype=f64, device=dev)
        gs, rh, rc = (torch.empty(nevt, dtype=f64, device=dev) for _ in range(3))
        wt = torch.empty(nevt, dtype=f64, device=dev) if want_weight else None
        s = stream if stream is not None else torch.cuda.current_stream(dev)
        if dev.index != self.device:
            raise MEError(f"device cuda:{dev.index} requested, but this handle was created for cuda:{self.device}")
        self._same_device(s)
        self._check(self._L.me_generate(self._h, int(seed), int(start), int(nevt), float(sqrts), float(alphas), _ptr(mom, f64),
                                        _ptr(gs, f64), _ptr(rh, f64), _ptr(rc, f64), _ptr(wt, f64), ctypes.c_void_p(s.cuda_stream)))
        return (mom, gs, rh, rc, wt) if want_weight else (mom, gs, rh, rc)

    def launch_info(self) -> dict:
        v = [ctypes.c_int() for _ in range(4)]
        self._check(self._L.me_launch_info(self._h, *[ctypes.byref(x) for x in v]))
        d = dict(zip(("threads", "blocks", "regs", "local_bytes"), (x.value for x in v)))
        n, c, b = ctypes.c_int(), ctypes.c_int64(), ctypes.c_int64()
        self._check(self._L.me_launch_stats(self._h, ctypes.byref(n), ctypes.byref(c), ctypes.byref(b)))
        d.update(launches=n.value, chunk_events=c.value, scratch_bytes=b.value)
        return d


NOALLOC_MAX_EVENTS = 16384   # ME_NOALLOC_MAX_EVENTS of include/me_b200.h


def compute_noalloc(momenta, gs, rndhel=None, rndcol=None, good_mask=None, params: dict | None = None, out=None,
                    selhel=None, selcol=None, stream=None):
    """me_compute_noalloc: gg -> t tbar g in fp64 without a handle and without any device allocation by the library.

    For callers that cannot let a library call cudaMalloc (the GPU's memory belongs to the application's own pool or
    budget, or an allocation's device-wide stall is not affordable): the kernel's scratch is a fixed 4 MiB array inside
    the library, so at most NOALLOC_MAX_EVENTS events per call; more raises MEError.  Calls on one GPU share that
    array: keep them on one stream (overlapping calls corrupt each other's helicity choice).

    momenta: cuda float64 [nevt, 5, 4]; gs, rndhel, rndcol: cuda float64 [nevt]; good_mask: 32 uint8 (None = all).
    This binding allocates nothing either if out (float64 [nevt]) and, with random numbers, selhel / selcol (int32
    [nevt]) are passed in; otherwise it makes them with torch.  Returns (me, selhel, selcol), enqueued on `stream`.
    """
    import torch
    L = load_library()
    nevt = momenta.shape[0]
    if tuple(momenta.shape[1:]) != (5, 4):
        raise MEError("momenta must be [nevt, 5, 4]")
    dev = momenta.device
    if out is None:
        out = torch.empty(nevt, dtype=torch.float64, device=dev)
    if rndhel is not None and selhel is None:
        selhel = torch.empty(nevt, dtype=torch.int32, device=dev)
    if rndcol is not None and selcol is None:
        selcol = torch.empty(nevt, dtype=torch.int32, device=dev)
    s = stream if stream is not None else torch.cuda.current_stream(dev)
    p = None
    if params is not None:
        d = dict(mt=173.0, wt=1.4915, mz=91.188, wz=2.441, aewm1=132.507, gf=1.16639e-5)
        d.update(params)
        p = me_params(**d)
    m = None
    if good_mask is not None:
        m = np.ascontiguousarray(good_mask, dtype=np.uint8)
        if m.shape != (32,):
            raise MEError("good_mask must have 32 entries")
    err = ctypes.create_string_buffer(256)
    f64, di = torch.float64, dev.index
    with torch.cuda.device(dev):   # the entry point works on the calling thread's current device
        rc = L.me_compute_noalloc(ctypes.byref(p) if p is not None else None, _hptr(m), _ptr(momenta, f64, di), _ptr(gs, f64, di),
                                  _ptr(rndhel, f64, di), _ptr(rndcol, f64, di), nevt, _ptr(out, f64, di),
                                  _ptr(selhel, torch.int32, di), _ptr(selcol, torch.int32, di), ctypes.c_void_p(s.cuda_stream),
                                  err, len(err))
    if rc != 0:
        raise MEError(f"error {rc}: {err.value.decode()}")
    return out, selhel, selcol


def fma_peak(precision: str = "fp64", device: int = 0) -> float:
    """Measured FMA peak in TFLOP/s (me_fma_peak)."""
    v = ctypes.c_double()
    rc = load_library().me_fma_peak(PRECISIONS[precision], device, ctypes.byref(v))
    if rc != 0:
        raise MEError(f"me_fma_peak failed ({rc})")
    return v.value


def mma_peak(kind: str = "dmma", device: int = 0) -> float:
    """Measured tensor-pipe peak in TFLOP/s (me_mma_peak): kind "dmma" (m8n8k4 f64) or "tf32" (m16n8k8)."""
    v = ctypes.c_double()
    rc = load_library().me_mma_peak({"dmma": 0, "tf32": 1}[kind], device, ctypes.byref(v))
    if rc != 0:
        raise MEError(f"me_mma_peak failed ({rc})")
    return v.value


def _as_np(a, dtype):
    if a is None:
        return None
    if not isinstance(a, np.ndarray):
        a = a.numpy()  # CPU torch tensor (pinned or not): zero-copy view
    if a.dtype != dtype or not a.flags["C_CONTIGUOUS"]:
        raise MEError(f"expected a C-contiguous {dtype} host array")
    return a
