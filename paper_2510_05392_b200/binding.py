"""Thin ctypes binding over the C ABI in include/mg5_b200.h -- argument marshalling only.

Every step of the hot path runs inside libmg5_b200.so (hand-written CUDA for sm_100a).  PyTorch is used
here only for device memory and streams.  There is NO CPU fallback: a missing library or a device that is
not a B200 raises.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmg5_b200.so")

MG_FP64, MG_MIXED, MG_FP32 = 0, 1, 2
MG_CS_FUSED, MG_CS_TENSOR = 0, 1
MG_SCHED_GRID, MG_SCHED_STREAMS = 0, 1
PRECISIONS = {"fp64": MG_FP64, "d": MG_FP64, "mixed": MG_MIXED, "m": MG_MIXED, "fp32": MG_FP32, "f": MG_FP32}

_ERR = {-1: "MG_EINVAL", -2: "MG_ENODEV", -3: "MG_ENOMEM", -4: "MG_ECUDA", -5: "MG_ESTATE"}

EXPORTS = ["mg_init_process", "mg_process_info", "mg_process_flops", "mg_set_parameters", "mg_set_option", "mg_get_option",
           "mg_workspace_bytes", "mg_workspace_bytes_ex", "mg_helicity_filter", "mg_set_good_helicities", "mg_sigma_batch",
           "mg_sigma_batch_ex", "mg_sigma_batch_noalloc",
           "mg_sigma_batch_host", "mg_last_helicity_terms", "mg_last_stage_ms", "mg_last_launch_count", "mg_color_sum", "mg_color_matrix",
           "mg_measure_peak", "mg_last_error", "mg_destroy"]

NOALLOC_MAX_EVENTS = 256          # MG_NOALLOC_MAX_EVENTS of include/mg5_b200.h

_lib = None


class MGError(RuntimeError):
    pass


def load_library() -> ctypes.CDLL:
    """dlopen the in-tree CUDA library; raises if it has not been built (no fallback of any kind)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise MGError(f"{LIB_PATH} is missing: build it with `python -m paper_2510_05392_b200.build` "
                      "(or __graft_entry__.build()); there is no CPU fallback")
    lib = ctypes.CDLL(LIB_PATH)
    vp, ip, dp = ctypes.c_void_p, ctypes.POINTER(ctypes.c_int), ctypes.POINTER(ctypes.c_double)
    lib.mg_init_process.argtypes = [ctypes.c_char_p, ctypes.c_int, ctypes.c_int, ctypes.POINTER(vp)]
    lib.mg_process_info.argtypes = [vp, ip, ip, ip, ip, ip]
    lib.mg_process_flops.argtypes = [vp, dp, dp]
    lib.mg_set_parameters.argtypes = [vp, ctypes.POINTER(ctypes.c_char_p), dp, ctypes.c_int]
    lib.mg_set_option.argtypes = [vp, ctypes.c_char_p, ctypes.c_int]
    lib.mg_get_option.argtypes = [vp, ctypes.c_char_p, ip]
    lib.mg_workspace_bytes.argtypes = [vp, ctypes.c_int]
    lib.mg_workspace_bytes.restype = ctypes.c_size_t
    lib.mg_helicity_filter.argtypes = [vp, vp, ctypes.c_int, vp, ctypes.c_size_t, vp, ctypes.POINTER(ctypes.c_ubyte), ip]
    lib.mg_set_good_helicities.argtypes = [vp, ctypes.POINTER(ctypes.c_ubyte)]
    lib.mg_sigma_batch.argtypes = [vp, vp, ctypes.c_int, vp, vp, ctypes.c_size_t, vp]
    lib.mg_sigma_batch_noalloc.argtypes = [vp, vp, ctypes.c_int, vp, vp, ctypes.c_size_t, vp]
    lib.mg_sigma_batch_ex.argtypes = [vp, vp, ctypes.c_int, vp, vp, vp, vp, vp, vp, vp, ctypes.c_size_t, vp]
    lib.mg_workspace_bytes_ex.argtypes = [vp, ctypes.c_int, ctypes.c_int]
    lib.mg_workspace_bytes_ex.restype = ctypes.c_size_t
    lib.mg_sigma_batch_host.argtypes = [vp, vp, ctypes.c_int, vp]
    lib.mg_last_helicity_terms.argtypes = [vp, ctypes.c_int, vp, vp, vp]
    lib.mg_last_stage_ms.argtypes = [vp, ctypes.POINTER(ctypes.c_float)]
    lib.mg_last_launch_count.argtypes = [vp, ip]
    lib.mg_color_sum.argtypes = [vp, ctypes.c_int, vp, ctypes.c_long, vp, vp]
    lib.mg_color_matrix.argtypes = [vp, ip, ip]
    lib.mg_measure_peak.argtypes = [ctypes.c_int, ctypes.c_int, dp]
    lib.mg_last_error.argtypes = [vp]
    lib.mg_last_error.restype = ctypes.c_char_p
    lib.mg_destroy.argtypes = [vp]
    lib.mg_destroy.restype = None
    _lib = lib
    return lib


def measure_peak(kind: int, device: int = 0) -> float:
    """TFLOP/s of a probe kernel: 0 fp64 FMA, 1 fp32 FMA, 2 DMMA f64, 3 tcgen05 TF32."""
    lib = load_library()
    v = ctypes.c_double(0.0)
    rc = lib.mg_measure_peak(device, kind, ctypes.byref(v))
    if rc != 0:
        raise MGError(f"mg_measure_peak({kind}) -> {_ERR.get(rc, rc)}")
    return v.value


class Process:
    """One physics process on one GPU: init_process / set_parameters / sigma_batch (same names as the C ABI)."""

    def __init__(self, name: str, precision="fp64", device: int = 0):
        import torch  # device memory and streams only
        self._torch = torch
        self.lib = load_library()
        self.name = name
        self.precision = PRECISIONS[precision] if isinstance(precision, str) else int(precision)
        self.device = device
        h = ctypes.c_void_p()
        rc = self.lib.mg_init_process(name.encode(), self.precision, device, ctypes.byref(h))
        if rc != 0:
            raise MGError(f"mg_init_process({name}) -> {_ERR.get(rc, rc)}: {self.lib.mg_last_error(None).decode()}")
        self.h = h
        v = [ctypes.c_int() for _ in range(5)]
        self._check(self.lib.mg_process_info(self.h, *[ctypes.byref(x) for x in v]))
        self.npar, self.ncomb, self.ncolor, self.ndiagrams, self.ngroups = [x.value for x in v]
        self._read_flops()
        self._ws = None
        self.ngood = None

    def _read_flops(self):
        a, b = ctypes.c_double(), ctypes.c_double()
        self._check(self.lib.mg_process_flops(self.h, ctypes.byref(a), ctypes.byref(b)))
        self.diagram_flops, self.color_flops = a.value, b.value

    # -- plumbing -----------------------------------------------------------------------------------
    def _check(self, rc):
        if rc != 0:
            raise MGError(f"{_ERR.get(rc, rc)}: {self.lib.mg_last_error(self.h).decode()}")

    def close(self):
        if getattr(self, "h", None):
            self.lib.mg_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _stream(self):
        return ctypes.c_void_p(self._torch.cuda.current_stream(self.device).cuda_stream)

    def _workspace(self, nevt, want_selcol=False):
        need = self.lib.mg_workspace_bytes_ex(self.h, nevt, 1 if want_selcol else 0)
        if self._ws is None or self._ws.numel() < need:
            self._ws = self._torch.empty(max(need, 256), dtype=self._torch.uint8, device=f"cuda:{self.device}")
        return self._ws

    # -- C ABI, same names ----------------------------------------------------------------------------
    def set_parameters(self, **kw):
        keys = (ctypes.c_char_p * len(kw))(*[k.encode() for k in kw])
        vals = (ctypes.c_double * len(kw))(*[float(v) for v in kw.values()])
        self._check(self.lib.mg_set_parameters(self.h, keys, vals, len(kw)))

    def set_option(self, key: str, value: int):
        self._check(self.lib.mg_set_option(self.h, key.encode(), int(value)))
        self._read_flops()
        self._ws = None

    def get_option(self, key: str) -> int:
        v = ctypes.c_int()
        self._check(self.lib.mg_get_option(self.h, key.encode(), ctypes.byref(v)))
        return v.value

    def helicity_filter(self, d_momenta, nprobe=None):
        nevt = d_momenta.shape[0]
        nprobe = min(nevt, self.get_option("probe_events")) if nprobe is None else nprobe
        ws = self._workspace(max(nevt, nprobe))
        mask = (ctypes.c_ubyte * self.ncomb)()
        ng = ctypes.c_int()
        self._check(self.lib.mg_helicity_filter(self.h, d_momenta.data_ptr(), nprobe, ws.data_ptr(), ws.numel(),
                                                self._stream(), mask, ctypes.byref(ng)))
        self.ngood = ng.value
        self._ws = None
        return np.array(list(mask), dtype=np.uint8)

    def set_good_helicities(self, mask):
        m = (ctypes.c_ubyte * self.ncomb)(*[int(x) for x in mask])
        self._check(self.lib.mg_set_good_helicities(self.h, m))
        self.ngood = int(sum(int(x) != 0 for x in mask))
        self._ws = None

    def sigma_batch(self, d_momenta, d_me=None):
        """d_momenta: cuda fp64 tensor [nevt][npar][4]; returns (or fills) d_me: cuda fp64 [nevt]. Asynchronous."""
        t = self._torch
        assert d_momenta.is_cuda and d_momenta.dtype == t.float64 and d_momenta.is_contiguous()
        nevt = d_momenta.shape[0]
        assert tuple(d_momenta.shape[1:]) == (self.npar, 4)
        if d_me is None:
            d_me = t.empty(nevt, dtype=t.float64, device=d_momenta.device)
        if self.ngood is None and nevt > 0:
            # the library would run the filter itself; do it here so that the workspace is sized for the result
            self.helicity_filter(d_momenta)
        ws = self._workspace(nevt)
        self._check(self.lib.mg_sigma_batch(self.h, d_momenta.data_ptr(), nevt, d_me.data_ptr(), ws.data_ptr(), ws.numel(),
                                            self._stream()))
        return d_me

    def sigma_batch_noalloc(self, d_momenta, d_me=None):
        """mg_sigma_batch_noalloc: as sigma_batch, the library allocating nothing (gg_ttxgggg, <= NOALLOC_MAX_EVENTS events, a
        helicity list already installed).  The output and the workspace are allocated HERE, by the caller's side."""
        t = self._torch
        assert d_momenta.is_cuda and d_momenta.dtype == t.float64 and d_momenta.is_contiguous()
        nevt = d_momenta.shape[0]
        if d_me is None:
            d_me = t.empty(nevt, dtype=t.float64, device=d_momenta.device)
        ws = self._workspace(nevt)
        self._check(self.lib.mg_sigma_batch_noalloc(self.h, d_momenta.data_ptr(), nevt, d_me.data_ptr(), ws.data_ptr(), ws.numel(),
                                                    self._stream()))
        return d_me

    def sigma_batch_ex(self, d_momenta, alphas=None, rndhel=None, rndcol=None):
        """mg_sigma_batch_ex: optional per-event alpha_s and the two random numbers per event (cuda fp64 [nevt] each);
        returns (d_me, d_selhel or None, d_selcol or None), the selections as cuda int32 [nevt]. Asynchronous."""
        t = self._torch
        assert d_momenta.is_cuda and d_momenta.dtype == t.float64 and d_momenta.is_contiguous()
        nevt = d_momenta.shape[0]
        for x in (alphas, rndhel, rndcol):
            assert x is None or (x.is_cuda and x.dtype == t.float64 and x.is_contiguous() and x.shape == (nevt,))
        d_me = t.empty(nevt, dtype=t.float64, device=d_momenta.device)
        selhel = t.empty(nevt, dtype=t.int32, device=d_momenta.device) if rndhel is not None else None
        selcol = t.empty(nevt, dtype=t.int32, device=d_momenta.device) if rndcol is not None else None
        if self.ngood is None and nevt > 0:
            self.helicity_filter(d_momenta)
        ws = self._workspace(nevt, rndcol is not None)
        ptr = lambda x: x.data_ptr() if x is not None else None
        self._check(self.lib.mg_sigma_batch_ex(self.h, d_momenta.data_ptr(), nevt, ptr(alphas), ptr(rndhel), ptr(rndcol),
                                               d_me.data_ptr(), ptr(selhel), ptr(selcol), ws.data_ptr(), ws.numel(), self._stream()))
        return d_me, selhel, selcol

    def sigma_batch_host(self, h_momenta: np.ndarray, h_me: np.ndarray | None = None):
        """host buffers in, host buffer out (copies inside the library, synchronous)"""
        h_momenta = np.ascontiguousarray(h_momenta, dtype=np.float64)
        nevt = h_momenta.shape[0]
        if h_me is None:
            h_me = np.empty(nevt, dtype=np.float64)
        self._check(self.lib.mg_sigma_batch_host(self.h, h_momenta.ctypes.data, nevt, h_me.ctypes.data))
        return h_me

    def last_helicity_terms(self, nevt):
        t = self._torch
        out = t.empty((self.ngood, nevt), dtype=t.float64, device=f"cuda:{self.device}")
        self._check(self.lib.mg_last_helicity_terms(self.h, nevt, self._ws.data_ptr(), out.data_ptr(), self._stream()))
        return out

    def last_stage_ms(self):
        ms = (ctypes.c_float * 3)()
        self._check(self.lib.mg_last_stage_ms(self.h, ms))
        return [ms[0], ms[1], ms[2]]

    def last_launch_count(self):
        n = ctypes.c_int()
        self._check(self.lib.mg_last_launch_count(self.h, ctypes.byref(n)))
        return n.value

    def color_sum(self, d_jamps, impl=MG_CS_TENSOR):
        """d_jamps: cuda tensor [2][ncolor][nrows] (fp64 for MG_FP64, fp32 otherwise) -> cuda fp64 [nrows] (numerators only)"""
        t = self._torch
        nrows = d_jamps.shape[2]
        out = t.empty(nrows, dtype=t.float64, device=d_jamps.device)
        self._check(self.lib.mg_color_sum(self.h, impl, d_jamps.data_ptr(), nrows, out.data_ptr(), self._stream()))
        return out

    def color_matrix(self):
        num = (ctypes.c_int * (self.ncolor * self.ncolor))()
        den = ctypes.c_int()
        self._check(self.lib.mg_color_matrix(self.h, num, ctypes.byref(den)))
        return np.array(list(num), dtype=np.int64).reshape(self.ncolor, self.ncolor), den.value


def init_process(name: str, precision="fp64", device: int = 0) -> Process:
    return Process(name, precision, device)
