"""paper_0906_1887_b200 -- Python binding of the B200 X-engine C ABI (include/corr.h).

Argument marshalling only: every step of the hot path runs in the CUDA kernels of libcorr.so.
Names mirror the C entry points (corr_create / corr_xengine / corr_destroy).
torch is used for device memory and streams, nothing else.  There is no CPU fallback: if
libcorr.so is missing or cannot be loaded, importing the binding's functions raises.
"""
from __future__ import annotations

import ctypes
import os

from . import build as _build

CORR_CI8, CORR_CF32, CORR_CI4 = 0, 1, 2
CORR_OK, CORR_EINVAL, CORR_EUNSUPPORTED, CORR_EALLOC, CORR_ECUDA, CORR_EARCH = range(6)
CORR_TURN_FUSED, CORR_TURN_STANDALONE = 0, 1
CORR_STATIC_BATCH_BYTES = 16 << 20   # include/corr.h: capacity of corr_accumulate_wide_static's built-in batch buffer
CORR_OPT_DIAG_PLAN, CORR_OPT_PAIRS, CORR_OPT_WIDE, CORR_OPT_UNITS, CORR_OPT_F32_GENERIC, CORR_OPT_PDL, CORR_OPT_COLLECT, CORR_OPT_RESIDENT, CORR_OPT_MIX = 1, 2, 3, 4, 5, 6, 7, 8, 9

# include/corr.h (the product ABI, libcorr.so)
EXPORTS = ("corr_create", "corr_xengine", "corr_destroy", "corr_last_error", "corr_last_status",
           "corr_in_bytes", "corr_vis_bytes", "corr_launches_per_call", "corr_set_turn",
           "corr_corner_turn", "corr_stream_run", "corr_set_accumulate", "corr_accumulate_count", "corr_normalize",
           "corr_accumulate_wide", "corr_accumulate_wide_static", "corr_normalize_wide", "corr_acc_bytes", "corr_xengine_batch", "corr_set_chan_window",
           "corr_set_option", "corr_plan_info",
           "corr_fstage_create", "corr_fstage_run", "corr_fstage_destroy", "corr_fstage_in_bytes", "corr_fstage_out_bytes", "corr_stream_run_fx", "corr_fstage_set_input")
# include/corr_diag.h (diagnostics, libcorr_diag.so only)
DIAG_EXPORTS = ("corr_set_probe", "corr_probe_stats", "corr_probe_mma", "corr_probe_ffma")

_lib = None
_diag = False


class CorrError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"[corr status {status}] {msg}")
        self.status = status


def use_diag_build():
    """Route the whole binding through libcorr_diag.so (the -DCORR_DIAG build: include/corr_diag.h), for the
    where-the-time-goes study.  Must be called before the first lib()."""
    global _diag
    if _lib is not None and not _diag:
        raise RuntimeError("use_diag_build() must come before the library is first loaded")
    _diag = True


def _bind(path, diag):
    L = ctypes.CDLL(path)
    vp, ci = ctypes.c_void_p, ctypes.c_int
    L.corr_create.restype, L.corr_create.argtypes = vp, [ci, ci, ci, ci]
    L.corr_xengine.restype, L.corr_xengine.argtypes = ci, [vp, vp, vp, vp]
    L.corr_destroy.restype, L.corr_destroy.argtypes = ci, [vp]
    L.corr_last_error.restype, L.corr_last_error.argtypes = ctypes.c_char_p, []
    L.corr_last_status.restype, L.corr_last_status.argtypes = ci, []
    L.corr_in_bytes.restype, L.corr_in_bytes.argtypes = ctypes.c_size_t, [vp]
    L.corr_vis_bytes.restype, L.corr_vis_bytes.argtypes = ctypes.c_size_t, [vp]
    L.corr_launches_per_call.restype, L.corr_launches_per_call.argtypes = ci, [vp]
    L.corr_set_turn.restype, L.corr_set_turn.argtypes = ci, [vp, ci]
    L.corr_set_accumulate.restype, L.corr_set_accumulate.argtypes = ci, [vp, ci]
    L.corr_accumulate_count.restype, L.corr_accumulate_count.argtypes = ctypes.c_longlong, [vp]
    L.corr_normalize.restype = ci
    L.corr_normalize.argtypes = [vp, vp, ctypes.c_double, vp, vp]
    L.corr_normalize_wide.restype = ci
    L.corr_normalize_wide.argtypes = [vp, vp, ctypes.c_double, vp, vp]
    L.corr_accumulate_wide.restype, L.corr_accumulate_wide.argtypes = ci, [vp, vp, vp, vp]
    L.corr_accumulate_wide_static.restype, L.corr_accumulate_wide_static.argtypes = ci, [vp, vp, vp, vp]
    L.corr_acc_bytes.restype, L.corr_acc_bytes.argtypes = ctypes.c_size_t, [vp]
    L.corr_xengine_batch.restype = ci
    L.corr_xengine_batch.argtypes = [vp, ctypes.POINTER(vp), ctypes.POINTER(vp), ci, vp]
    L.corr_set_chan_window.restype, L.corr_set_chan_window.argtypes = ci, [vp, ci, ci]
    L.corr_set_option.restype, L.corr_set_option.argtypes = ci, [vp, ci, ci]
    L.corr_plan_info.restype = ci
    L.corr_plan_info.argtypes = [vp, ctypes.POINTER(ci), ctypes.c_char_p, ctypes.c_size_t]
    if diag:
        L.corr_set_probe.restype, L.corr_set_probe.argtypes = ci, [vp, ci]
        L.corr_probe_stats.restype, L.corr_probe_stats.argtypes = ci, [vp, ctypes.POINTER(ctypes.c_double)]
        L.corr_probe_mma.restype = ci
        L.corr_probe_mma.argtypes = [ci, ci, ci, ci, ctypes.POINTER(ctypes.c_double)]
        L.corr_probe_ffma.restype = ci
        L.corr_probe_ffma.argtypes = [ci, ci, ctypes.POINTER(ctypes.c_double)]
    L.corr_corner_turn.restype, L.corr_corner_turn.argtypes = ci, [vp, vp, vp, vp]
    L.corr_fstage_create.restype, L.corr_fstage_create.argtypes = vp, [ci, ci, ci]
    L.corr_fstage_run.restype, L.corr_fstage_run.argtypes = ci, [vp, vp, vp, vp]
    L.corr_fstage_destroy.restype, L.corr_fstage_destroy.argtypes = ci, [vp]
    L.corr_fstage_set_input.restype, L.corr_fstage_set_input.argtypes = ci, [vp, ci]
    L.corr_fstage_in_bytes.restype, L.corr_fstage_in_bytes.argtypes = ctypes.c_size_t, [vp]
    L.corr_fstage_out_bytes.restype, L.corr_fstage_out_bytes.argtypes = ctypes.c_size_t, [vp]
    L.corr_stream_run_fx.restype = ci
    L.corr_stream_run_fx.argtypes = [vp, vp, ctypes.POINTER(vp), ci, vp, ctypes.POINTER(ctypes.c_double)]
    L.corr_stream_run.restype = ci
    L.corr_stream_run.argtypes = [vp, ctypes.POINTER(vp), ci, vp, ctypes.POINTER(ctypes.c_double)]
    return L


def lib():
    """Load libcorr.so (building it in-tree first if it is stale and nvcc is present)."""
    global _lib
    if _lib is None:
        path = _build.LIB_DIAG if _diag else _build.LIB
        if _build.stale(_diag):
            path = _build.build(diag=_diag)
        _lib = _bind(path, _diag)
    return _lib


_diag_lib = None


def diag_lib():
    """libcorr_diag.so (include/corr_diag.h): peak probes and engine switches.  Diagnostics only."""
    global _diag_lib
    if _diag:
        return lib()
    if _diag_lib is None:
        path = _build.LIB_DIAG
        if _build.stale(True):
            path = _build.build(diag=True)
        _diag_lib = _bind(path, True)
    return _diag_lib


def _raise(L=None):
    L = L or lib()
    raise CorrError(L.corr_last_status(), L.corr_last_error().decode())


def _stream_ptr(stream):
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    return getattr(stream, "cuda_stream", stream)


class Correlator:
    """One planned X-engine shape.  Tensors are torch CUDA tensors (device memory only)."""

    def __init__(self, n_inputs, n_chan, n_time, dtype):
        self.n_inputs, self.n_chan, self.n_time = n_inputs, n_chan, n_time
        self.dtype = {"ci8": CORR_CI8, "cf32": CORR_CF32, "ci4": CORR_CI4}.get(dtype, dtype)
        self._h = lib().corr_create(n_inputs, n_chan, n_time, self.dtype)
        if not self._h:
            _raise()
        self.n_baselines = n_inputs * (n_inputs + 1) // 2
        self.in_bytes = lib().corr_in_bytes(self._h)
        self.vis_bytes = lib().corr_vis_bytes(self._h)

    # -- corr_destroy
    def destroy(self):
        if getattr(self, "_h", None):
            lib().corr_destroy(self._h)
            self._h = None

    __del__ = destroy

    @property
    def launches_per_call(self):
        return lib().corr_launches_per_call(self._h)

    def set_turn(self, mode):
        if lib().corr_set_turn(self._h, mode) != CORR_OK:
            _raise()

    # -- corr_set_option / corr_set_chan_window
    def set_option(self, key, value):
        if lib().corr_set_option(self._h, key, value) != CORR_OK:
            _raise()

    def plan_info(self):
        """corr_plan_info: {"kernel": name, "kernel_id", "gsize", "slices", "grid", "mixed", "stages", "wide", "smem"}."""
        info = (ctypes.c_int * 8)()
        name = ctypes.create_string_buffer(64)
        if lib().corr_plan_info(self._h, info, name, 64) != CORR_OK:
            _raise()
        keys = ("kernel_id", "gsize", "slices", "grid", "mixed", "stages", "wide", "smem")
        out = {k: int(info[i]) for i, k in enumerate(keys)}
        out["kernel"] = name.value.decode()
        out["resident"] = out["kernel_id"] == 2
        return out

    def set_chan_window(self, n_chan_total, chan0):
        """Read channels chan0 .. chan0 + n_chan - 1 of a [T][n_chan_total][N] buffer in place."""
        if lib().corr_set_chan_window(self._h, n_chan_total, chan0) != CORR_OK:
            _raise()
        self.in_bytes = lib().corr_in_bytes(self._h)

    def set_probe(self, mode):
        """Diagnostics build only (use_diag_build())."""
        if lib().corr_set_probe(self._h, mode) != CORR_OK:
            _raise()

    def probe_stats(self):
        """Diagnostics build only: mean cycles per CTA (pair) of the last launch with probe bit 128."""
        out = (ctypes.c_double * 4)()
        if lib().corr_probe_stats(self._h, out) != CORR_OK:
            _raise()
        return {"cycles": out[0], "mma_wait_loads": out[1], "mma_wait_tmem": out[2], "producer_wait_stage": out[3]}

    # -- corr_set_accumulate / corr_normalize
    def set_accumulate(self, on=True):
        if lib().corr_set_accumulate(self._h, 1 if on else 0) != CORR_OK:
            _raise()

    @property
    def accumulate_count(self):
        return lib().corr_accumulate_count(self._h)

    # -- corr_accumulate_wide / corr_normalize_wide
    def empty_acc(self):
        """Zeroed wide accumulators [C][N(N+1)/2][2]: int64 (CI8, CI4) or float64 (CF32)."""
        import torch
        dt = torch.float64 if self.dtype == CORR_CF32 else torch.int64
        return torch.zeros((self.n_chan, self.n_baselines, 2), dtype=dt, device="cuda")

    def accumulate_wide(self, d_in, d_acc, stream=None):
        self._check_in(d_in)
        if not d_acc.is_cuda or not d_acc.is_contiguous() or d_acc.numel() * d_acc.element_size() != 2 * self.vis_bytes:
            raise ValueError(f"d_acc must be a contiguous CUDA tensor of {2 * self.vis_bytes} bytes")
        if lib().corr_accumulate_wide(self._h, d_in.data_ptr(), d_acc.data_ptr(), _stream_ptr(stream)) != CORR_OK:
            _raise()
        return d_acc

    def accumulate_wide_static(self, d_in, d_acc, stream=None):
        """corr_accumulate_wide_static: accumulate_wide() for code that must not allocate device memory (a real-time
        loop that cannot take cudaMalloc's device-wide stall, a host application whose pool owns all of the GPU).  The
        batch is staged in a fixed array inside the library (CORR_STATIC_BATCH_BYTES; larger vis_bytes raise CorrError),
        shared by every handle on the GPU: keep calls stream-ordered, and make the first call during set-up."""
        self._check_in(d_in)
        if not d_acc.is_cuda or not d_acc.is_contiguous() or d_acc.numel() * d_acc.element_size() != 2 * self.vis_bytes:
            raise ValueError(f"d_acc must be a contiguous CUDA tensor of {2 * self.vis_bytes} bytes")
        if lib().corr_accumulate_wide_static(self._h, d_in.data_ptr(), d_acc.data_ptr(), _stream_ptr(stream)) != CORR_OK:
            _raise()
        return d_acc

    def normalize_wide(self, d_acc, count, d_out=None, stream=None):
        import torch
        if d_out is None:
            d_out = torch.empty(d_acc.shape, dtype=torch.float32, device="cuda")
        if lib().corr_normalize_wide(self._h, d_acc.data_ptr(), float(count), d_out.data_ptr(), _stream_ptr(stream)) != CORR_OK:
            _raise()
        return d_out

    # -- corr_xengine_batch
    def xengine_batch(self, d_in_list, d_vis_list=None, stream=None):
        """n integrations in one launch: lists of CUDA tensors, as xengine()."""
        n = len(d_in_list)
        if d_vis_list is None:
            d_vis_list = [self.empty_vis() for _ in range(n)]
        for d_in, d_vis in zip(d_in_list, d_vis_list):
            self._check_in(d_in)
            if not d_vis.is_cuda or not d_vis.is_contiguous() or d_vis.numel() * d_vis.element_size() != self.vis_bytes:
                raise ValueError(f"every d_vis must be a contiguous CUDA tensor of {self.vis_bytes} bytes")
        pin = (ctypes.c_void_p * n)(*[t.data_ptr() for t in d_in_list])
        pout = (ctypes.c_void_p * n)(*[t.data_ptr() for t in d_vis_list])
        if lib().corr_xengine_batch(self._h, pin, pout, n, _stream_ptr(stream)) != CORR_OK:
            _raise()
        return d_vis_list

    def normalize(self, d_vis, count, d_out=None, stream=None):
        """d_vis (raw sums) / count -> float32 [C][N(N+1)/2][2] (PAPER.md:84 read-out)."""
        import torch
        if d_out is None:
            d_out = torch.empty(d_vis.shape, dtype=torch.float32, device="cuda")
        rc = lib().corr_normalize(self._h, d_vis.data_ptr(), float(count), d_out.data_ptr(), _stream_ptr(stream))
        if rc != CORR_OK:
            _raise()
        return d_out

    def empty_vis(self, n=1):
        import torch
        dt = torch.float32 if self.dtype == CORR_CF32 else torch.int32
        shape = (self.n_chan, self.n_baselines, 2) if n == 1 else (n, self.n_chan, self.n_baselines, 2)
        return torch.empty(shape, dtype=dt, device="cuda")

    def _check_in(self, d_in):
        if not d_in.is_cuda or not d_in.is_contiguous() or d_in.numel() * d_in.element_size() != self.in_bytes:
            raise ValueError(f"d_in must be a contiguous CUDA tensor of {self.in_bytes} bytes "
                             f"([T][C][N][2] int8 or float32)")

    # -- corr_xengine
    def xengine(self, d_in, d_vis=None, stream=None):
        """d_in: CUDA [T][C][N][2] int8|float32 -> d_vis: CUDA [C][N(N+1)/2][2] int32|float32 (raw sums)."""
        self._check_in(d_in)
        if d_vis is None:
            d_vis = self.empty_vis()
        if not d_vis.is_cuda or not d_vis.is_contiguous() or d_vis.numel() * d_vis.element_size() != self.vis_bytes:
            raise ValueError(f"d_vis must be a contiguous CUDA tensor of {self.vis_bytes} bytes")
        rc = lib().corr_xengine(self._h, d_in.data_ptr(), d_vis.data_ptr(), _stream_ptr(stream))
        if rc != CORR_OK:
            _raise()
        return d_vis

    # -- corr_corner_turn
    def corner_turn(self, d_in, d_out=None, stream=None):
        import torch
        self._check_in(d_in)
        if d_out is None:
            d_out = torch.empty_like(d_in)
        rc = lib().corr_corner_turn(self._h, d_in.data_ptr(), d_out.data_ptr(), _stream_ptr(stream))
        if rc != CORR_OK:
            _raise()
        return d_out

    # -- corr_stream_run
    def stream_run(self, h_in_list, d_vis=None, fstage=None):
        """h_in_list: pinned host tensors, one per integration (raw int8 voltages when `fstage` is given:
        corr_stream_run_fx).  Returns (d_vis, stats dict)."""
        n = len(h_in_list)
        want = self.in_bytes if fstage is None else fstage.in_bytes
        for t in h_in_list:
            if t.is_cuda or not t.is_pinned() or t.numel() * t.element_size() != want:
                raise ValueError(f"stream_run needs pinned host tensors of {want} bytes each")
        if d_vis is None:
            d_vis = self.empty_vis(n)
        ptrs = (ctypes.c_void_p * n)(*[t.data_ptr() for t in h_in_list])
        stats = (ctypes.c_double * 4)()
        if fstage is None:
            rc = lib().corr_stream_run(self._h, ptrs, n, d_vis.data_ptr(), stats)
        else:
            rc = lib().corr_stream_run_fx(self._h, fstage._f, ptrs, n, d_vis.data_ptr(), stats)
        if rc != CORR_OK:
            _raise()
        return d_vis, {"wall_s": stats[0], "device_s": stats[1], "kernel_s": stats[2], "h2d_s": stats[3]}


def probe_mma(m=128, n=256, mn_major=True, iters=4096, random_fill=False):
    """tcgen05 int8 MMA issue-rate probe (corr_probe_mma, include/corr_diag.h; runs in libcorr_diag.so)."""
    out = (ctypes.c_double * 4)()
    L = diag_lib()
    if L.corr_probe_mma(m, n, (1 if mn_major else 0) | (2 if random_fill else 0), iters, out) != CORR_OK:
        _raise(L)
    return {"ms": out[0], "cycles_per_mma": out[1], "tops": out[2], "sm_mhz": out[3]}


def probe_ffma(packed=True, iters=8192):
    """FP32 FMA issue-rate probe (corr_probe_ffma, include/corr_diag.h; runs in libcorr_diag.so)."""
    out = (ctypes.c_double * 3)()
    L = diag_lib()
    if L.corr_probe_ffma(1 if packed else 0, iters, out) != CORR_OK:
        _raise(L)
    return {"ms": out[0], "tflops": out[1], "sm_mhz": out[2]}


class FStage:
    """The F-stage in front of the float X-engine (corr_fstage_*): raw complex-int8 voltages
    [n_batch][n_fft][n_inputs][2] -> float32 spectra [n_batch][n_fft][n_inputs][2]."""

    def __init__(self, n_inputs, n_fft, n_batch):
        self.n_inputs, self.n_fft, self.n_batch = n_inputs, n_fft, n_batch
        self._f = lib().corr_fstage_create(n_inputs, n_fft, n_batch)
        if not self._f:
            _raise()
        self.in_bytes = lib().corr_fstage_in_bytes(self._f)
        self.out_bytes = lib().corr_fstage_out_bytes(self._f)

    def set_input(self, dtype):
        """"ci8" (int8 pairs, default) or "ci4" (one byte per sample, the paper's 1-byte mode)."""
        code = {"ci8": CORR_CI8, "ci4": CORR_CI4}.get(dtype, dtype)
        if lib().corr_fstage_set_input(self._f, code) != CORR_OK:
            _raise()
        self.in_bytes = lib().corr_fstage_in_bytes(self._f)

    def run(self, d_raw, d_spec=None, stream=None):
        import torch
        if not d_raw.is_cuda or not d_raw.is_contiguous() or d_raw.numel() * d_raw.element_size() != self.in_bytes:
            raise ValueError(f"d_raw must be a contiguous CUDA tensor of {self.in_bytes} bytes ([B][n_fft][N][2] int8, or [B][n_fft][N] bytes in the 4+4-bit mode)")
        if d_spec is None:
            d_spec = torch.empty((self.n_batch, self.n_fft, self.n_inputs, 2), dtype=torch.float32, device="cuda")
        if not d_spec.is_cuda or not d_spec.is_contiguous() or d_spec.numel() * d_spec.element_size() != self.out_bytes:
            raise ValueError(f"d_spec must be a contiguous CUDA tensor of {self.out_bytes} bytes")
        if lib().corr_fstage_run(self._f, d_raw.data_ptr(), d_spec.data_ptr(), _stream_ptr(stream)) != CORR_OK:
            _raise()
        return d_spec

    def destroy(self):
        if getattr(self, "_f", None) and lib is not None:
            lib().corr_fstage_destroy(self._f)
            self._f = None

    __del__ = destroy


def corr_fstage_create(n_inputs, n_fft, n_batch):
    return FStage(n_inputs, n_fft, n_batch)


def corr_fstage_run(f, d_raw, d_spec=None, stream=None):
    return f.run(d_raw, d_spec, stream)


def corr_fstage_destroy(f):
    f.destroy()


def corr_create(n_inputs, n_chan, n_time, dtype):
    return Correlator(n_inputs, n_chan, n_time, dtype)


def corr_xengine(handle, d_in, d_vis=None, stream=None):
    return handle.xengine(d_in, d_vis, stream)


def corr_xengine_batch(handle, d_in_list, d_vis_list=None, stream=None):
    return handle.xengine_batch(d_in_list, d_vis_list, stream)


def corr_destroy(handle):
    handle.destroy()
