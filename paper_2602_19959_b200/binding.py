"""Thin ctypes binding of include/pvf.h -- argument marshalling only.

Every step of the hot path runs inside libpvf.so's CUDA kernels; PyTorch appears here only for
device memory (``tensor.data_ptr()``) and streams (``torch.cuda.Stream.cuda_stream``).  There is no
CPU fallback: if the shared library is missing or fails to load, importing raises.
Function and struct names are those of include/pvf.h.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpvf.so")

PVF_OK, PVF_ERR_ARG, PVF_ERR_CONFIG, PVF_ERR_CAPACITY, PVF_ERR_CUDA, PVF_ERR_UNSUPPORTED = range(6)
PVF_PREC_FP32, PVF_PREC_TF32, PVF_PREC_BF16, PVF_PREC_FP16 = 0, 1, 2, 3
PRECISIONS = {"fp32": PVF_PREC_FP32, "tf32": PVF_PREC_TF32, "bf16": PVF_PREC_BF16, "fp16": PVF_PREC_FP16}
FLAG_PEAK_OVERFLOW, FLAG_TRACK_DROPPED, FLAG_NONFINITE, FLAG_BAD_OFFSETS = 1, 2, 4, 8
N_INTERVALS, N_BINS, N_GLOBAL_BINS, MAX_PEAKS = 40, 100, 4000, 32
NOALLOC_MAX_EVENTS, NOALLOC_MAX_TRACKS = 64, 16384      # pvf_histogram_noalloc (include/pvf.h)

EXPORTS = [
    "pvf_default_config", "pvf_workspace_bytes", "pvf_create", "pvf_create_in_pool", "pvf_run",
    "pvf_run_host", "pvf_find_peaks", "pvf_run_unet", "pvf_debug_copy_histogram", "pvf_histogram_noalloc",
    "pvf_stage_times_ms", "pvf_launches_per_run", "pvf_destroy", "pvf_status_string",
    "pvf_last_cuda_error", "pvf_build_info",
]


class pvf_config(C.Structure):
    _fields_ = [
        ("n_intervals", C.c_int32), ("n_bins", C.c_int32), ("z_min_mm", C.c_float), ("bin_width_mm", C.c_float),
        ("fc_in", C.c_int32), ("fc_hidden", C.c_int32), ("hist_channels", C.c_int32), ("unet_channels", C.c_int32),
        ("k_e1", C.c_int32), ("k_e2", C.c_int32), ("k_b", C.c_int32), ("k_d2", C.c_int32), ("k_d1", C.c_int32),
        ("leaky_slope", C.c_float), ("peak_threshold", C.c_float), ("peak_halfwidth", C.c_int32),
        ("max_peaks", C.c_int32), ("precision", C.c_int32), ("split_mask", C.c_int32),
        ("max_events", C.c_int32), ("max_tracks", C.c_int64), ("enable_stage_timing", C.c_int32),
        ("enable_host_io", C.c_int32), ("elide_empty_intervals", C.c_int32),
        ("boundary_margin_mm", C.c_float), ("unet_cta_pair", C.c_int32), ("l2_chunk_events", C.c_int32),
    ]


class pvf_weights(C.Structure):
    _fields_ = [("fc_w", C.c_void_p * 6), ("fc_b", C.c_void_p * 6), ("conv_w", C.c_void_p * 6), ("conv_b", C.c_void_p * 6)]


class pvf_tracks(C.Structure):
    _fields_ = [("feat", C.c_void_p * 9), ("event_offsets", C.c_void_p), ("n_tracks", C.c_int64)]


class pvf_peaks(C.Structure):
    _fields_ = [("z_mm", C.c_void_p), ("prob", C.c_void_p), ("bin", C.c_void_p), ("count", C.c_void_p),
                ("event_flags", C.c_void_p)]


def load_library(path: str = LIB_PATH) -> C.CDLL:
    if not os.path.exists(path):
        raise ImportError(f"{path} not found: build it with `python -m paper_2602_19959_b200.build` "
                          "(there is no CPU fallback)")
    lib = C.CDLL(path)
    lib.pvf_default_config.argtypes = [C.POINTER(pvf_config), C.c_int32, C.c_int64]
    lib.pvf_default_config.restype = None
    lib.pvf_workspace_bytes.argtypes = [C.POINTER(pvf_config)]
    lib.pvf_workspace_bytes.restype = C.c_size_t
    lib.pvf_create.argtypes = [C.POINTER(pvf_weights), C.POINTER(pvf_config), C.POINTER(C.c_void_p)]
    lib.pvf_create_in_pool.argtypes = [C.POINTER(pvf_weights), C.POINTER(pvf_config), C.c_void_p, C.c_size_t,
                                       C.POINTER(C.c_void_p)]
    lib.pvf_run.argtypes = [C.c_void_p, C.POINTER(pvf_tracks), C.c_int32, C.c_void_p, C.POINTER(pvf_peaks), C.c_void_p]
    lib.pvf_run_host.argtypes = lib.pvf_run.argtypes
    lib.pvf_find_peaks.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.POINTER(pvf_peaks), C.c_void_p]
    lib.pvf_run_unet.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p]
    lib.pvf_debug_copy_histogram.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p]
    lib.pvf_histogram_noalloc.argtypes = [C.c_void_p, C.POINTER(pvf_tracks), C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p]
    lib.pvf_stage_times_ms.argtypes = [C.c_void_p, C.POINTER(C.c_float * 4)]
    lib.pvf_launches_per_run.argtypes = [C.c_void_p, C.c_int32]
    lib.pvf_launches_per_run.restype = C.c_int32
    lib.pvf_destroy.argtypes = [C.c_void_p]
    lib.pvf_status_string.argtypes = [C.c_int]
    lib.pvf_status_string.restype = C.c_char_p
    lib.pvf_last_cuda_error.argtypes = [C.c_void_p]
    lib.pvf_last_cuda_error.restype = C.c_char_p
    lib.pvf_build_info.argtypes = []
    lib.pvf_build_info.restype = C.c_char_p
    for name in ("pvf_create", "pvf_create_in_pool", "pvf_run", "pvf_run_host", "pvf_find_peaks", "pvf_run_unet",
                 "pvf_debug_copy_histogram", "pvf_histogram_noalloc", "pvf_stage_times_ms", "pvf_destroy"):
        getattr(lib, name).restype = C.c_int
    return lib


class PVFError(RuntimeError):
    def __init__(self, status: int, what: str, detail: str = ""):
        self.status = status
        super().__init__(f"{what}: status {status}" + (f" ({detail})" if detail else ""))


def default_config(lib, max_events: int, max_tracks: int, **over) -> pvf_config:
    cfg = pvf_config()
    lib.pvf_default_config(C.byref(cfg), int(max_events), int(max_tracks))
    for k, v in over.items():
        setattr(cfg, k, v)
    return cfg


def _weights_struct(w):
    """w: object with fc_w, fc_b, conv_w, conv_b lists of float32 numpy arrays (PyTorch layouts).
    Returns (struct, keepalive)."""
    s = pvf_weights()
    keep = []
    for field in ("fc_w", "fc_b", "conv_w", "conv_b"):
        arrs = getattr(w, field)
        assert len(arrs) == 6
        for k in range(6):
            a = np.ascontiguousarray(arrs[k], dtype=np.float32)
            keep.append(a)
            getattr(s, field)[k] = a.ctypes.data
    return s, keep


class PVFinder:
    """One pvf_handle.  Methods mirror the C entry points; tensors are torch CUDA tensors."""

    def __init__(self, weights, max_events: int, max_tracks: int, precision="fp32", channels: int | None = None,
                 split_mask: int = 0, stage_timing: bool = False, host_io: bool = False, elide_empty: bool = False,
                 boundary_margin_mm: float = 0.0, cta_pair: bool | None = None, pool=None, lib=None,
                 **cfg_over):
        import torch  # device memory + streams only
        self.torch = torch
        self.lib = lib or load_library()
        ch = channels if channels is not None else getattr(weights, "channels", 64)
        prec = PRECISIONS[precision] if isinstance(precision, str) else int(precision)
        if cta_pair is None:                 # CTA pairs (cta_group::2) by default: faster, same bits; precision "fp32" with
            cta_pair = True                  # cta_pair=False selects the CUDA-core kernels (bisecting reference)
        self.cfg = default_config(self.lib, max_events, max_tracks, unet_channels=ch, precision=prec,
                                  split_mask=split_mask, enable_stage_timing=int(stage_timing),
                                  enable_host_io=int(host_io), elide_empty_intervals=int(elide_empty),
                                  boundary_margin_mm=float(boundary_margin_mm), unet_cta_pair=int(cta_pair),
                                  **cfg_over)
        ws, keep = _weights_struct(weights)
        self.handle = C.c_void_p()
        if pool is None:
            st = self.lib.pvf_create(C.byref(ws), C.byref(self.cfg), C.byref(self.handle))
        else:
            self._pool = pool
            st = self.lib.pvf_create_in_pool(C.byref(ws), C.byref(self.cfg), pool.data_ptr(),
                                             pool.numel() * pool.element_size(), C.byref(self.handle))
        del keep
        if st != PVF_OK:
            self.handle = None
            raise PVFError(st, "pvf_create", self.lib.pvf_status_string(st).decode())

    # ------------------------------------------------------------------ helpers
    def _check(self, st, what):
        if st != PVF_OK:
            detail = self.lib.pvf_status_string(st).decode()
            if st == PVF_ERR_CUDA:
                detail += " " + self.lib.pvf_last_cuda_error(self.handle).decode()
            raise PVFError(st, what, detail)

    def _stream(self, stream):
        s = stream if stream is not None else self.torch.cuda.current_stream()
        return C.c_void_p(s.cuda_stream)

    def alloc_peaks(self, n_events, device="cuda", pinned=False):
        t = self.torch
        kw = dict(device="cpu", pin_memory=True) if pinned else dict(device=device)
        return dict(z=t.zeros(n_events, MAX_PEAKS, dtype=t.float32, **kw),
                    prob=t.zeros(n_events, MAX_PEAKS, dtype=t.float32, **kw),
                    bin=t.full((n_events, MAX_PEAKS), -1, dtype=t.int32, **kw),
                    count=t.zeros(n_events, dtype=t.int32, **kw),
                    flags=t.zeros(n_events, dtype=t.int32, **kw))

    @staticmethod
    def _peaks_struct(pk):
        s = pvf_peaks()
        s.z_mm, s.prob, s.bin, s.count = pk["z"].data_ptr(), pk["prob"].data_ptr(), pk["bin"].data_ptr(), pk["count"].data_ptr()
        s.event_flags = pk["flags"].data_ptr() if pk.get("flags") is not None else None
        return s

    @staticmethod
    def _tracks_struct(feat, event_offsets):
        """feat: float32 tensor [9, n_tracks] (rows contiguous = SoA); event_offsets int32 [E+1]."""
        assert feat.dim() == 2 and feat.shape[0] == 9 and (feat.shape[1] == 0 or feat.stride(1) == 1)
        s = pvf_tracks()
        for k in range(9):
            s.feat[k] = feat[k].data_ptr()
        s.event_offsets = event_offsets.data_ptr()
        s.n_tracks = int(feat.shape[1])
        return s

    # ------------------------------------------------------------------ entry points
    def run(self, feat, event_offsets, n_events, out_probs, out_peaks, stream=None):
        ts = self._tracks_struct(feat, event_offsets)
        ps = self._peaks_struct(out_peaks)
        st = self.lib.pvf_run(self.handle, C.byref(ts), int(n_events), C.c_void_p(out_probs.data_ptr()),
                              C.byref(ps), self._stream(stream))
        self._check(st, "pvf_run")

    def run_host(self, feat, event_offsets, n_events, host_probs, host_peaks, stream=None):
        ts = self._tracks_struct(feat, event_offsets)
        ps = self._peaks_struct(host_peaks)
        hp = C.c_void_p(host_probs.data_ptr()) if host_probs is not None else None
        st = self.lib.pvf_run_host(self.handle, C.byref(ts), int(n_events), hp, C.byref(ps), self._stream(stream))
        self._check(st, "pvf_run_host")

    def find_peaks(self, probs, n_events, out_peaks, stream=None):
        ps = self._peaks_struct(out_peaks)
        st = self.lib.pvf_find_peaks(self.handle, C.c_void_p(probs.data_ptr()), int(n_events), C.byref(ps),
                                     self._stream(stream))
        self._check(st, "pvf_find_peaks")

    def run_unet(self, hist, n_events, out_probs, stream=None):
        st = self.lib.pvf_run_unet(self.handle, C.c_void_p(hist.data_ptr()), int(n_events),
                                   C.c_void_p(out_probs.data_ptr()), self._stream(stream))
        self._check(st, "pvf_run_unet")

    def debug_copy_histogram(self, dev_out, n_events, stream=None):
        st = self.lib.pvf_debug_copy_histogram(self.handle, C.c_void_p(dev_out.data_ptr()), int(n_events),
                                               self._stream(stream))
        self._check(st, "pvf_debug_copy_histogram")

    def histogram_noalloc(self, feat, event_offsets, n_events, dev_hist, dev_flags=None, stream=None):
        """pvf_histogram_noalloc: H [n_events, 40, 8, 100] of a small batch (<= NOALLOC_MAX_EVENTS events,
        <= NOALLOC_MAX_TRACKS tracks) with the kernels' scratch in the library's static device array: no allocation."""
        ts = self._tracks_struct(feat, event_offsets)
        st = self.lib.pvf_histogram_noalloc(self.handle, C.byref(ts), int(n_events), C.c_void_p(dev_hist.data_ptr()),
                                            C.c_void_p(dev_flags.data_ptr()) if dev_flags is not None else None,
                                            self._stream(stream))
        if st != PVF_OK:
            raise PVFError(st, "pvf_histogram_noalloc", self.lib.pvf_status_string(st).decode() + " "
                           + self.lib.pvf_last_cuda_error(self.handle).decode())

    def stage_times_ms(self):
        out = (C.c_float * 4)()
        self._check(self.lib.pvf_stage_times_ms(self.handle, C.byref(out)), "pvf_stage_times_ms")
        return [float(v) for v in out]

    def launches_per_run(self, n_events):
        return int(self.lib.pvf_launches_per_run(self.handle, int(n_events)))

    def workspace_bytes(self):
        return int(self.lib.pvf_workspace_bytes(C.byref(self.cfg)))

    def destroy(self):
        if getattr(self, "handle", None):
            self.lib.pvf_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass
