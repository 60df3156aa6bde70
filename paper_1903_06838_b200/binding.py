"""Thin ctypes binding over the C ABI of include/pdp.h (libpdp.so).

Argument marshalling only: every step of the chain runs in the CUDA kernels behind the
boundary.  PyTorch is used for device memory and streams.  There is no fallback: if
libpdp.so is missing or no sm_100 device is present, calls raise.
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpdp.so")

CM_MEDIAN, CM_MEAN_GUARDED, CM_NONE = 0, 1, 2
STATUS_HIT_OVERFLOW = 1

EXPORTS = ("pdp_create", "pdp_process", "pdp_process_pinned", "pdp_process_host", "pdp_debug_set", "pdp_histograms", "pdp_process_dense", "pdp_set_cm_stages", "pdp_set_params", "pdp_destroy",
           "pdp_last_launch_count", "pdp_last_kernel_name", "pdp_keep_common_mode", "pdp_get_common_mode", "pdp_strerror",
           "pdp_last_error", "pdp_version", "pdp_histograms_static", "pdp_static_last_error")
STATIC_HIST_MAX_BINS = 4096   # PDP_STATIC_HIST_MAX_BINS


class pdp_geometry(ctypes.Structure):
    _fields_ = [("panels", ctypes.c_int32), ("rows", ctypes.c_int32), ("cols", ctypes.c_int32),
                ("seg_cols", ctypes.c_int32), ("max_frames_per_batch", ctypes.c_int32)]


class pdp_params(ctypes.Structure):
    _fields_ = [("seed_adu", ctypes.c_float), ("cm_adu", ctypes.c_float), ("photon_adu", ctypes.c_float),
                ("cm_mode", ctypes.c_int32), ("cm_min_count", ctypes.c_int32)]


class pdp_batch(ctypes.Structure):
    _fields_ = [("data", ctypes.c_void_p), ("n_frames", ctypes.c_int32)]


class pdp_output(ctypes.Structure):
    _fields_ = [("hit_capacity", ctypes.c_uint32), ("hit_count", ctypes.c_void_p),
                ("hit_pixel", ctypes.c_void_p), ("hit_charge", ctypes.c_void_p),
                ("hit_nphot", ctypes.c_void_p), ("hit_dx", ctypes.c_void_p), ("hit_dy", ctypes.c_void_p),
                ("frame_photons", ctypes.c_void_p), ("accum", ctypes.c_void_p), ("status", ctypes.c_void_p)]


class pdp_hist_spec(ctypes.Structure):
    _fields_ = [("lo", ctypes.c_float), ("width", ctypes.c_float), ("nbins", ctypes.c_int32)]


class pdp_cm_stage(ctypes.Structure):
    _fields_ = [("group_rows", ctypes.c_int32), ("group_cols", ctypes.c_int32), ("cm_mode", ctypes.c_int32),
                ("cm_min_count", ctypes.c_int32)]


class PdpError(RuntimeError):
    def __init__(self, code: int, where: str, detail: str = ""):
        self.code = code
        super().__init__(f"{where} failed with {code} ({_strerror(code)}){': ' + detail if detail else ''}")


_lib = None


def load_library(path: str | None = None) -> ctypes.CDLL:
    """Load libpdp.so; raises if it has not been built (python -m paper_1903_06838_b200.build)."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    p = path or LIB_PATH
    if not os.path.exists(p):
        raise FileNotFoundError(f"{p} not found: build it with `python -m paper_1903_06838_b200.build` "
                                "(there is no CPU or PyTorch fallback)")
    lib = ctypes.CDLL(p)
    lib.pdp_create.argtypes = [ctypes.POINTER(pdp_geometry), ctypes.c_void_p, ctypes.c_void_p,
                               ctypes.POINTER(pdp_params), ctypes.POINTER(ctypes.c_void_p)]
    lib.pdp_process.argtypes = [ctypes.c_void_p, ctypes.POINTER(pdp_batch), ctypes.c_void_p,
                                ctypes.POINTER(pdp_output)]
    lib.pdp_process_host.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int32, ctypes.c_int32,
                                     ctypes.c_void_p, ctypes.POINTER(pdp_output)]
    lib.pdp_process_pinned.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int32, ctypes.c_int32,
                                       ctypes.c_void_p, ctypes.c_void_p, ctypes.POINTER(pdp_output)]
    lib.pdp_debug_set.argtypes = [ctypes.c_void_p, ctypes.c_char_p, ctypes.c_int64]
    lib.pdp_histograms.argtypes = [ctypes.c_void_p, ctypes.POINTER(pdp_output), ctypes.c_int32, ctypes.POINTER(pdp_hist_spec),
                                   ctypes.c_void_p, ctypes.POINTER(pdp_hist_spec), ctypes.c_void_p, ctypes.c_void_p,
                                   ctypes.c_void_p]
    lib.pdp_process_dense.argtypes = [ctypes.c_void_p, ctypes.POINTER(pdp_batch), ctypes.c_void_p, ctypes.c_float,
                                      ctypes.c_void_p, ctypes.c_void_p]
    lib.pdp_set_cm_stages.argtypes = [ctypes.c_void_p, ctypes.POINTER(pdp_cm_stage), ctypes.c_int32]
    lib.pdp_set_params.argtypes = [ctypes.c_void_p, ctypes.POINTER(pdp_params)]
    lib.pdp_destroy.argtypes = [ctypes.c_void_p]
    lib.pdp_last_launch_count.argtypes = [ctypes.c_void_p]
    lib.pdp_last_kernel_name.argtypes = [ctypes.c_void_p]
    lib.pdp_last_kernel_name.restype = ctypes.c_char_p
    lib.pdp_keep_common_mode.argtypes = [ctypes.c_void_p, ctypes.c_int32]
    lib.pdp_get_common_mode.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int64, ctypes.c_void_p]
    lib.pdp_strerror.argtypes = [ctypes.c_int]
    lib.pdp_strerror.restype = ctypes.c_char_p
    lib.pdp_last_error.argtypes = [ctypes.c_void_p]
    lib.pdp_last_error.restype = ctypes.c_char_p
    lib.pdp_version.restype = ctypes.c_int
    lib.pdp_histograms_static.argtypes = [ctypes.POINTER(pdp_output), ctypes.c_int32, ctypes.POINTER(pdp_hist_spec),
                                          ctypes.c_void_p, ctypes.POINTER(pdp_hist_spec), ctypes.c_void_p, ctypes.c_void_p,
                                          ctypes.c_void_p]
    lib.pdp_static_last_error.restype = ctypes.c_char_p
    if path is None:
        _lib = lib
    return lib


def _strerror(code: int) -> str:
    try:
        return load_library().pdp_strerror(code).decode()
    except Exception:  # library missing: keep the original error readable
        return "?"


@dataclass
class Output:
    """Device buffers of one pdp_process call (torch tensors own the memory)."""
    hit_capacity: int
    hit_count: torch.Tensor      # [n] int32 (bit pattern uint32)
    hit_pixel: torch.Tensor      # [n, cap] int32 (bit pattern uint32)
    hit_charge: torch.Tensor     # [n, cap] float32
    hit_nphot: torch.Tensor      # [n, cap] int32
    hit_dx: torch.Tensor         # [n, cap] float32
    hit_dy: torch.Tensor         # [n, cap] float32
    frame_photons: torch.Tensor  # [n] int32 (bit pattern uint32)
    accum: torch.Tensor          # [npix] int32 (bit pattern uint32)
    status: torch.Tensor         # [1] int32

    def c_struct(self) -> pdp_output:
        return pdp_output(self.hit_capacity, self.hit_count.data_ptr(), self.hit_pixel.data_ptr(),
                          self.hit_charge.data_ptr(), self.hit_nphot.data_ptr(), self.hit_dx.data_ptr(),
                          self.hit_dy.data_ptr(), self.frame_photons.data_ptr(), self.accum.data_ptr(),
                          self.status.data_ptr())

    @property
    def bytes_per_frame_slots(self) -> int:
        return 20 * self.hit_capacity + 8


def histograms_static(out: "Output", n_frames: int, *, energy=None, dxy=None, hist_energy=None, hist_dx=None, hist_dy=None,
                      stream: torch.cuda.Stream | None = None):
    """pdp_histograms_static: the histogram summarization with its workspace in a static device array (no context, no
    allocation).  energy / dxy: (lo, width, nbins) or None, nbins_e + 2 * nbins_d <= STATIC_HIST_MAX_BINS; histograms:
    CUDA int32 tensors of nbins words on the current device, +=.  Calls that overlap on the GPU race (include/pdp.h)."""
    lib = load_library()
    s = stream if stream is not None else torch.cuda.current_stream()
    o = out.c_struct()
    es = pdp_hist_spec(*energy) if energy is not None else None
    ds = pdp_hist_spec(*dxy) if dxy is not None else None
    ptr = lambda t: t.data_ptr() if t is not None else None
    rc = lib.pdp_histograms_static(ctypes.byref(o), n_frames, ctypes.byref(es) if es else None, ptr(hist_energy),
                                   ctypes.byref(ds) if ds else None, ptr(hist_dx), ptr(hist_dy),
                                   ctypes.c_void_p(s.cuda_stream))
    if rc != 0:
        raise PdpError(rc, "pdp_histograms_static", lib.pdp_static_last_error().decode())


def alloc_output(n_frames: int, npix: int, hit_capacity: int, device="cuda", accum: torch.Tensor | None = None) -> Output:
    z = lambda *s, dt=torch.int32: torch.zeros(s, dtype=dt, device=device)
    return Output(hit_capacity, z(n_frames), z(n_frames, hit_capacity),
                  z(n_frames, hit_capacity, dt=torch.float32), z(n_frames, hit_capacity),
                  z(n_frames, hit_capacity, dt=torch.float32), z(n_frames, hit_capacity, dt=torch.float32),
                  z(n_frames), accum if accum is not None else z(npix), z(1))


class Context:
    """pdp_create / pdp_process / pdp_destroy with torch tensors."""

    def __init__(self, *, panels: int, rows: int, cols: int, seg_cols: int, max_frames_per_batch: int,
                 pedestal, gain, seed_adu: float, cm_adu: float, photon_adu: float,
                 cm_mode: int = CM_MEDIAN, cm_min_count: int = 0):
        self._lib = load_library()
        self._h = ctypes.c_void_p()
        self.panels, self.rows, self.cols, self.seg_cols = panels, rows, cols, seg_cols
        self.npix = panels * rows * cols
        self.max_frames = max_frames_per_batch
        ped = torch.as_tensor(pedestal, dtype=torch.float32).contiguous().cpu().reshape(-1)
        gn = torch.as_tensor(gain, dtype=torch.float32).contiguous().cpu().reshape(-1)
        if ped.numel() != self.npix or gn.numel() != self.npix:
            raise ValueError("pedestal/gain must have panels*rows*cols elements")
        geo = pdp_geometry(panels, rows, cols, seg_cols, max_frames_per_batch)
        prm = pdp_params(seed_adu, cm_adu, photon_adu, cm_mode, cm_min_count)
        rc = self._lib.pdp_create(ctypes.byref(geo), ped.data_ptr(), gn.data_ptr(), ctypes.byref(prm),
                                  ctypes.byref(self._h))
        if rc != 0:
            raise PdpError(rc, "pdp_create", self._lib.pdp_last_error(None).decode())

    @property
    def max_hits(self) -> int:
        return ((self.rows + 1) // 2) * ((self.cols + 1) // 2) * self.panels

    def _check(self, rc: int, where: str):
        if rc != 0:
            raise PdpError(rc, where, self._lib.pdp_last_error(self._h).decode())

    def set_params(self, *, seed_adu, cm_adu, photon_adu, cm_mode=CM_MEDIAN, cm_min_count=0):
        prm = pdp_params(seed_adu, cm_adu, photon_adu, cm_mode, cm_min_count)
        self._check(self._lib.pdp_set_params(self._h, ctypes.byref(prm)), "pdp_set_params")

    def process(self, raw: torch.Tensor, out: Output, stream: torch.cuda.Stream | None = None, n_frames: int | None = None):
        """raw: CUDA uint16 (or int16 bit pattern) tensor [n, P, H, W], contiguous.  Asynchronous."""
        if not raw.is_cuda or not raw.is_contiguous() or raw.element_size() != 2:
            raise ValueError("raw must be a contiguous CUDA tensor of 16-bit elements")
        n = raw.numel() // self.npix if n_frames is None else n_frames
        s = stream if stream is not None else torch.cuda.current_stream(raw.device)
        b = pdp_batch(raw.data_ptr(), n)
        o = out.c_struct()
        self._check(self._lib.pdp_process(self._h, ctypes.byref(b), ctypes.c_void_p(s.cuda_stream), ctypes.byref(o)),
                    "pdp_process")

    def process_host(self, raw_host: torch.Tensor, out: Output, chunk_frames: int,
                     stream: torch.cuda.Stream | None = None, copy_stream: torch.cuda.Stream | None = None):
        """raw_host: CPU (pinned) 16-bit tensor [n, P, H, W]; chunks are copied on `copy_stream` (default: the
        context's own side stream) while `stream` computes (pdp_process_pinned)."""
        if raw_host.is_cuda or not raw_host.is_contiguous() or raw_host.element_size() != 2:
            raise ValueError("raw_host must be a contiguous CPU tensor of 16-bit elements")
        n = raw_host.numel() // self.npix
        s = stream if stream is not None else torch.cuda.current_stream()
        o = out.c_struct()
        cs = ctypes.c_void_p(copy_stream.cuda_stream) if copy_stream is not None else None
        self._check(self._lib.pdp_process_pinned(self._h, raw_host.data_ptr(), n, chunk_frames,
                                                 ctypes.c_void_p(s.cuda_stream), cs, ctypes.byref(o)), "pdp_process_pinned")

    def histograms(self, out: Output, n_frames: int, *, energy=None, dxy=None, hist_energy=None, hist_dx=None,
                   hist_dy=None, stream: torch.cuda.Stream | None = None):
        """energy / dxy: (lo, width, nbins) or None; histograms: CUDA int32 tensors of nbins words, += (pdp_histograms)."""
        s = stream if stream is not None else torch.cuda.current_stream()
        o = out.c_struct()
        es = pdp_hist_spec(*energy) if energy is not None else None
        ds = pdp_hist_spec(*dxy) if dxy is not None else None
        ptr = lambda t: t.data_ptr() if t is not None else None
        self._check(self._lib.pdp_histograms(self._h, ctypes.byref(o), n_frames, ctypes.byref(es) if es else None,
                                             ptr(hist_energy), ctypes.byref(ds) if ds else None, ptr(hist_dx),
                                             ptr(hist_dy), ctypes.c_void_p(s.cuda_stream)), "pdp_histograms")

    def process_dense(self, raw: torch.Tensor, image: torch.Tensor, frame_totals: torch.Tensor | None = None,
                      zero_below_adu: float = float("-inf"), stream: torch.cuda.Stream | None = None):
        """Dense photon counting (pdp_process_dense): image int32[npix] +=, frame_totals int32[n] or None."""
        if not raw.is_cuda or not raw.is_contiguous() or raw.element_size() != 2:
            raise ValueError("raw must be a contiguous CUDA tensor of 16-bit elements")
        s = stream if stream is not None else torch.cuda.current_stream(raw.device)
        b = pdp_batch(raw.data_ptr(), raw.numel() // self.npix)
        self._check(self._lib.pdp_process_dense(self._h, ctypes.byref(b), ctypes.c_void_p(s.cuda_stream), zero_below_adu,
                                                image.data_ptr(), frame_totals.data_ptr() if frame_totals is not None else None),
                    "pdp_process_dense")

    def set_cm_stages(self, stages):
        """stages: list of up to 3 (group_rows, group_cols, cm_mode[, cm_min_count]); [] restores the hot path."""
        arr = (pdp_cm_stage * max(1, len(stages)))(*[pdp_cm_stage(int(s[0]), int(s[1]), int(s[2]), int(s[3]) if len(s) > 3 else 0)
                                                     for s in stages])
        self._check(self._lib.pdp_set_cm_stages(self._h, arr, len(stages)), "pdp_set_cm_stages")

    def debug_set(self, key: str, value: int):
        """Diagnostic switches of include/pdp.h (kernel, chunk_frames, sparse_warps, variant)."""
        self._check(self._lib.pdp_debug_set(self._h, key.encode(), int(value)), "pdp_debug_set")

    def keep_common_mode(self, enable: bool = True):
        self._check(self._lib.pdp_keep_common_mode(self._h, int(enable)), "pdp_keep_common_mode")

    def common_mode(self, n_frames: int, stream: torch.cuda.Stream | None = None) -> torch.Tensor:
        nseg = self.cols // self.seg_cols
        t = torch.empty((n_frames, self.panels, self.rows, nseg), dtype=torch.float32, device="cuda")
        s = stream if stream is not None else torch.cuda.current_stream()
        self._check(self._lib.pdp_get_common_mode(self._h, t.data_ptr(), t.numel(), ctypes.c_void_p(s.cuda_stream)),
                    "pdp_get_common_mode")
        return t

    @property
    def last_launch_count(self) -> int:
        return int(self._lib.pdp_last_launch_count(self._h))

    @property
    def last_kernel_name(self) -> str:
        return self._lib.pdp_last_kernel_name(self._h).decode()

    def close(self):
        if self._h:
            self._lib.pdp_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
