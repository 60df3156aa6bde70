"""ctypes wrapper around oracle/pdp_oracle.c — TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this module.  It imports nothing from paper_1903_06838_b200.
The arithmetic lives in pdp_oracle.c (each step cites PAPER.md there); this file
only builds the shared object, marshals numpy arrays and trims the hit lists.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pdp_oracle.c")
_LIB = os.path.join(_HERE, "libpdp_oracle.so")

CM_MEDIAN, CM_MEAN_GUARDED, CM_NONE = 0, 1, 2
F1, F2, F3, F4 = 1, 2, 4, 8


class _Geometry(ctypes.Structure):
    _fields_ = [("panels", ctypes.c_int32), ("rows", ctypes.c_int32),
                ("cols", ctypes.c_int32), ("seg_cols", ctypes.c_int32)]


class _Stage(ctypes.Structure):
    _fields_ = [("gh", ctypes.c_int32), ("gw", ctypes.c_int32), ("mode", ctypes.c_int32),
                ("min_count", ctypes.c_int32)]


class _Params(ctypes.Structure):
    _fields_ = [("seed_adu", ctypes.c_double), ("cm_adu", ctypes.c_double),
                ("photon_adu", ctypes.c_double), ("cm_mode", ctypes.c_int32),
                ("cm_min_count", ctypes.c_int32), ("band", ctypes.c_double),
                ("n_stages", ctypes.c_int32), ("stage", _Stage * 3), ("zero_below_adu", ctypes.c_double)]


def _params(seed_adu, cm_adu, photon_adu, cm_mode, cm_min_count, band, stages=None, zero_below_adu=-np.inf):
    """thresholds reach the library as float32; the oracle promotes those to double.
    stages: optional list of up to 3 (gh, gw, mode[, min_count]) common-mode stages."""
    p = _Params(float(np.float32(seed_adu)), float(np.float32(cm_adu)), float(np.float32(photon_adu)),
                cm_mode, cm_min_count, band)
    stages = list(stages or [])
    assert len(stages) <= 3
    p.n_stages = len(stages)
    for i, st in enumerate(stages):
        p.stage[i] = _Stage(int(st[0]), int(st[1]), int(st[2]), int(st[3]) if len(st) > 3 else 0)
    p.zero_below_adu = float(np.float32(zero_below_adu)) if np.isfinite(zero_below_adu) else float(zero_below_adu)
    return p


def _n_groups(npix, seg_cols, stages):
    return npix // (stages[-1][0] * stages[-1][1]) if stages else npix // seg_cols


def build(force: bool = False) -> str:
    """Compile pdp_oracle.c with gcc -O2 (no SIMD intrinsics, OpenMP over frames).

    PDP_ORACLE_SANITIZE=1 builds a separate AddressSanitizer + UndefinedBehaviorSanitizer library instead
    (run the CPU tests with LD_PRELOAD=$(gcc -print-file-name=libasan.so) ASAN_OPTIONS=detect_leaks=0)."""
    if os.environ.get("PDP_ORACLE_SANITIZE") == "1":
        lib = _LIB.replace(".so", "_san.so")
        if force or not os.path.exists(lib) or os.path.getmtime(lib) < os.path.getmtime(_SRC):
            subprocess.check_call(["gcc", "-O1", "-g", "-std=c11", "-fopenmp", "-fsanitize=address,undefined",
                                   "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer", "-shared", "-fPIC",
                                   _SRC, "-o", lib, "-lm"])
        return lib
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-fopenmp", "-shared", "-fPIC", _SRC,
                               "-o", _LIB, "-lm"])
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.pdp_oracle_frame.restype = ctypes.c_int64
        _lib.pdp_oracle_batch.restype = ctypes.c_int
        _lib.pdp_oracle_dense_batch.restype = ctypes.c_int
        _lib.pdp_oracle_histogram.restype = None
    return _lib


def _ptr(a, ctype):
    return None if a is None else a.ctypes.data_as(ctypes.POINTER(ctype))


@dataclass
class OracleResult:
    hit_count: np.ndarray      # [n] int64, true seed count per frame
    hit_pixel: list            # per frame uint32[count]
    hit_charge: list           # per frame float64[count]
    hit_nphot: list            # per frame int32[count]
    hit_dx: list               # per frame float64[count]
    hit_dy: list               # per frame float64[count]
    frame_photons: np.ndarray  # [n] uint64
    accum: np.ndarray          # [npix] uint32 (this batch only)
    cm: np.ndarray | None      # [n, npix/S] float64
    cm_count: np.ndarray | None = None  # [n, npix/S] int32: #M, number of segmented pixels of each group
    fragile: np.ndarray | None = None  # [n, npix] uint8


def max_hits(panels: int, rows: int, cols: int) -> int:
    """Seeds are never 8-adjacent, so this capacity cannot overflow."""
    return ((rows + 1) // 2) * ((cols + 1) // 2) * panels


def process(raw, pedestal, gain, *, panels, rows, cols, seg_cols, seed_adu, cm_adu, photon_adu,
            cm_mode=CM_MEDIAN, cm_min_count=0, band=1e-4, threads=1, hit_capacity=None,
            want_cm=False, want_fragile=False, stages=None) -> OracleResult:
    """Run the oracle over raw[n, panels*rows*cols] (uint16).  stages: see _params."""
    lib = _load()
    npix = panels * rows * cols
    raw = np.ascontiguousarray(raw, dtype=np.uint16).reshape(-1, npix)
    n = raw.shape[0]
    pedestal = np.ascontiguousarray(pedestal, dtype=np.float32).reshape(npix)
    gain = np.ascontiguousarray(gain, dtype=np.float32).reshape(npix)
    assert cols % seg_cols == 0
    cap = int(hit_capacity) if hit_capacity is not None else max_hits(panels, rows, cols)
    g = _Geometry(panels, rows, cols, seg_cols)
    p = _params(seed_adu, cm_adu, photon_adu, cm_mode, cm_min_count, band, stages)
    ngr = _n_groups(npix, seg_cols, stages)
    hit_count = np.zeros(n, np.int64)
    hp = np.zeros((n, cap), np.uint32)
    he = np.zeros((n, cap), np.float64)
    hn = np.zeros((n, cap), np.int32)
    hx = np.zeros((n, cap), np.float64)
    hy = np.zeros((n, cap), np.float64)
    fp = np.zeros(n, np.uint64)
    accum = np.zeros(npix, np.uint32)
    cm = np.zeros((n, ngr), np.float64) if want_cm else None
    frag = np.zeros((n, npix), np.uint8) if want_fragile else None
    cmn = np.zeros((n, ngr), np.int32) if (want_cm or want_fragile) else None
    rc = lib.pdp_oracle_batch(
        ctypes.byref(g), _ptr(pedestal, ctypes.c_float), _ptr(gain, ctypes.c_float),
        ctypes.byref(p), _ptr(raw, ctypes.c_uint16), ctypes.c_int32(n), ctypes.c_int32(threads),
        ctypes.c_int64(cap), _ptr(hit_count, ctypes.c_int64), _ptr(hp, ctypes.c_uint32),
        _ptr(he, ctypes.c_double), _ptr(hn, ctypes.c_int32), _ptr(hx, ctypes.c_double),
        _ptr(hy, ctypes.c_double), _ptr(fp, ctypes.c_uint64), _ptr(accum, ctypes.c_uint32),
        _ptr(cm, ctypes.c_double), _ptr(cmn, ctypes.c_int32), _ptr(frag, ctypes.c_uint8))
    if rc != 0:
        raise MemoryError("pdp_oracle_batch failed")
    k = np.minimum(hit_count, cap)
    return OracleResult(
        hit_count=hit_count,
        hit_pixel=[hp[f, :k[f]].copy() for f in range(n)],
        hit_charge=[he[f, :k[f]].copy() for f in range(n)],
        hit_nphot=[hn[f, :k[f]].copy() for f in range(n)],
        hit_dx=[hx[f, :k[f]].copy() for f in range(n)],
        hit_dy=[hy[f, :k[f]].copy() for f in range(n)],
        frame_photons=fp, accum=accum, cm=cm, cm_count=cmn, fragile=frag)


def frame_v2(raw, pedestal, gain, *, panels, rows, cols, seg_cols, seed_adu, cm_adu, photon_adu,
             cm_mode=CM_MEDIAN, cm_min_count=0, band=1e-4, stages=None):
    """v2 (after dark, gain, common mode) and the per-group c (last stage) of ONE frame, fp64."""
    lib = _load()
    npix = panels * rows * cols
    raw = np.ascontiguousarray(raw, dtype=np.uint16).reshape(npix)
    pedestal = np.ascontiguousarray(pedestal, dtype=np.float32).reshape(npix)
    gain = np.ascontiguousarray(gain, dtype=np.float32).reshape(npix)
    g = _Geometry(panels, rows, cols, seg_cols)
    p = _params(seed_adu, cm_adu, photon_adu, cm_mode, cm_min_count, band, stages)
    v2 = np.zeros(npix, np.float64)
    cm = np.zeros(_n_groups(npix, seg_cols, stages), np.float64)
    ph = ctypes.c_uint64(0)
    cnt = lib.pdp_oracle_frame(
        ctypes.byref(g), _ptr(pedestal, ctypes.c_float), _ptr(gain, ctypes.c_float),
        ctypes.byref(p), _ptr(raw, ctypes.c_uint16), _ptr(v2, ctypes.c_double),
        _ptr(cm, ctypes.c_double), None, None, ctypes.c_int64(0), None, None, None, None, None,
        ctypes.byref(ph), None)
    if cnt < 0:
        raise MemoryError("pdp_oracle_frame failed")
    if stages:
        return v2.reshape(panels, rows, cols), cm.reshape(panels, rows // stages[-1][0], cols // stages[-1][1])
    return v2.reshape(panels, rows, cols), cm.reshape(panels, rows, cols // seg_cols)


def histogram(values, lo, width, nbins, hist=None):
    """O11: uniform-bin histogram of `values` (float64), out-of-range dropped; hist (uint64[nbins]) += counts."""
    lib = _load()
    x = np.ascontiguousarray(values, dtype=np.float64).reshape(-1)
    if hist is None:
        hist = np.zeros(nbins, np.uint64)
    lib.pdp_oracle_histogram(_ptr(x, ctypes.c_double), ctypes.c_int64(x.size), ctypes.c_double(float(np.float32(lo))),
                             ctypes.c_double(float(np.float32(width))), ctypes.c_int32(nbins), _ptr(hist, ctypes.c_uint64))
    return hist


def dense(raw, pedestal, gain, *, panels, rows, cols, seg_cols, cm_adu, photon_adu, cm_mode=CM_MEDIAN,
          cm_min_count=0, band=1e-4, stages=None, zero_below_adu=-np.inf, want_fragile=False):
    """O12: dense photon-counting image (uint32[npix], summed over the frames), per-frame totals, fragile flags."""
    lib = _load()
    npix = panels * rows * cols
    raw = np.ascontiguousarray(raw, dtype=np.uint16).reshape(-1, npix)
    n = raw.shape[0]
    pedestal = np.ascontiguousarray(pedestal, dtype=np.float32).reshape(npix)
    gain = np.ascontiguousarray(gain, dtype=np.float32).reshape(npix)
    g = _Geometry(panels, rows, cols, seg_cols)
    p = _params(0.0, cm_adu, photon_adu, cm_mode, cm_min_count, band, stages, zero_below_adu)
    image = np.zeros(npix, np.uint32)
    totals = np.zeros(n, np.uint64)
    frag = np.zeros((n, npix), np.uint8) if want_fragile else None
    rc = lib.pdp_oracle_dense_batch(ctypes.byref(g), _ptr(pedestal, ctypes.c_float), _ptr(gain, ctypes.c_float),
                                    ctypes.byref(p), _ptr(raw, ctypes.c_uint16), ctypes.c_int32(n),
                                    _ptr(image, ctypes.c_uint32), _ptr(totals, ctypes.c_uint64), _ptr(frag, ctypes.c_uint8))
    if rc != 0:
        raise ValueError("pdp_oracle_dense_batch failed (allocation, or a stage that does not tile the panel)")
    return image, totals, frag
