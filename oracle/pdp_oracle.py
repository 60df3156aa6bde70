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


class _Params(ctypes.Structure):
    _fields_ = [("seed_adu", ctypes.c_double), ("cm_adu", ctypes.c_double),
                ("photon_adu", ctypes.c_double), ("cm_mode", ctypes.c_int32),
                ("cm_min_count", ctypes.c_int32), ("band", ctypes.c_double)]


def build(force: bool = False) -> str:
    """Compile pdp_oracle.c with gcc -O2 (no SIMD intrinsics, OpenMP over frames)."""
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
            want_cm=False, want_fragile=False) -> OracleResult:
    """Run the oracle over raw[n, panels*rows*cols] (uint16)."""
    lib = _load()
    npix = panels * rows * cols
    raw = np.ascontiguousarray(raw, dtype=np.uint16).reshape(-1, npix)
    n = raw.shape[0]
    pedestal = np.ascontiguousarray(pedestal, dtype=np.float32).reshape(npix)
    gain = np.ascontiguousarray(gain, dtype=np.float32).reshape(npix)
    assert cols % seg_cols == 0
    cap = int(hit_capacity) if hit_capacity is not None else max_hits(panels, rows, cols)
    g = _Geometry(panels, rows, cols, seg_cols)
    # thresholds reach the library as float32; the oracle promotes those to double
    p = _Params(float(np.float32(seed_adu)), float(np.float32(cm_adu)),
                float(np.float32(photon_adu)), cm_mode, cm_min_count, band)
    hit_count = np.zeros(n, np.int64)
    hp = np.zeros((n, cap), np.uint32)
    he = np.zeros((n, cap), np.float64)
    hn = np.zeros((n, cap), np.int32)
    hx = np.zeros((n, cap), np.float64)
    hy = np.zeros((n, cap), np.float64)
    fp = np.zeros(n, np.uint64)
    accum = np.zeros(npix, np.uint32)
    cm = np.zeros((n, npix // seg_cols), np.float64) if want_cm else None
    frag = np.zeros((n, npix), np.uint8) if want_fragile else None
    cmn = np.zeros((n, npix // seg_cols), np.int32) if (want_cm or want_fragile) else None
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
             cm_mode=CM_MEDIAN, cm_min_count=0, band=1e-4):
    """v2 (after dark, gain, common mode) and the per-segment c of ONE frame, fp64."""
    lib = _load()
    npix = panels * rows * cols
    raw = np.ascontiguousarray(raw, dtype=np.uint16).reshape(npix)
    pedestal = np.ascontiguousarray(pedestal, dtype=np.float32).reshape(npix)
    gain = np.ascontiguousarray(gain, dtype=np.float32).reshape(npix)
    g = _Geometry(panels, rows, cols, seg_cols)
    p = _Params(float(np.float32(seed_adu)), float(np.float32(cm_adu)),
                float(np.float32(photon_adu)), cm_mode, cm_min_count, band)
    v2 = np.zeros(npix, np.float64)
    cm = np.zeros(npix // seg_cols, np.float64)
    ph = ctypes.c_uint64(0)
    cnt = lib.pdp_oracle_frame(
        ctypes.byref(g), _ptr(pedestal, ctypes.c_float), _ptr(gain, ctypes.c_float),
        ctypes.byref(p), _ptr(raw, ctypes.c_uint16), _ptr(v2, ctypes.c_double),
        _ptr(cm, ctypes.c_double), None, None, ctypes.c_int64(0), None, None, None, None, None,
        ctypes.byref(ph), None)
    if cnt < 0:
        raise MemoryError("pdp_oracle_frame failed")
    return v2.reshape(panels, rows, cols), cm.reshape(panels, rows, cols // seg_cols)
