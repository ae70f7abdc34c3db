"""ctypes wrapper + build step for oracle_c.c (plain C fp64 oracle).  TEST INFRASTRUCTURE, NOT THE PRODUCT."""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle_c.c")
_LIB = os.path.join(_HERE, "liboracle_c.so")
_lib = None


def build(force: bool = False) -> str:
    """gcc -O2, no fast-math, no FMA contraction: the arithmetic stays the written fp64 arithmetic."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-std=c99", "-ffp-contract=off", "-fPIC", "-shared",
                               "-o", _LIB, _SRC, "-lm"])
    return _LIB


def _load():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.oracle_grid.restype = ctypes.c_int
        _lib.oracle_dft.restype = ctypes.c_int
    return _lib


def _p(a):
    return a.ctypes.data_as(ctypes.c_void_p)


def grid(uvw_m, freq_hz, vis, weight, nx, ny, cell_arcsec, Q, supports, tables, wc=None, grid_id=None, ngrids=1,
         offset=(0.0, 0.0), counts=False):
    """O1+O3 (2-D: supports=int S, tables=real table) or O1+O6 (w-mode: wc, supports[p], complex tables[p]).
    offset = (dl, dm): phase correction of the visibilities first (NEXT-3); counts=True: also the hit-count grid (NEXT-2).
    Returns G complex128 [ngrids,ny,nx], Gw (float64, or complex128 in w-mode), stats dict (with "cnt" if asked)."""
    lib = _load()
    wmode = wc is not None
    uvw = np.ascontiguousarray(uvw_m, np.float32)
    f = np.ascontiguousarray(freq_hz, np.float64)
    v = np.ascontiguousarray(vis, np.complex64)
    w = np.ascontiguousarray(weight, np.float32)
    nvis = v.shape[0]
    if wmode:
        wc_a = np.ascontiguousarray(wc, np.float64)
        sup = np.ascontiguousarray(supports, np.int32)
        tabs = [np.ascontiguousarray(t, np.complex128) for t in tables]
    else:
        wc_a = np.zeros(1, np.float64)
        sup = np.array([int(supports)], np.int32)
        tabs = [np.ascontiguousarray(tables, np.float64)]
    for t, S in zip(tabs, sup):
        assert t.shape[0] == int(S) * Q + 1
    tptr = (ctypes.c_void_p * len(tabs))(*[t.ctypes.data for t in tabs])
    G = np.zeros((ngrids, ny, nx), np.complex128)
    Gw = np.zeros((ngrids, ny, nx), np.complex128 if wmode else np.float64)
    stats = np.zeros(4, np.float64)
    cnt = np.zeros((ngrids, ny, nx), np.int64) if counts else None
    gid = None if grid_id is None else np.ascontiguousarray(grid_id, np.int32)
    rc = lib.oracle_grid(_p(uvw), _p(f), _p(v), _p(w), None if gid is None else _p(gid),
                         ctypes.c_longlong(nvis), ctypes.c_int(nx), ctypes.c_int(ny),
                         ctypes.c_double(cell_arcsec), ctypes.c_int(Q), ctypes.c_int(len(tabs)),
                         _p(wc_a), _p(sup), tptr, ctypes.c_int(1 if wmode else 0), ctypes.c_double(offset[0]),
                         ctypes.c_double(offset[1]), _p(G), _p(Gw), None if cnt is None else _p(cnt), _p(stats))
    assert rc == 0
    out = dict(sum_weights=float(stats[0]), n_gridded=int(stats[1]), n_dropped=int(stats[2]), n_flagged=int(stats[3]))
    if counts:
        out["cnt"] = cnt
    return G, Gw, out


def dft(u, v, w, val, l, m, use_w=False):
    """(I) at direction cosines (l, m); u, v, w in wavelengths; val complex."""
    lib = _load()
    u = np.ascontiguousarray(u, np.float64); v = np.ascontiguousarray(v, np.float64)
    w = np.ascontiguousarray(w, np.float64)
    val = np.asarray(val, np.complex128)
    vr = np.ascontiguousarray(val.real); vi = np.ascontiguousarray(val.imag)
    l = np.ascontiguousarray(l, np.float64); m = np.ascontiguousarray(m, np.float64)
    ore = np.empty(l.shape[0], np.float64); oim = np.empty(l.shape[0], np.float64)
    rc = lib.oracle_dft(ctypes.c_longlong(u.shape[0]), _p(u), _p(v), _p(w), _p(vr), _p(vi),
                        ctypes.c_longlong(l.shape[0]), _p(l), _p(m), ctypes.c_int(1 if use_w else 0),
                        _p(ore), _p(oim))
    assert rc == 0
    return ore + 1j * oim
