"""oracle — TEST INFRASTRUCTURE: the plain CPU fp64 LSQR the CUDA path is checked against.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference``
legs may import this package; the product (``paper_2604_11920_b200``) never does and shares no code
with it.  The arithmetic lives in ``lsqr_oracle.cpp`` (single-threaded C++17, ``-O2
-ffp-contract=off``), which follows Paige & Saunders' LSQR (ref. PAPER.md:268) step by
step as written in DESIGN.md "Oracle"; this file only marshals numpy arrays.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lsqr_oracle.cpp")
_LIB = os.path.join(_HERE, "liblsqr_oracle.so")
_lib = None

PLAIN, DD = 0, 1


def build(force: bool = False) -> str:
    if not force and os.path.exists(_LIB) and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC):
        return _LIB
    cmd = ["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-ffp-contract=off", "-mfma", _SRC, "-o", _LIB + ".tmp"]
    subprocess.run(cmd, check=True)
    os.replace(_LIB + ".tmp", _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        vp, i64, i32, f64, ci = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int32, ctypes.c_double, ctypes.c_int
        lib.oracle_spmv.argtypes = [i64, i64, vp, vp, vp, vp, vp, ci]
        lib.oracle_spmv.restype = None
        lib.oracle_spmv_t.argtypes = [i64, i64, vp, vp, vp, vp, vp, ci]
        lib.oracle_spmv_t.restype = None
        lib.oracle_spmv_x.argtypes = [i64, i64, vp, vp, vp, vp, vp, vp, ci]
        lib.oracle_spmv_x.restype = None
        lib.oracle_spmv_t_x.argtypes = [i64, i64, vp, vp, vp, vp, vp, vp, ci]
        lib.oracle_spmv_t_x.restype = None
        lib.oracle_lsqr_solve_x.argtypes = [i64, i64, vp, vp, vp, vp, vp, f64, f64, f64, i32, ci, vp, vp, vp, vp, i32, vp, vp]
        lib.oracle_lsqr_solve_x.restype = None
        lib.oracle_lsmr_solve_x.argtypes = lib.oracle_lsqr_solve_x.argtypes
        lib.oracle_lsmr_solve_x.restype = None
        lib.oracle_csr_to_csc.argtypes = [i64, i64, vp, vp, vp, vp, vp, vp]
        lib.oracle_csr_to_csc.restype = None
        lib.oracle_lsqr_new.argtypes = [i64, i64, vp, vp, vp, vp, f64, f64, f64, i32, ci]
        lib.oracle_lsqr_new.restype = vp
        lib.oracle_lsqr_step.argtypes = [vp]
        lib.oracle_lsqr_step.restype = i32
        lib.oracle_lsqr_done.argtypes = [vp]
        lib.oracle_lsqr_done.restype = i32
        lib.oracle_lsqr_free.argtypes = [vp]
        lib.oracle_lsqr_free.restype = None
        lib.oracle_lsqr_get_vec.argtypes = [vp, ci, vp]
        lib.oracle_lsqr_get_vec.restype = None
        lib.oracle_lsqr_get_scalars.argtypes = [vp, vp]
        lib.oracle_lsqr_get_scalars.restype = None
        lib.oracle_lsqr_solve.argtypes = [i64, i64, vp, vp, vp, vp, f64, f64, f64, i32, ci, vp, vp, vp, vp, i32, vp, vp]
        lib.oracle_lsqr_solve.restype = None
        lib.oracle_lsmr_solve.argtypes = lib.oracle_lsqr_solve.argtypes
        lib.oracle_lsmr_solve.restype = None
        _lib = lib
    return _lib


def _p(a):
    return None if a is None else ctypes.c_void_p(a.ctypes.data)


def _csr(rowptr, colind, vals):
    rp = np.ascontiguousarray(rowptr, dtype=np.int64)
    ci = np.ascontiguousarray(colind, dtype=np.int32)
    va = np.ascontiguousarray(vals, dtype=np.float64)
    return rp, ci, va


def spmv(m, n, rowptr, colind, vals, x, mode=PLAIN, vals_lo=None):
    """vals_lo: optional second word of every entry (entry = vals + vals_lo, dd mode; oracle/factored.py expand_exact)."""
    rp, ci, va = _csr(rowptr, colind, vals)
    x = np.ascontiguousarray(x, dtype=np.float64)
    y = np.empty(m, dtype=np.float64)
    if vals_lo is not None:
        lo = np.ascontiguousarray(vals_lo, dtype=np.float64)
        _load().oracle_spmv_x(m, n, _p(rp), _p(ci), _p(va), _p(lo), _p(x), _p(y), mode)
        return y
    _load().oracle_spmv(m, n, _p(rp), _p(ci), _p(va), _p(x), _p(y), mode)
    return y


def spmv_t(m, n, rowptr, colind, vals, u, mode=PLAIN, vals_lo=None):
    rp, ci, va = _csr(rowptr, colind, vals)
    u = np.ascontiguousarray(u, dtype=np.float64)
    v = np.empty(n, dtype=np.float64)
    if vals_lo is not None:
        lo = np.ascontiguousarray(vals_lo, dtype=np.float64)
        _load().oracle_spmv_t_x(m, n, _p(rp), _p(ci), _p(va), _p(lo), _p(u), _p(v), mode)
        return v
    _load().oracle_spmv_t(m, n, _p(rp), _p(ci), _p(va), _p(u), _p(v), mode)
    return v


def csr_to_csc(m, n, rowptr, colind, vals):
    rp, ci, va = _csr(rowptr, colind, vals)
    colptr = np.empty(n + 1, dtype=np.int64)
    rowind = np.empty(len(ci), dtype=np.int32)
    cvals = np.empty(len(ci), dtype=np.float64)
    _load().oracle_csr_to_csc(m, n, _p(rp), _p(ci), _p(va), _p(colptr), _p(rowind), _p(cvals))
    return colptr, rowind, cvals


@dataclass
class Result:
    x: np.ndarray
    itn: int
    istop: int
    r1norm: float
    r2norm: float
    arnorm: float
    anorm: float
    acond: float
    xnorm: float
    r2norm_hist: np.ndarray
    arnorm_hist: np.ndarray
    snapshots: dict


def lsqr(m, n, rowptr, colind, vals, b, damp=0.0, atol=0.0, btol=0.0, max_iters=50, mode=PLAIN, snapshots=(), vals_lo=None):
    """Run the oracle LSQR.  ``snapshots``: iteration numbers whose iterate x_k is also returned.
    ``vals_lo``: optional second word of every entry (entry = vals + vals_lo; used in dd mode)."""
    rp, ci, va = _csr(rowptr, colind, vals)
    lo = None if vals_lo is None else np.ascontiguousarray(vals_lo, dtype=np.float64)
    b = np.ascontiguousarray(b, dtype=np.float64)
    assert len(b) == m and len(rp) == m + 1
    x = np.zeros(n, dtype=np.float64)
    res = np.zeros(8, dtype=np.float64)
    r2h = np.full(max(max_iters, 1), np.nan)
    arh = np.full(max(max_iters, 1), np.nan)
    snaps = np.ascontiguousarray(sorted(int(k) for k in snapshots), dtype=np.int32)
    sx = np.full((len(snaps), n), np.nan)
    _load().oracle_lsqr_solve_x(m, n, _p(rp), _p(ci), _p(va), _p(lo), _p(b), damp, atol, btol, int(max_iters), mode,
                                _p(x), _p(res), _p(r2h), _p(arh), len(snaps), _p(snaps) if len(snaps) else None,
                                _p(sx) if len(snaps) else None)
    itn = int(res[0])
    return Result(x, itn, int(res[1]), res[2], res[3], res[4], res[5], res[6], res[7], r2h[:itn].copy(), arh[:itn].copy(),
                  {int(k): sx[i] for i, k in enumerate(snaps)})


@dataclass
class LsmrResult:
    x: np.ndarray
    itn: int
    istop: int
    normr: float
    normar: float
    normA: float
    condA: float
    normx: float
    normr_hist: np.ndarray
    normar_hist: np.ndarray
    snapshots: dict


def lsmr(m, n, rowptr, colind, vals, b, damp=0.0, atol=0.0, btol=0.0, max_iters=50, mode=PLAIN, snapshots=(), vals_lo=None):
    """Run the oracle LSMR (Fong & Saunders; the paper's own solver).  vals_lo: as in lsqr."""
    rp, ci, va = _csr(rowptr, colind, vals)
    lo = None if vals_lo is None else np.ascontiguousarray(vals_lo, dtype=np.float64)
    b = np.ascontiguousarray(b, dtype=np.float64)
    assert len(b) == m and len(rp) == m + 1
    x = np.zeros(n, dtype=np.float64)
    res = np.zeros(8, dtype=np.float64)
    nrh = np.full(max(max_iters, 1), np.nan)
    narh = np.full(max(max_iters, 1), np.nan)
    snaps = np.ascontiguousarray(sorted(int(k) for k in snapshots), dtype=np.int32)
    sx = np.full((len(snaps), n), np.nan)
    _load().oracle_lsmr_solve_x(m, n, _p(rp), _p(ci), _p(va), _p(lo), _p(b), damp, atol, btol, int(max_iters), mode,
                                _p(x), _p(res), _p(nrh), _p(narh), len(snaps), _p(snaps) if len(snaps) else None,
                                _p(sx) if len(snaps) else None)
    itn = int(res[0])
    return LsmrResult(x, itn, int(res[1]), res[2], res[3], res[4], res[5], res[6], nrh[:itn].copy(), narh[:itn].copy(),
                      {int(k): sx[i] for i, k in enumerate(snaps)})


_SCALARS = ("itn", "istop", "alpha", "beta", "rhobar", "phibar", "bnorm", "anorm", "ddnorm", "res2", "xxnorm", "z",
            "cs2", "sn2", "acond", "r2norm", "arnorm", "xnorm", "r1norm", "done")


class Stepper:
    """Step-by-step oracle (used by the one-step parity tests): exposes u, v, w, x and the scalars."""

    def __init__(self, m, n, rowptr, colind, vals, b, damp=0.0, atol=0.0, btol=0.0, max_iters=50, mode=PLAIN):
        self._keep = _csr(rowptr, colind, vals) + (np.ascontiguousarray(b, dtype=np.float64),)
        rp, ci, va, bb = self._keep
        self.m, self.n = m, n
        self._h = _load().oracle_lsqr_new(m, n, _p(rp), _p(ci), _p(va), _p(bb), damp, atol, btol, int(max_iters), mode)

    def step(self) -> int:
        return int(_load().oracle_lsqr_step(self._h))

    @property
    def done(self) -> bool:
        return bool(_load().oracle_lsqr_done(self._h))

    def vec(self, name: str) -> np.ndarray:
        which = {"u": 0, "v": 1, "w": 2, "x": 3}[name]
        out = np.empty(self.m if which == 0 else self.n, dtype=np.float64)
        _load().oracle_lsqr_get_vec(self._h, which, _p(out))
        return out

    def scalars(self) -> dict:
        out = np.zeros(20, dtype=np.float64)
        _load().oracle_lsqr_get_scalars(self._h, _p(out))
        return dict(zip(_SCALARS, out.tolist()))

    def close(self):
        if self._h:
            _load().oracle_lsqr_free(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
