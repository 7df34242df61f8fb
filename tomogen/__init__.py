"""tomogen — seeded synthetic tomography systems for the five BASELINE.json configs.

Input generator only: serves both the CPU oracle (``oracle/``) and the CUDA library
(``paper_2604_11920_b200/``) and holds none of the LSQR method's arithmetic.  The recipe is in
DESIGN.md ("Input recipe"); the row structure follows PAPER.md Eq. 1, Eq. 5 and
the depth-fastest unknown ordering of Eq. 7.  The native part is ``csrc/tomogen.cpp``
(C++/OpenMP, own PRNG), built in-tree by :func:`build`.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "csrc", "tomogen.cpp")
_LIB = os.path.join(_HERE, "libtomogen.so")
_lib = None

# Solve parameters of each config (BASELINE.json configs; reading G12 in DESIGN.md).
SOLVE = {
    0: dict(atol=0.0, btol=0.0, max_iters=50),
    1: dict(atol=1e-6, btol=1e-6, max_iters=300),
    2: dict(atol=0.0, btol=0.0, max_iters=100),
    3: dict(atol=0.0, btol=0.0, max_iters=100),
    4: dict(atol=0.0, btol=0.0, max_iters=100),
}


def build(force: bool = False) -> str:
    """Compile csrc/tomogen.cpp -> libtomogen.so (in-tree) if missing or stale."""
    if not force and os.path.exists(_LIB) and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC):
        return _LIB
    cmd = ["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off", _SRC, "-o", _LIB + ".tmp"]
    subprocess.run(cmd, check=True)
    os.replace(_LIB + ".tmp", _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        lib.tomogen_open.restype = ctypes.c_void_p
        lib.tomogen_open.argtypes = [ctypes.c_int]
        for name in ("tomogen_close",):
            getattr(lib, name).argtypes = [ctypes.c_void_p]
            getattr(lib, name).restype = None
        for name in ("tomogen_dims", "tomogen_params", "tomogen_rowptr", "tomogen_raylen", "tomogen_stations", "tomogen_pairs"):
            getattr(lib, name).argtypes = [ctypes.c_void_p, ctypes.c_void_p]
            getattr(lib, name).restype = None
        lib.tomogen_fill.argtypes = [ctypes.c_void_p, ctypes.c_int64, ctypes.c_int64, ctypes.c_void_p, ctypes.c_void_p]
        lib.tomogen_fill.restype = None
        lib.tomogen_lateral_ptr.argtypes = [ctypes.c_void_p, ctypes.c_void_p]
        lib.tomogen_lateral_ptr.restype = None
        lib.tomogen_lateral_fill.argtypes = [ctypes.c_void_p, ctypes.c_int64, ctypes.c_int64, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
        lib.tomogen_lateral_fill.restype = None
        lib.tomogen_kernels.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
        lib.tomogen_kernels.restype = None
        for name in ("tomogen_xtrue", "tomogen_rhs"):
            getattr(lib, name).argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_void_p]
            getattr(lib, name).restype = None
        _lib = lib
    return _lib


def _p(a: np.ndarray):
    return ctypes.c_void_p(a.ctypes.data)


@dataclass
class Dims:
    m: int
    n: int
    nnz: int
    m_data: int
    nx: int
    ny: int
    nz: int
    nper: int
    npairs: int
    keep: int
    nrhs: int
    nst: int


class System:
    """Handle on one config's generator.  Arrays are produced on request (config 2 is 45 GB of CSR,
    so rows can be generated block by block with :meth:`fill`)."""

    def __init__(self, config: int):
        lib = _load()
        self._h = lib.tomogen_open(int(config))
        if not self._h:
            raise ValueError(f"unknown config {config}")
        self.config = int(config)
        d = np.zeros(12, dtype=np.int64)
        lib.tomogen_dims(self._h, _p(d))
        self.dims = Dims(*[int(v) for v in d])
        pr = np.zeros(3, dtype=np.float64)
        lib.tomogen_params(self._h, _p(pr))
        self.damp, self.wsm, self.sigma = (float(v) for v in pr)
        self.solve = dict(SOLVE[self.config])

    def close(self):
        if self._h:
            _load().tomogen_close(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # --- matrix -----------------------------------------------------------------------------
    def rowptr(self) -> np.ndarray:
        rp = np.empty(self.dims.m + 1, dtype=np.int64)
        _load().tomogen_rowptr(self._h, _p(rp))
        return rp

    def fill(self, r0: int, r1: int, colind: np.ndarray, vals: np.ndarray) -> None:
        """Write rows [r0, r1) into colind/vals, entry e at index e - rowptr[r0]."""
        assert colind.dtype == np.int32 and vals.dtype == np.float64
        assert colind.flags.c_contiguous and vals.flags.c_contiguous
        _load().tomogen_fill(self._h, int(r0), int(r1), _p(colind), _p(vals))

    def csr(self):
        """(rowptr int64[m+1], colind int32[nnz], vals float64[nnz]) of the whole matrix."""
        rp = self.rowptr()
        ci = np.empty(self.dims.nnz, dtype=np.int32)
        va = np.empty(self.dims.nnz, dtype=np.float64)
        self.fill(0, self.dims.m, ci, va)
        return rp, ci, va

    def rows(self, rows) -> tuple:
        """CSR (rowptr, colind, vals) of the sub-matrix made of the given rows (sampled-row checks at
        sizes where the whole matrix is too big to hold twice)."""
        rp = self.rowptr()
        rows = np.asarray(rows, dtype=np.int64)
        srp = np.zeros(len(rows) + 1, dtype=np.int64)
        srp[1:] = np.cumsum(rp[rows + 1] - rp[rows])
        ci = np.empty(int(srp[-1]), dtype=np.int32)
        va = np.empty(int(srp[-1]), dtype=np.float64)
        for k, r in enumerate(rows):
            self.fill(int(r), int(r) + 1, ci[srp[k]:srp[k + 1]], va[srp[k]:srp[k + 1]])
        return srp, ci, va

    def csr_cuda(self, block_rows: int = 100000):
        """The whole matrix as torch CUDA tensors (rowptr, colind, vals), generated and uploaded block by
        block so that the host never holds more than one block (config 2: 45 GB of CSR)."""
        import torch
        rp = self.rowptr()
        nnz = int(rp[-1])
        ci_d = torch.empty(nnz, dtype=torch.int32, device="cuda")
        va_d = torch.empty(nnz, dtype=torch.float64, device="cuda")
        for r0 in range(0, self.dims.m, block_rows):
            r1 = min(self.dims.m, r0 + block_rows)
            e0, e1 = int(rp[r0]), int(rp[r1])
            ci = np.empty(e1 - e0, dtype=np.int32)
            va = np.empty(e1 - e0, dtype=np.float64)
            self.fill(r0, r1, ci, va)
            ci_d[e0:e1] = torch.from_numpy(ci).cuda()
            va_d[e0:e1] = torch.from_numpy(va).cuda()
        return torch.from_numpy(rp).cuda(), ci_d, va_d

    # --- the same matrix in factored form (Eq. 5: lateral footprint x depth kernel) --------------
    def factored(self):
        """The parts tomogen multiplies out into the CSR values: a dict with
        npairs, nper, nnodes, nz, klen; lptr int64[npairs+1], lnode int32[E], lw float64[E] (the pairs' lateral
        footprints W, nodes ascending); kj0 int32[nper], kern float64[nper, klen] (depth-kernel windows);
        sptr/sidx/svals: the smoothing rows as a CSR block of their own (ms = n rows).
        Row q*nper + p of the data block has value lw[e] * kern[p, t] at column lnode[e]*nz + kj0[p] + t."""
        d = self.dims
        lib = _load()
        lptr = np.empty(d.npairs + 1, dtype=np.int64)
        lib.tomogen_lateral_ptr(self._h, _p(lptr))
        E = int(lptr[-1])
        lnode = np.empty(E, dtype=np.int32)
        lw = np.empty(E, dtype=np.float64)
        lib.tomogen_lateral_fill(self._h, 0, d.npairs, _p(lptr), _p(lnode), _p(lw))
        kj0 = np.empty(d.nper, dtype=np.int32)
        kern = np.empty((d.nper, d.keep), dtype=np.float64)
        lib.tomogen_kernels(self._h, _p(kj0), _p(kern))
        rp = self.rowptr()
        s0 = int(rp[d.m_data])
        sptr = (rp[d.m_data:] - s0).astype(np.int64)
        snnz = int(sptr[-1])
        sidx = np.empty(snnz, dtype=np.int32)
        svals = np.empty(snnz, dtype=np.float64)
        self.fill(d.m_data, d.m, sidx, svals)
        return dict(npairs=d.npairs, nper=d.nper, nnodes=d.nx * d.ny, nz=d.nz, klen=d.keep, lptr=lptr, lnode=lnode, lw=lw,
                    kj0=kj0, kern=kern, sptr=sptr, sidx=sidx, svals=svals)

    # --- vectors ----------------------------------------------------------------------------
    def x_true(self, rhs: int = 0) -> np.ndarray:
        x = np.empty(self.dims.n, dtype=np.float64)
        _load().tomogen_xtrue(self._h, int(rhs), _p(x))
        return x

    def rhs(self, rhs: int = 0) -> np.ndarray:
        b = np.empty(self.dims.m, dtype=np.float64)
        _load().tomogen_rhs(self._h, int(rhs), _p(b))
        return b

    def rhs_block(self) -> np.ndarray:
        """All right-hand sides as an m x nrhs row-major block (config 3: 8 columns)."""
        return np.ascontiguousarray(np.stack([self.rhs(r) for r in range(self.dims.nrhs)], axis=1))

    def ray_lengths(self) -> np.ndarray:
        L = np.empty(self.dims.npairs, dtype=np.float64)
        _load().tomogen_raylen(self._h, _p(L))
        return L

    def stations(self) -> np.ndarray:
        xy = np.empty((self.dims.nst, 2), dtype=np.float64)
        _load().tomogen_stations(self._h, _p(xy))
        return xy

    def pairs(self) -> np.ndarray:
        ab = np.empty((self.dims.npairs, 2), dtype=np.int32)
        _load().tomogen_pairs(self._h, _p(ab))
        return ab


def random_csr(m: int, n: int, row_lengths, seed: int, dtype=np.float64):
    """Unstructured canonical CSR with the given row lengths (unit tests: skew, empty rows, tails)."""
    rng = np.random.default_rng(seed)
    row_lengths = np.minimum(np.asarray(row_lengths, dtype=np.int64), n)
    assert len(row_lengths) == m
    rp = np.zeros(m + 1, dtype=np.int64)
    np.cumsum(row_lengths, out=rp[1:])
    ci = np.empty(rp[-1], dtype=np.int32)
    for i in range(m):
        k = int(row_lengths[i])
        if k == 0:
            continue
        if k * 4 >= n:
            cols = np.sort(rng.permutation(n)[:k])
        else:
            cols = np.unique(rng.integers(0, n, size=2 * k + 8))
            while len(cols) < k:
                cols = np.unique(np.concatenate([cols, rng.integers(0, n, size=2 * k)]))
            cols = np.sort(rng.permutation(cols)[:k])
        ci[rp[i]:rp[i + 1]] = cols
    va = rng.standard_normal(rp[-1]).astype(dtype)
    va[va == 0] = 1.0
    return rp, ci, va


def random_factored(npairs, nper, nnodes, nz, klen, seed, ms=None, empty_pairs=0.1, empty_nodes=0.1, max_entries=40, nodal=False):
    """Unstructured factored system (unit tests: odd shapes, empty pairs and nodes, windows at the rim): the dict
    :meth:`System.factored` returns, with random footprints, windows and a random short-row extra block (ms rows;
    None: nnodes*nz rows of 0..7 entries; 0: no extra block)."""
    rng = np.random.default_rng(seed)
    live = np.flatnonzero(rng.random(nnodes) >= empty_nodes)
    if len(live) == 0:
        live = np.array([0])
    cnt = rng.integers(1, min(max_entries, len(live)) + 1, size=npairs)
    cnt[rng.random(npairs) < empty_pairs] = 0
    lptr = np.zeros(npairs + 1, dtype=np.int64)
    np.cumsum(cnt, out=lptr[1:])
    lnode = np.empty(int(lptr[-1]), dtype=np.int32)
    for q in range(npairs):
        lnode[lptr[q]:lptr[q + 1]] = np.sort(rng.choice(live, size=int(cnt[q]), replace=False))
    lw = rng.standard_normal(int(lptr[-1]))
    lw[lw == 0] = 1.0
    kj0 = rng.integers(0, nz - klen + 1, size=nper).astype(np.int32)
    kern = rng.standard_normal((nper, klen))
    if nodal:   # a kernel table per lateral node (the paper's Theta_k): kern[k, p, t], kj0[k, p]
        kj0 = rng.integers(0, nz - klen + 1, size=(nnodes, nper)).astype(np.int32)
        kern = rng.standard_normal((nnodes, nper, klen))
    n = nnodes * nz
    if ms is None:
        ms = n
    out = dict(npairs=npairs, nper=nper, nnodes=nnodes, nz=nz, klen=klen, lptr=lptr, lnode=lnode, lw=lw, kj0=kj0, kern=kern,
               sptr=None, sidx=None, svals=None)
    if ms:
        sp_, si_, sv_ = random_csr(ms, n, rng.integers(0, min(8, n + 1), size=ms), seed + 1)
        out.update(sptr=sp_, sidx=si_, svals=sv_)
    return out
