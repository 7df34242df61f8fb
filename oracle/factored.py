"""oracle/factored.py — TEST INFRASTRUCTURE (only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline may use it).

The factored form of the sensitivity block, written out as its plain definition (Eq. 5: a row of G
is the ray's lateral footprint times the depth kernel of the period; unknowns depth-fastest, Eq. 7):

    A = [ A_data ; A_extra ]
    A_data[q * nper + p, k * nz + j] = fl( W[q, k] * g_p[j - j0_p] )     for j0_p <= j < j0_p + klen, W[q, k] stored

`expand` multiplies it out into the canonical CSR matrix; everything else the factored operator computes is, by
definition, what the CSR oracle (oracle.lsqr / oracle.spmv) computes on that matrix.  One rounding per stored value
(the fp64 product), exactly as a CSR assembly of G stores it.  numpy only, no blocking, no shared code with the CUDA
path.  Pins (tests/test_oracle_factored_pins.py): the dense triple loop of the definition on small cases; the
generator's own CSR assembly of configs 0, 1, 4 (bitwise, sampled pairs at the large sizes); row sums = ray length.
"""
from __future__ import annotations

import numpy as np


def expand(npairs, nper, nnodes, nz, lptr, lnode, lw, kj0, kern, sptr=None, sidx=None, svals=None):
    """(rowptr int64[m+1], colind int32[nnz], vals float64[nnz]) of A, m = npairs*nper + ms, n = nnodes*nz.

    lptr/lnode/lw: W in CSR form (nodes strictly ascending inside a pair); kj0 int[nper]; kern float64[nper, klen];
    sptr/sidx/svals: A_extra in CSR form (or None)."""
    lptr = np.asarray(lptr, dtype=np.int64)
    lnode = np.asarray(lnode, dtype=np.int64)
    lw = np.asarray(lw, dtype=np.float64)
    kern = np.asarray(kern, dtype=np.float64)
    kj0 = np.asarray(kj0, dtype=np.int64)
    nodal = kern.ndim == 3       # kernel table per lateral node (the paper's Theta_k): kern[k, p, t], kj0[k, p]
    if not nodal:
        kern = kern.reshape(nper, -1)
    klen = kern.shape[-1]
    assert lptr.shape == (npairs + 1,) and kj0.shape == ((nnodes, nper) if nodal else (nper,))
    assert np.all(kj0 >= 0) and np.all(kj0 + klen <= nz)
    cnt = np.diff(lptr)                                   # lateral entries per pair
    ms = 0 if sptr is None else len(sptr) - 1
    m_data = npairs * nper
    rowlen = np.repeat(cnt * klen, nper)                  # every period row of a pair has cnt * klen entries
    rowptr = np.zeros(m_data + ms + 1, dtype=np.int64)
    np.cumsum(rowlen, out=rowptr[1:m_data + 1])
    nnz_data = int(rowptr[m_data])
    colind = np.empty(nnz_data, dtype=np.int32)
    vals = np.empty(nnz_data, dtype=np.float64)
    t = np.arange(klen, dtype=np.int64)
    for q in range(npairs):                               # pair by pair, period by period: the definition
        k = lnode[lptr[q]:lptr[q + 1]]
        w = lw[lptr[q]:lptr[q + 1]]
        for p in range(nper):
            r = q * nper + p
            if nodal:
                cols = (k[:, None] * nz + kj0[k, p][:, None] + t[None, :]).reshape(-1)
                v = (w[:, None] * kern[k, p, :]).reshape(-1)
            else:
                cols = (k[:, None] * nz + kj0[p] + t[None, :]).reshape(-1)
                v = (w[:, None] * kern[p][None, :]).reshape(-1)     # one fp64 rounding per value
            colind[rowptr[r]:rowptr[r + 1]] = cols
            vals[rowptr[r]:rowptr[r + 1]] = v
    if ms:
        sptr = np.asarray(sptr, dtype=np.int64)
        rowptr[m_data + 1:] = nnz_data + sptr[1:]
        colind = np.concatenate([colind, np.asarray(sidx, dtype=np.int32)])
        vals = np.concatenate([vals, np.asarray(svals, dtype=np.float64)])
    return rowptr, colind, vals


def two_prod(a, b):
    """(p, e) with p = fl(a * b) and p + e = a * b exactly (Dekker's product through Veltkamp splitting: no FMA needed,
    exact in fp64 barring over/underflow; elementwise on numpy arrays)."""
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    p = a * b
    c = 134217729.0  # 2^27 + 1
    ah = c * a; ah = ah - (ah - a); al = a - ah
    bh = c * b; bh = bh - (bh - b); bl = b - bh
    e = ((ah * bh - p) + ah * bl + al * bh) + al * bl
    return p, e


def expand_exact(npairs, nper, nnodes, nz, lptr, lnode, lw, kj0, kern, sptr=None, sidx=None, svals=None):
    """The factored operator with EXACT entries W[q, k] * g_p[t] (reading F-fac3) as two-word CSR values:
    (rowptr, colind, vals, vals_lo) with vals = fl(W g) (what `expand` returns) and vals + vals_lo = W g exactly; the
    extra block's entries are one word (vals_lo = 0).  oracle.spmv / spmv_t / lsqr(..., mode=DD, vals_lo=...) then sum the
    exact products of both words and round once: the definition  y_i = RN( sum_j (W g)_ij x_j )  written out."""
    rowptr, colind, vals = expand(npairs, nper, nnodes, nz, lptr, lnode, lw, kj0, kern, sptr, sidx, svals)
    lw = np.asarray(lw, dtype=np.float64)
    kern = np.asarray(kern, dtype=np.float64)
    nodal = kern.ndim == 3
    if not nodal:
        kern = kern.reshape(nper, -1)
    lptr = np.asarray(lptr, dtype=np.int64)
    lnode = np.asarray(lnode, dtype=np.int64)
    lo = np.zeros_like(vals)
    for q in range(npairs):
        w = lw[lptr[q]:lptr[q + 1]]
        k = lnode[lptr[q]:lptr[q + 1]]
        for p in range(nper):
            r = q * nper + p
            pr, er = two_prod(w[:, None], kern[k, p, :] if nodal else kern[p][None, :])
            assert np.array_equal(pr.reshape(-1), vals[rowptr[r]:rowptr[r + 1]])
            lo[rowptr[r]:rowptr[r + 1]] = er.reshape(-1)
    return rowptr, colind, vals, lo
