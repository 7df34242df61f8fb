"""Pins of oracle/factored.py (the factored sensitivity block multiplied out, Eq. 5, Eq. 7)
against things other than itself: the dense triple loop of the definition, the generator's own CSR assembly of the
BASELINE.json systems (an independent code path: tomogen_fill), and the row-sum invariant (sum of a data row = ray
length, because every depth kernel sums to 1)."""
import numpy as np
import pytest

import tomogen
from oracle import factored


def dense_by_definition(f):
    """A as a dense array, entry by entry from the definition (pure-Python loops; tiny cases only)."""
    nper, nz, klen = f["nper"], f["nz"], f["klen"]
    ms = 0 if f["sptr"] is None else len(f["sptr"]) - 1
    A = np.zeros((f["npairs"] * nper + ms, f["nnodes"] * nz))
    for q in range(f["npairs"]):
        for e in range(f["lptr"][q], f["lptr"][q + 1]):
            k, w = int(f["lnode"][e]), float(f["lw"][e])
            for p in range(nper):
                for t in range(klen):
                    A[q * nper + p, k * nz + int(f["kj0"][p]) + t] = w * float(f["kern"][p][t])
    for r in range(ms):
        for e in range(f["sptr"][r], f["sptr"][r + 1]):
            A[f["npairs"] * nper + r, f["sidx"][e]] = f["svals"][e]
    return A


def expand(f):
    return factored.expand(f["npairs"], f["nper"], f["nnodes"], f["nz"], f["lptr"], f["lnode"], f["lw"], f["kj0"], f["kern"],
                           f["sptr"], f["sidx"], f["svals"])


@pytest.mark.parametrize("shape", [(7, 3, 9, 6, 4, None), (5, 1, 4, 5, 5, 0), (9, 10, 12, 20, 12, 17), (4, 32, 3, 40, 1, None)])
def test_expand_is_the_definition(shape):
    npairs, nper, nnodes, nz, klen, ms = shape
    f = tomogen.random_factored(npairs, nper, nnodes, nz, klen, seed=11 + npairs, ms=ms)
    rp, ci, va = expand(f)
    A = dense_by_definition(f)
    m, n = A.shape
    assert rp.shape == (m + 1,) and rp[0] == 0 and rp[-1] == len(ci) == len(va)
    B = np.zeros_like(A)
    for r in range(m):
        cols = ci[rp[r]:rp[r + 1]]
        assert np.all(np.diff(cols) > 0), "columns strictly ascending inside a row (canonical CSR)"
        assert cols.size == 0 or (cols[0] >= 0 and cols[-1] < n)
        B[r, cols] = va[rp[r]:rp[r + 1]]
    assert np.array_equal(A, B)          # bitwise: one rounding per value on both sides
    assert np.count_nonzero(A) <= len(va)


def test_expand_equals_generator_csr_config0():
    s = tomogen.System(0)
    rp, ci, va = s.csr()
    rp2, ci2, va2 = expand(s.factored())
    assert np.array_equal(rp, rp2) and np.array_equal(ci, ci2) and np.array_equal(va, va2)


@pytest.mark.parametrize("config", [1, 4])
def test_expand_equals_generator_rows_sampled_pairs(config):
    """configs 1 / 4 (194 M nonzeros): 40 sampled pairs, all their period rows, and the first / last smoothing rows."""
    s = tomogen.System(config)
    d = s.dims
    f = s.factored()
    rng = np.random.default_rng(5 + config)
    pairs = np.unique(np.concatenate([[0, d.npairs - 1], rng.integers(0, d.npairs, size=38)]))
    sub = dict(f)
    cnt = np.diff(f["lptr"])[pairs]
    lptr = np.zeros(len(pairs) + 1, dtype=np.int64)
    np.cumsum(cnt, out=lptr[1:])
    sel = np.concatenate([np.arange(f["lptr"][q], f["lptr"][q + 1]) for q in pairs])
    sub.update(npairs=len(pairs), lptr=lptr, lnode=f["lnode"][sel], lw=f["lw"][sel], sptr=None, sidx=None, svals=None)
    rp2, ci2, va2 = expand(sub)
    rows = (pairs[:, None] * d.nper + np.arange(d.nper)[None, :]).reshape(-1)
    rp, ci, va = s.rows(rows)
    assert np.array_equal(rp, rp2) and np.array_equal(ci, ci2) and np.array_equal(va, va2)
    # the extra block is the generator's smoothing rows, unchanged
    srows = np.array([d.m_data, d.m_data + 1, d.m - 1])
    rps, cis, vas = s.rows(srows)
    for i, r in enumerate(srows - d.m_data):
        a, b = f["sptr"][r], f["sptr"][r + 1]
        assert np.array_equal(cis[rps[i]:rps[i + 1]], f["sidx"][a:b]) and np.array_equal(vas[rps[i]:rps[i + 1]], f["svals"][a:b])


def test_row_sums_are_ray_lengths():
    s = tomogen.System(0)
    d = s.dims
    rp, ci, va = expand(s.factored())
    L = s.ray_lengths()
    sums = np.add.reduceat(va, rp[:d.m_data])
    assert np.allclose(sums, np.repeat(L, d.nper), rtol=1e-13, atol=0)
    assert np.abs(np.add.reduceat(va[rp[d.m_data]:], rp[d.m_data:-1] - rp[d.m_data])).max() < 1e-12   # smoothing rows sum to 0
