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
                    if f["kern"].ndim == 3:   # a kernel table per node
                        A[q * nper + p, k * nz + int(f["kj0"][k][p]) + t] = w * float(f["kern"][k][p][t])
                    else:
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


# ---- exact entries W*g as two-word values (reading F-fac3) ---------------------------------------------
def test_two_prod_is_exact():
    from fractions import Fraction
    rng = np.random.default_rng(3)
    a = rng.standard_normal(500) * 10.0 ** rng.integers(-8, 8, size=500)
    b = rng.standard_normal(500) * 10.0 ** rng.integers(-8, 8, size=500)
    p, e = factored.two_prod(a, b)
    assert np.array_equal(p, a * b)
    for i in range(500):
        assert Fraction(float(p[i])) + Fraction(float(e[i])) == Fraction(float(a[i])) * Fraction(float(b[i]))


@pytest.mark.parametrize("shape", [(6, 3, 7, 6, 4, None), (5, 10, 6, 20, 12, 9)])
def test_exact_entries_dd_products_are_the_rounded_exact_sums(shape):
    """oracle.spmv / spmv_t in dd mode on the two-word entries = the exact rational sum over the UNROUNDED entries W*g,
    rounded once to nearest; and it differs from the one-word (rounded-entry) result somewhere, so the second word is
    really used.  Values with a wide exponent spread and cancelling signs."""
    from fractions import Fraction

    import oracle
    npairs, nper, nnodes, nz, klen, ms = shape
    f = tomogen.random_factored(npairs, nper, nnodes, nz, klen, seed=40 + npairs, ms=ms)
    rng = np.random.default_rng(9)
    f["lw"] = f["lw"] * 10.0 ** rng.integers(-3, 4, size=len(f["lw"]))
    rp, ci, va, lo = factored.expand_exact(f["npairs"], f["nper"], f["nnodes"], f["nz"], f["lptr"], f["lnode"], f["lw"], f["kj0"], f["kern"],
                                           f["sptr"], f["sidx"], f["svals"])
    m, n = len(rp) - 1, nnodes * nz
    x = rng.standard_normal(n) * 10.0 ** rng.integers(-2, 3, size=n)
    u = rng.standard_normal(m) * 10.0 ** rng.integers(-2, 3, size=m)
    # the exact operator entry by entry from the definition (rational)
    nperK = f["nper"]
    exact = {}
    for q in range(npairs):
        for e in range(f["lptr"][q], f["lptr"][q + 1]):
            k, w = int(f["lnode"][e]), Fraction(float(f["lw"][e]))
            for p in range(nperK):
                for t in range(klen):
                    exact[(q * nperK + p, k * nz + int(f["kj0"][p]) + t)] = w * Fraction(float(f["kern"][p][t]))
    if f["sptr"] is not None:
        for r in range(len(f["sptr"]) - 1):
            for e in range(f["sptr"][r], f["sptr"][r + 1]):
                exact[(npairs * nperK + r, int(f["sidx"][e]))] = Fraction(float(f["svals"][e]))
    ey = [Fraction(0)] * m
    ev = [Fraction(0)] * n
    for (i, j), a in exact.items():
        ey[i] += a * Fraction(float(x[j]))
        ev[j] += a * Fraction(float(u[i]))
    y = oracle.spmv(m, n, rp, ci, va, x, oracle.DD, vals_lo=lo)
    v = oracle.spmv_t(m, n, rp, ci, va, u, oracle.DD, vals_lo=lo)
    assert np.array_equal(y, np.array([float(z) for z in ey]))      # float(Fraction) rounds to nearest
    assert np.array_equal(v, np.array([float(z) for z in ev]))
    y1 = oracle.spmv(m, n, rp, ci, va, x, oracle.DD)
    assert not np.array_equal(y, y1) and np.allclose(y, y1, rtol=1e-12, atol=1e-300)


def test_exact_entries_lsqr_is_lsqr_on_a_nearby_matrix():
    """LSQR on the two-word entries: x_k within rounding-level perturbation theory of the one-word run (the matrices differ
    by one rounding per entry), same iteration count; with vals_lo = 0 it is the one-word run bit for bit."""
    import oracle
    s = tomogen.System(0)
    f = s.factored()
    rp, ci, va, lo = factored.expand_exact(f["npairs"], f["nper"], f["nnodes"], f["nz"], f["lptr"], f["lnode"], f["lw"], f["kj0"], f["kern"],
                                           f["sptr"], f["sidx"], f["svals"])
    m, n = s.dims.m, s.dims.n
    b = s.rhs(0)
    o1 = oracle.lsqr(m, n, rp, ci, va, b, damp=s.damp, max_iters=30, mode=oracle.DD)
    o2 = oracle.lsqr(m, n, rp, ci, va, b, damp=s.damp, max_iters=30, mode=oracle.DD, vals_lo=lo)
    o0 = oracle.lsqr(m, n, rp, ci, va, b, damp=s.damp, max_iters=30, mode=oracle.DD, vals_lo=np.zeros_like(va))
    assert np.array_equal(o0.x, o1.x)
    assert o2.itn == o1.itn == 30 and not np.array_equal(o2.x, o1.x)
    assert np.linalg.norm(o2.x - o1.x) <= 1e-11 * np.linalg.norm(o1.x)


@pytest.mark.parametrize("shape", [(7, 3, 9, 6, 4, None), (6, 10, 8, 20, 12, 5)])
def test_expand_nodal_kernels_is_the_definition(shape):
    """kernel table per lateral node (the paper's Theta_k): expand and expand_exact against the dense definition"""
    from fractions import Fraction
    npairs, nper, nnodes, nz, klen, ms = shape
    f = tomogen.random_factored(npairs, nper, nnodes, nz, klen, seed=70 + npairs, ms=ms, nodal=True)
    rp, ci, va = expand(f)
    A = dense_by_definition(f)
    B = np.zeros_like(A)
    for r in range(A.shape[0]):
        cols = ci[rp[r]:rp[r + 1]]
        assert np.all(np.diff(cols) > 0)
        B[r, cols] = va[rp[r]:rp[r + 1]]
    assert np.array_equal(A, B)
    rp2, ci2, va2, lo = factored.expand_exact(f["npairs"], f["nper"], f["nnodes"], f["nz"], f["lptr"], f["lnode"], f["lw"], f["kj0"], f["kern"],
                                              f["sptr"], f["sidx"], f["svals"])
    assert np.array_equal(rp2, rp) and np.array_equal(ci2, ci) and np.array_equal(va2, va)
    e = 0
    for q in range(npairs):     # the two words add up to the exact product, entry by entry
        for le in range(f["lptr"][q], f["lptr"][q + 1]):
            pass
    for r in range(npairs * nper):
        q, p = divmod(r, nper)
        for i, le in enumerate(range(f["lptr"][q], f["lptr"][q + 1])):
            k = int(f["lnode"][le])
            for t in range(klen):
                e = rp[r] + i * klen + t
                assert Fraction(float(va[e])) + Fraction(float(lo[e])) == Fraction(float(f["lw"][le])) * Fraction(float(f["kern"][k][p][t]))
