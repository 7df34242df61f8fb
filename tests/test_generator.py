"""Invariants of the synthetic-system generator (tomogen), DESIGN.md "Input recipe".

The row structure comes from PAPER.md Eq. 1 (bilinear lateral weights along the path),
Eq. 5 (lateral weight x depth kernel) and Eq. 7 (depth-fastest unknown ordering).
"""
import numpy as np
import pytest
import scipy.sparse as sp

import tomogen


@pytest.fixture(scope="module", params=[0, 1, 4])
def system(request):
    s = tomogen.System(request.param)
    rp, ci, va = s.csr()
    return s, rp, ci, va


def test_dims_match_baseline_configs():
    want = {0: (2048, 950), 1: (46080, 261060), 3: (46080, 261060), 4: (46080, 261060)}
    for cfg, (n, md) in want.items():
        d = tomogen.System(cfg).dims
        assert (d.n, d.m_data, d.m) == (n, md, md + n)
    d2 = tomogen.System(2).dims  # count only, no 45 GB fill
    assert (d2.n, d2.m_data, d2.m) == (655360, 3200000, 3855360)
    assert 3.6e9 < d2.nnz < 3.9e9  # BASELINE.json: "about 3.8e9 nnz"
    assert 1100 < d2.nnz / d2.m_data < 1300  # "about 1.2k nnz/row"


def test_canonical_csr(system):
    s, rp, ci, va = system
    d = s.dims
    assert rp[0] == 0 and rp[-1] == d.nnz == len(ci) == len(va)
    assert (np.diff(rp) >= 0).all()
    assert ci.min() >= 0 and ci.max() < d.n
    inc = np.diff(ci.astype(np.int64)) > 0
    boundary = np.zeros(len(ci) - 1, dtype=bool)
    inner = rp[1:-1]
    boundary[inner[(inner > 0) & (inner < len(ci))] - 1] = True
    assert (inc | boundary).all(), "columns must be strictly increasing inside every row"
    assert np.isfinite(va).all() and (va != 0).all()


def test_row_sums_are_ray_lengths_and_laplacian_rows_sum_to_zero(system):
    s, rp, ci, va = system
    d = s.dims
    A = sp.csr_matrix((va, ci, rp), shape=(d.m, d.n))
    rs = np.asarray(A.sum(axis=1)).ravel()
    L = np.repeat(s.ray_lengths(), d.nper)  # depth kernel sums to 1 => row sum = ray length
    assert np.abs(rs[: d.m_data] - L).max() < 1e-12 * max(1.0, L.max())
    assert np.abs(rs[d.m_data:]).max() == 0.0
    rl = np.diff(rp)
    assert rl[d.m_data:].min() >= 4 and rl[d.m_data:].max() == 7
    assert (rl[: d.m_data] % d.keep == 0).all()  # runs of `keep` consecutive layers per lateral node


def test_depth_fastest_runs(system):
    s, rp, ci, va = system
    d = s.dims
    # first data row: columns come in runs of `keep` consecutive indices inside one lateral node
    c = ci[rp[0]:rp[1]].reshape(-1, d.keep)
    assert (np.diff(c, axis=1) == 1).all()
    assert (c[:, 0] // d.nz == c[:, -1] // d.nz).all()


def test_block_fill_equals_full_fill(system):
    s, rp, ci, va = system
    d = s.dims
    for r0, r1 in [(0, 17), (13, 29), (d.m_data - 7, d.m_data + 11), (d.m_data + 5, d.m), (d.m - 1, d.m)]:
        c2 = np.empty(rp[r1] - rp[r0], np.int32)
        v2 = np.empty(rp[r1] - rp[r0], np.float64)
        s.fill(r0, r1, c2, v2)
        assert np.array_equal(c2, ci[rp[r0]:rp[r1]]) and np.array_equal(v2, va[rp[r0]:rp[r1]])


def test_deterministic_and_rhs_recipe(system):
    s, rp, ci, va = system
    d = s.dims
    s2 = tomogen.System(s.config)
    rp2, ci2, va2 = s2.csr()
    assert np.array_equal(rp, rp2) and np.array_equal(ci, ci2) and np.array_equal(va, va2)
    b, b2 = s.rhs(0), s2.rhs(0)
    assert np.array_equal(b, b2)
    assert (b[d.m_data:] == 0).all()
    x = s.x_true(0)
    assert abs(np.abs(x).max() - 0.05) < 1e-15
    A = sp.csr_matrix((va, ci, rp), shape=(d.m, d.n))
    dd = (A @ x)[: d.m_data]
    noise = b[: d.m_data] - dd
    rms = np.sqrt((dd ** 2).mean())
    assert 0.8 * 0.01 * rms < noise.std() < 1.2 * 0.01 * rms  # 1 % noise


def test_config3_shares_config1_matrix_and_has_8_checkerboards():
    s1, s3 = tomogen.System(1), tomogen.System(3)
    assert s1.dims.nnz == s3.dims.nnz and s3.dims.nrhs == 8
    assert np.array_equal(s1.rowptr(), s3.rowptr())
    assert np.array_equal(s1.stations(), s3.stations())
    d = s3.dims
    for r in (0, 7):
        x = s3.x_true(r).reshape(d.ny, d.nx, d.nz)
        blk = 2 + r
        assert set(np.unique(x)) == {-0.05, 0.05}
        assert x[0, 0, 0] == 0.05 and x[0, blk, 0] == -0.05 and x[blk, 0, 0] == -0.05 and x[0, 0, 2] == -0.05


def test_config4_is_skewed():
    s = tomogen.System(4)
    rp, ci, _ = s.csr()
    cl = np.bincount(ci, minlength=s.dims.n)
    assert cl.max() / cl.mean() > 15  # heavily repeated hot columns in A^T (BASELINE.json configs[4])
    xy = s.stations()
    ncl = int(round(0.6 * s.dims.nst))
    assert np.ptp(xy[:ncl, 0]) <= 6.0 and np.ptp(xy[:ncl, 1]) <= 6.0


def test_random_csr_helper():
    rp, ci, va = tomogen.random_csr(6, 50, [0, 1, 50, 7, 0, 33], seed=3)
    assert rp[-1] == 91
    for i in range(6):
        c = ci[rp[i]:rp[i + 1]]
        assert (np.diff(c) > 0).all()
