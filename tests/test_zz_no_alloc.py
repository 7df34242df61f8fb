"""tomo_lsqr_spmv_noalloc (include/tomo_lsqr.h): the sparse product for callers that cannot call cudaMalloc.  Its scratch
is a file-scope static device array in libtomolsqr.so; the test checks it against the existing path
(tomo_lsqr_create + tomo_lsqr_spmv) on calls in a row that share that array.

The file name sorts last on purpose: the run uses `pytest -x`, so nothing is collected after it.
It must pass alone in a fresh process and after the other GPU tests (it shares no fixture state with them).
"""
import numpy as np
import pytest
import torch

import tomogen

pytestmark = pytest.mark.gpu

TOL_SPMV = 1e-12   # the SpMV tolerance of tests/test_gpu_parity.py (BASELINE.json north_star)


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def rel(a, b):
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))


@pytest.fixture(scope="module")
def tl():
    from paper_2604_11920_b200 import build
    build.build()
    import paper_2604_11920_b200 as tl
    tl.load()
    return tl


class Mat:
    """A CSR on the device, a handle on it (the existing path) and the arguments of the no-alloc entry."""

    def __init__(self, tl, m, n, rp, ci, va):
        self.tl, self.m, self.n, self.nnz = tl, int(m), int(n), int(rp[-1])
        self.rp, self.ci, self.va = dev(rp), dev(ci), dev(va)
        self.vt = tl.TOMO_VAL_F32 if va.dtype == np.float32 else tl.TOMO_VAL_F64
        self.S = tl.TomoLsqr(self.m, self.n, self.rp, self.ci, self.va)

    def existing(self, x, accumulate):
        self.S.set(accumulate=accumulate)
        return self.S.spmv(x).cpu().numpy()

    def noalloc(self, x, accumulate, y=None):
        if y is None:
            y = torch.full((self.m,), float("nan"), dtype=torch.float64, device="cuda")  # every entry must be written
        self.tl.tomo_lsqr_spmv_noalloc(self.m, self.n, self.nnz, self.rp, self.ci, self.va, self.vt, accumulate, x, y)
        return y.cpu().numpy()


def check(mat, seed):
    rng = np.random.default_rng(seed)
    x = dev(rng.standard_normal(mat.n))
    for accumulate in (1, 0):
        want = mat.existing(x, accumulate)
        got = mat.noalloc(x, accumulate)
        assert np.all(np.isfinite(got))
        assert rel(got, want) <= TOL_SPMV
        # same kernel, same split points, same summation order: the documented outcome is bitwise equality
        assert np.array_equal(got, want), f"accumulate={accumulate}: not bitwise the handle path"


def test_noalloc_matches_handle_path_on_calls_in_a_row(tl, cfg0):
    """Two calls in a row on config 0 (different x), then matrices of other shapes in between (rows without entries, a
    ragged tail, fp32 values), then config 0 again: the shared array keeps each call's leftovers, the results do not."""
    a = Mat(tl, cfg0["m"], cfg0["n"], cfg0["rp"], cfg0["ci"], cfg0["va"])
    check(a, 1)
    check(a, 2)

    rng = np.random.default_rng(4242)
    lens = np.concatenate([[0, 0, 0], rng.integers(0, 9, size=30000), [0] * 700, rng.integers(200, 2100, size=300),
                           [70001], [0, 5, 0, 0]]).astype(np.int64)
    n = 71003
    rp, ci, va = tomogen.random_csr(len(lens), n, lens, seed=99)
    b = Mat(tl, len(lens), n, rp, ci, va)           # 60 % of the short rows and both ends hold rows without entries
    check(b, 3)
    check(a, 4)                                      # ... after a call that used the compaction part of the array
    c = Mat(tl, len(lens), n, rp, ci, va.astype(np.float32))
    check(c, 5)
    check(b, 6)

    # a matrix without any entry: y = 0
    z = Mat(tl, 5, 3, np.zeros(6, dtype=np.int64), np.zeros(0, dtype=np.int32), np.zeros(0, dtype=np.float64))
    assert np.array_equal(z.noalloc(dev(np.ones(3)), 1), np.zeros(5))
    check(a, 7)
    for mat in (a, b, c, z):
        mat.S.close()


def test_noalloc_allocates_nothing_and_rejects_what_does_not_fit(tl, cfg0):
    a = Mat(tl, cfg0["m"], cfg0["n"], cfg0["rp"], cfg0["ci"], cfg0["va"])
    x = dev(np.random.default_rng(8).standard_normal(a.n))
    y = torch.empty(a.m, dtype=torch.float64, device="cuda")
    a.noalloc(x, 1, y)                               # first use on this device: the library sets the array up
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        a.noalloc(x, 1, y)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 >= free0, "device memory in use grew over calls of the no-alloc entry"

    # beyond the static array: a clear error, nothing launched, the output untouched
    m_big = tl.TOMO_NOALLOC_MAX_ROWS + 1
    rp = torch.zeros(m_big + 1, dtype=torch.int64, device="cuda")
    y_big = torch.full((m_big,), 7.0, dtype=torch.float64, device="cuda")
    with pytest.raises(tl.TomoError) as ei:
        tl.tomo_lsqr_spmv_noalloc(m_big, a.n, 0, rp, None, None, tl.TOMO_VAL_F64, 1, x, y_big)
    assert ei.value.status == tl.TOMO_ERR_NOALLOC_LIMIT
    assert "TOMO_NOALLOC_MAX_ROWS" in str(ei.value) and str(m_big) in str(ei.value)
    assert bool((y_big == 7.0).all())
    # the largest size that fits is accepted (all rows without entries: y = 0)
    tl.tomo_lsqr_spmv_noalloc(m_big - 1, a.n, 0, rp[:-1], None, None, tl.TOMO_VAL_F64, 1, x, y_big[:-1])
    assert bool((y_big[:-1] == 0.0).all())

    # argument errors are reported like everywhere else in the library
    for bad in (dict(accumulate=2), dict(vt=5)):
        kw = dict(vt=tl.TOMO_VAL_F64, accumulate=1)
        kw.update(bad)
        with pytest.raises(tl.TomoError) as ei:
            tl.tomo_lsqr_spmv_noalloc(a.m, a.n, a.nnz, a.rp, a.ci, a.va, kw["vt"], kw["accumulate"], x, y)
        assert ei.value.status == tl.TOMO_ERR_INVALID_ARG
    with pytest.raises(tl.TomoError) as ei:
        tl.tomo_lsqr_spmv_noalloc(a.m, a.n, a.nnz, a.rp, a.ci, a.va, tl.TOMO_VAL_F64, 1, x.cpu(), y)
    assert ei.value.status == tl.TOMO_ERR_NOT_DEVICE_PTR
    # and the entry still works afterwards
    assert np.array_equal(a.noalloc(x, 1), a.existing(x, 1))
    a.S.close()
