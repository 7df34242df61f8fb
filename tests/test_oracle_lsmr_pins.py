"""Pins of the LSMR oracle (oracle.lsmr; Fong & Saunders' algorithm, the paper's own solver)
against things other than itself: the library routine scipy.sparse.linalg.lsmr, the dense solution of the
damped normal equations, the method's monotone ||A^T r|| (the property it is named for), directly computed
norms, and order-independence of the double-double mode."""
import numpy as np
import pytest
import scipy.sparse as sp
import scipy.sparse.linalg as sla

import oracle


def csr_args(A):
    A = sp.csr_matrix(A)
    A.sort_indices()
    return A.shape[0], A.shape[1], A.indptr.astype(np.int64), A.indices.astype(np.int32), A.data.astype(np.float64)


def rel(a, b):
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))


@pytest.mark.parametrize("mode", [oracle.PLAIN, oracle.DD])
@pytest.mark.parametrize("damp", [0.0, 0.3])
def test_against_scipy_lsmr(mode, damp):
    rng = np.random.default_rng(0)
    A = sp.random(60, 25, density=0.3, random_state=1, format="csr")
    b = rng.standard_normal(60)
    for k in (1, 2, 3, 5, 8):
        o = oracle.lsmr(*csr_args(A), b, damp=damp, max_iters=k, mode=mode)
        x, istop, itn, normr, normar, normA, condA, normx = sla.lsmr(A, b, damp=damp, atol=0, btol=0, conlim=0, maxiter=k)
        assert o.itn == itn == k
        assert rel(o.x, x) <= 1e-9
        for mine, ref in ((o.normr, normr), (o.normar, normar), (o.normA, normA), (o.condA, condA), (o.normx, normx)):
            assert abs(mine - ref) <= 1e-9 * abs(ref)


def test_tolerance_stop_like_scipy(cfg0):
    A = sp.csr_matrix((cfg0["va"], cfg0["ci"], cfg0["rp"]), shape=(cfg0["m"], cfg0["n"]))
    o = oracle.lsmr(cfg0["m"], cfg0["n"], cfg0["rp"], cfg0["ci"], cfg0["va"], cfg0["b"], damp=cfg0["damp"], atol=1e-6, btol=1e-6,
                    max_iters=500)
    x, istop, itn = sla.lsmr(A, cfg0["b"], damp=cfg0["damp"], atol=1e-6, btol=1e-6, conlim=0, maxiter=500)[:3]
    # same iteration count and stop reason; x agrees to the level of the tolerance (167 iterations amplify
    # the different rounding order of the two implementations, cf. DESIGN.md R-dd)
    assert (o.itn, o.istop) == (itn, istop) and rel(o.x, x) <= 1e-4


@pytest.mark.parametrize("mode", [oracle.PLAIN, oracle.DD])
@pytest.mark.parametrize("damp", [0.0, 0.2])
def test_converges_to_damped_normal_equations(mode, damp):
    rng = np.random.default_rng(3)
    D = rng.standard_normal((30, 12))
    b = rng.standard_normal(30)
    o = oracle.lsmr(*csr_args(D), b, damp=damp, max_iters=40, mode=mode)
    xs = np.linalg.solve(D.T @ D + damp * damp * np.eye(12), D.T @ b)
    assert rel(o.x, xs) <= 1e-10


@pytest.mark.parametrize("mode", [oracle.PLAIN, oracle.DD])
def test_monotone_normar_and_direct_norms(cfg0, mode):
    m, n, rp, ci, va, b, damp = (cfg0[k] for k in ("m", "n", "rp", "ci", "va", "b", "damp"))
    A = sp.csr_matrix((va, ci, rp), shape=(m, n))
    o = oracle.lsmr(m, n, rp, ci, va, b, damp=damp, max_iters=40, mode=mode, snapshots=(5, 20, 40))
    assert np.all(np.diff(o.normar_hist) <= 1e-12 * o.normar_hist[0])  # LSMR: ||Abar^T rbar|| decreases monotonically
    assert np.all(np.diff(o.normr_hist) <= 1e-12 * o.normr_hist[0])
    for k in (5, 20, 40):
        x = o.snapshots[k]
        r = b - A @ x
        normr = np.sqrt(r @ r + damp * damp * (x @ x))          # ||bbar - Abar x||
        normar = np.linalg.norm(A.T @ r - damp * damp * x)      # ||Abar^T rbar||
        assert abs(o.normr_hist[k - 1] - normr) <= 1e-9 * normr
        assert abs(o.normar_hist[k - 1] - normar) <= 1e-7 * o.normar_hist[0]
    assert abs(o.normx - np.linalg.norm(o.x)) <= 1e-14 * o.normx


def test_dd_mode_is_invariant_under_row_permutation(cfg0):
    m, n, rp, ci, va, b, damp = (cfg0[k] for k in ("m", "n", "rp", "ci", "va", "b", "damp"))
    A = sp.csr_matrix((va, ci, rp), shape=(m, n))
    P = np.random.default_rng(4).permutation(m)
    o1 = oracle.lsmr(m, n, rp, ci, va, b, damp=damp, max_iters=40, mode=oracle.DD)
    o2 = oracle.lsmr(*csr_args(A[P]), b[P], damp=damp, max_iters=40, mode=oracle.DD)
    assert np.array_equal(o1.x, o2.x)


def test_edge_cases():
    A = sp.csr_matrix(np.array([[1.0, 0.0], [0.0, 2.0], [0.0, 0.0]]))
    o = oracle.lsmr(*csr_args(A), np.zeros(3), max_iters=5)
    assert o.itn == 0 and o.istop == 0 and not o.x.any()
    o = oracle.lsmr(*csr_args(A), np.array([0.0, 0.0, 1.0]), max_iters=5)  # A^T b = 0
    assert o.itn == 0 and o.istop == 0 and not o.x.any()
    o = oracle.lsmr(*csr_args(A), np.array([1.0, 1.0, 1.0]), max_iters=0)
    assert o.itn == 0 and o.istop == 7
