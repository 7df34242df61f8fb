"""Pins of the CPU oracle (oracle/lsqr_oracle.cpp) against things other than itself.

The paper prints no worked numerical example for the solver (PAPER.md has only ratios), so the
pins are what the mathematics fixes: dense normal equations / QR on tiny systems, brute-force exact
arithmetic, the adjoint identity, the closed form of x_1, finite termination, exact recovery, the
monotone decrease of ||r|| that the paper states for LSQR, the identities the norm estimates
satisfy, and a library routine (scipy.sparse.linalg.lsqr) that implements the same algorithm.
Each test is chosen so that a plausible mistake (dropped term, sign, index, transposed operand) fails.
"""
from fractions import Fraction

import numpy as np
import pytest
import scipy.sparse as sp
from scipy.sparse.linalg import lsqr as scipy_lsqr

import oracle
import tomogen


def rel(a, b):
    return np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300)


def small_system(m, n, density, seed, cond_boost=False):
    rng = np.random.default_rng(seed)
    A = sp.random(m, n, density=density, random_state=rng, format="csr", data_rvs=rng.standard_normal)
    A = (A + sp.eye(m, n, format="csr") * (2.0 if cond_boost else 0.0)).tocsr()
    A.sort_indices()
    A.eliminate_zeros()
    b = rng.standard_normal(m)
    return A, b


def csr_args(A):
    return A.shape[0], A.shape[1], A.indptr.astype(np.int64), A.indices.astype(np.int32), A.data.astype(np.float64)


# ---------------------------------------------------------------- SpMV, both directions ---------------
@pytest.mark.parametrize("mode", [oracle.PLAIN, oracle.DD])
def test_spmv_matches_dense(mode):
    A, _ = small_system(37, 23, 0.3, 1)
    rng = np.random.default_rng(2)
    x, u = rng.standard_normal(23), rng.standard_normal(37)
    D = A.toarray()
    assert rel(oracle.spmv(*csr_args(A), x, mode), D @ x) < 1e-14
    assert rel(oracle.spmv_t(*csr_args(A), u, mode), D.T @ u) < 1e-14  # a transposed operand fails here


def test_dd_spmv_is_correctly_rounded_exact_sum():
    # brute force in exact rational arithmetic, ill-conditioned sums (massive cancellation)
    rng = np.random.default_rng(5)
    m, n = 9, 40
    D = rng.standard_normal((m, n)) * 10.0 ** rng.integers(-8, 8, size=(m, n))
    D[:, n // 2:] = -D[:, : n // 2] * (1 + 1e-9 * rng.standard_normal((m, n // 2)))
    x = np.ones(n) + 1e-7 * rng.standard_normal(n)
    A = sp.csr_matrix(D)
    y = oracle.spmv(*csr_args(A), x, oracle.DD)
    for i in range(m):
        exact = sum(Fraction(D[i, j]) * Fraction(x[j]) for j in range(n))
        assert y[i] == float(exact)  # float(Fraction) rounds to nearest
    # the transposed product (a scatter with one (hi, lo) pair per column) on sums that cancel just as
    # badly: the transpose of the same construction, so every COLUMN sum loses ~9 digits; a scatter that
    # dropped or mis-paired the low word would be off by ~1e-9 relative here
    Dt = np.ascontiguousarray(D.T)          # n x m: column i of Dt is row i of D
    At = sp.csr_matrix(Dt)
    yt = oracle.spmv_t(*csr_args(At), x, oracle.DD)   # (Dt)^T x = D x, computed by the scatter
    for i in range(m):
        exact = sum(Fraction(Dt[j, i]) * Fraction(x[j]) for j in range(n))
        assert yt[i] == float(exact)
    assert np.array_equal(yt, y)            # both routes give the one correctly rounded value
    u = np.ones(m) + 1e-7 * rng.standard_normal(m)
    yu = oracle.spmv_t(*csr_args(A), u, oracle.DD)
    for j in range(n):
        exact = sum(Fraction(D[i, j]) * Fraction(u[i]) for i in range(m))
        assert yu[j] == float(exact)


def test_fused_axpy_terms_and_norms_are_exact_in_dd_mode():
    """spmv / spmv_t with c != 0 (u <- A v - alpha u, v <- A^T u - beta v: the fused term enters the same
    (hi, lo) sum and the total is rounded once) and the dd norms, pinned through the first iteration of the
    Stepper against exact rational arithmetic.  A dropped or separately rounded -alpha*u_i / -beta*v_j
    term, a wrong sign or a norm that is not the rounded exact sum changes the last bits checked here."""
    rng = np.random.default_rng(15)
    m, n = 14, 9
    D = rng.standard_normal((m, n)) * (rng.random((m, n)) < 0.6)
    D[0, :] = 0.0
    D[0, 0] = 1.0  # keep every column and row non-trivial enough
    A = sp.csr_matrix(D)
    A.sort_indices()
    b = rng.standard_normal(m)
    st = oracle.Stepper(*csr_args(A), b, damp=0.3, max_iters=3, mode=oracle.DD)
    F = Fraction

    def rsum(terms):  # correctly rounded exact sum
        return float(sum(terms, F(0)))

    # state after init: u = b/||b||, v = A^T u / alpha (both rounded as the algorithm states)
    beta1 = np.sqrt(rsum(F(t) * F(t) for t in b))
    u0 = b * (1.0 / beta1)
    assert np.array_equal(st.vec("u"), u0)
    vh = np.array([rsum(F(D[i, j]) * F(u0[i]) for i in range(m)) for j in range(n)])
    alpha1 = np.sqrt(rsum(F(t) * F(t) for t in vh))
    v0 = vh * (1.0 / alpha1)
    assert np.array_equal(st.vec("v"), v0)
    sc = st.scalars()
    assert sc["alpha"] == alpha1 and sc["beta"] == beta1
    # one iteration: u^ = A v - alpha u, beta, u = u^/beta ; v^ = A^T u - beta v, alpha, v = v^/alpha
    st.step()
    uh = np.array([rsum([F(-alpha1) * F(u0[i])] + [F(D[i, j]) * F(v0[j]) for j in range(n)]) for i in range(m)])
    beta2 = np.sqrt(rsum(F(t) * F(t) for t in uh))
    u1 = uh * (1.0 / beta2)
    assert np.array_equal(st.vec("u"), u1)
    vh2 = np.array([rsum([F(-beta2) * F(v0[j])] + [F(D[i, j]) * F(u1[i]) for i in range(m)]) for j in range(n)])
    alpha2 = np.sqrt(rsum(F(t) * F(t) for t in vh2))
    assert np.array_equal(st.vec("v"), vh2 * (1.0 / alpha2))
    sc = st.scalars()
    assert sc["alpha"] == alpha2 and sc["beta"] == beta2
    # plain mode takes the same terms in fp64 with the fused term LAST (fma(c, y_i, s)): pinned to rounding
    sp_ = oracle.Stepper(*csr_args(A), b, damp=0.3, max_iters=3, mode=oracle.PLAIN)
    sp_.step()
    assert rel(sp_.vec("u"), u1) < 1e-14 and rel(sp_.vec("v"), vh2 * (1.0 / alpha2)) < 1e-13


def test_adjoint_identity(cfg0):
    rng = np.random.default_rng(7)
    for mode in (oracle.PLAIN, oracle.DD):
        v, u = rng.standard_normal(cfg0["n"]), rng.standard_normal(cfg0["m"])
        Av = oracle.spmv(cfg0["m"], cfg0["n"], cfg0["rp"], cfg0["ci"], cfg0["va"], v, mode)
        Atu = oracle.spmv_t(cfg0["m"], cfg0["n"], cfg0["rp"], cfg0["ci"], cfg0["va"], u, mode)
        lhs, rhs = Av @ u, v @ Atu
        assert abs(lhs - rhs) <= 1e-13 * (np.linalg.norm(Av) * np.linalg.norm(u))


def test_A_times_ones_is_ray_length(cfg0):
    s = cfg0["sys"]
    y = oracle.spmv(cfg0["m"], cfg0["n"], cfg0["rp"], cfg0["ci"], cfg0["va"], np.ones(cfg0["n"]), oracle.DD)
    L = np.repeat(s.ray_lengths(), s.dims.nper)
    assert np.abs(y[: s.dims.m_data] - L).max() < 1e-12
    assert np.abs(y[s.dims.m_data:]).max() == 0.0


def test_csr_to_csc_matches_scipy(cfg0):
    colptr, rowind, cvals = oracle.csr_to_csc(cfg0["m"], cfg0["n"], cfg0["rp"], cfg0["ci"], cfg0["va"])
    C = sp.csr_matrix((cfg0["va"], cfg0["ci"], cfg0["rp"]), shape=(cfg0["m"], cfg0["n"])).tocsc()
    C.sort_indices()
    assert np.array_equal(colptr, C.indptr) and np.array_equal(rowind, C.indices) and np.array_equal(cvals, C.data)


# ---------------------------------------------------------------- LSQR iterates -----------------------
@pytest.mark.parametrize("mode", [oracle.PLAIN, oracle.DD])
@pytest.mark.parametrize("damp", [0.0, 0.3])
def test_x1_closed_form(mode, damp):
    # x_1 = t g, g = A^T b, t = |g|^2 / (|A g|^2 + damp^2 |g|^2)  (first Krylov step of CG on the normal eqs)
    A, b = small_system(60, 25, 0.2, 11)
    r = oracle.lsqr(*csr_args(A), b, damp=damp, max_iters=1, mode=mode)
    g = A.T @ b
    t = (g @ g) / ((A @ g) @ (A @ g) + damp ** 2 * (g @ g))
    assert rel(r.x, t * g) < 1e-14
    assert r.itn == 1 and r.istop == 7


@pytest.mark.parametrize("mode", [oracle.PLAIN, oracle.DD])
def test_finite_termination_on_diagonal(mode):
    # diagonal A with l distinct singular values: x_l = a_i b_i / (a_i^2 + damp^2) after exactly l iterations
    vals = np.array([1.0, 2.0, 3.5, 5.0])
    n = 12
    a = np.tile(vals, n // 4)
    A = sp.diags(a).tocsr()
    b = np.arange(1, n + 1, dtype=float)
    damp = 0.7
    want = a * b / (a ** 2 + damp ** 2)
    r4 = oracle.lsqr(*csr_args(A), b, damp=damp, max_iters=4, mode=mode)
    r3 = oracle.lsqr(*csr_args(A), b, damp=damp, max_iters=3, mode=mode)
    assert rel(r4.x, want) < 1e-12
    assert rel(r3.x, want) > 1e-3


@pytest.mark.parametrize("mode", [oracle.PLAIN, oracle.DD])
@pytest.mark.parametrize("seed,damp", [(21, 0.0), (22, 0.1), (23, 1.5)])
def test_converges_to_normal_equations_and_qr(mode, seed, damp):
    A, b = small_system(40, 12, 0.4, seed, cond_boost=True)
    D = A.toarray()
    n = D.shape[1]
    x_ne = np.linalg.solve(D.T @ D + damp ** 2 * np.eye(n), D.T @ b)
    x_qr = np.linalg.lstsq(np.vstack([D, damp * np.eye(n)]), np.concatenate([b, np.zeros(n)]), rcond=None)[0]
    r = oracle.lsqr(*csr_args(A), b, damp=damp, max_iters=n + 1, mode=mode)  # <= n+1 iterations suffice
    assert rel(r.x, x_qr) < 1e-10 and rel(r.x, x_ne) < 1e-9
    # estimates against the directly computed quantities at the end
    rr = b - D @ r.x
    assert abs(r.r1norm - np.linalg.norm(rr)) <= 1e-8 * np.linalg.norm(b)
    assert abs(r.r2norm - np.sqrt(rr @ rr + damp ** 2 * (r.x @ r.x))) <= 1e-10 * np.linalg.norm(b)
    assert abs(r.xnorm - np.linalg.norm(r.x)) <= 1e-10 * np.linalg.norm(r.x)


def test_exact_recovery_noise_free():
    A, _ = small_system(80, 20, 0.3, 31, cond_boost=True)
    xt = np.random.default_rng(32).standard_normal(20)
    b = A @ xt
    r = oracle.lsqr(*csr_args(A), b, damp=0.0, atol=1e-14, btol=1e-14, max_iters=200, mode=oracle.PLAIN)
    assert rel(r.x, xt) < 1e-10
    assert r.istop in (1, 2, 4, 5)


@pytest.mark.parametrize("mode", [oracle.PLAIN, oracle.DD])
def test_monotone_residual_and_estimate_identities(cfg0, mode):
    m, n, damp = cfg0["m"], cfg0["n"], cfg0["damp"]
    snaps = (1, 2, 5, 10, 25, 50)
    r = oracle.lsqr(m, n, cfg0["rp"], cfg0["ci"], cfg0["va"], cfg0["b"], damp=damp, max_iters=50, mode=mode, snapshots=snaps)
    assert r.itn == 50 and r.istop == 7
    assert (np.diff(r.r2norm_hist) <= 0).all()  # LSQR: monotone ||r||
    A = sp.csr_matrix((cfg0["va"], cfg0["ci"], cfg0["rp"]), shape=(m, n))
    bn = np.linalg.norm(cfg0["b"])
    for k in snaps:
        x = r.snapshots[k]
        res = cfg0["b"] - A @ x
        r2 = np.sqrt(res @ res + damp ** 2 * (x @ x))
        ar = np.linalg.norm(A.T @ res - damp ** 2 * x)
        assert abs(r.r2norm_hist[k - 1] - r2) <= 1e-10 * bn
        assert abs(r.arnorm_hist[k - 1] - ar) <= 1e-9 * max(ar, 1e-3 * r.arnorm_hist[0])
    assert abs(r.xnorm - np.linalg.norm(r.x)) <= 1e-10 * np.linalg.norm(r.x)
    assert abs(r.r1norm - np.linalg.norm(cfg0["b"] - A @ r.x)) <= 1e-8 * bn


def test_against_scipy_lsqr(cfg0):
    m, n, damp = cfg0["m"], cfg0["n"], cfg0["damp"]
    A = sp.csr_matrix((cfg0["va"], cfg0["ci"], cfg0["rp"]), shape=(m, n))
    for k, tol in ((1, 1e-13), (10, 1e-11), (50, 1e-10)):
        ref = scipy_lsqr(A, cfg0["b"], damp=damp, atol=0, btol=0, conlim=0, iter_lim=k)
        for mode in (oracle.PLAIN, oracle.DD):
            r = oracle.lsqr(m, n, cfg0["rp"], cfg0["ci"], cfg0["va"], cfg0["b"], damp=damp, max_iters=k, mode=mode)
            assert rel(r.x, ref[0]) < tol, (k, mode)
            assert abs(r.r2norm - ref[4]) <= 1e-10 * ref[4] and abs(r.anorm - ref[5]) <= 1e-10 * ref[5]
            assert abs(r.acond - ref[6]) <= 1e-8 * ref[6] and abs(r.arnorm - ref[7]) <= 1e-7 * max(ref[7], 1e-12)
    # tolerance run: same stopping iteration and reason as the library
    ref = scipy_lsqr(A, cfg0["b"], damp=damp, atol=1e-6, btol=1e-6, conlim=0, iter_lim=2000)
    r = oracle.lsqr(m, n, cfg0["rp"], cfg0["ci"], cfg0["va"], cfg0["b"], damp=damp, atol=1e-6, btol=1e-6, max_iters=2000)
    assert (r.istop, r.itn) == (ref[1], ref[2])


def test_edge_cases():
    A, b = small_system(15, 6, 0.4, 41)
    args = csr_args(A)
    r = oracle.lsqr(*args, np.zeros(15), damp=0.1, max_iters=10)  # b = 0
    assert r.itn == 0 and r.istop == 0 and not r.x.any()
    r = oracle.lsqr(*args, b, damp=0.1, max_iters=0)  # no iterations allowed
    assert r.itn == 0 and r.istop == 7 and not r.x.any()
    # b orthogonal to range(A): A^T b = 0 => x = 0
    D = A.toarray()
    q = np.linalg.svd(D, full_matrices=True)[0][:, -1]
    Dz = D.copy()
    Dz[np.abs(Dz) < 1e-300] = 0
    r = oracle.lsqr(*args, q, damp=0.0, atol=1e-10, btol=1e-10, max_iters=10)
    assert np.linalg.norm(r.x) < 1e-10
    # empty rows and an empty column are legal CSR
    rp, ci, va = tomogen.random_csr(8, 10, [0, 3, 0, 10, 1, 0, 2, 4], seed=9)
    va[ci == 4] = 0.0
    r = oracle.lsqr(8, 10, rp, ci, va, np.arange(8.0), damp=0.5, max_iters=12)
    D = sp.csr_matrix((va, ci, rp), shape=(8, 10)).toarray()
    want = np.linalg.solve(D.T @ D + 0.25 * np.eye(10), D.T @ np.arange(8.0))
    assert rel(r.x, want) < 1e-9


def test_stepper_equals_solve(cfg0):
    m, n = cfg0["m"], cfg0["n"]
    st = oracle.Stepper(m, n, cfg0["rp"], cfg0["ci"], cfg0["va"], cfg0["b"], damp=cfg0["damp"], max_iters=7, mode=oracle.DD)
    while not st.done:
        st.step()
    r = oracle.lsqr(m, n, cfg0["rp"], cfg0["ci"], cfg0["va"], cfg0["b"], damp=cfg0["damp"], max_iters=7, mode=oracle.DD)
    assert np.array_equal(st.vec("x"), r.x) and st.scalars()["itn"] == 7
    # Golub-Kahan: u and v are unit vectors
    assert abs(np.linalg.norm(st.vec("u")) - 1) < 1e-14 and abs(np.linalg.norm(st.vec("v")) - 1) < 1e-14


# ---------------------------------------------------------------- dd mode: order independence ---------
def _subsystem(nrows_data=12000):
    """Config-1 grid with the first `nrows_data` data rows + all smoothing rows (fast enough for CPU CI)."""
    s = tomogen.System(1)
    d = s.dims
    rp = s.rowptr()
    e1 = rp[nrows_data]
    ci = np.empty(e1, np.int32)
    va = np.empty(e1, np.float64)
    s.fill(0, nrows_data, ci, va)
    es = rp[d.m] - rp[d.m_data]
    cs = np.empty(es, np.int32)
    vs = np.empty(es, np.float64)
    s.fill(d.m_data, d.m, cs, vs)
    rp2 = np.concatenate([rp[: nrows_data + 1], rp[d.m_data + 1:] - rp[d.m_data] + e1])
    b = s.rhs(0)
    b2 = np.concatenate([b[:nrows_data], b[d.m_data:]])
    return nrows_data + d.n, d.n, rp2, np.concatenate([ci, cs]), np.concatenate([va, vs]), b2, s.damp


def test_dd_mode_is_invariant_under_row_and_column_permutation():
    m, n, rp, ci, va, b, damp = _subsystem()
    A = sp.csr_matrix((va, ci, rp), shape=(m, n))
    rng = np.random.default_rng(77)
    P, Q = rng.permutation(m), rng.permutation(n)
    AP = A[P].tocsr()
    AP.sort_indices()
    AQ = A[:, Q].tocsr()
    AQ.sort_indices()
    k = 40
    base = oracle.lsqr(m, n, rp, ci, va, b, damp=damp, max_iters=k, mode=oracle.DD, snapshots=(10, 20, 30, 40))
    rowp = oracle.lsqr(*csr_args(AP), b[P], damp=damp, max_iters=k, mode=oracle.DD, snapshots=(10, 20, 30, 40))
    colp = oracle.lsqr(*csr_args(AQ), b, damp=damp, max_iters=k, mode=oracle.DD, snapshots=(10, 20, 30, 40))
    for kk in (10, 20, 30, 40):
        assert np.array_equal(base.snapshots[kk], rowp.snapshots[kk]), kk  # bitwise
        assert np.array_equal(base.snapshots[kk][Q], colp.snapshots[kk]), kk
    assert np.array_equal(base.r2norm_hist, rowp.r2norm_hist)
    # plain mode agrees with dd to rounding at k = 10 (before order sensitivity sets in)
    pl = oracle.lsqr(m, n, rp, ci, va, b, damp=damp, max_iters=10, mode=oracle.PLAIN)
    assert rel(pl.x, base.snapshots[10]) < 1e-9
