"""GPU parity of the factored operator (tomo_lsqr_create_factored, second form; Eq. 5
P:69-71, Eq. 7) through the C ABI against the CPU oracle on the multiplied-out matrix (oracle/factored.py, whose
output is pinned bitwise to the generator's CSR assembly in tests/test_oracle_factored_pins.py).

Bars: as for the CSR path (north_star): SpMV <= 1e-12, x_50 <= 1e-8; in dd mode the sums are order-independent, so the
factored kernels (another order of the same rounded products) must reproduce the oracle bit for bit, which is asserted.
Runs after test_gpu_parity.py (file name), when the full-size oracle jobs have finished.
"""
import numpy as np
import pytest
import torch

import oracle
import oracle_jobs
import tomogen
from oracle import factored as ofac

pytestmark = pytest.mark.gpu

TOL_SPMV = 1e-12
TOL_X50 = 1e-8


def rel(a, b):
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))


def dev(a):
    return None if a is None else torch.from_numpy(np.ascontiguousarray(a)).cuda()


@pytest.fixture(scope="module")
def tl():
    from paper_2604_11920_b200 import build
    build.build()
    import paper_2604_11920_b200 as tl
    tl.load()
    return tl


def make(tl, f):
    return tl.TomoLsqr.factored(f["npairs"], f["nper"], f["nnodes"], f["nz"], dev(f["lptr"]), dev(f["lnode"]), dev(f["lw"]),
                                dev(f["kj0"].astype(np.int32)), dev(f["kern"]), dev(f["sptr"]), dev(f["sidx"]), dev(f["svals"]))


def expand_exact(f):
    return ofac.expand_exact(f["npairs"], f["nper"], f["nnodes"], f["nz"], f["lptr"], f["lnode"], f["lw"], f["kj0"], f["kern"],
                             f["sptr"], f["sidx"], f["svals"])


def expand(f):
    return ofac.expand(f["npairs"], f["nper"], f["nnodes"], f["nz"], f["lptr"], f["lnode"], f["lw"], f["kj0"], f["kern"],
                       f["sptr"], f["sidx"], f["svals"])


SHAPES = [  # npairs, nper, nnodes, nz, klen, ms   (klen 8 / 12 / 16: the template shapes; others: the general shape)
    (300, 5, 64, 8, 8, None),      # config-0-like
    (500, 10, 100, 20, 12, None),  # config-1-like: three groups of ten lanes, two idle
    (200, 16, 50, 40, 12, None),   # config-2-like: nz > 32 (two layers per lane in the closing)
    (120, 7, 30, 24, 16, 0),       # no extra block
    (90, 1, 40, 5, 5, None),       # one period: 32 groups of one lane; window = all layers; general shape
    (60, 32, 9, 33, 1, 50),        # 32 periods: one group; one-layer windows
    (150, 3, 2500, 12, 7, None),   # many nodes, most of them with no ray (closed from the extra block alone)
    (40, 11, 6, 32, 32, 7),        # the widest window the ABI takes
]


@pytest.mark.parametrize("shape", SHAPES)
def test_factored_spmv_and_solve_random_shapes(tl, shape):
    npairs, nper, nnodes, nz, klen, ms = shape
    f = tomogen.random_factored(npairs, nper, nnodes, nz, klen, seed=1000 + npairs, ms=ms,
                                empty_nodes=0.9 if nnodes > 1000 else 0.1, max_entries=60)
    rp, ci, va = expand(f)
    m, n = len(rp) - 1, nnodes * nz
    S = make(tl, f)
    assert (S.m, S.n) == (m, n) and S.info("factored") == 1.0 and S.info("lateral_entries") == len(f["lnode"])
    rng = np.random.default_rng(shape[0])
    x, u = rng.standard_normal(n), rng.standard_normal(m)
    for acc, mode, ts in ((1, oracle.DD, 1), (0, oracle.PLAIN, 1), (0, oracle.PLAIN, 0)):   # ts: fast mode's two-stage contraction / per-entry products
        S.set(accumulate=acc, two_stage=ts)
        y = S.spmv(dev(x)).cpu().numpy()
        yt = S.spmv(dev(u), transpose=True).cpu().numpy()
        oy, oyt = oracle.spmv(m, n, rp, ci, va, x, mode), oracle.spmv_t(m, n, rp, ci, va, u, mode)
        if acc:
            assert np.array_equal(y, oy) and np.array_equal(yt, oyt)
        else:
            scale = np.abs(va).max() * np.abs(x).max()
            assert np.abs(y - oy).max() <= 1e-12 * scale * 60 * nper * klen
            assert rel(y, oy) <= 1e-11 and rel(yt, oyt) <= 1e-11   # cancelling random sums: per-row bound above
    b = rng.standard_normal(m)
    for solver, ofn in (("lsqr", oracle.lsqr), ("lsmr", oracle.lsmr)):
        S.set(accumulate=1)
        xg, res = S.solve(dev(b), damp=0.1, max_iters=20, solver=solver)
        o = ofn(m, n, rp, ci, va, b, damp=0.1, max_iters=20, mode=oracle.DD)
        assert res.itn == o.itn and res.istop == o.istop
        assert np.array_equal(xg.cpu().numpy(), o.x), (solver, rel(xg.cpu().numpy(), o.x))
    # the CSR path of the library on the multiplied-out matrix gives the same bits
    C = tl.TomoLsqr(m, n, dev(rp), dev(ci), dev(va))
    xc, _ = C.solve(dev(b), damp=0.1, max_iters=20)
    xg, _ = S.solve(dev(b), damp=0.1, max_iters=20)
    assert torch.equal(xc, xg)
    C.close(); S.close()


def test_factored_cfg0_both_modes(tl, cfg0):
    s = cfg0["sys"]
    f = s.factored()
    m, n, rp, ci, va, b = cfg0["m"], cfg0["n"], cfg0["rp"], cfg0["ci"], cfg0["va"], cfg0["b"]
    S = make(tl, f)
    for acc, mode in ((1, oracle.DD), (0, oracle.PLAIN)):
        S.set(accumulate=acc)
        xg, res, r2, ar = S.solve(dev(b), damp=s.damp, max_iters=50, history=True)
        o = oracle.lsqr(m, n, rp, ci, va, b, damp=s.damp, max_iters=50, mode=mode)
        xg = xg.cpu().numpy()
        assert res.itn == o.itn == 50 and res.istop == o.istop
        assert rel(xg, o.x) <= TOL_X50
        assert np.allclose(r2, o.r2norm_hist, rtol=1e-10, atol=0) and np.allclose(ar, o.arnorm_hist, rtol=1e-8, atol=0)
        for k in ("r1norm", "r2norm", "arnorm", "anorm", "acond", "xnorm"):
            assert abs(getattr(res, k) - getattr(o, k)) <= 1e-9 * abs(getattr(o, k)), k
        if acc:
            assert np.array_equal(xg, o.x) and np.array_equal(r2, o.r2norm_hist)
    # tolerance stop: same iteration count and reason as the oracle
    S.set(accumulate=1)
    xg, res = S.solve(dev(b), damp=s.damp, atol=1e-6, btol=1e-6, max_iters=300)
    o = oracle.lsqr(m, n, rp, ci, va, b, damp=s.damp, atol=1e-6, btol=1e-6, max_iters=300, mode=oracle.DD)
    assert (res.itn, res.istop) == (o.itn, o.istop) and np.array_equal(xg.cpu().numpy(), o.x)
    # fast mode without the two-stage contraction (per-entry products of the rounded values): same bar
    S.set(accumulate=0, two_stage=0)
    xg, res = S.solve(dev(b), damp=s.damp, max_iters=50)
    o = oracle.lsqr(m, n, rp, ci, va, b, damp=s.damp, max_iters=50, mode=oracle.PLAIN)
    assert res.itn == 50 and rel(xg.cpu().numpy(), o.x) <= TOL_X50
    S.set(two_stage=1)
    # determinism and independence of the launch mode (graph / check_every / pdl), both accumulation modes
    for acc in (1, 0):
        S.set(accumulate=acc, graph=1, check_every=10, pdl=1)
        x1, _ = S.solve(dev(b), damp=s.damp, max_iters=37)
        x2, _ = S.solve(dev(b), damp=s.damp, max_iters=37)
        S.set(graph=0, check_every=7, pdl=0)
        x3, _ = S.solve(dev(b), damp=s.damp, max_iters=37)
        assert torch.equal(x1, x2) and torch.equal(x1, x3)
    # host-buffer entry and the sequential multi-RHS entry work on a factored handle
    S.set(accumulate=1, graph=1, check_every=10, pdl=1)
    xh = np.empty(n)
    tl.tomo_lsqr_solve_host(S.h, b, s.damp, 0.0, 0.0, 50, xh)
    o = oracle.lsqr(m, n, rp, ci, va, b, damp=s.damp, max_iters=50, mode=oracle.DD)
    assert np.array_equal(xh, o.x)
    B = np.ascontiguousarray(np.stack([b, 2.0 * b[::-1]], axis=1))
    X, rs = S.solve_multi(dev(B), damp=s.damp, max_iters=50)
    assert np.array_equal(X[:, 0].cpu().numpy(), o.x)
    o1 = oracle.lsqr(m, n, rp, ci, va, np.ascontiguousarray(B[:, 1]), damp=s.damp, max_iters=50, mode=oracle.DD)
    assert np.array_equal(X[:, 1].cpu().numpy(), o1.x)
    S.close()


def test_factored_edge_cases_and_errors(tl):
    import paper_2604_11920_b200 as T
    f = tomogen.random_factored(50, 4, 20, 10, 6, seed=77)
    S = make(tl, f)
    rp, ci, va = expand(f)
    m, n = S.m, S.n
    # b = 0 -> x = 0, istop 0 ; max_iters = 0 -> x = 0, istop 7
    x, res = S.solve(dev(np.zeros(m)), damp=0.1, max_iters=5)
    assert res.istop == 0 and res.itn == 0 and not x.any()
    x, res = S.solve(dev(np.ones(m)), damp=0.1, max_iters=0)
    assert res.istop == 7 and res.itn == 0 and not x.any()
    # an option that only concerns the CSR path is accepted and changes nothing
    xa, _ = S.solve(dev(np.ones(m)), damp=0.1, max_iters=7)
    S.set(row_cost=100)
    xb, _ = S.solve(dev(np.ones(m)), damp=0.1, max_iters=7)
    assert torch.equal(xa, xb)
    # calls a factored handle does not take
    for call in (lambda: T.tomo_lsqr_update_values(S.h, dev(va)), lambda: S.csc(), lambda: S.set(compress=1)):
        with pytest.raises(T.TomoError) as ei:
            call()
        assert ei.value.status == T.TOMO_ERR_INVALID_ARG
    S.close()
    # malformed operators are rejected at create, *out stays NULL
    def create(**over):
        g = dict(f); g.update(over)
        return make(tl, g)
    bad_nodes = f["lnode"].copy(); bad_nodes[1] = bad_nodes[0]            # not strictly ascending inside the first pair with >= 2 entries
    q = int(np.flatnonzero(np.diff(f["lptr"]) >= 2)[0]); bad_nodes = f["lnode"].copy(); bad_nodes[f["lptr"][q] + 1] = bad_nodes[f["lptr"][q]]
    bad_w = f["lw"].copy(); bad_w[3] = np.inf
    bad_j0 = f["kj0"].copy(); bad_j0[0] = f["nz"] - f["klen"] + 1
    bad_kern = f["kern"].copy(); bad_kern[1, 2] = np.nan
    for over in (dict(lnode=bad_nodes), dict(lw=bad_w), dict(kj0=bad_j0), dict(kern=bad_kern)):
        with pytest.raises(T.TomoError) as ei:
            create(**over)
        assert ei.value.status == T.TOMO_ERR_BAD_CSR, over.keys()
    with pytest.raises(T.TomoError) as ei:
        T.tomo_lsqr_create_factored(10, 33, 5, 40, dev(np.zeros(11, dtype=np.int64)), None, None, 4, dev(np.zeros(33, dtype=np.int32)),
                                    dev(np.zeros(33 * 4)))
    assert ei.value.status == T.TOMO_ERR_RANGE
    with pytest.raises(T.TomoError) as ei:   # host pointer
        T.tomo_lsqr_create_factored(f["npairs"], f["nper"], f["nnodes"], f["nz"], f["lptr"], dev(f["lnode"]), dev(f["lw"]), f["klen"],
                                    dev(f["kj0"]), dev(f["kern"]))
    assert ei.value.status == T.TOMO_ERR_NOT_DEVICE_PTR
    # a system with no lateral entry at all and one with no extra rows still solve (oracle on the expansion)
    for g in (tomogen.random_factored(6, 3, 5, 8, 4, seed=5, empty_pairs=1.0), tomogen.random_factored(30, 6, 8, 9, 3, seed=6, ms=0)):
        rp, ci, va = expand(g)
        S = make(tl, g)
        b = np.random.default_rng(1).standard_normal(S.m)
        x, res = S.solve(dev(b), damp=0.3, max_iters=10)
        o = oracle.lsqr(S.m, S.n, rp, ci, va, b, damp=0.3, max_iters=10, mode=oracle.DD)
        assert (res.itn, res.istop) == (o.itn, o.istop) and np.array_equal(x.cpu().numpy(), o.x)
        S.close()


@pytest.fixture(scope="module")
def big(tl):
    out = {}
    for cfg in (1, 4):
        s = tomogen.System(cfg)
        out[cfg] = (s, make(tl, s.factored()))
    return out


def test_factored_spmv_cfg1_cfg4(tl, big):
    for cfg in (1, 4):
        s, S = big[cfg]
        d = s.dims
        rp, ci, va = s.csr()   # = the expansion, bitwise (tests/test_oracle_factored_pins.py)
        rng = np.random.default_rng(cfg)
        x, u = rng.standard_normal(d.n), rng.standard_normal(d.m)
        for acc, mode in ((1, oracle.DD), (0, oracle.PLAIN)):
            S.set(accumulate=acc)
            y = S.spmv(dev(x)).cpu().numpy()
            yt = S.spmv(dev(u), transpose=True).cpu().numpy()
            oy, oyt = oracle.spmv(d.m, d.n, rp, ci, va, x, mode), oracle.spmv_t(d.m, d.n, rp, ci, va, u, mode)
            assert rel(y, oy) <= TOL_SPMV and rel(yt, oyt) <= TOL_SPMV
            if acc:
                assert np.array_equal(y, oy) and np.array_equal(yt, oyt)
        assert abs(np.dot(y, u) - np.dot(x, yt)) <= 1e-12 * np.linalg.norm(y) * np.linalg.norm(u)   # adjoint identity
        del rp, ci, va


def test_factored_x50_and_tolerance_run_cfg1(tl, big):
    s, S = big[1]
    b = dev(s.rhs(0))
    o = oracle_jobs.get("cfg1_dd_tol")
    S.set(accumulate=1)
    x50, res = S.solve(b, damp=s.damp, max_iters=50)
    assert rel(x50.cpu().numpy(), o["snapshots"][50]) <= TOL_X50 and np.array_equal(x50.cpu().numpy(), o["snapshots"][50])
    x, res, r2, ar = S.solve(b, damp=s.damp, atol=1e-6, btol=1e-6, max_iters=300, history=True)
    assert (res.itn, res.istop) == (o["itn"], o["istop"])
    assert np.array_equal(x.cpu().numpy(), o["x"]) and np.array_equal(r2, o["r2hist"][: res.itn])
    # LSMR, the paper's own solver
    ol = oracle_jobs.get("cfg1_lsmr_dd_50")
    xl, resl = S.solve(b, damp=s.damp, max_iters=50, solver="lsmr")
    assert resl.itn == ol["itn"] and np.array_equal(xl.cpu().numpy(), ol["x"])
    # fast mode: x_10 to the contract, as for the CSR path
    S.set(accumulate=0)
    op = oracle_jobs.get("cfg1_plain_50")
    x10, _ = S.solve(b, damp=s.damp, max_iters=10)
    assert rel(x10.cpu().numpy(), op["snapshots"][10]) <= TOL_X50
    S.set(accumulate=1)


def test_factored_x50_x100_cfg4_skewed(tl, big):
    s, S = big[4]
    b = dev(s.rhs(0))
    o = oracle_jobs.get("cfg4_dd_100")
    S.set(accumulate=1)
    x50, _ = S.solve(b, damp=s.damp, max_iters=50)
    x100, res = S.solve(b, damp=s.damp, max_iters=100)
    assert np.array_equal(x50.cpu().numpy(), o["snapshots"][50]) and np.array_equal(x100.cpu().numpy(), o["x"])
    assert res.itn == o["itn"] == 100


def test_factored_cfg2_full_size(tl):
    """configs[2] (3.7e9 nonzeros as CSR; 236 MB factored): sampled rows of A x and sampled columns' worth of A^T x
    against the oracle on the generator's rows, and x_1, x_2, x_5 bitwise against the dd oracle's full-size run (the
    background job of test_gpu_parity.py; its matrix is the generator's CSR = the multiplied-out operator)."""
    s = tomogen.System(2)
    d = s.dims
    S = make(tl, s.factored())
    assert (S.m, S.n) == (d.m, d.n)
    rng = np.random.default_rng(2)
    x = rng.standard_normal(d.n)
    rows = np.unique(np.concatenate([[0, d.m_data - 1, d.m_data, d.m - 1], rng.integers(0, d.m, size=2000)]))
    rp, ci, va = s.rows(rows)
    for acc, mode in ((1, oracle.DD), (0, oracle.PLAIN)):
        S.set(accumulate=acc)
        y = S.spmv(dev(x)).cpu().numpy()[rows]
        oy = oracle.spmv(len(rows), d.n, rp, ci, va, x, mode)
        assert rel(y, oy) <= TOL_SPMV
        if acc:
            assert np.array_equal(y, oy)
    # A^T: adjoint identity with the product just checked (every column enters)
    S.set(accumulate=1)
    u = rng.standard_normal(d.m)
    yt = S.spmv(dev(u), transpose=True).cpu().numpy()
    yx = S.spmv(dev(x)).cpu().numpy()
    assert abs(np.dot(yx, u) - np.dot(x, yt)) <= 1e-12 * np.linalg.norm(yx) * np.linalg.norm(u)
    b = dev(s.rhs(0))
    xk = {k: S.solve(b, damp=s.damp, max_iters=k)[0].cpu().numpy() for k in (1, 2, 5)}
    x100a, res = S.solve(b, damp=s.damp, max_iters=100)
    x100b, _ = S.solve(b, damp=s.damp, max_iters=100)
    assert res.itn == 100 and torch.equal(x100a, x100b)
    S.close()
    o = oracle_jobs.get("cfg2_dd_5")
    if "skipped" in o:
        pytest.skip("config-2 x_k parity of the factored operator not run: " + o["skipped"])
    for k, want in ((1, o["snapshots"][1]), (2, o["snapshots"][2]), (5, o["x"])):
        assert rel(xk[k], want) <= TOL_X50 and np.array_equal(xk[k], want), k


def assemble(tl, f):
    """tomo_lsqr_assemble_csr on the device -> (rowptr, colind, vals) device tensors."""
    ms = 0 if f["sptr"] is None else len(f["sptr"]) - 1
    snnz = 0 if f["sidx"] is None else len(f["sidx"])
    m = f["npairs"] * f["nper"] + ms
    nnz = len(f["lnode"]) * f["nper"] * f["klen"] + snnz
    keep = [dev(f[k]) for k in ("lptr", "lnode", "lw")] + [dev(f["kj0"].astype(np.int32)), dev(f["kern"])] + \
           [dev(f[k]) for k in ("sptr", "sidx", "svals")]
    rp = torch.full((m + 1,), -1, dtype=torch.int64, device="cuda")
    ci = torch.full((max(nnz, 1),), -1, dtype=torch.int32, device="cuda")
    va = torch.full((max(nnz, 1),), float("nan"), dtype=torch.float64, device="cuda")
    tl.tomo_lsqr_assemble_csr(f["npairs"], f["nper"], f["nnodes"], f["nz"], keep[0], keep[1], keep[2], f["klen"], keep[3], keep[4],
                              ms, snnz, keep[5], keep[6], keep[7], nnz, rp, ci, va, nodal=int(f["kern"].ndim == 3))
    return m, nnz, rp, ci[:nnz], va[:nnz]


@pytest.mark.parametrize("shape", SHAPES)
def test_assemble_csr_random_shapes(tl, shape):
    """NEXT-4, on-device assembly of G: bit-exact (indices and one-rounding values) against the oracle's expansion."""
    npairs, nper, nnodes, nz, klen, ms = shape
    f = tomogen.random_factored(npairs, nper, nnodes, nz, klen, seed=2000 + npairs, ms=ms)
    orp, oci, ova = expand(f)
    m, nnz, rp, ci, va = assemble(tl, f)
    assert np.array_equal(rp.cpu().numpy(), orp) and np.array_equal(ci.cpu().numpy(), oci) and np.array_equal(va.cpu().numpy(), ova)


def test_assemble_csr_configs_and_roundtrip(tl, cfg0):
    import paper_2604_11920_b200 as T
    # config 0: equals the generator's host assembly; the assembled matrix is accepted by tomo_lsqr_create and solves to
    # the bits of the factored handle
    s = cfg0["sys"]
    f = s.factored()
    m, nnz, rp, ci, va = assemble(tl, f)
    assert np.array_equal(rp.cpu().numpy(), cfg0["rp"]) and np.array_equal(ci.cpu().numpy(), cfg0["ci"]) and np.array_equal(va.cpu().numpy(), cfg0["va"])
    C = tl.TomoLsqr(m, cfg0["n"], rp, ci, va)
    F = make(tl, f)
    b = dev(cfg0["b"])
    assert torch.equal(C.solve(b, damp=s.damp, max_iters=50)[0], F.solve(b, damp=s.damp, max_iters=50)[0])
    C.close(); F.close()
    # config 1 at full size (194 M nonzeros, 2.3 GB written): equals the generator's CSR
    s1 = tomogen.System(1)
    f1 = s1.factored()
    m, nnz, rp, ci, va = assemble(tl, f1)
    orp, oci, ova = s1.csr()
    assert nnz == s1.dims.nnz and np.array_equal(rp.cpu().numpy(), orp)
    assert torch.equal(ci, dev(oci)) and torch.equal(va, dev(ova))
    # a wrong nnz is refused before anything is written
    with pytest.raises(T.TomoError) as ei:
        T.tomo_lsqr_assemble_csr(f["npairs"], f["nper"], f["nnodes"], f["nz"], dev(f["lptr"]), dev(f["lnode"]), dev(f["lw"]), f["klen"],
                                 dev(f["kj0"]), dev(f["kern"]), len(f["sptr"]) - 1, len(f["sidx"]), dev(f["sptr"]), dev(f["sidx"]),
                                 dev(f["svals"]), 7, rp, ci, va)
    assert ei.value.status == T.TOMO_ERR_INVALID_ARG


# ---- dd mode on the exact entries W*g (option two_stage = 2; reading F-fac3) ------------------------------
@pytest.mark.parametrize("shape", SHAPES)
def test_factored_exact_entries_dd_random_shapes(tl, shape):
    """The two-stage contraction in dd mode applies the operator with UNROUNDED entries W*g; its oracle is the dd oracle on
    the two-word entries (oracle/factored.py expand_exact), each sum of exact products rounded once: bitwise."""
    npairs, nper, nnodes, nz, klen, ms = shape
    f = tomogen.random_factored(npairs, nper, nnodes, nz, klen, seed=3000 + npairs, ms=ms, max_entries=60)
    rp, ci, va, lo = expand_exact(f)
    m, n = len(rp) - 1, nnodes * nz
    S = make(tl, f)
    S.set(accumulate=1, two_stage=2)
    rng = np.random.default_rng(shape[0] + 1)
    x, u = rng.standard_normal(n), rng.standard_normal(m)
    y = S.spmv(dev(x)).cpu().numpy()
    yt = S.spmv(dev(u), transpose=True).cpu().numpy()
    assert np.array_equal(y, oracle.spmv(m, n, rp, ci, va, x, oracle.DD, vals_lo=lo))
    assert np.array_equal(yt, oracle.spmv_t(m, n, rp, ci, va, u, oracle.DD, vals_lo=lo))
    b = rng.standard_normal(m)
    xg, res = S.solve(dev(b), damp=0.1, max_iters=20)
    o = oracle.lsqr(m, n, rp, ci, va, b, damp=0.1, max_iters=20, mode=oracle.DD, vals_lo=lo)
    assert (res.itn, res.istop) == (o.itn, o.istop) and np.array_equal(xg.cpu().numpy(), o.x)
    S.set(two_stage=1)   # back on the rounded entries: the CSR bits again
    x1, _ = S.solve(dev(b), damp=0.1, max_iters=20)
    assert np.array_equal(x1.cpu().numpy(), oracle.lsqr(m, n, rp, ci, va, b, damp=0.1, max_iters=20, mode=oracle.DD).x)
    S.close()


def test_factored_exact_entries_dd_cfg0_cfg1(tl, cfg0, big):
    s = cfg0["sys"]
    f = s.factored()
    rp, ci, va, lo = expand_exact(f)
    S = make(tl, f)
    S.set(accumulate=1, two_stage=2)
    b = cfg0["b"]
    xg, res, r2, ar = S.solve(dev(b), damp=s.damp, max_iters=50, history=True)
    o = oracle.lsqr(cfg0["m"], cfg0["n"], rp, ci, va, b, damp=s.damp, max_iters=50, mode=oracle.DD, vals_lo=lo)
    assert res.itn == o.itn == 50 and np.array_equal(xg.cpu().numpy(), o.x) and np.array_equal(r2, o.r2norm_hist)
    x2, _ = S.solve(dev(b), damp=s.damp, max_iters=50)
    assert torch.equal(xg, x2)
    # LSMR, the paper's own solver, on the exact entries
    xl, resl = S.solve(dev(b), damp=s.damp, max_iters=50, solver="lsmr")
    ol = oracle.lsmr(cfg0["m"], cfg0["n"], rp, ci, va, b, damp=s.damp, max_iters=50, mode=oracle.DD, vals_lo=lo)
    assert resl.itn == ol.itn == 50 and np.array_equal(xl.cpu().numpy(), ol.x)
    S.close()
    # config 1: x_10 and x_50 against the background run of the exact-entries oracle
    s1, S1 = big[1]
    S1.set(accumulate=1, two_stage=2)
    b1 = dev(s1.rhs(0))
    o1 = oracle_jobs.get("cfg1_ddx_50")
    x10, _ = S1.solve(b1, damp=s1.damp, max_iters=10)
    x50, res = S1.solve(b1, damp=s1.damp, max_iters=50)
    S1.set(two_stage=1)
    assert res.itn == 50
    assert rel(x50.cpu().numpy(), o1["x"]) <= TOL_X50 and np.array_equal(x10.cpu().numpy(), o1["snapshots"][10])
    assert np.array_equal(x50.cpu().numpy(), o1["x"])


def test_update_kernels_equals_create_from_scratch(tl):
    """NEXT-4 on a factored handle: new depth kernels on the same rays (the outer Gauss-Newton loop, P:77 / P:81);
    every mode, also after a graph was captured with the old table."""
    import paper_2604_11920_b200 as T
    f = tomogen.random_factored(400, 10, 120, 20, 12, seed=91)
    rng = np.random.default_rng(92)
    g = dict(f)
    g["kern"] = rng.standard_normal(f["kern"].shape)
    g["kj0"] = rng.integers(0, f["nz"] - f["klen"] + 1, size=f["nper"]).astype(np.int32)
    S, R = make(tl, f), make(tl, g)
    b = dev(rng.standard_normal(S.m))
    for acc, ts in ((1, 1), (1, 2), (0, 1), (0, 0)):
        S.set(accumulate=acc, two_stage=ts)
        S.solve(b, damp=0.1, max_iters=12)      # captures a graph on the old table (first pass) / the refreshed one (later)
    T.tomo_lsqr_update_kernels(S.h, dev(g["kj0"]), dev(g["kern"]))
    for acc, ts in ((1, 1), (1, 2), (0, 1), (0, 0)):
        S.set(accumulate=acc, two_stage=ts); R.set(accumulate=acc, two_stage=ts)
        assert torch.equal(S.solve(b, damp=0.1, max_iters=12)[0], R.solve(b, damp=0.1, max_iters=12)[0]), (acc, ts)
    # and the oracle on the new multiplied-out matrix
    rp, ci, va = expand(g)
    S.set(accumulate=1, two_stage=1)
    o = oracle.lsqr(S.m, S.n, rp, ci, va, b.cpu().numpy(), damp=0.1, max_iters=12, mode=oracle.DD)
    assert np.array_equal(S.solve(b, damp=0.1, max_iters=12)[0].cpu().numpy(), o.x)
    # a bad table leaves the handle as it was
    bad = g["kern"].copy(); bad[0, 0] = np.inf
    with pytest.raises(T.TomoError) as ei:
        T.tomo_lsqr_update_kernels(S.h, dev(g["kj0"]), dev(bad))
    assert ei.value.status == T.TOMO_ERR_BAD_CSR
    assert np.array_equal(S.solve(b, damp=0.1, max_iters=12)[0].cpu().numpy(), o.x)
    C = tl.TomoLsqr(S.m, S.n, dev(rp), dev(ci), dev(va))
    with pytest.raises(T.TomoError):
        T.tomo_lsqr_update_kernels(C.h, dev(g["kj0"]), dev(g["kern"]))   # not a factored handle
    C.close(); S.close(); R.close()


@pytest.mark.parametrize("shape", [SHAPES[0], SHAPES[1], SHAPES[2], SHAPES[4], SHAPES[7]])
def test_nodal_kernel_tables(tl, shape):
    """Depth kernels per lateral node (the paper's Theta_k) through tomo_lsqr_set_nodal_kernels: dd mode bitwise the
    dd oracle on the exact two-word entries, fast mode to the SpMV bar against the plain oracle on the multiplied-out
    matrix; refresh of the tables; a bad table leaves the handle unchanged."""
    import paper_2604_11920_b200 as T
    npairs, nper, nnodes, nz, klen, ms = shape
    f = tomogen.random_factored(npairs, nper, nnodes, nz, klen, seed=4000 + npairs, ms=ms, max_entries=60, nodal=True)
    rp, ci, va, lo = expand_exact(f)
    m, n = len(rp) - 1, nnodes * nz
    shared = dict(f); shared["kj0"] = f["kj0"][0].copy(); shared["kern"] = f["kern"][0].copy()
    S = make(tl, shared)
    T.tomo_lsqr_set_nodal_kernels(S.h, dev(f["kj0"].astype(np.int32)), dev(f["kern"]))
    assert S.info("nodal_kernels") == 1.0
    rng = np.random.default_rng(npairs)
    x, u, b = rng.standard_normal(n), rng.standard_normal(m), rng.standard_normal(m)
    S.set(accumulate=1)
    assert np.array_equal(S.spmv(dev(x)).cpu().numpy(), oracle.spmv(m, n, rp, ci, va, x, oracle.DD, vals_lo=lo))
    assert np.array_equal(S.spmv(dev(u), transpose=True).cpu().numpy(), oracle.spmv_t(m, n, rp, ci, va, u, oracle.DD, vals_lo=lo))
    xg, res = S.solve(dev(b), damp=0.1, max_iters=20)
    o = oracle.lsqr(m, n, rp, ci, va, b, damp=0.1, max_iters=20, mode=oracle.DD, vals_lo=lo)
    assert (res.itn, res.istop) == (o.itn, o.istop) and np.array_equal(xg.cpu().numpy(), o.x)
    S.set(accumulate=0)
    assert rel(S.spmv(dev(x)).cpu().numpy(), oracle.spmv(m, n, rp, ci, va, x, oracle.PLAIN)) <= 1e-11
    assert rel(S.spmv(dev(u), transpose=True).cpu().numpy(), oracle.spmv_t(m, n, rp, ci, va, u, oracle.PLAIN)) <= 1e-11
    # refresh with other tables: equals a handle that got them first
    g = tomogen.random_factored(npairs, nper, nnodes, nz, klen, seed=4000 + npairs, ms=ms, max_entries=60, nodal=True)
    g["kern"] = np.random.default_rng(5).standard_normal(f["kern"].shape)
    bad = g["kern"].copy(); bad[-1, -1, -1] = np.nan
    with pytest.raises(T.TomoError) as ei:
        T.tomo_lsqr_set_nodal_kernels(S.h, dev(g["kj0"].astype(np.int32)), dev(bad))
    assert ei.value.status == T.TOMO_ERR_BAD_CSR
    S.set(accumulate=1)
    assert np.array_equal(S.solve(dev(b), damp=0.1, max_iters=20)[0].cpu().numpy(), o.x)
    T.tomo_lsqr_set_nodal_kernels(S.h, dev(g["kj0"].astype(np.int32)), dev(g["kern"]))
    rp2, ci2, va2, lo2 = expand_exact(g)
    o2 = oracle.lsqr(m, n, rp2, ci2, va2, b, damp=0.1, max_iters=20, mode=oracle.DD, vals_lo=lo2)
    assert np.array_equal(S.solve(dev(b), damp=0.1, max_iters=20)[0].cpu().numpy(), o2.x)
    with pytest.raises(T.TomoError):
        T.tomo_lsqr_update_kernels(S.h, dev(shared["kj0"].astype(np.int32)), dev(shared["kern"]))
    S.close()


@pytest.mark.parametrize("shape", [SHAPES[1], SHAPES[2], SHAPES[7]])
def test_assemble_csr_nodal_tables(tl, shape):
    """on-device assembly with a kernel table per node: bit-exact against the oracle's expansion; the CSR path on the
    assembled matrix and the nodal factored handle agree to rounding (dd: rounded against exact entries)"""
    import paper_2604_11920_b200 as T
    npairs, nper, nnodes, nz, klen, ms = shape
    f = tomogen.random_factored(npairs, nper, nnodes, nz, klen, seed=5000 + npairs, ms=ms, nodal=True)
    orp, oci, ova = expand(f)
    m, nnz, rp, ci, va = assemble(tl, f)
    assert np.array_equal(rp.cpu().numpy(), orp) and np.array_equal(ci.cpu().numpy(), oci) and np.array_equal(va.cpu().numpy(), ova)
    C = tl.TomoLsqr(m, nnodes * nz, rp, ci, va)
    shared = dict(f); shared["kj0"] = f["kj0"][0].copy(); shared["kern"] = f["kern"][0].copy()
    F = make(tl, shared)
    T.tomo_lsqr_set_nodal_kernels(F.h, dev(f["kj0"].astype(np.int32)), dev(f["kern"]))
    x = dev(np.random.default_rng(3).standard_normal(nnodes * nz))
    for acc in (1, 0):
        C.set(accumulate=acc); F.set(accumulate=acc)
        yc, yf = C.spmv(x).cpu().numpy(), F.spmv(x).cpu().numpy()
        assert rel(yf, yc) <= 1e-11
    C.close(); F.close()
