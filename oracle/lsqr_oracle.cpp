// oracle/lsqr_oracle.cpp — TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, slow, single-threaded fp64 CPU implementation of the hot path of this repository: the damped
// sparse least-squares solve  min ||A x - b||^2 + damp^2 ||x||^2  by LSQR (Golub-Kahan
// bidiagonalisation; Paige & Saunders 1982, the reference the paper names at PAPER.md:142 and lists at
// PAPER.md:268) for the system  Delta d = G Delta m  of PAPER.md Eq. 6.  Only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call it; it shares
// no code, header, table or data layout with the CUDA path (A^T u is a scatter over CSR rows here, the
// CUDA path gathers over a CSC copy).
//
// LSQR is an iteration, so the oracle IS the algorithm, step by step, in the order and notation of
// SURVEY.md §8(c) / DESIGN.md "Oracle" (Paige & Saunders' Algorithm LSQR with the standard second
// rotation for damping).  No blocking, fusion or reordering.  Compile with -ffp-contract=off: a fused
// multiply-add appears only where std::fma is written.
//
// Accumulation modes (reading R-dd; needed because fixed-k iterates are summation-order
// sensitive beyond toy size):
//   mode 0 "plain": every inner product is a left-to-right fp64 loop, s = fma(a, b, s).
//   mode 1 "dd"   : every inner product (row sums of A v including the -alpha*u_i term, column sums of
//                   A^T u including -beta*v_j, the norms, sum (w_j/rho)^2) is accumulated as an
//                   unevaluated double-double (hi, lo) and rounded to fp64 once => the result is the
//                   correctly rounded exact sum (up to ~1e-10-probability ties), independent of order.
// x, w updates, normalisations and all scalars are identical in both modes.
//
// Pins (tests/test_oracle_*.py, -m "not gpu"): dense normal equations and QR on tiny systems, adjoint
// identity, closed form of x_1, finite termination on diagonal systems, exact recovery, monotone
// ||r||, estimate identities against directly computed norms, scipy.sparse.linalg.lsqr, dd-mode
// permutation invariance, brute-force long-double SpMV.  No function here is "parity unpinned".
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>

namespace {

// ---- double-double primitives (Knuth TwoSum, fma TwoProd, Dekker FastTwoSum) -------------------------
struct dd { double hi, lo; };

inline void two_sum(double a, double b, double& s, double& t) {
  s = a + b;
  double bb = s - a;
  t = (a - (s - bb)) + (b - bb);
}
inline void two_prod(double a, double b, double& p, double& e) {
  p = a * b;
  e = std::fma(a, b, -p);
}
// acc <- acc + a*b   (per term: TwoProd, TwoSum(hi, p), t += lo + e, FastTwoSum)
inline void dd_fma(dd& acc, double a, double b) {
  double p, e, s, t;
  two_prod(a, b, p, e);
  two_sum(acc.hi, p, s, t);
  t = t + (acc.lo + e);
  acc.hi = s + t;
  acc.lo = t - (acc.hi - s);
}
inline double dd_round(const dd& a) { return a.hi + a.lo; }

struct Csr {
  int64_t m, n;
  const int64_t* rowptr;
  const int32_t* colind;
  const double* vals;
  // optional second word of every entry: the entry is the unevaluated sum vals[e] + vals_lo[e] (the factored
  // operator with exact entries W*g, reading F-fac3: vals = fl(W g), vals_lo = W g - fl(W g) exactly).
  // Used in dd mode only (the entry's two words are two exact products); NULL: the entry is vals[e].
  const double* vals_lo = nullptr;
};

// y_i = sum_j a_ij x_j + c * y_i   (c = 0: plain product; c = -alpha: the LSQR u-update)
void spmv(const Csr& A, const double* x, double c, double* y, int mode) {
  for (int64_t i = 0; i < A.m; ++i) {
    if (mode == 0) {
      double s = 0.0;
      for (int64_t e = A.rowptr[i]; e < A.rowptr[i + 1]; ++e) s = std::fma(A.vals[e], x[A.colind[e]], s);
      y[i] = (c == 0.0) ? s : std::fma(c, y[i], s);
    } else {
      dd acc{0.0, 0.0};
      if (c != 0.0) dd_fma(acc, c, y[i]);
      for (int64_t e = A.rowptr[i]; e < A.rowptr[i + 1]; ++e) {
        dd_fma(acc, A.vals[e], x[A.colind[e]]);
        if (A.vals_lo) dd_fma(acc, A.vals_lo[e], x[A.colind[e]]);
      }
      y[i] = dd_round(acc);
    }
  }
}

// v_j = sum_i a_ij u_i + c * v_j   as a scatter over the rows of A (no transposed copy)
void spmv_t(const Csr& A, const double* u, double c, double* v, int mode, std::vector<dd>& work) {
  if (mode == 0) {
    for (int64_t j = 0; j < A.n; ++j) v[j] = (c == 0.0) ? 0.0 : c * v[j];
    for (int64_t i = 0; i < A.m; ++i) {
      double ui = u[i];
      for (int64_t e = A.rowptr[i]; e < A.rowptr[i + 1]; ++e) v[A.colind[e]] = std::fma(A.vals[e], ui, v[A.colind[e]]);
    }
  } else {
    work.assign((size_t)A.n, dd{0.0, 0.0});
    if (c != 0.0) for (int64_t j = 0; j < A.n; ++j) dd_fma(work[j], c, v[j]);
    for (int64_t i = 0; i < A.m; ++i) {
      double ui = u[i];
      for (int64_t e = A.rowptr[i]; e < A.rowptr[i + 1]; ++e) {
        dd_fma(work[A.colind[e]], A.vals[e], ui);
        if (A.vals_lo) dd_fma(work[A.colind[e]], A.vals_lo[e], ui);
      }
    }
    for (int64_t j = 0; j < A.n; ++j) v[j] = dd_round(work[j]);
  }
}

double sumsq(const double* z, int64_t len, int mode) {
  if (mode == 0) {
    double s = 0.0;
    for (int64_t i = 0; i < len; ++i) s = std::fma(z[i], z[i], s);
    return s;
  }
  dd acc{0.0, 0.0};
  for (int64_t i = 0; i < len; ++i) dd_fma(acc, z[i], z[i]);
  return dd_round(acc);
}

struct Lsqr {
  Csr A;
  int mode;
  double damp, atol, btol;
  int32_t max_iters;
  std::vector<double> u, v, w, x;
  std::vector<dd> work;
  // scalars, Paige & Saunders' names
  double alpha = 0, beta = 0, rhobar = 0, phibar = 0, bnorm = 0;
  double anorm = 0, ddnorm = 0, res2 = 0, xxnorm = 0, z = 0, cs2 = -1, sn2 = 0;
  double acond = 0, rnorm = 0, arnorm = 0, xnorm = 0, r1norm = 0, r2norm = 0;
  int32_t itn = 0, istop = 0;
  bool done = false;

  void init(const double* b) {
    u.assign(b, b + A.m);
    v.assign((size_t)A.n, 0.0); w.assign((size_t)A.n, 0.0); x.assign((size_t)A.n, 0.0);
    beta = std::sqrt(sumsq(u.data(), A.m, mode));
    bnorm = beta;
    if (beta == 0.0) { done = true; istop = 0; return; }
    double rb = 1.0 / beta;
    for (int64_t i = 0; i < A.m; ++i) u[i] = u[i] * rb;
    spmv_t(A, u.data(), 0.0, v.data(), mode, work);
    alpha = std::sqrt(sumsq(v.data(), A.n, mode));
    rnorm = r1norm = r2norm = bnorm;
    if (alpha == 0.0) { done = true; istop = 0; return; }
    double ra = 1.0 / alpha;
    for (int64_t j = 0; j < A.n; ++j) v[j] = v[j] * ra;
    w = v;
    rhobar = alpha; phibar = beta;
    arnorm = alpha * beta;
    if (max_iters <= 0) { done = true; istop = 7; }
  }

  // one LSQR iteration; returns istop (0 = continue)
  int32_t step() {
    if (done) return istop;
    ++itn;
    // bidiagonalisation: beta*u = A v - alpha*u ; alpha*v = A^T u - beta*v
    spmv(A, v.data(), -alpha, u.data(), mode);
    beta = std::sqrt(sumsq(u.data(), A.m, mode));
    if (beta > 0.0) {
      double rb = 1.0 / beta;
      for (int64_t i = 0; i < A.m; ++i) u[i] = u[i] * rb;
      anorm = std::sqrt(anorm * anorm + alpha * alpha + beta * beta + damp * damp);
      spmv_t(A, u.data(), -beta, v.data(), mode, work);
      alpha = std::sqrt(sumsq(v.data(), A.n, mode));
      if (alpha > 0.0) {
        double ra = 1.0 / alpha;
        for (int64_t j = 0; j < A.n; ++j) v[j] = v[j] * ra;
      }
    }
    // damping rotation
    double rhobar1 = std::sqrt(rhobar * rhobar + damp * damp);
    double cs1 = rhobar / rhobar1, sn1 = damp / rhobar1;
    double psi = sn1 * phibar;
    phibar = cs1 * phibar;
    // plane rotation eliminating beta
    double rho = std::sqrt(rhobar1 * rhobar1 + beta * beta);
    double cs = rhobar1 / rho, sn = beta / rho;
    double theta = sn * alpha;
    rhobar = -cs * alpha;
    double phi = cs * phibar;
    phibar = sn * phibar;
    double tau = sn * phi;
    // update x and w; ddnorm uses the old w
    double t1 = phi / rho, t2 = -theta / rho, rrho = 1.0 / rho;
    {
      double s;
      if (mode == 0) {
        s = 0.0;
        for (int64_t j = 0; j < A.n; ++j) { double d = w[j] * rrho; s = std::fma(d, d, s); }
      } else {
        dd acc{0.0, 0.0};
        for (int64_t j = 0; j < A.n; ++j) { double d = w[j] * rrho; dd_fma(acc, d, d); }
        s = dd_round(acc);
      }
      ddnorm = ddnorm + s;
    }
    for (int64_t j = 0; j < A.n; ++j) {
      double wj = w[j];
      x[j] = std::fma(t1, wj, x[j]);
      w[j] = std::fma(t2, wj, v[j]);
    }
    // norm estimates
    double delta = sn2 * rho, gambar = -cs2 * rho, rhs = phi - delta * z, zbar = rhs / gambar;
    xnorm = std::sqrt(xxnorm + zbar * zbar);
    double gamma = std::sqrt(gambar * gambar + theta * theta);
    cs2 = gambar / gamma; sn2 = theta / gamma; z = rhs / gamma;
    xxnorm = xxnorm + z * z;
    acond = anorm * std::sqrt(ddnorm);
    res2 = res2 + psi * psi;
    rnorm = std::sqrt(phibar * phibar + res2);
    arnorm = alpha * std::fabs(tau);
    r2norm = rnorm;
    {
      double r1sq = r2norm * r2norm - damp * damp * (xnorm * xnorm);
      r1norm = std::sqrt(r1sq > 0.0 ? r1sq : 0.0);
    }
    // stopping tests (conlim disabled: ctol = 0)
    double test1 = rnorm / bnorm;
    double den2 = anorm * rnorm;
    double test2 = den2 > 0.0 ? arnorm / den2 : 0.0;
    double test3 = acond > 0.0 ? 1.0 / acond : INFINITY;
    double ax = anorm * xnorm / bnorm;
    double tt1 = test1 / (1.0 + ax);
    double rtol = btol + atol * ax;
    istop = 0;
    if (itn >= max_iters) istop = 7;
    if (1.0 + test3 <= 1.0) istop = 6;
    if (1.0 + test2 <= 1.0) istop = 5;
    if (1.0 + tt1 <= 1.0) istop = 4;
    if (test3 <= 0.0) istop = 3;
    if (test2 <= atol) istop = 2;
    if (test1 <= rtol) istop = 1;
    if (istop != 0) done = true;
    return istop;
  }
};


// ---- LSMR (Fong & Saunders 2011): the solver the paper itself uses (ref. PAPER.md:249) ----
// Same Golub-Kahan steps as LSQR; the solution is updated through h, hbar so that ||A^T r|| decreases
// monotonically.  Step by step as published (damping by the extra rotation Qhat), inner products in the
// same two accumulation modes; the vector updates are single fused multiply-adds.  NEXT-1 of SURVEY.md.

// stable Givens rotation: [c s; -s c] [a; b] = [r; 0]
inline void sym_ortho(double a, double b, double& c, double& s, double& r) {
  if (b == 0.0) { c = (a > 0.0) - (a < 0.0); s = 0.0; r = std::fabs(a); }
  else if (a == 0.0) { c = 0.0; s = (b > 0.0) - (b < 0.0); r = std::fabs(b); }
  else if (std::fabs(b) > std::fabs(a)) {
    double tau = a / b;
    s = ((b > 0.0) ? 1.0 : -1.0) / std::sqrt(1.0 + tau * tau);
    c = s * tau; r = b / s;
  } else {
    double tau = b / a;
    c = ((a > 0.0) ? 1.0 : -1.0) / std::sqrt(1.0 + tau * tau);
    s = c * tau; r = a / c;
  }
}

struct Lsmr {
  Csr A;
  int mode;
  double damp, atol, btol;
  int32_t max_iters;
  std::vector<double> u, v, h, hbar, x;
  std::vector<dd> work;
  double alpha = 0, beta = 0, normb = 0;
  double zetabar = 0, alphabar = 0, rho = 1, rhobar = 1, cbar = 1, sbar = 0;
  double betadd = 0, betad = 0, rhodold = 1, tautildeold = 0, thetatilde = 0, zeta = 0, d = 0;
  double normA2 = 0, maxrbar = 0, minrbar = 1e100;
  double normA = 0, condA = 1, normx = 0, normr = 0, normar = 0;
  int32_t itn = 0, istop = 0;
  bool done = false;

  void init(const double* b) {
    u.assign(b, b + A.m);
    v.assign((size_t)A.n, 0.0); h.assign((size_t)A.n, 0.0); hbar.assign((size_t)A.n, 0.0); x.assign((size_t)A.n, 0.0);
    beta = std::sqrt(sumsq(u.data(), A.m, mode));
    normb = beta; normr = beta;
    if (beta == 0.0) { done = true; istop = 0; return; }
    double rb = 1.0 / beta;
    for (int64_t i = 0; i < A.m; ++i) u[i] = u[i] * rb;
    spmv_t(A, u.data(), 0.0, v.data(), mode, work);
    alpha = std::sqrt(sumsq(v.data(), A.n, mode));
    normar = alpha * beta;
    if (alpha == 0.0) { done = true; istop = 0; return; }
    double ra = 1.0 / alpha;
    for (int64_t j = 0; j < A.n; ++j) v[j] = v[j] * ra;
    h = v;
    zetabar = alpha * beta; alphabar = alpha;
    betadd = beta;
    normA2 = alpha * alpha; normA = std::sqrt(normA2);
    if (max_iters <= 0) { done = true; istop = 7; }
  }

  int32_t step() {
    if (done) return istop;
    ++itn;
    spmv(A, v.data(), -alpha, u.data(), mode);
    beta = std::sqrt(sumsq(u.data(), A.m, mode));
    if (beta > 0.0) {
      double rb = 1.0 / beta;
      for (int64_t i = 0; i < A.m; ++i) u[i] = u[i] * rb;
      spmv_t(A, u.data(), -beta, v.data(), mode, work);
      alpha = std::sqrt(sumsq(v.data(), A.n, mode));
      if (alpha > 0.0) {
        double ra = 1.0 / alpha;
        for (int64_t j = 0; j < A.n; ++j) v[j] = v[j] * ra;
      }
    }
    // rotation Qhat for the damping term, then the rotations Q_k and Qbar_k
    double chat, shat, alphahat;
    sym_ortho(alphabar, damp, chat, shat, alphahat);
    double rhoold = rho, c, s;
    sym_ortho(alphahat, beta, c, s, rho);
    double thetanew = s * alpha;
    alphabar = c * alpha;
    double rhobarold = rhobar, zetaold = zeta;
    double thetabar = sbar * rho, rhotemp = cbar * rho;
    sym_ortho(cbar * rho, thetanew, cbar, sbar, rhobar);
    zeta = cbar * zetabar;
    zetabar = -sbar * zetabar;
    // hbar = h - (thetabar rho / (rhoold rhobarold)) hbar ;  x = x + (zeta / (rho rhobar)) hbar ;  h = v - (thetanew / rho) h
    double f1 = -(thetabar * rho / (rhoold * rhobarold)), f2 = zeta / (rho * rhobar), f3 = -(thetanew / rho);
    for (int64_t j = 0; j < A.n; ++j) {
      double hb = std::fma(f1, hbar[j], h[j]);
      hbar[j] = hb;
      x[j] = std::fma(f2, hb, x[j]);
      h[j] = std::fma(f3, h[j], v[j]);
    }
    // estimate of ||r||
    double betaacute = chat * betadd, betacheck = -shat * betadd;
    double betahat = c * betaacute;
    betadd = -s * betaacute;
    double thetatildeold = thetatilde, ctildeold, stildeold, rhotildeold;
    sym_ortho(rhodold, thetabar, ctildeold, stildeold, rhotildeold);
    thetatilde = stildeold * rhobar;
    rhodold = ctildeold * rhobar;
    betad = -stildeold * betad + ctildeold * betahat;
    tautildeold = (zetaold - thetatildeold * tautildeold) / rhotildeold;
    double taud = (zeta - thetatilde * tautildeold) / rhodold;
    d = d + betacheck * betacheck;
    normr = std::sqrt(d + (betad - taud) * (betad - taud) + betadd * betadd);
    // estimates of ||A||, cond(A), ||A^T r||, ||x||
    normA2 = normA2 + beta * beta;
    normA = std::sqrt(normA2);
    normA2 = normA2 + alpha * alpha;
    maxrbar = std::fmax(maxrbar, rhobarold);
    if (itn > 1) minrbar = std::fmin(minrbar, rhobarold);
    condA = std::fmax(maxrbar, rhotemp) / std::fmin(minrbar, rhotemp);
    normar = std::fabs(zetabar);
    normx = std::sqrt(sumsq(x.data(), A.n, mode));
    // stopping tests (conlim disabled)
    double test1 = normr / normb;
    double den2 = normA * normr;
    double test2 = den2 > 0.0 ? normar / den2 : INFINITY;
    double test3 = 1.0 / condA;
    double ax = normA * normx / normb;
    double tt1 = test1 / (1.0 + ax);
    double rtol = btol + atol * ax;
    istop = 0;
    if (itn >= max_iters) istop = 7;
    if (1.0 + test3 <= 1.0) istop = 6;
    if (1.0 + test2 <= 1.0) istop = 5;
    if (1.0 + tt1 <= 1.0) istop = 4;
    if (test3 <= 0.0) istop = 3;
    if (test2 <= atol) istop = 2;
    if (test1 <= rtol) istop = 1;
    if (istop != 0) done = true;
    return istop;
  }
};

}  // namespace

extern "C" {

// y = A x  (mode 0 plain / 1 dd)
void oracle_spmv(int64_t m, int64_t n, const int64_t* rowptr, const int32_t* colind, const double* vals,
                 const double* x, double* y, int mode) {
  Csr A{m, n, rowptr, colind, vals};
  spmv(A, x, 0.0, y, mode);
}
// the same with two-word entries vals + vals_lo (dd mode)
void oracle_spmv_x(int64_t m, int64_t n, const int64_t* rowptr, const int32_t* colind, const double* vals, const double* vals_lo,
                   const double* x, double* y, int mode) {
  Csr A{m, n, rowptr, colind, vals, vals_lo};
  spmv(A, x, 0.0, y, mode);
}
void oracle_spmv_t_x(int64_t m, int64_t n, const int64_t* rowptr, const int32_t* colind, const double* vals, const double* vals_lo,
                     const double* u, double* v, int mode) {
  Csr A{m, n, rowptr, colind, vals, vals_lo};
  std::vector<dd> work;
  spmv_t(A, u, 0.0, v, mode, work);
}

// v = A^T u  (scatter over rows)
void oracle_spmv_t(int64_t m, int64_t n, const int64_t* rowptr, const int32_t* colind, const double* vals,
                   const double* u, double* v, int mode) {
  Csr A{m, n, rowptr, colind, vals};
  std::vector<dd> work;
  spmv_t(A, u, 0.0, v, mode, work);
}

// Stable CSR -> CSC (rows ascending inside each column): the plain definition of the transpose the
// CUDA library builds at create time; counting sort, one pass in row order.
void oracle_csr_to_csc(int64_t m, int64_t n, const int64_t* rowptr, const int32_t* colind, const double* vals,
                       int64_t* colptr, int32_t* rowind, double* cvals) {
  for (int64_t j = 0; j <= n; ++j) colptr[j] = 0;
  int64_t nnz = rowptr[m];
  for (int64_t e = 0; e < nnz; ++e) colptr[colind[e] + 1]++;
  for (int64_t j = 0; j < n; ++j) colptr[j + 1] += colptr[j];
  std::vector<int64_t> cur(colptr, colptr + n);
  for (int64_t i = 0; i < m; ++i)
    for (int64_t e = rowptr[i]; e < rowptr[i + 1]; ++e) {
      int64_t d = cur[colind[e]]++;
      rowind[d] = (int32_t)i; cvals[d] = vals[e];
    }
}

void* oracle_lsqr_new(int64_t m, int64_t n, const int64_t* rowptr, const int32_t* colind, const double* vals,
                      const double* b, double damp, double atol, double btol, int32_t max_iters, int mode) {
  Lsqr* s = new Lsqr();
  s->A = Csr{m, n, rowptr, colind, vals};
  s->mode = mode; s->damp = damp; s->atol = atol; s->btol = btol; s->max_iters = max_iters;
  s->init(b);
  return s;
}
int32_t oracle_lsqr_step(void* h) { return ((Lsqr*)h)->step(); }
int32_t oracle_lsqr_done(void* h) { return ((Lsqr*)h)->done ? 1 : 0; }
void oracle_lsqr_free(void* h) { delete (Lsqr*)h; }

// which: 0 u (m), 1 v (n), 2 w (n), 3 x (n)
void oracle_lsqr_get_vec(void* h, int which, double* out) {
  Lsqr* s = (Lsqr*)h;
  const std::vector<double>& src = which == 0 ? s->u : which == 1 ? s->v : which == 2 ? s->w : s->x;
  std::memcpy(out, src.data(), sizeof(double) * src.size());
}

// out[0..19]: itn, istop, alpha, beta, rhobar, phibar, bnorm, anorm, ddnorm, res2, xxnorm, z, cs2, sn2,
//             acond, rnorm(r2norm), arnorm, xnorm, r1norm, done
void oracle_lsqr_get_scalars(void* h, double* out) {
  Lsqr* s = (Lsqr*)h;
  double v[20] = {(double)s->itn, (double)s->istop, s->alpha, s->beta, s->rhobar, s->phibar, s->bnorm, s->anorm,
                  s->ddnorm, s->res2, s->xxnorm, s->z, s->cs2, s->sn2, s->acond, s->r2norm, s->arnorm, s->xnorm,
                  s->r1norm, s->done ? 1.0 : 0.0};
  std::memcpy(out, v, sizeof(v));
}

// Whole solve.  res[0..7] = itn, istop, r1norm, r2norm, arnorm, anorm, acond, xnorm.
// r2hist / arhist: [max_iters] or NULL.  snap_iters[nsnap] ascending iteration numbers whose x is
// copied to snap_x[nsnap][n] (NULL for none).
void oracle_lsqr_solve_x(int64_t m, int64_t n, const int64_t* rowptr, const int32_t* colind, const double* vals, const double* vals_lo,
                         const double* b, double damp, double atol, double btol, int32_t max_iters, int mode,
                         double* x, double* res, double* r2hist, double* arhist,
                         int32_t nsnap, const int32_t* snap_iters, double* snap_x);
void oracle_lsqr_solve(int64_t m, int64_t n, const int64_t* rowptr, const int32_t* colind, const double* vals,
                       const double* b, double damp, double atol, double btol, int32_t max_iters, int mode,
                       double* x, double* res, double* r2hist, double* arhist,
                       int32_t nsnap, const int32_t* snap_iters, double* snap_x) {
  oracle_lsqr_solve_x(m, n, rowptr, colind, vals, nullptr, b, damp, atol, btol, max_iters, mode, x, res, r2hist, arhist, nsnap, snap_iters,
                      snap_x);
}
// the same on two-word entries vals + vals_lo (NULL: one-word entries)
void oracle_lsqr_solve_x(int64_t m, int64_t n, const int64_t* rowptr, const int32_t* colind, const double* vals, const double* vals_lo,
                         const double* b, double damp, double atol, double btol, int32_t max_iters, int mode,
                         double* x, double* res, double* r2hist, double* arhist,
                         int32_t nsnap, const int32_t* snap_iters, double* snap_x) {
  Lsqr* s = new Lsqr();
  s->A = Csr{m, n, rowptr, colind, vals, vals_lo};
  s->mode = mode; s->damp = damp; s->atol = atol; s->btol = btol; s->max_iters = max_iters;
  s->init(b);
  int32_t sn = 0;
  while (!s->done) {
    s->step();
    if (r2hist) r2hist[s->itn - 1] = s->r2norm;
    if (arhist) arhist[s->itn - 1] = s->arnorm;
    while (sn < nsnap && snap_iters[sn] == s->itn) {
      std::memcpy(snap_x + (int64_t)sn * n, s->x.data(), sizeof(double) * n);
      ++sn;
    }
  }
  std::memcpy(x, s->x.data(), sizeof(double) * n);
  res[0] = s->itn; res[1] = s->istop; res[2] = s->r1norm; res[3] = s->r2norm; res[4] = s->arnorm;
  res[5] = s->anorm; res[6] = s->acond; res[7] = s->xnorm;
  delete s;
}

// LSMR, whole solve.  res[0..7] = itn, istop, normr, normar, normA, condA, normx, 0.
// nrhist / narhist: [max_iters] or NULL; snapshots as in oracle_lsqr_solve.
void oracle_lsmr_solve_x(int64_t m, int64_t n, const int64_t* rowptr, const int32_t* colind, const double* vals, const double* vals_lo,
                         const double* b, double damp, double atol, double btol, int32_t max_iters, int mode,
                         double* x, double* res, double* nrhist, double* narhist,
                         int32_t nsnap, const int32_t* snap_iters, double* snap_x);
void oracle_lsmr_solve(int64_t m, int64_t n, const int64_t* rowptr, const int32_t* colind, const double* vals,
                       const double* b, double damp, double atol, double btol, int32_t max_iters, int mode,
                       double* x, double* res, double* nrhist, double* narhist,
                       int32_t nsnap, const int32_t* snap_iters, double* snap_x) {
  oracle_lsmr_solve_x(m, n, rowptr, colind, vals, nullptr, b, damp, atol, btol, max_iters, mode, x, res, nrhist, narhist, nsnap, snap_iters,
                      snap_x);
}
// the same on two-word entries vals + vals_lo (NULL: one-word entries)
void oracle_lsmr_solve_x(int64_t m, int64_t n, const int64_t* rowptr, const int32_t* colind, const double* vals, const double* vals_lo,
                         const double* b, double damp, double atol, double btol, int32_t max_iters, int mode,
                         double* x, double* res, double* nrhist, double* narhist,
                         int32_t nsnap, const int32_t* snap_iters, double* snap_x) {
  Lsmr* s = new Lsmr();
  s->A = Csr{m, n, rowptr, colind, vals, vals_lo};
  s->mode = mode; s->damp = damp; s->atol = atol; s->btol = btol; s->max_iters = max_iters;
  s->init(b);
  int32_t sn = 0;
  while (!s->done) {
    s->step();
    if (nrhist) nrhist[s->itn - 1] = s->normr;
    if (narhist) narhist[s->itn - 1] = s->normar;
    while (sn < nsnap && snap_iters[sn] == s->itn) {
      std::memcpy(snap_x + (int64_t)sn * n, s->x.data(), sizeof(double) * n);
      ++sn;
    }
  }
  std::memcpy(x, s->x.data(), sizeof(double) * n);
  res[0] = s->itn; res[1] = s->istop; res[2] = s->normr; res[3] = s->normar; res[4] = s->normA;
  res[5] = s->condA; res[6] = s->normx; res[7] = 0.0;
  delete s;
}

}  // extern "C"
