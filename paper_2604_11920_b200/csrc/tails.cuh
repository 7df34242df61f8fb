// tails.cuh — the O(1) scalar part of an LSQR iteration, run by ONE thread of the last block of a
// kernel.  Step by step Paige & Saunders' Algorithm LSQR with the second rotation
// for damping (ref. P:268), in fp64 with IEEE sqrt and
// division and no FMA contraction (--fmad=false), so that it reproduces a host evaluation of the same
// formulas bit for bit.
#pragma once
#include "state.cuh"

namespace tomo {

// after  u^ = b :  s = ||b||^2
__device__ inline void tail_init_u(Scalars* sc, double s) {
  double beta = sqrt(s);
  sc->beta = beta;
  sc->bnorm = beta;
  sc->rnorm = beta; sc->r1norm = beta; sc->r2norm = beta;
  if (beta == 0.0) {            // b = 0  =>  x = 0 is exact
    sc->rbeta = 0.0;
    sc->rnorm = 0.0; sc->r1norm = 0.0; sc->r2norm = 0.0;
    sc->istop = 0; sc->stop = 1;
    return;
  }
  sc->rbeta = 1.0 / beta;
}

// after  v^ = A^T u  (first pass):  s = ||v^||^2
__device__ inline void tail_init_v(Scalars* sc, double s) {
  double alpha = sqrt(s);
  sc->alpha = alpha;
  if (alpha == 0.0) {           // A^T b = 0  =>  x = 0 is exact
    sc->ralpha = 0.0;
    sc->arnorm = 0.0;
    sc->istop = 0; sc->stop = 1;
    return;
  }
  sc->ralpha = 1.0 / alpha;
  sc->rhobar = alpha;
  sc->phibar = sc->beta;
  sc->arnorm = alpha * sc->beta;
  if (sc->solver == 1) {  // LSMR start values
    sc->zetabar = alpha * sc->beta; sc->alphabar = alpha;
    sc->lrho = 1.0; sc->lrhobar = 1.0; sc->cbar = 1.0; sc->sbar = 0.0;
    sc->betadd = sc->beta; sc->betad = 0.0; sc->rhodold = 1.0; sc->tautildeold = 0.0; sc->thetatilde = 0.0;
    sc->zeta = 0.0; sc->dsum = 0.0;
    sc->normA2 = alpha * alpha; sc->maxrbar = 0.0; sc->minrbar = 1e100;
    sc->anorm = sqrt(sc->normA2); sc->acond = 1.0;
  }
  if (sc->max_iters <= 0) { sc->istop = 7; sc->stop = 1; }
}

// stable Givens rotation [c s; -s c][a; b] = [r; 0] (Fong & Saunders' SymOrtho)
__device__ inline void sym_ortho(double a, double b, double& c, double& s, double& r) {
  if (b == 0.0) { c = (a > 0.0) ? 1.0 : (a < 0.0 ? -1.0 : 0.0); s = 0.0; r = fabs(a); }
  else if (a == 0.0) { c = 0.0; s = (b > 0.0) ? 1.0 : -1.0; r = fabs(b); }
  else if (fabs(b) > fabs(a)) {
    const double tau = a / b;
    s = ((b > 0.0) ? 1.0 : -1.0) / sqrt(1.0 + tau * tau);
    c = s * tau; r = b / s;
  } else {
    const double tau = b / a;
    c = ((a > 0.0) ? 1.0 : -1.0) / sqrt(1.0 + tau * tau);
    s = c * tau; r = a / c;
  }
}

// LSMR: after v^ = A^T u - beta v.  The three rotations, the update factors f1, f2, f3 and the estimate of ||r||.
__device__ inline void tail_k2_lsmr(Scalars* sc, double ssq) {
  double alpha = sc->alpha;
  sc->norm_v = 0;
  if (!sc->beta_zero) {
    alpha = sqrt(ssq);
    sc->alpha = alpha;
    if (alpha > 0.0) { sc->ralpha = 1.0 / alpha; sc->norm_v = 1; }
  }
  const double beta = sc->beta, damp = sc->damp;
  double chat, shat, alphahat;
  sym_ortho(sc->alphabar, damp, chat, shat, alphahat);
  const double rhoold = sc->lrho;
  double c, s, rho;
  sym_ortho(alphahat, beta, c, s, rho);
  const double thetanew = s * alpha;
  sc->alphabar = c * alpha;
  const double rhobarold = sc->lrhobar, zetaold = sc->zeta;
  const double thetabar = sc->sbar * rho, rhotemp = sc->cbar * rho;
  double cbar, sbar, rhobar;
  sym_ortho(sc->cbar * rho, thetanew, cbar, sbar, rhobar);
  const double zeta = cbar * sc->zetabar;
  sc->zetabar = -sbar * sc->zetabar;
  sc->cbar = cbar; sc->sbar = sbar; sc->lrho = rho; sc->lrhobar = rhobar; sc->zeta = zeta;
  sc->f1 = -(thetabar * rho / (rhoold * rhobarold));
  sc->f2 = zeta / (rho * rhobar);
  sc->f3 = -(thetanew / rho);
  // estimate of ||r||
  const double betaacute = chat * sc->betadd, betacheck = -shat * sc->betadd;
  const double betahat = c * betaacute;
  sc->betadd = -s * betaacute;
  const double thetatildeold = sc->thetatilde;
  double ctildeold, stildeold, rhotildeold;
  sym_ortho(sc->rhodold, thetabar, ctildeold, stildeold, rhotildeold);
  sc->thetatilde = stildeold * rhobar;
  sc->rhodold = ctildeold * rhobar;
  sc->betad = -stildeold * sc->betad + ctildeold * betahat;
  sc->tautildeold = (zetaold - thetatildeold * sc->tautildeold) / rhotildeold;
  const double taud = (zeta - sc->thetatilde * sc->tautildeold) / sc->rhodold;
  sc->dsum = sc->dsum + betacheck * betacheck;
  const double bt = sc->betad - taud;
  sc->rnorm = sqrt(sc->dsum + bt * bt + sc->betadd * sc->betadd);
  sc->r2norm = sc->rnorm;
  // estimates of ||A||, cond(A), ||A^T r||
  double normA2 = sc->normA2 + beta * beta;
  sc->anorm = sqrt(normA2);
  sc->normA2 = normA2 + alpha * alpha;
  const double maxrbar = fmax(sc->maxrbar, rhobarold);
  sc->maxrbar = maxrbar;
  if (sc->itn + 1 > 1) sc->minrbar = fmin(sc->minrbar, rhobarold);
  sc->acond = fmax(maxrbar, rhotemp) / fmin(sc->minrbar, rhotemp);
  sc->arnorm = fabs(sc->zetabar);
}

// LSMR: after the h / hbar / x update:  ssq = ||x||^2.  Stopping tests, history.
__device__ inline void tail_k4_lsmr(Scalars* sc, double ssq) {
  const double normx = sqrt(ssq);
  sc->xnorm = normx;
  const double normA = sc->anorm, normr = sc->rnorm, normar = sc->arnorm, normb = sc->bnorm, damp = sc->damp;
  const double r1sq = normr * normr - damp * damp * (normx * normx);
  sc->r1norm = sqrt(r1sq > 0.0 ? r1sq : 0.0);
  const int itn = sc->itn + 1;
  sc->itn = itn;
  const double test1 = normr / normb;
  const double den2 = normA * normr;
  const double test2 = den2 > 0.0 ? normar / den2 : __longlong_as_double(0x7ff0000000000000LL);
  const double test3 = 1.0 / sc->acond;
  const double ax = normA * normx / normb;
  const double tt1 = test1 / (1.0 + ax);
  const double rtol = sc->btol + sc->atol * ax;
  int istop = 0;
  if (itn >= sc->max_iters) istop = 7;
  if (1.0 + test3 <= 1.0) istop = 6;
  if (1.0 + test2 <= 1.0) istop = 5;
  if (1.0 + tt1 <= 1.0) istop = 4;
  if (test3 <= 0.0) istop = 3;
  if (test2 <= sc->atol) istop = 2;
  if (test1 <= rtol) istop = 1;
  if (itn <= sc->hist_cap) {
    if (sc->hist_r2) sc->hist_r2[itn - 1] = normr;
    if (sc->hist_ar) sc->hist_ar[itn - 1] = normar;
  }
  sc->istop = istop;
  if (istop != 0) sc->stop = 1;
}

// after  u^ = A v - alpha u :  s = ||u^||^2
__device__ inline void tail_k1(Scalars* sc, double s) {
  double beta = sqrt(s);
  sc->beta = beta;
  if (beta > 0.0) {
    sc->rbeta = 1.0 / beta;
    if (sc->solver == 0) {
      double alpha = sc->alpha, damp = sc->damp, anorm = sc->anorm;
      sc->anorm = sqrt(anorm * anorm + alpha * alpha + beta * beta + damp * damp);
    }
    sc->beta_zero = 0;
  } else {
    sc->rbeta = 0.0;
    sc->beta_zero = 1;
  }
}

// after  v^ = A^T u - beta v :  s = ||v^||^2  (ignored when the pass was skipped because beta = 0).
// Computes the two rotations and every estimate that does not need ddnorm.
__device__ inline void tail_k2_lsmr(Scalars* sc, double ssq);
__device__ inline void tail_k2(Scalars* sc, double s) {
  if (sc->solver == 1) { tail_k2_lsmr(sc, s); return; }
  double alpha = sc->alpha;
  sc->norm_v = 0;
  if (!sc->beta_zero) {
    alpha = sqrt(s);
    sc->alpha = alpha;
    if (alpha > 0.0) { sc->ralpha = 1.0 / alpha; sc->norm_v = 1; }
  }
  const double beta = sc->beta, damp = sc->damp;
  double rhobar = sc->rhobar, phibar = sc->phibar;
  // rotation that eliminates damp
  double rhobar1 = sqrt(rhobar * rhobar + damp * damp);
  double cs1 = rhobar / rhobar1, sn1 = damp / rhobar1;
  double psi = sn1 * phibar;
  phibar = cs1 * phibar;
  // rotation that eliminates beta
  double rho = sqrt(rhobar1 * rhobar1 + beta * beta);
  double cs = rhobar1 / rho, sn = beta / rho;
  double theta = sn * alpha;
  rhobar = -cs * alpha;
  double phi = cs * phibar;
  phibar = sn * phibar;
  double tau = sn * phi;
  sc->rhobar = rhobar; sc->phibar = phibar;
  sc->t1 = phi / rho;
  sc->t2 = -theta / rho;
  sc->rrho = 1.0 / rho;
  // estimates of ||x||, ||r||, ||A^T r||
  double z = sc->z, cs2 = sc->cs2, sn2 = sc->sn2, xxnorm = sc->xxnorm;
  double delta = sn2 * rho, gambar = -cs2 * rho, rhs = phi - delta * z, zbar = rhs / gambar;
  double xnorm = sqrt(xxnorm + zbar * zbar);
  double gamma = sqrt(gambar * gambar + theta * theta);
  sc->cs2 = gambar / gamma; sc->sn2 = theta / gamma;
  z = rhs / gamma;
  sc->z = z;
  sc->xxnorm = xxnorm + z * z;
  sc->xnorm = xnorm;
  double res2 = sc->res2 + psi * psi;
  sc->res2 = res2;
  double rnorm = sqrt(phibar * phibar + res2);
  sc->rnorm = rnorm;
  sc->arnorm = alpha * fabs(tau);
  sc->r2norm = rnorm;
  double r1sq = rnorm * rnorm - damp * damp * (xnorm * xnorm);
  sc->r1norm = sqrt(r1sq > 0.0 ? r1sq : 0.0);
}

// after the x / w update:  s = sum_j (w_j / rho)^2 .  ddnorm, acond, the stopping tests, history.
__device__ inline void tail_k4(Scalars* sc, double s) {
  double ddnorm = sc->ddnorm + s;
  sc->ddnorm = ddnorm;
  const double anorm = sc->anorm, rnorm = sc->rnorm, arnorm = sc->arnorm, xnorm = sc->xnorm, bnorm = sc->bnorm;
  double acond = anorm * sqrt(ddnorm);
  sc->acond = acond;
  int itn = sc->itn + 1;
  sc->itn = itn;
  double test1 = rnorm / bnorm;
  double den2 = anorm * rnorm;
  double test2 = den2 > 0.0 ? arnorm / den2 : 0.0;
  double test3 = acond > 0.0 ? 1.0 / acond : __longlong_as_double(0x7ff0000000000000LL);
  double ax = anorm * xnorm / bnorm;
  double tt1 = test1 / (1.0 + ax);
  double rtol = sc->btol + sc->atol * ax;
  int istop = 0;
  if (itn >= sc->max_iters) istop = 7;
  if (1.0 + test3 <= 1.0) istop = 6;
  if (1.0 + test2 <= 1.0) istop = 5;
  if (1.0 + tt1 <= 1.0) istop = 4;
  if (test3 <= 0.0) istop = 3;
  if (test2 <= sc->atol) istop = 2;
  if (test1 <= rtol) istop = 1;
  if (itn <= sc->hist_cap) {
    if (sc->hist_r2) sc->hist_r2[itn - 1] = sc->r2norm;
    if (sc->hist_ar) sc->hist_ar[itn - 1] = arnorm;
  }
  sc->istop = istop;
  if (istop != 0) sc->stop = 1;
}

}  // namespace tomo
