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
  if (sc->max_iters <= 0) { sc->istop = 7; sc->stop = 1; }
}

// after  u^ = A v - alpha u :  s = ||u^||^2
__device__ inline void tail_k1(Scalars* sc, double s) {
  double beta = sqrt(s);
  sc->beta = beta;
  if (beta > 0.0) {
    sc->rbeta = 1.0 / beta;
    double alpha = sc->alpha, damp = sc->damp, anorm = sc->anorm;
    sc->anorm = sqrt(anorm * anorm + alpha * alpha + beta * beta + damp * damp);
    sc->beta_zero = 0;
  } else {
    sc->rbeta = 0.0;
    sc->beta_zero = 1;
  }
}

// after  v^ = A^T u - beta v :  s = ||v^||^2  (ignored when the pass was skipped because beta = 0).
// Computes the two rotations and every estimate that does not need ddnorm.
__device__ inline void tail_k2(Scalars* sc, double s) {
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
