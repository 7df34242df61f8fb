// state.cuh — device-resident LSQR state shared by the kernels of one handle (one per right-hand side).
//
// All scalars of Paige & Saunders' recurrences (ref. P:268)
// live here, in device memory: a kernel's tail block writes them, the next kernel reads them, the host
// only ever reads {stop, itn} once per `check_every` iterations.
#pragma once
#include <stdint.h>

namespace tomo {

struct Scalars {
  // bidiagonalisation
  double alpha, beta;      // alpha_k, beta_{k+1}
  double ralpha, rbeta;    // guarded reciprocals: 1/alpha, 1/beta (0 if the norm is 0)
  // QR of the bidiagonal matrix and the damped problem
  double rhobar, phibar, bnorm;
  double anorm, ddnorm, res2, xxnorm, z, cs2, sn2;
  double t1, t2, rrho;     // x += t1 w ; w = v + t2 w ; ddnorm += sum (w * rrho)^2
  // estimates reported to the caller
  double acond, rnorm, arnorm, xnorm, r1norm, r2norm;
  // problem parameters (written by the host at the start of a solve)
  double damp, atol, btol;
  double* hist_r2;         // device fp64[hist_cap] or nullptr
  double* hist_ar;
  int32_t hist_cap;
  int32_t max_iters;
  // control
  int32_t itn, istop;
  int32_t stop;            // 1: every later kernel of this solve returns immediately (x is frozen)
  int32_t beta_zero;       // beta_{k+1} == 0 in this iteration: the A^T pass is skipped
  int32_t norm_v;          // K4 must normalise v (alpha > 0 and the A^T pass ran)
  int32_t pad_;
  // LSMR (solver = 1; Fong & Saunders 2011, the paper's own solver): same bidiagonalisation,
  // other recurrences.  Results are reported through the fields above: r2norm = ||rbar||, arnorm = ||Abar^T rbar||,
  // anorm = ||Abar|| estimate, acond, xnorm = ||x|| (computed, not estimated).
  int32_t solver, pad2_;
  double zetabar, alphabar, lrho, lrhobar, cbar, sbar;
  double betadd, betad, rhodold, tautildeold, thetatilde, zeta, dsum;
  double normA2, maxrbar, minrbar;
  double f1, f2, f3;       // hbar = h + f1 hbar ; x = x + f2 hbar ; h = v + f3 h
  // last-block tickets, one per kernel kind (reset to 0 by the tail that consumed them)
  unsigned int ticket[4];
};

// what a fused SpMV launch is for
enum SpmvOp : int {
  OP_PLAIN = 0,   // y = A x                       (tomo_lsqr_spmv)
  OP_K1 = 1,      // u^ = A v - alpha u  , ||u^||^2 ; tail: beta, anorm
  OP_K2 = 2,      // v^ = A^T u - beta v , ||v^||^2 ; tail: alpha, rotations, estimates
  OP_K2_INIT = 3, // v^ = A^T u          , ||v^||^2 ; tail: alpha_1, rhobar, phibar
  // row-sharded solve (shard.cuh): one row block of A per launch, the sums over blocks are closed after an exchange
  OP_K1S = 4,     // u^_p = A_p v - alpha u_p ; the block's ||u^_p||^2 as an unrounded (hi, lo) pair, no tail
  OP_K2S = 5      // t_p = A_p^T u_p as UNROUNDED (hi, lo) pairs per column (y is a double2 array), no norm, no tail
};

enum VecOp : int {
  VOP_INIT_U = 0,  // u^ = b, ||b||^2 ; tail: beta_1
  VOP_INIT_VW = 1, // v = v^/alpha, w = v, x = 0
  VOP_K4 = 2,      // v = v^/alpha ; ddnorm partial ; x += t1 w ; w = v + t2 w ; tail: stop tests
  VOP_K4_LSMR = 3, // v = v^/alpha ; hbar = h + f1 hbar ; x += f2 hbar ; h = v + f3 h ; ||x||^2 ; tail: stop tests
  VOP_INIT_US = 4  // sharded: u^_p = b_p ; ||b_p||^2 as an unrounded pair to a3[0..1], no tail
};

}  // namespace tomo
