// kernels.cuh — the fused vector kernels of the LSQR hot path.  The two sparse
// products live in stream.cuh.
//
// One iteration of LSQR (PAPER.md P:142 names the method; the paper's GPU solver offloads "sparse
// matrix-vector multiplications and vector norm calculations") is three launches:
//   K1  u^ <- A v - alpha u     + ||u^||^2 -> tail: beta, 1/beta, anorm                    (stream.cuh)
//   K2  v^ <- A^T u - beta v    + ||v^||^2 -> tail: alpha, rotations, t1, t2, estimates    (stream.cuh)
//   K4  v <- v^/alpha; ddnorm partial; x <- x + t1 w; w <- v + t2 w -> tail: stop tests, history
// u is kept un-normalised (u^); the factor 1/beta is applied where u is read (fl(u^_i * (1/beta)) is
// exactly the value a normalising pass would have stored).
#pragma once
#include "accum.cuh"
#include "state.cuh"
#include "tails.cuh"

namespace tomo {

constexpr int kThreads = 256;
constexpr int kWarps = kThreads / 32;

// Fused vector kernels: one pass, scale + axpy + norm^2, static grid-stride
// assignment so that the fast-mode partial sums have a fixed order.
//   VOP_INIT_U : u^ = b ; ||b||^2                               (len = m; in0 = b, out0 = u^)
//   VOP_INIT_VW: v = v^ * (1/alpha) ; w = v                     (len = n; io0 = v, out1 = w)
//   VOP_K4     : v = v^ * (1/alpha) ; sum (w*rrho)^2 ; x += t1 w ; w = v + t2 w   (io0 = v, io1 = w, io2 = x)
template <int MODE, int VOP>
__global__ void __launch_bounds__(kThreads) k_vec(const double* __restrict__ in0, double* __restrict__ a0,
                                                  double* __restrict__ a1, double* __restrict__ a2,
                                                  double* __restrict__ a3, int64_t len, Scalars* sc, double2* partials) {
  __shared__ double2 s_slots[kWarps];
  __shared__ int s_flag;
  grid_dependency_wait();
  if (VOP != VOP_INIT_U && VOP != VOP_INIT_US && sc->stop) return;
  Acc<MODE> acc;
  acc.zero();
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  const int64_t i0 = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (VOP == VOP_INIT_U || VOP == VOP_INIT_US) {
    for (int64_t i = i0; i < len; i += stride) {
      double b = in0[i];
      a0[i] = b;
      acc.mac(b, b);
    }
  } else if (VOP == VOP_INIT_VW) {
    const double ra = sc->ralpha;
    for (int64_t i = i0; i < len; i += stride) {
      double v = a0[i] * ra;
      a0[i] = v;
      a1[i] = v;
    }
    return;
  } else if (VOP == VOP_K4_LSMR) {  // a0 = v, a1 = h, a2 = x, a3 = hbar (Fong & Saunders' update)
    const double ra = sc->ralpha, f1 = sc->f1, f2 = sc->f2, f3 = sc->f3;
    const bool norm_v = sc->norm_v != 0;
    for (int64_t i = i0; i < len; i += stride) {
      double v = a0[i];
      if (norm_v) { v = v * ra; a0[i] = v; }
      const double h = a1[i];
      const double hb = fma(f1, a3[i], h);
      a3[i] = hb;
      const double xn = fma(f2, hb, a2[i]);
      a2[i] = xn;
      a1[i] = fma(f3, h, v);
      acc.mac(xn, xn);
    }
  } else {
    const double ra = sc->ralpha, t1 = sc->t1, t2 = sc->t2, rrho = sc->rrho;
    const bool norm_v = sc->norm_v != 0;
    int64_t i = i0;
    for (; i + 3 * stride < len; i += 4 * stride) {  // four independent elements per trip: 12 loads in flight
      double v[4], w[4], xo[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) { v[u] = a0[i + u * stride]; w[u] = a1[i + u * stride]; xo[u] = a2[i + u * stride]; }
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        if (norm_v) { v[u] = v[u] * ra; a0[i + u * stride] = v[u]; }
        const double d = w[u] * rrho;
        acc.mac(d, d);
        a2[i + u * stride] = fma(t1, w[u], xo[u]);
        a1[i + u * stride] = fma(t2, w[u], v[u]);
      }
    }
    for (; i < len; i += stride) {
      double v = a0[i];
      if (norm_v) { v = v * ra; a0[i] = v; }
      double w = a1[i];
      double d = w * rrho;
      acc.mac(d, d);
      a2[i] = fma(t1, w, a2[i]);
      a1[i] = fma(t2, w, v);
    }
  }
  lanes_reduce<32, MODE>(acc);
  block_combine<MODE>(acc, s_slots);
  grid_launch_dependents();
  if (publish_and_ticket(partials, acc.pack(), &sc->ticket[1], &s_flag)) {
    const double2 pair = final_sum_pair<MODE>(partials, gridDim.x, s_slots);
    if (threadIdx.x == 0) {
      Acc<MODE> t;
      t.unpack(pair);
      const double total = t.value();
      if (VOP == VOP_INIT_US) reinterpret_cast<double2*>(a3)[0] = pair;
      if (VOP == VOP_INIT_U) tail_init_u(sc, total);
      if (VOP == VOP_K4) tail_k4(sc, total);
      if (VOP == VOP_K4_LSMR) tail_k4_lsmr(sc, total);
      sc->ticket[1] = 0u;
    }
  }
}

}  // namespace tomo
