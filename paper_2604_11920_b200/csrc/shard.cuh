// shard.cuh — the closing kernels of the row-sharded solve.
//
// A = [A_1; ...; A_P] by row blocks (one or more blocks per GPU).  u, b and the CSR / CSC of a block are local to
// its owner; v, w, x and the scalars are replicated.  A_p v is local.  A^T u = sum_p A_p^T u_p and ||u||^2 =
// sum_p ||u_p||^2 need ONE exchange each per iteration.  To keep the double-double sums order-independent, what
// is exchanged is UNROUNDED: every block leaves (hi, lo) pairs (k_wstream OP_K1S / OP_K2S), the exchange is an
// all-gather in block order, and these kernels add the P pairs in that fixed order, add the fused axpy term and round
// once — in dd mode bit for bit the unsharded result, in fast mode a deterministic sum in block order.
#pragma once
#include "accum.cuh"
#include "state.cuh"
#include "tails.cuh"

namespace tomo {

// ||.||^2 = sum of the P blocks' pairs -> the scalar step.  WHICH 0: ||b||^2 (tail_init_u), 1: ||u^||^2 (tail_k1).
template <int MODE, int WHICH>
__global__ void k_shard_norm(const double2* __restrict__ all, int P, Scalars* sc) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  if (WHICH == 1 && sc->stop) return;
  Acc<MODE> a;
  a.zero();
  for (int p = 0; p < P; ++p) { Acc<MODE> o; o.unpack(all[p]); a.merge(o); }
  if (WHICH == 0) tail_init_u(sc, a.value()); else tail_k1(sc, a.value());
}

// v^_j = sum_p t_p[j] (+ (-beta) v_j), ||v^||^2 -> tail.  t_all: double2[P][n] in block order.  INIT: first pass
// (no axpy term, tail_init_v); else tail_k2.
template <int MODE, bool INIT>
__global__ void __launch_bounds__(256) k_shard_combine(const double2* __restrict__ t_all, int P, int64_t n, double* __restrict__ v,
                                                       Scalars* sc, double2* partials) {
  __shared__ double2 s_slots[8];
  __shared__ int s_flag;
  if (sc->stop) return;
  if (!INIT && sc->beta_zero) {  // beta = 0: the A^T pass was skipped, the scalar step still runs
    if (blockIdx.x == 0 && threadIdx.x == 0) tail_k2(sc, 0.0);
    return;
  }
  const double c = INIT ? 0.0 : -sc->beta;
  Acc<MODE> nsq;
  nsq.zero();
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; j < n; j += stride) {
    Acc<MODE> a;
    a.zero();
    for (int p = 0; p < P; ++p) { Acc<MODE> o; o.unpack(t_all[(int64_t)p * n + j]); a.merge(o); }
    double vn;
    if (INIT) vn = a.value();
    else if (MODE == 0) vn = fma(c, v[j], a.value());
    else { a.mac(c, v[j]); vn = a.value(); }
    v[j] = vn;
    nsq.mac(vn, vn);
  }
  lanes_reduce<32, MODE>(nsq);
  block_combine<MODE>(nsq, s_slots);
  if (publish_and_ticket(partials, nsq.pack(), &sc->ticket[1], &s_flag)) {
    const double total = final_sum<MODE>(partials, gridDim.x, s_slots);
    if (threadIdx.x == 0) {
      if (INIT) tail_init_v(sc, total); else tail_k2(sc, total);
      sc->ticket[1] = 0u;
    }
  }
}

}  // namespace tomo
