// multi.cuh — the fused vector kernels of the multi-right-hand-side variant (BASELINE
// configs[3]): eight independent LSQR / LSMR recurrences that SHARE every pass over A and A^T.  Vectors are
// row-major blocks (len x 8); the two sparse products live in wspmm.cuh.
//
// Each right-hand side has its own device-resident Scalars (sc[0..8)), its own stopping tests and stop
// flag; a stopped side is frozen: its columns are no longer written.  Fewer than eight sides are padded
// with zero columns (b = 0 stops at once with istop 0).
#pragma once
#include "accum.cuh"
#include "state.cuh"
#include "tails.cuh"
#include "wspmm.cuh"

namespace tomo {

constexpr int kMThreads = 256;    // block size of the multi kernels
constexpr int kMWarps = kMThreads / 32;

// block-level: lanes 0..7 of every warp hold a per-column partial -> thread k (< 8) returns the block sum
template <int MODE>
__device__ __forceinline__ Acc<MODE> block_columns(Acc<MODE> mine, double2 (*slots)[kR]) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (lane < kR) slots[warp][lane] = mine.pack();
  __syncthreads();
  Acc<MODE> t;
  t.zero();
  if (threadIdx.x < kR) {
    t.unpack(slots[0][threadIdx.x]);
    for (int w = 1; w < kMWarps; ++w) { Acc<MODE> o; o.unpack(slots[w][threadIdx.x]); t.merge(o); }
  }
  return t;
}

// Publish the block's eight partials; the last-arriving block sums them per column in block order.
// Returns true in the threads k < 8 of the last block, with `total` = the column sum.
template <int MODE>
__device__ __forceinline__ bool finish_columns(Acc<MODE> blocksum, double2* partials, unsigned int* ticket, int* s_flag,
                                               double& total) {
  if (threadIdx.x < kR) __stcg(partials + (size_t)blockIdx.x * kR + threadIdx.x, blocksum.pack());
  __threadfence();
  __syncthreads();
  if (threadIdx.x == 0) {
    const unsigned int t = atomicAdd(ticket, 1u);
    *s_flag = (t == gridDim.x - 1) ? 1 : 0;
  }
  __syncthreads();
  if (*s_flag == 0) return false;
  __threadfence();
  if (threadIdx.x >= kR) return false;
  Acc<MODE> a;
  a.zero();
  for (int b = 0; b < (int)gridDim.x; ++b) { Acc<MODE> o; o.unpack(__ldcg(partials + (size_t)b * kR + threadIdx.x)); a.merge(o); }
  total = a.value();
  return true;
}

// Fused vector kernels on len x 8 blocks; element e = i*8 + k belongs to side k = e & 7, which is fixed per
// thread because every stride is a multiple of 8.
//   VOP_INIT_U : U = B (B is len x nrhs, nrhs <= 8; missing columns are zero) ; ||b_k||^2
//   VOP_INIT_VW: V = V * (1/alpha_k) ; W = V ; (X zeroed by the host)
//   VOP_K4     : as the single-side kernel, with the scalars of side k
//   VOP_K4_LSMR: LSMR's three-vector update (hbar, x, h) and ||x_k||^2, with the scalars of side k
template <int MODE, int VOP>
__global__ void __launch_bounds__(kMThreads) k_vec8(const double* __restrict__ in0, int nrhs, double* __restrict__ a0,
                                                    double* __restrict__ a1, double* __restrict__ a2, int64_t len, Scalars* sc,
                                                    double2* partials, double* __restrict__ a3 = nullptr) {
  __shared__ double2 s_slots[kMWarps][kR];
  __shared__ int s_flag;
  const int k = threadIdx.x & 7;
  Scalars* s = sc + k;
  const bool stopped = (VOP != VOP_INIT_U) && s->stop;
  Acc<MODE> acc;
  acc.zero();
  const int64_t total_e = len * kR;
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  const int64_t e0 = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (VOP == VOP_INIT_U) {
    for (int64_t e = e0; e < total_e; e += stride) {
      const double b = (k < nrhs) ? in0[(e >> 3) * nrhs + k] : 0.0;
      a0[e] = b;
      acc.mac(b, b);
    }
  } else if (VOP == VOP_INIT_VW) {
    if (!stopped) {
      const double ra = s->ralpha;
      for (int64_t e = e0; e < total_e; e += stride) {
        const double v = a0[e] * ra;
        a0[e] = v;
        a1[e] = v;
      }
    }
    return;
  } else if (VOP == VOP_K4_LSMR) {  // a0 = V, a1 = H, a2 = X, a3 = Hbar (Fong & Saunders' update with the scalars of side k)
    if (!stopped) {
      const double ra = s->ralpha, f1 = s->f1, f2 = s->f2, f3 = s->f3;
      const bool norm_v = s->norm_v != 0;
      for (int64_t e = e0; e < total_e; e += stride) {
        double v = a0[e];
        if (norm_v) { v = v * ra; a0[e] = v; }
        const double h = a1[e];
        const double hb = fma(f1, a3[e], h);
        a3[e] = hb;
        const double xn = fma(f2, hb, a2[e]);
        a2[e] = xn;
        a1[e] = fma(f3, h, v);
        acc.mac(xn, xn);
      }
    }
  } else if (!stopped) {
    const double ra = s->ralpha, t1 = s->t1, t2 = s->t2, rrho = s->rrho;
    const bool norm_v = s->norm_v != 0;
    for (int64_t e = e0; e < total_e; e += stride) {
      double v = a0[e];
      if (norm_v) { v = v * ra; a0[e] = v; }
      const double w = a1[e];
      const double d = w * rrho;
      acc.mac(d, d);
      a2[e] = fma(t1, w, a2[e]);
      a1[e] = fma(t2, w, v);
    }
  }
  // lanes with the same k: offsets 8 and 16
#pragma unroll
  for (int off = 16; off >= 8; off >>= 1) {
    Acc<MODE> o;
    double2 p = acc.pack();
    p.x = __shfl_xor_sync(0xffffffffu, p.x, off);
    p.y = __shfl_xor_sync(0xffffffffu, p.y, off);
    o.unpack(p);
    if ((threadIdx.x & 31) & off) { o.merge(acc); acc = o; } else { acc.merge(o); }
  }
  Acc<MODE> bs = block_columns<MODE>(acc, s_slots);
  double total = 0.0;
  if (finish_columns<MODE>(bs, partials, &sc->ticket[1], &s_flag, total)) {
    Scalars* t = sc + threadIdx.x;
    if (VOP == VOP_INIT_U) tail_init_u(t, total);
    else if (!t->stop) { if (VOP == VOP_K4_LSMR) tail_k4_lsmr(t, total); else tail_k4(t, total); }
    if (threadIdx.x == 0) sc->ticket[1] = 0u;
  }
}

}  // namespace tomo
