// multi.cuh — the multi-right-hand-side variant (BASELINE configs[3]): eight independent
// LSQR recurrences that SHARE every pass over A and A^T.  Vectors are row-major blocks (len x 8): one
// element of the matrix is read once and multiplied with a 64-byte row of the gathered block, so the
// HBM stream of `idx`/`val` is paid once per iteration for all eight systems; the gather (64 B per
// nonzero through L1/L2) and, in dd mode, the fp64 pipe become the limits.
//
// Each right-hand side has its own device-resident Scalars (sc[0..8)), its own stopping tests and stop
// flag; a stopped side is frozen: its columns are no longer written.  Fewer than eight sides are padded
// with zero columns (b = 0 stops at once with istop 0).
#pragma once
#include "accum.cuh"
#include "state.cuh"
#include "tails.cuh"

namespace tomo {

constexpr int kR = 8;             // right-hand sides per pass
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

// Y[r][k] <- sum_j a_rj X[j][k] (+ c_k * Y[r][k] * sy_k), ||Y[:,k]||^2, for k = 0..7; rows of the CSR-like
// triple are dealt to the warps of a block round-robin inside the block's static range part[b]..part[b+1].
template <int MODE, typename VT, int OP>
__global__ void __launch_bounds__(kMThreads) k_spmm8(const int64_t* __restrict__ ptr, const int32_t* __restrict__ idx,
                                                     const VT* __restrict__ val, const double* __restrict__ X,
                                                     double* __restrict__ Y, const int32_t* __restrict__ part, Scalars* sc,
                                                     double2* partials) {
  __shared__ double2 s_slots[kMWarps][kR];
  __shared__ double s_c[kR], s_sx[kR], s_sy[kR];
  __shared__ int s_skip[kR], s_flag, s_any;
  if (threadIdx.x < kR) {
    const Scalars* s = sc + threadIdx.x;
    const int skip = s->stop || (OP == OP_K2 && s->beta_zero);
    s_skip[threadIdx.x] = skip;
    s_c[threadIdx.x] = (OP == OP_K1) ? -s->alpha : (OP == OP_K2 ? -s->beta : 0.0);
    s_sx[threadIdx.x] = (OP == OP_K2 || OP == OP_K2_INIT) ? s->rbeta : 1.0;
    s_sy[threadIdx.x] = (OP == OP_K1) ? s->rbeta : 1.0;
  }
  if (threadIdx.x == 0) s_any = 0;
  __syncthreads();
  if (threadIdx.x < kR && !sc[threadIdx.x].stop) s_any = 1;
  __syncthreads();
  if (!s_any) return;  // every side has stopped: nothing changes any more
  constexpr bool SCALE_X = (OP == OP_K2 || OP == OP_K2_INIT);
  // Lane layout: lane = 4*es + j.  The warp takes 8 consecutive elements per step (es = 0..7); the four
  // lanes of an element each gather 16 bytes (sides 2j, 2j+1) of its 64-byte row of X, so one warp load
  // touches 8 rows = 8 L1 wavefronts for 8 elements (a lane-per-element layout with 64-byte gathers costs
  // four times as many wavefronts and is bound by them).
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, es = lane >> 2, j = lane & 3;
  const double sx0 = s_sx[2 * j], sx1 = s_sx[2 * j + 1];
  const double c0 = s_c[2 * j], c1 = s_c[2 * j + 1], sy0 = s_sy[2 * j], sy1 = s_sy[2 * j + 1];
  const bool skip0 = s_skip[2 * j] != 0, skip1 = s_skip[2 * j + 1] != 0;
  Acc<MODE> nsq0, nsq1;
  nsq0.zero(); nsq1.zero();
  const int R0 = part[blockIdx.x], R1 = part[blockIdx.x + 1];
  const double2* X2 = reinterpret_cast<const double2*>(X);
  for (int r = R0 + warp; r < R1; r += kMWarps) {
    const int64_t s = ptr[r], e = ptr[r + 1];
    Acc<MODE> a0, a1;
    a0.zero(); a1.zero();
    int64_t q = s + es;
    for (; q + 56 < e; q += 64) {  // eight steps in flight
      int32_t cc[8];
      double vv[8];
      double2 xx[8];
#pragma unroll
      for (int u = 0; u < 8; ++u) { cc[u] = idx[q + 8 * u]; vv[u] = (double)val[q + 8 * u]; }
#pragma unroll
      for (int u = 0; u < 8; ++u) xx[u] = __ldg(X2 + (size_t)cc[u] * (kR / 2) + j);
#pragma unroll
      for (int u = 0; u < 8; ++u) {
        if (SCALE_X) { xx[u].x = xx[u].x * sx0; xx[u].y = xx[u].y * sx1; }
        a0.mac(vv[u], xx[u].x);
        a1.mac(vv[u], xx[u].y);
      }
    }
    for (; q < e; q += 8) {
      const int32_t c = idx[q];
      const double v = (double)val[q];
      double2 x2 = __ldg(X2 + (size_t)c * (kR / 2) + j);
      if (SCALE_X) { x2.x = x2.x * sx0; x2.y = x2.y * sx1; }
      a0.mac(v, x2.x);
      a1.mac(v, x2.y);
    }
    // sum over the eight element slots (lane bits 2..4), same order in both partners
#pragma unroll
    for (int off = 16; off >= 4; off >>= 1) {
      Acc<MODE> o0, o1;
      double2 p0 = a0.pack(), p1 = a1.pack();
      p0.x = __shfl_xor_sync(0xffffffffu, p0.x, off); p0.y = __shfl_xor_sync(0xffffffffu, p0.y, off);
      p1.x = __shfl_xor_sync(0xffffffffu, p1.x, off); p1.y = __shfl_xor_sync(0xffffffffu, p1.y, off);
      o0.unpack(p0); o1.unpack(p1);
      if (lane & off) { o0.merge(a0); a0 = o0; o1.merge(a1); a1 = o1; } else { a0.merge(o0); a1.merge(o1); }
    }
    if (lane < 4) {  // lane j: sides 2j and 2j+1 of this row
      double2* yp = reinterpret_cast<double2*>(Y + (size_t)r * kR) + j;
      double2 yo = make_double2(0.0, 0.0);
      if (OP == OP_K1 || OP == OP_K2) yo = *yp;
      double yn0, yn1;
      if (OP == OP_K1 || OP == OP_K2) {
        double y0 = yo.x, y1 = yo.y;
        if (OP == OP_K1) { y0 = y0 * sy0; y1 = y1 * sy1; }
        if (MODE == 0) { yn0 = fma(c0, y0, a0.value()); yn1 = fma(c1, y1, a1.value()); }
        else { a0.mac(c0, y0); yn0 = a0.value(); a1.mac(c1, y1); yn1 = a1.value(); }
      } else {
        yn0 = a0.value(); yn1 = a1.value();
      }
      if (OP == OP_K1 || OP == OP_K2) {  // a stopped side keeps its old column
        if (skip0) yn0 = yo.x;
        if (skip1) yn1 = yo.y;
        *yp = make_double2(yn0, yn1);
      } else if (!(skip0 && skip1)) {
        double2 old = (skip0 || skip1) ? *yp : make_double2(0.0, 0.0);
        *yp = make_double2(skip0 ? old.x : yn0, skip1 ? old.y : yn1);
      }
      if (OP != OP_PLAIN) {
        if (!skip0) nsq0.mac(yn0, yn0);
        if (!skip1) nsq1.mac(yn1, yn1);
      }
    }
  }
  // lanes 0..3 hold the sums of sides (2j, 2j+1): spread them to lanes 0..7 as side = lane
  Acc<MODE> nsq;
  {
    const int src = (lane & 7) >> 1;
    double2 p0 = nsq0.pack(), p1 = nsq1.pack();
    p0.x = __shfl_sync(0xffffffffu, p0.x, src); p0.y = __shfl_sync(0xffffffffu, p0.y, src);
    p1.x = __shfl_sync(0xffffffffu, p1.x, src); p1.y = __shfl_sync(0xffffffffu, p1.y, src);
    nsq.unpack((lane & 1) ? p1 : p0);
  }
  if (OP == OP_PLAIN) return;
  Acc<MODE> bs = block_columns<MODE>(nsq, s_slots);
  double total = 0.0;
  if (finish_columns<MODE>(bs, partials, &sc->ticket[0], &s_flag, total)) {
    Scalars* s = sc + threadIdx.x;
    if (!s->stop) {
      const bool skipped = (OP == OP_K2 && s->beta_zero);
      if (OP == OP_K1) tail_k1(s, total);
      if (OP == OP_K2) tail_k2(s, skipped ? 0.0 : total);
      if (OP == OP_K2_INIT) tail_init_v(s, total);
    }
    if (threadIdx.x == 0) sc->ticket[0] = 0u;
  }
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
