// kernels.cuh — the hot kernels: fused SpMV (+axpy +norm^2 +scalar tail) used for both A v (over the
// caller's CSR) and A^T u (over the CSC copy, i.e. the CSR of A^T), and the fused vector kernels.
//
// One iteration of LSQR (PAPER.md P:142 names the method; the paper's GPU solver offloads "sparse
// matrix-vector multiplications and vector norm calculations") is three launches:
//   K1  u^ <- A v - alpha u     + ||u^||^2 -> tail: beta, 1/beta, anorm
//   K2  v^ <- A^T u - beta v    + ||v^||^2 -> tail: alpha, rotations, t1, t2, estimates
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
constexpr int kRowGroup = 4;      // rows per warp task; partitions are aligned to it
constexpr int kShortRow = 8;      // rows of <= 8 nnz are done four at a time, 8 lanes each

// streaming loads of the matrix arrays: read once per pass, keep them out of L1 so that the gathered
// vector stays resident there
__device__ __forceinline__ int32_t ld_stream(const int32_t* p) {
  int32_t r;
  asm volatile("ld.global.nc.L1::no_allocate.s32 %0, [%1];" : "=r"(r) : "l"(p));
  return r;
}
__device__ __forceinline__ double ld_stream(const double* p) {
  double r;
  asm volatile("ld.global.nc.L1::no_allocate.f64 %0, [%1];" : "=d"(r) : "l"(p));
  return r;
}
__device__ __forceinline__ double ld_stream(const float* p) {
  float r;
  asm volatile("ld.global.nc.L1::no_allocate.f32 %0, [%1];" : "=f"(r) : "l"(p));
  return (double)r;
}

// per-lane partial of  sum_{e in [s,e)} val[e] * (x[idx[e]] * sx)  for one row, whole warp cooperating
template <int MODE, typename VT, bool SCALE_X>
__device__ __forceinline__ Acc<MODE> row_dot(const int32_t* __restrict__ idx, const VT* __restrict__ val,
                                             const double* __restrict__ x, int64_t s, int64_t e, int lane, double sx) {
  Acc<MODE> a0, a1, a2, a3;
  a0.zero(); a1.zero(); a2.zero(); a3.zero();
  for (int64_t base = s; base < e; base += 128) {
    const int64_t q = base + lane;
    if (base + 128 <= e) {  // warp-uniform: four full 32-element slices
      int32_t c0 = ld_stream(idx + q), c1 = ld_stream(idx + q + 32), c2 = ld_stream(idx + q + 64), c3 = ld_stream(idx + q + 96);
      double v0 = ld_stream(val + q), v1 = ld_stream(val + q + 32), v2 = ld_stream(val + q + 64), v3 = ld_stream(val + q + 96);
      double x0 = __ldg(x + c0), x1 = __ldg(x + c1), x2 = __ldg(x + c2), x3 = __ldg(x + c3);
      if (SCALE_X) { x0 = x0 * sx; x1 = x1 * sx; x2 = x2 * sx; x3 = x3 * sx; }
      a0.mac(v0, x0); a1.mac(v1, x1); a2.mac(v2, x2); a3.mac(v3, x3);
    } else {               // ragged tail: masked lanes contribute an exact zero
      const bool k0 = q < e, k1 = q + 32 < e, k2 = q + 64 < e, k3 = q + 96 < e;
      int32_t c0 = k0 ? ld_stream(idx + q) : 0, c1 = k1 ? ld_stream(idx + q + 32) : 0;
      int32_t c2 = k2 ? ld_stream(idx + q + 64) : 0, c3 = k3 ? ld_stream(idx + q + 96) : 0;
      double v0 = k0 ? ld_stream(val + q) : 0.0, v1 = k1 ? ld_stream(val + q + 32) : 0.0;
      double v2 = k2 ? ld_stream(val + q + 64) : 0.0, v3 = k3 ? ld_stream(val + q + 96) : 0.0;
      double x0 = k0 ? __ldg(x + c0) : 0.0, x1 = k1 ? __ldg(x + c1) : 0.0;
      double x2 = k2 ? __ldg(x + c2) : 0.0, x3 = k3 ? __ldg(x + c3) : 0.0;
      if (SCALE_X) { x0 = x0 * sx; x1 = x1 * sx; x2 = x2 * sx; x3 = x3 * sx; }
      a0.mac(v0, x0); a1.mac(v1, x1); a2.mac(v2, x2); a3.mac(v3, x3);
    }
  }
  a0.merge(a1); a2.merge(a3); a0.merge(a2);
  return a0;
}

// y_r <- dot + c * (y_r * sy)  and the running ||y||^2 ; executed by the lane that holds the row sum
template <int MODE, int OP>
__device__ __forceinline__ void row_epilogue(Acc<MODE>& dot, double* __restrict__ y, int64_t r, double c, double sy,
                                             Acc<MODE>& nsq) {
  double yn;
  if (OP == OP_K1 || OP == OP_K2) {
    double yo = y[r];
    if (OP == OP_K1) yo = yo * sy;
    if (MODE == 0) {
      yn = fma(c, yo, dot.value());
    } else {
      dot.mac(c, yo);
      yn = dot.value();
    }
  } else {
    yn = dot.value();
  }
  y[r] = yn;
  if (OP != OP_PLAIN) nsq.mac(yn, yn);
}

// Fused SpMV over a CSR-like triple (ptr, idx, val) with `nrows` rows.  Block b owns the contiguous
// row range [part[b], part[b+1]) (nnz-balanced, aligned to kRowGroup); inside it warps take groups of
// four consecutive rows round-robin, so both the assignment and every summation order are static.
template <int MODE, typename VT, int OP>
__global__ void __launch_bounds__(kThreads) k_spmv(const int64_t* __restrict__ ptr, const int32_t* __restrict__ idx,
                                                   const VT* __restrict__ val, const double* __restrict__ x,
                                                   double* __restrict__ y, const int32_t* __restrict__ part,
                                                   Scalars* sc, double2* partials) {
  __shared__ double2 s_slots[kWarps];
  __shared__ int s_flag;
  double c = 0.0, sx = 1.0, sy = 1.0;
  if (OP != OP_PLAIN) {
    if (sc->stop) return;
    if (OP == OP_K2 && sc->beta_zero) {  // beta = 0: A^T pass skipped, the scalar step still runs
      if (blockIdx.x == 0 && threadIdx.x == 0) tail_k2(sc, 0.0);
      return;
    }
    if (OP == OP_K1) { c = -sc->alpha; sy = sc->rbeta; }
    if (OP == OP_K2) { c = -sc->beta; sx = sc->rbeta; }
    if (OP == OP_K2_INIT) { sx = sc->rbeta; }
  }
  constexpr bool SCALE_X = (OP == OP_K2 || OP == OP_K2_INIT);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int R0 = part[blockIdx.x], R1 = part[blockIdx.x + 1];
  Acc<MODE> nsq;
  nsq.zero();
  for (int g = R0 + kRowGroup * warp; g < R1; g += kRowGroup * kWarps) {
    const int nr = min(kRowGroup, R1 - g);
    // lanes 0..nr fetch the row pointers of the group; p[k] .. p[k+1] delimit row g+k
    int64_t pv = (lane <= nr) ? ptr[g + lane] : 0;
    int64_t p[kRowGroup + 1];
#pragma unroll
    for (int k = 0; k <= kRowGroup; ++k) p[k] = __shfl_sync(0xffffffffu, pv, k);
    bool all_short = (nr == kRowGroup);
#pragma unroll
    for (int k = 0; k < kRowGroup; ++k) all_short = all_short && (p[k + 1] - p[k] <= kShortRow);
    if (all_short) {
      const int sub = lane >> 3, sl = lane & 7;
      const int64_t s = sub == 0 ? p[0] : sub == 1 ? p[1] : sub == 2 ? p[2] : p[3];
      const int64_t e = sub == 0 ? p[1] : sub == 1 ? p[2] : sub == 2 ? p[3] : p[4];
      const int64_t q = s + sl;
      const bool ok = q < e;
      int32_t cc = ok ? ld_stream(idx + q) : 0;
      double vv = ok ? ld_stream(val + q) : 0.0;
      double xx = ok ? __ldg(x + cc) : 0.0;
      if (SCALE_X) xx = xx * sx;
      Acc<MODE> a;
      a.zero();
      a.mac(vv, xx);
      lanes_reduce<8, MODE>(a);
      if (sl == 0) row_epilogue<MODE, OP>(a, y, (int64_t)g + sub, c, sy, nsq);
    } else {
#pragma unroll
      for (int k = 0; k < kRowGroup; ++k) {
        if (k < nr) {
          Acc<MODE> a = row_dot<MODE, VT, SCALE_X>(idx, val, x, p[k], p[k + 1], lane, sx);
          lanes_reduce<32, MODE>(a);
          if (lane == 0) row_epilogue<MODE, OP>(a, y, (int64_t)g + k, c, sy, nsq);
        }
      }
    }
  }
  if (OP == OP_PLAIN) return;
  lanes_reduce<32, MODE>(nsq);
  block_combine<MODE>(nsq, s_slots);
  if (publish_and_ticket(partials, nsq.pack(), &sc->ticket[0], &s_flag)) {
    double total = final_sum<MODE>(partials, gridDim.x, s_slots);
    if (threadIdx.x == 0) {
      if (OP == OP_K1) tail_k1(sc, total);
      if (OP == OP_K2) tail_k2(sc, total);
      if (OP == OP_K2_INIT) tail_init_v(sc, total);
      sc->ticket[0] = 0u;
    }
  }
}

// Fused vector kernels: one pass, scale + axpy + norm^2, static grid-stride
// assignment so that the fast-mode partial sums have a fixed order.
//   VOP_INIT_U : u^ = b ; ||b||^2                               (len = m; in0 = b, out0 = u^)
//   VOP_INIT_VW: v = v^ * (1/alpha) ; w = v                     (len = n; io0 = v, out1 = w)
//   VOP_K4     : v = v^ * (1/alpha) ; sum (w*rrho)^2 ; x += t1 w ; w = v + t2 w   (io0 = v, io1 = w, io2 = x)
template <int MODE, int VOP>
__global__ void __launch_bounds__(kThreads) k_vec(const double* __restrict__ in0, double* __restrict__ a0,
                                                  double* __restrict__ a1, double* __restrict__ a2, int64_t len,
                                                  Scalars* sc, double2* partials) {
  __shared__ double2 s_slots[kWarps];
  __shared__ int s_flag;
  if (VOP != VOP_INIT_U && sc->stop) return;
  Acc<MODE> acc;
  acc.zero();
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  const int64_t i0 = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (VOP == VOP_INIT_U) {
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
  } else {
    const double ra = sc->ralpha, t1 = sc->t1, t2 = sc->t2, rrho = sc->rrho;
    const bool norm_v = sc->norm_v != 0;
    for (int64_t i = i0; i < len; i += stride) {
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
  if (publish_and_ticket(partials, acc.pack(), &sc->ticket[1], &s_flag)) {
    double total = final_sum<MODE>(partials, gridDim.x, s_slots);
    if (threadIdx.x == 0) {
      if (VOP == VOP_INIT_U) tail_init_u(sc, total);
      if (VOP == VOP_K4) tail_k4(sc, total);
      sc->ticket[1] = 0u;
    }
  }
}

}  // namespace tomo
