// accum.cuh — accumulators for the inner products of the LSQR hot path (device code only).
//
// Two accumulation modes (reading R-dd):
//   MODE 0 "fast": fp64 FMA chains, several per lane, combined in a fixed order  -> deterministic,
//                  within rounding of any other summation order.
//   MODE 1 "dd"  : every product is formed exactly (TwoProd by FMA) and added into an unevaluated
//                  double-double (hi, lo) (Knuth TwoSum); partial sums of lanes / warps / blocks are
//                  combined by a dd+dd addition and the total is rounded to fp64 ONCE.  The rounded
//                  result is a faithful rounding of the exact sum, and the correctly rounded one unless the
//                  exact sum lies within ~2^-100 relative of a rounding boundary (probability ~1e-14 * cond
//                  per sum), hence independent of the order of summation in practice, which is what makes
//                  the fixed-k iterate reproducible at scale (the tests assert it bitwise and record it).
// This translation unit is compiled with --fmad=false: a fused multiply-add exists only where fma() is
// written, so the error-free transformations below are not contracted away.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace tomo {

struct dd_t {
  double hi, lo;
};

// Programmatic dependent launch (the kernels of an iteration are chained with
// cudaLaunchAttributeProgrammaticStreamSerialization): everything above grid_dependency_wait() may run while
// the previous kernel drains; nothing that kernel writes is read before it.  launch_dependents() lets the next
// kernel's CTAs start their prologue.  Both are no-ops in a launch without the attribute.
__device__ __forceinline__ void grid_dependency_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void grid_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

__device__ __forceinline__ void two_sum(double a, double b, double& s, double& t) {
  s = a + b;
  double bb = s - a;
  t = (a - (s - bb)) + (b - bb);
}

__device__ __forceinline__ dd_t dd_add(dd_t a, dd_t b) {
  double s, t;
  two_sum(a.hi, b.hi, s, t);
  t = t + (a.lo + b.lo);
  dd_t r;
  r.hi = s + t;
  r.lo = t - (r.hi - s);
  return r;
}

__device__ __forceinline__ double shfl_down_f64(double v, int off) { return __shfl_down_sync(0xffffffffu, v, off); }

template <int MODE>
struct Acc;

template <>
struct Acc<0> {
  double s;
  __device__ __forceinline__ void zero() { s = 0.0; }
  __device__ __forceinline__ void mac(double a, double b) { s = fma(a, b, s); }
  __device__ __forceinline__ void merge(const Acc& o) { s = s + o.s; }
  __device__ __forceinline__ void mac8(const double (&a)[8], const double (&b)[8]) {  // fixed tree
    const double t0 = fma(a[1], b[1], a[0] * b[0]), t1 = fma(a[3], b[3], a[2] * b[2]);
    const double t2 = fma(a[5], b[5], a[4] * b[4]), t3 = fma(a[7], b[7], a[6] * b[6]);
    s = s + ((t0 + t1) + (t2 + t3));
  }
  __device__ __forceinline__ Acc down(int off) const {
    Acc r;
    r.s = shfl_down_f64(s, off);
    return r;
  }
  __device__ __forceinline__ double value() const { return s; }
  __device__ __forceinline__ double2 pack() const { return make_double2(s, 0.0); }
  __device__ __forceinline__ void unpack(double2 p) { s = p.x; }
};

template <>
struct Acc<1> {
  dd_t v;
  __device__ __forceinline__ void zero() { v.hi = 0.0; v.lo = 0.0; }
  // hi carries the fp64 running sum, lo the running sum of the exact rounding errors of every product
  // (TwoProd by FMA) and every addition (Knuth TwoSum); (hi, lo) is not renormalised per term (the
  // loop-carried dependency is one add on hi and one on lo), merge() and value() take it as it is.
  __device__ __forceinline__ void mac(double a, double b) {
    double p = a * b;
    double e = fma(a, b, -p);
    double s, q;
    two_sum(v.hi, p, s, q);
    v.hi = s;
    v.lo = v.lo + (q + e);
  }
  __device__ __forceinline__ void merge(const Acc& o) {  // TwoSum of the his, errors collected in lo
    double s, q;
    two_sum(v.hi, o.v.hi, s, q);
    v.hi = s;
    v.lo = (v.lo + o.v.lo) + q;
  }
  // the products of eight (a, b) pairs at once: exact products (TwoProd), a TwoSum tree over them and
  // one plain sum of all the rounding errors; same flop count as eight mac() calls, a third of the depth
  __device__ __forceinline__ void mac8(const double (&a)[8], const double (&b)[8]) {
    double p[8], e[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) { p[u] = a[u] * b[u]; e[u] = fma(a[u], b[u], -p[u]); }
    double s01, q01, s23, q23, s45, q45, s67, q67, s03, q03, s47, q47, s07, q07;
    two_sum(p[0], p[1], s01, q01); two_sum(p[2], p[3], s23, q23);
    two_sum(p[4], p[5], s45, q45); two_sum(p[6], p[7], s67, q67);
    two_sum(s01, s23, s03, q03); two_sum(s45, s67, s47, q47);
    two_sum(s03, s47, s07, q07);
    const double err = ((((e[0] + e[1]) + (e[2] + e[3])) + ((e[4] + e[5]) + (e[6] + e[7]))) +
                        ((q01 + q23) + (q45 + q67))) + ((q03 + q47) + q07);
    double s, q;
    two_sum(v.hi, s07, s, q);
    v.hi = s;
    v.lo = v.lo + (q + err);
  }
  __device__ __forceinline__ Acc down(int off) const {
    Acc r;
    r.v.hi = shfl_down_f64(v.hi, off);
    r.v.lo = shfl_down_f64(v.lo, off);
    return r;
  }
  __device__ __forceinline__ double value() const { return v.hi + v.lo; }
  __device__ __forceinline__ double2 pack() const { return make_double2(v.hi, v.lo); }
  __device__ __forceinline__ void unpack(double2 p) { v.hi = p.x; v.lo = p.y; }
};

// Sum over the lanes [base, base+WIDTH) of a warp, result valid in lane `base` (WIDTH = 32 or 8).
template <int WIDTH, int MODE>
__device__ __forceinline__ void lanes_reduce(Acc<MODE>& a) {
#pragma unroll
  for (int off = WIDTH / 2; off >= 1; off >>= 1) a.merge(a.down(off));
}

// Fixed-order block combine of one accumulator per warp (valid in lane 0 of each warp): result in
// thread 0.  `slots` is shared memory for blockDim.x/32 double2.
template <int MODE>
__device__ __forceinline__ void block_combine(Acc<MODE>& a, double2* slots) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
  if (lane == 0) slots[warp] = a.pack();
  __syncthreads();
  if (threadIdx.x == 0) {
    a.unpack(slots[0]);
    for (int w = 1; w < nw; ++w) {
      Acc<MODE> o;
      o.unpack(slots[w]);
      a.merge(o);
    }
  }
}

// The last-arriving block of a launch sums the per-block partials in index order (bitwise
// reproducible) and returns the total in thread 0.  Call with all threads of that block.
template <int MODE>
__device__ __forceinline__ double final_sum(const double2* partials, int count, double2* slots) {
  Acc<MODE> a;
  a.zero();
  for (int i = threadIdx.x; i < count; i += blockDim.x) {
    Acc<MODE> o;
    o.unpack(__ldcg(partials + i));
    a.merge(o);
  }
  lanes_reduce<32, MODE>(a);
  __syncthreads();
  block_combine<MODE>(a, slots);
  return a.value();
}

// the same, unrounded: the (hi, lo) pair of the total in thread 0 (sharded solve: the sum is closed after an exchange)
template <int MODE>
__device__ __forceinline__ double2 final_sum_pair(const double2* partials, int count, double2* slots) {
  Acc<MODE> a;
  a.zero();
  for (int i = threadIdx.x; i < count; i += blockDim.x) {
    Acc<MODE> o;
    o.unpack(__ldcg(partials + i));
    a.merge(o);
  }
  lanes_reduce<32, MODE>(a);
  __syncthreads();
  block_combine<MODE>(a, slots);
  return a.pack();
}

// Publish this block's partial and find out whether it is the last block of the launch.
__device__ __forceinline__ bool publish_and_ticket(double2* partials, double2 mine, unsigned int* ticket, int* s_flag) {
  if (threadIdx.x == 0) {
    __stcg(partials + blockIdx.x, mine);
    __threadfence();
    unsigned int t = atomicAdd(ticket, 1u);
    *s_flag = (t == gridDim.x - 1) ? 1 : 0;
  }
  __syncthreads();
  bool last = (*s_flag != 0);
  if (last) __threadfence();
  return last;
}

}  // namespace tomo
