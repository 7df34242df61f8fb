// wstream.cuh — the streaming SpMV kernel of the LSQR hot path, warp-private streams:
//     K1  u^ <- A v - alpha u     + ||u^||^2 -> tail: beta, 1/beta, anorm           (over the caller's CSR)
//     K2  v^ <- A^T u - beta v    + ||v^||^2 -> tail: alpha, rotations, estimates   (over the CSC copy)
// "sparse matrix-vector multiplications and vector norm calculations" are what the paper's GPU solver
// offloads; here both are one kernel, with the axpy and the norm fused in.
//
// Design (B200: 148 SMs, HBM3e-bound, TMA engine, 227 KB shared memory per SM):
//   * One persistent CTA per SM, W warps.  Every WARP owns one contiguous ELEMENT range [E_w, E_{w+1}) of the
//     matrix arrays (cost-balanced, boundaries at multiples of the tile size, not aligned to rows) and streams
//     it through its own NS-stage shared-memory ring: lane 0 issues the cp.async.bulk copies (TMA engine, L2
//     evict-first) of the next tile as soon as the warp has moved the previous one to registers, completion
//     is signalled on the warp's own mbarrier.  No warp ever waits for another warp: there is no CTA-wide
//     barrier, no producer and no resolver warp between the first and the last element of a launch.
//   * A tile is consumed in rounds of 256 elements (eight 32-element steps): the round's matrix entries go
//     to registers and all eight gathers of x are issued at once; the gathers of round r+1 are in flight
//     while round r is multiplied and summed (two register sets), which hides the L2 latency of the gather; the
//     values are read from the ring when the round is summed.
//   * The per-lane accumulator of the open row lives across rounds and tiles.  A round that lies inside one row
//     is eight exact products and a TwoSum tree (`mac8`); pairs of such rounds run a straight-line copy of the
//     round in which the two gather register sets swap roles.  Where a row ends, its 32 per-lane partials are
//     parked in shared memory and every fourth row end one common reduction closes four rows (close_row /
//     flush_rows).  A step with several row ends (short rows: the 4-7-entry smoothing rows) uses a segmented
//     warp reduction whose cost does not depend on the number of rows in the step.  Row starts come from a 64-entry register window of the row pointers
//     (two registers per lane, refilled 32 rows at a time, one refill ahead).
//   * The two rows a warp range may cut (the one open at its start, the one open at its end) leave one
//     record per warp; warp 0 chains the W records of the CTA with a log-step scan over "carry maps" (fixed
//     tree order: deterministic) and leaves one record per CTA; the last-arriving CTA of the launch chains
//     those, sums the per-CTA ||.||^2 partials in index order and runs the scalar step (tails.cuh).
//   * Rows without entries never enter the stream: create compacts them away (ptr = starts of the non-empty
//     rows, rid = their row numbers) and lists them; the kernel gives them y_r <- c y_r in a side pass.
//   * FMT 1 (run-compressed index; structure from Eq. 5 P:69-71 and the
//     depth-fastest ordering Eq. 7): instead of one int32 per element the tile carries one bit per
//     element ("starts a run of consecutive indices") and one int32 per run head (a head is forced at every
//     32-element step); the lane rebuilds its index with one popc and one shared load (compress.cuh).
// Every assignment (ranges, tiles, rounds, reduction trees) is static, so results are bitwise reproducible in
// both accumulation modes; in dd mode they are moreover independent of all of it (DESIGN.md R-dd).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "accum.cuh"
#include "state.cuh"
#include "tails.cuh"

namespace tomo {

// ---- shapes -------------------------------------------------------------------------------------
template <int TILE_, int NS_, int W_>
struct WCfg {
  static constexpr int TILE = TILE_;      // elements per tile (multiple of 256); range boundaries are multiples of it
  static constexpr int NS = NS_;          // ring stages per warp
  static constexpr int W = W_;            // warps per CTA
  static constexpr int RPT = TILE_ / 256; // rounds per tile
  static constexpr int THREADS = 32 * W_;
  static_assert(TILE_ % 256 == 0 && (RPT & (RPT - 1)) == 0, "tile = 256 * 2^k elements");
};

struct CtaRec {        // what a warp (shared memory) or a CTA (global memory) leaves for the chain over records
  double2 head;        // partial sum of the row that was open at the range start
  double2 tail;        // partial sum of the row that started in the range and continues behind it
  int head_state;      // 0 none, 1 that row continues behind the range, 2 it ended inside the range
  int tail_state;      // 0 none, 1 present
  int tail_row;        // (compact) row number of the tail
  int pad;             // CTA records: busy time of the CTA in 16-cycle units
};

constexpr int kBig = 0x3fffffff;  // "beyond the range" for relative element offsets
#ifndef TOMO_PEND
#define TOMO_PEND 4
#endif
constexpr int kPendRows = TOMO_PEND;  // finished rows whose per-lane partials wait in shared memory for one common reduction (1, 2, 4 or 8)

template <typename CFG, typename VT, int FMT>
struct WSmem {
  // FMT 0: int32 index per element.  FMT 1: TILE/8 bytes of run flags + up to TILE run heads (int32).
  static constexpr size_t kIdx = (FMT == 0) ? sizeof(int32_t) * CFG::TILE : sizeof(int32_t) * CFG::TILE + CFG::TILE / 8 + 16;
  static constexpr size_t kVal = sizeof(VT) * CFG::TILE;
  static constexpr size_t kStage = kIdx + kVal;
  static constexpr size_t kWarp = kStage * CFG::NS;
  static constexpr size_t kBars = 8 * CFG::NS * CFG::W;
  static constexpr size_t kRec = sizeof(CtaRec) * CFG::W;
  static constexpr size_t kSlots = sizeof(double2) * CFG::W + 16;
  static constexpr size_t kPendWarp = sizeof(double2) * 32 * kPendRows + 16 * kPendRows;  // batched row ends (close_row)
  static constexpr size_t kTotal = kWarp * CFG::W + kBars + kRec + kSlots + kPendWarp * CFG::W;
  static_assert(kStage % 16 == 0 && kIdx % 16 == 0, "bulk copies need 16-byte aligned destinations");
};

// ---- PTX wrappers: mbarrier, bulk async copy ------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1, 0x989680;\n"  // suspend-time hint (ns): sleep, do not spin
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx_a(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait_a(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1, 0x989680;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}" ::"r"(bar),
      "r"(parity)
      : "memory");
}
__device__ __forceinline__ void bulk_g2s_a(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar, uint64_t policy) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(dst),
               "l"(src), "r"(bytes), "r"(bar), "l"(policy)
               : "memory");
}
__device__ __forceinline__ uint64_t l2_evict_first_policy() {
  uint64_t p;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
  return p;
}
// global -> shared bulk copy executed by the TMA engine; dst, src 16-byte aligned, bytes % 16 == 0
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar, uint64_t policy) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(
                   smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar)), "l"(policy)
               : "memory");
}
// generic-proxy reads of a stage are ordered before the async-proxy (TMA) writes that refill it
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
// one lane of the (converged) warp
__device__ __forceinline__ bool elect_one() {
  uint32_t pred;
  asm volatile("{\n.reg .pred P;\nelect.sync _|P, 0xffffffff;\nselp.u32 %0, 1, 0, P;\n}" : "=r"(pred));
  return pred != 0;
}
// warp-uniform copies (lane 0's value): lets the compiler keep addresses of the bulk copies in uniform registers
__device__ __forceinline__ int uni(int v) { return __shfl_sync(0xffffffffu, v, 0); }
__device__ __forceinline__ int64_t uni(int64_t v) {
  const int lo = __shfl_sync(0xffffffffu, (int)(uint32_t)(uint64_t)v, 0), hi = __shfl_sync(0xffffffffu, (int)((uint64_t)v >> 32), 0);
  return (int64_t)(((uint64_t)(uint32_t)hi << 32) | (uint32_t)lo);
}
__device__ __forceinline__ void prefetch_l1(const void* p) { asm volatile("prefetch.global.L1 [%0];" ::"l"(p)); }

template <int MODE>
__device__ __forceinline__ Acc<MODE> acc_bcast(const Acc<MODE>& a, int src) {
  Acc<MODE> r;
  double2 p = a.pack();
  p.x = __shfl_sync(0xffffffffu, p.x, src);
  p.y = __shfl_sync(0xffffffffu, p.y, src);
  r.unpack(p);
  return r;
}
template <int MODE>
__device__ __forceinline__ Acc<MODE> acc_of(double2 p) {
  Acc<MODE> r;
  r.unpack(p);
  return r;
}

// y_r <- sum + c * (yo * sy) and the running ||y||^2 (the fused axpy + norm of K1 / K2); yo = old y_r
template <int MODE, int OP>
__device__ __forceinline__ void finish_row_with(Acc<MODE> sum, double yo, double* __restrict__ y, int64_t r, double c,
                                                double sy, Acc<MODE>& nsq) {
  if (OP == OP_K2S) {  // the unrounded partial column sum of this row block: closed after the exchange (shard.cuh)
    reinterpret_cast<double2*>(y)[r] = sum.pack();
    return;
  }
  double yn;
  if (OP == OP_K1 || OP == OP_K2 || OP == OP_K1S) {
    if (OP == OP_K1 || OP == OP_K1S) yo = yo * sy;
    if (MODE == 0) {
      yn = fma(c, yo, sum.value());
    } else {
      sum.mac(c, yo);
      yn = sum.value();
    }
  } else {
    yn = sum.value();
  }
  y[r] = yn;
  if (OP != OP_PLAIN) nsq.mac(yn, yn);
}

// The chain over records as a warp scan.  Lane l holds the record of range l: an optional head piece (state 1:
// its row continues, 2: its row ends here) followed by an optional tail piece (a row that starts here and
// continues).  Each record is a map on the carry (partial sum and id of the open row):
//   tail present -> carry := tail ;  head ends -> carry := none ;  else carry := carry + head
// Maps compose associatively, so all carries come out of a 5-step Kogge-Stone scan in a fixed tree order
// (deterministic) instead of a serial walk.  Returns, per lane, the row that ends in this record (emit_row >= 0,
// or -2: the row that entered the chained ranges from the left) with its complete sum.
template <int MODE>
__device__ __forceinline__ void chain_scan(int hs, int ts, Acc<MODE> head, Acc<MODE> tail, int tail_row,
                                           Acc<MODE>& carry, int& carry_row, bool& emit, Acc<MODE>& emit_sum,
                                           int& emit_row) {
  const int lane = threadIdx.x & 31;
  int A = (ts || hs == 2) ? 0 : 1;
  Acc<MODE> B;
  B.zero();
  if (ts) B = tail; else if (hs == 1) B = head;
  int R = ts ? tail_row : -1;
#pragma unroll 1  // not on the critical path: keep the code small
  for (int d = 1; d < 32; d <<= 1) {
    const int A1 = __shfl_up_sync(0xffffffffu, A, d);
    const int R1 = __shfl_up_sync(0xffffffffu, R, d);
    double2 bp = B.pack();
    bp.x = __shfl_up_sync(0xffffffffu, bp.x, d);
    bp.y = __shfl_up_sync(0xffffffffu, bp.y, d);
    if (lane >= d && A) {  // own map keeps the carry: the earlier map's result flows through
      Acc<MODE> B1 = acc_of<MODE>(bp);
      B1.merge(B);
      B = B1;
      R = R1;
      A = A1;
    }
  }
  int Aex = __shfl_up_sync(0xffffffffu, A, 1);
  int Rex = __shfl_up_sync(0xffffffffu, R, 1);
  double2 bex = B.pack();
  bex.x = __shfl_up_sync(0xffffffffu, bex.x, 1);
  bex.y = __shfl_up_sync(0xffffffffu, bex.y, 1);
  if (lane == 0) { Aex = 1; Rex = -1; bex = make_double2(0.0, 0.0); }
  Acc<MODE> cin = acc_of<MODE>(bex);
  int rin = Rex;
  if (Aex) { Acc<MODE> t = carry; t.merge(cin); cin = t; rin = carry_row; }
  emit = (hs == 2);
  emit_sum = cin;
  if (hs) emit_sum.merge(head);
  emit_row = rin;
  const int Al = __shfl_sync(0xffffffffu, A, 31), Rl = __shfl_sync(0xffffffffu, R, 31);
  Acc<MODE> Bl = acc_bcast<MODE>(B, 31);
  if (Al) { carry.merge(Bl); } else { carry = Bl; carry_row = Rl; }
}

// ---- per-warp sweep state -----------------------------------------------------------------------------
template <int MODE>
struct WSweep {
  Acc<MODE> acc;     // per-lane partial of the open row
  Acc<MODE> nsq;     // per-lane partial of ||y||^2
  double yold;       // lane 0: old y of the open row (requested when the row opens)
  double2 h_val;     // head record value (valid in lane 0)
  int h_state;       // head record state
  int cur;           // (compact) number of the open row; R0 - 1: the row that was open at the range start
  int next_b;        // relative offset where the open row ends (>= len: behind the range)
  int wbase;         // first row of the register window
  int S, S2;         // window: relative starts of rows wbase + lane and wbase + 32 + lane (kBig beyond row R1)
  int np;            // rows waiting in the pend buffer
  bool started;      // the open row starts inside this range
};

struct WCtx {        // uniform, read-only
  const int64_t* ptr; const int32_t* rid; double* y; int64_t E0; int R0, R1, len; double c, sy;
  double2* pend;     // per warp: [kPendRows][32] per-lane partials of finished rows, then [kPendRows] {old y, row number}
};

__device__ __forceinline__ int win_load(const WCtx& cx, int rbase) {
  const int lane = threadIdx.x & 31;
  const int r = rbase + lane;
  if (r > cx.R1 || r < 0) return kBig;
  const int64_t p = cx.ptr[r] - cx.E0;
  return p >= (int64_t)kBig ? kBig : (int)p;
}
// start of row r (uniform), wbase <= r < wbase + 64
template <typename ST>
__device__ __forceinline__ int win_get(const ST& st, int r) {
  const int i = r - st.wbase;
  const int a = __shfl_sync(0xffffffffu, st.S, i & 31), b = __shfl_sync(0xffffffffu, st.S2, i & 31);
  return i < 32 ? a : b;
}
// keep cur + 1 inside the first half of the window
template <typename ST>
__device__ __forceinline__ void win_advance(ST& st, const WCtx& cx) {
  while (st.cur + 1 - st.wbase >= 32) {
    st.S = st.S2;
    st.wbase += 32;
    st.S2 = win_load(cx, st.wbase + 32);
  }
}
__device__ __forceinline__ int64_t row_number(const WCtx& cx, int k) { return cx.rid ? (int64_t)cx.rid[k] : (int64_t)k; }

// The rows that ended since the last flush: their per-lane partials sit in shared memory, [slot][lane].  32 / kPendRows
// lanes per row add kPendRows partials each (with 4 rows: lane q takes lanes q, q+8, q+16, q+24: conflict-free), a
// butterfly closes the sum, the first lane of each group finishes its row.  One reduction for kPendRows rows instead of one (5 shuffle
// steps + the finish code in ONE lane) per row.
template <int MODE, int OP>
__device__ __forceinline__ void flush_rows(WSweep<MODE>& st, const WCtx& cx) {
  const int lane = threadIdx.x & 31;
  __syncwarp();
  constexpr int LPR = 32 / kPendRows;  // lanes per row
  const int k = lane / LPR, q = lane % LPR;
  const double2* p = cx.pend + k * 32 + q;
  Acc<MODE> a = acc_of<MODE>(p[0]);
#pragma unroll
  for (int i = 1; i < kPendRows; ++i) a.merge(acc_of<MODE>(p[LPR * i]));
#pragma unroll
  for (int off = 1; off < LPR; off <<= 1) {
    double2 o = a.pack();
    o.x = __shfl_xor_sync(0xffffffffu, o.x, off);
    o.y = __shfl_xor_sync(0xffffffffu, o.y, off);
    a.merge(acc_of<MODE>(o));
  }
  if (q == 0 && k < st.np) {
    const double2 meta = cx.pend[32 * kPendRows + k];  // {old y, row number}
    finish_row_with<MODE, OP>(a, meta.x, cx.y, row_number(cx, (int)__double_as_longlong(meta.y)), cx.c, cx.sy, st.nsq);
  }
  __syncwarp();
  st.np = 0;
}

// the open row ends here: st.acc holds its per-lane partials
template <int MODE, int OP>
__device__ __forceinline__ void close_row(WSweep<MODE>& st, const WCtx& cx) {
  const int lane = threadIdx.x & 31;
  if (!st.started) {  // the row that was open at the range start: its sum goes to the warp's record (once per range)
    lanes_reduce<32, MODE>(st.acc);
    if (lane == 0) { st.h_val = st.acc.pack(); st.h_state = 2; }
    return;
  }
  cx.pend[st.np * 32 + lane] = st.acc.pack();
  if (lane == 0) cx.pend[32 * kPendRows + st.np] = make_double2(st.yold, __longlong_as_double((long long)st.cur));
  if (++st.np == kPendRows) flush_rows<MODE, OP>(st, cx);
}

// One 32-element step [base, base+32) in which the open row ends (base < next_b <= base + 32): close it, then
// give the remaining lanes' products to the rows that follow; rows that end inside the step are reduced
// (segmented, 5 shuffle steps whatever their number) and finished, the last one becomes the open row if it
// runs on.  One copy in the code, called from a non-unrolled loop.
template <int MODE, int OP>
__device__ __forceinline__ void slow_step(WSweep<MODE>& st, const WCtx& cx, double v, double x, int base) {
  constexpr bool NEEDS_Y = (OP == OP_K1 || OP == OP_K2 || OP == OP_K1S);
  const int lane = threadIdx.x & 31;
  const int hi = min(base + 32, cx.len);
  const int pos = base + lane;
  // (1) the last piece of the open row
  {
    const bool mine = pos < st.next_b;
    st.acc.mac(mine ? v : 0.0, mine ? x : 0.0);  // other lanes add an exact zero
    close_row<MODE, OP>(st, cx);
    st.acc.zero();
  }
  const int lo = st.next_b;
  if (lo >= cx.len) { st.next_b = kBig; st.started = true; return; }  // the range ends with this row: nothing is open
  if (lo < hi) {
    // (2) rows cur+1, cur+2, ... start inside [lo, hi): T = starts of rows cur+2+lane; a lane's row is
    // cur + 1 + (number of those starts <= pos)
    const int i = st.cur + 2 - st.wbase + lane;
    const int ta = __shfl_sync(0xffffffffu, st.S, i & 31), tb = __shfl_sync(0xffffffffu, st.S2, i & 31);
    const int T = (i < 32) ? ta : ((i < 64) ? tb : kBig);
    const unsigned bit = (T < hi) ? (1u << (T - base)) : 0u;  // hi: a row starting at the range end is not ours
    const unsigned M = __reduce_or_sync(0xffffffffu, bit);
    const bool valid = pos >= lo && pos < hi;
    const int k = __popc(M & ((2u << lane) - 1u));
    const int klast = __popc(M);                                  // the last row that starts inside the step
    const int end_last = __shfl_sync(0xffffffffu, T, klast);      // where it ends
    const bool closes_last = end_last <= hi;
    Acc<MODE> t;
    t.zero();
    if (valid) t.mac(v, x);
    if (klast == 0 && !closes_last) {  // one row starts here and runs on (long rows): it is the open row, no reduction
      st.acc = t;
      st.cur = st.cur + 1;
      st.started = true;
      st.next_b = end_last;
      if (NEEDS_Y && lane == 0) st.yold = cx.y[row_number(cx, st.cur)];
      win_advance(st, cx);
      return;
    }
    const Acc<MODE> t0 = t;
    const int kk0 = valid ? k : -1;
    const int kprev = __shfl_up_sync(0xffffffffu, kk0, 1);
    const bool head = valid && (pos == lo || kprev != k);
    const bool fin = head && (k < klast || closes_last);
    double yo = 0.0;
    int64_t rn = 0;
    if (fin) { rn = row_number(cx, st.cur + 1 + k); if (NEEDS_Y) yo = cx.y[rn]; }
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      Acc<MODE> o = t.down(d);
      const int kd = __shfl_down_sync(0xffffffffu, kk0, d);
      if (lane + d < 32 && kd == kk0) t.merge(o);
    }
    if (fin) finish_row_with<MODE, OP>(t, yo, cx.y, rn, cx.c, cx.sy, st.nsq);
    st.cur = st.cur + 1 + klast;
    st.started = true;
    if (!closes_last) {  // the last row runs on: it is the open row, every lane keeps its own product
      if (valid && k == klast) st.acc = t0;
      st.next_b = end_last;
      if (NEEDS_Y && lane == 0) st.yold = cx.y[row_number(cx, st.cur)];
      win_advance(st, cx);
      return;
    }
    if (hi >= cx.len) { st.next_b = kBig; return; }  // range finished exactly at a row end
    // the step ends exactly at a row end: the next row opens at base + 32
  }
  st.cur = st.cur + 1;
  st.started = true;
  win_advance(st, cx);
  st.next_b = win_get(st, st.cur + 1);
  if (NEEDS_Y && lane == 0) st.yold = cx.y[row_number(cx, st.cur)];
}

// The products of one round (8 steps of 32 elements at relative offset pos0) go to the rows they belong to.
// Three shapes.  P0: the round lies inside the open row (long rows: the common case).  P1: exactly one row ends
// inside it and the next one runs on behind the round.  P2: anything else (short rows, the last round of the
// range), step by step through one shared copy of the general code.
template <int MODE, int OP, bool SCALE_X>
__device__ __forceinline__ void consume_round(WSweep<MODE>& st, const WCtx& cx, double (&vv)[8], double (&xx)[8], int pos0,
                                              double sx) {
  constexpr bool NEEDS_Y = (OP == OP_K1 || OP == OP_K2 || OP == OP_K1S);
  const int lane = threadIdx.x & 31;
  if (SCALE_X) {
#pragma unroll
    for (int u = 0; u < 8; ++u) xx[u] = xx[u] * sx;
  }
  const int pend = pos0 + 256;
  if (st.next_b > pend) {  // P0 (lanes behind the range hold zeros)
    st.acc.mac8(vv, xx);
    return;
  }
  if (pend <= cx.len) {
    const int nb2 = win_get(st, st.cur + 2);  // end of the row that starts where the open one ends
    if (st.next_b == pend || nb2 > pend) {    // P1
      const int pe = st.next_b;               // pos0 < pe <= pend
      const int us = (pe - pos0) >> 5;        // step that holds the row end (8: the round ends with the row)
      const bool first = pos0 + 32 * us + lane < pe;
      Acc<MODE> accB;
      accB.zero();
      double yold_new = 0.0;
      if (NEEDS_Y && lane == 0 && pe < cx.len) yold_new = cx.y[row_number(cx, st.cur + 1)];
#pragma unroll
      for (int u = 0; u < 8; ++u) {
        if (u < us) st.acc.mac(vv[u], xx[u]);
        else if (u > us) accB.mac(vv[u], xx[u]);
        else {
          st.acc.mac(first ? vv[u] : 0.0, first ? xx[u] : 0.0);
          accB.mac(first ? 0.0 : vv[u], first ? 0.0 : xx[u]);
        }
      }
      close_row<MODE, OP>(st, cx);
      st.acc = accB;
      st.started = true;
      if (pe >= cx.len) { st.next_b = kBig; return; }  // the range ends with this row
      st.cur = st.cur + 1;
      st.next_b = nb2;
      st.yold = yold_new;
      win_advance(st, cx);
      return;
    }
  }
#pragma unroll 1
  for (int u = 0; u < 8; ++u) {  // P2
    const int base = pos0 + 32 * u;
    if (base >= cx.len) break;
    double v = vv[0], x = xx[0];
#pragma unroll
    for (int k = 1; k < 8; ++k) { v = (u == k) ? vv[k] : v; x = (u == k) ? xx[k] : x; }
    if (st.next_b > base + 32) st.acc.mac(v, x);
    else slow_step<MODE, OP>(st, cx, v, x, base);
  }
}

// ---- the kernel -----------------------------------------------------------------------------------
// ptr/rid/idx/val: CSR-like triple over the NON-EMPTY rows (K1: the CSR of A; K2: the CSC copy, i.e. the CSR
// of A^T): ptr[k] = first element of the k-th non-empty row, ptr[nrows] = nnz, rid[k] = its row number (NULL:
// no empty rows, rid = identity).  erows[0..n_empty): the rows without elements.  wE[g], wR[g] (g = 0 ..
// gridDim.x * W): element split points (multiples of TILE, wE[last] = nnz) and the first row with
// ptr[row] >= wE[g] (wR[last] = nrows).  FMT 1: idx is unused; cidx/coff hold the run-compressed index
// (one record of TILE/8 flag bytes + 4 bytes per run head per tile, coff[t] = byte offset of tile t's record).
template <typename CFG, int MODE, typename VT, int OP, int FMT>
__global__ void __launch_bounds__(CFG::THREADS, 1)
k_wstream(const int64_t* __restrict__ ptr, const int32_t* __restrict__ rid, const int32_t* __restrict__ idx,
          const VT* __restrict__ val, const unsigned char* __restrict__ cidx, const int64_t* __restrict__ coff,
          int64_t nnz, int nrows, const int32_t* __restrict__ erows, int n_empty, const double* __restrict__ x,
          double* __restrict__ y, const int64_t* __restrict__ wE, const int32_t* __restrict__ wR, CtaRec* __restrict__ cta_rec,
          Scalars* sc, double2* partials) {
  constexpr int TILE = CFG::TILE, NS = CFG::NS, W = CFG::W, RPT = CFG::RPT;
  using SM = WSmem<CFG, VT, FMT>;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  constexpr bool NEEDS_Y = (OP == OP_K1 || OP == OP_K2 || OP == OP_K1S);
  constexpr bool SCALE_X = (OP == OP_K2 || OP == OP_K2_INIT || OP == OP_K2S);

  const int lane = threadIdx.x & 31, warp = uni((int)(threadIdx.x >> 5));
  const long long t_start = clock64();
  unsigned char* my_ring = smem_raw + (size_t)warp * SM::kWarp;
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem_raw + SM::kWarp * W);
  uint64_t* my_bar = bars + warp * NS;
  CtaRec* s_rec = reinterpret_cast<CtaRec*>(smem_raw + SM::kWarp * W + SM::kBars);
  double2* s_slots = reinterpret_cast<double2*>(smem_raw + SM::kWarp * W + SM::kBars + SM::kRec);
  int* s_flag = reinterpret_cast<int*>(s_slots + W);
  unsigned char* s_pend = smem_raw + SM::kWarp * W + SM::kBars + SM::kRec + SM::kSlots;

  // ---- prologue that depends on nothing the previous kernel writes: barriers, split points, first copies ----
  if (lane == 0) {
    for (int s = 0; s < NS; ++s) mbar_init(my_bar + s, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    fence_proxy_async();
  }
  __syncwarp();
  const int gw = blockIdx.x * W + warp;
  WCtx cx;
  cx.ptr = ptr; cx.rid = rid; cx.y = y;
  cx.pend = reinterpret_cast<double2*>(s_pend + (size_t)warp * SM::kPendWarp);
  cx.E0 = uni(wE[gw]);
  const int64_t E1 = uni(wE[gw + 1]);
  cx.R0 = uni(wR[gw]); cx.R1 = uni(wR[gw + 1]);
  cx.len = (int)(E1 - cx.E0);
  const int ntiles = (cx.len + TILE - 1) / TILE;
  const uint64_t policy = l2_evict_first_policy();

  // FMT 1: the tile records are issued in order, so a running byte position and a register window of 32 record
  // SIZES (refilled as the tiles go by) is all the bookkeeping the index stream needs
  const int64_t tile0 = cx.E0 / TILE;
  uint32_t csize_w = 0;  // bytes of the record of tile cbase + lane
  int cbase = 0;
  const unsigned char* cpos = cidx;
  auto csize_load = [&](int base) {
    if (FMT == 1) {
      const int t = base + lane;
      csize_w = (t < ntiles) ? (uint32_t)(coff[tile0 + t + 1] - coff[tile0 + t]) : 0u;
      cbase = base;
    }
  };
  if (FMT == 1 && ntiles > 0) { csize_load(0); cpos = cidx + uni(coff[tile0]); }

  auto stage_ptr = [&](int s) { return my_ring + (size_t)s * SM::kStage; };
  // one lane requests tile t into stage t % NS (all lanes call, converged; every operand is warp-uniform).
  // `refill`: the stage was read before (generic proxy): order those reads before the async-proxy writes.
  const uint32_t ring_a = smem_u32(my_ring), bar_a = smem_u32(my_bar);
  const VT* val0 = val + cx.E0;
  const int32_t* idx0 = (FMT == 0) ? idx + cx.E0 : nullptr;
  auto issue_tile = [&](int t, bool refill) {
    const int s = t % NS;
    if (FMT == 0 && t != ntiles - 1) {  // a full tile: constant sizes, nothing but the two copies
      __syncwarp();
      if (elect_one()) {
        if (refill) fence_proxy_async();
        const uint32_t dst = ring_a + (uint32_t)s * (uint32_t)SM::kStage, bar = bar_a + 8u * (uint32_t)s;
        mbar_arrive_expect_tx_a(bar, (uint32_t)(TILE * (4 + sizeof(VT))));
        bulk_g2s_a(dst, idx0 + (size_t)t * TILE, (uint32_t)(TILE * 4), bar, policy);
        bulk_g2s_a(dst + (uint32_t)SM::kIdx, val0 + (size_t)t * TILE, (uint32_t)(TILE * sizeof(VT)), bar, policy);
      }
      return;
    }
    if (FMT == 1 && t - cbase >= 32) csize_load(t);
    const uint32_t crec = (FMT == 1) ? (uint32_t)__shfl_sync(0xffffffffu, csize_w, t - cbase) : 0u;
    const unsigned char* csrc = cpos;
    if (FMT == 1) cpos += crec;
    if (FMT == 1 && t != ntiles - 1) {  // a full tile of the run-compressed stream: the record (variable size) and the values
      __syncwarp();
      if (elect_one()) {
        if (refill) fence_proxy_async();
        const uint32_t dst = ring_a + (uint32_t)s * (uint32_t)SM::kStage, bar = bar_a + 8u * (uint32_t)s;
        mbar_arrive_expect_tx_a(bar, crec + (uint32_t)(TILE * sizeof(VT)));
        bulk_g2s_a(dst, csrc, crec, bar, policy);
        bulk_g2s_a(dst + (uint32_t)SM::kIdx, val0 + (size_t)t * TILE, (uint32_t)(TILE * sizeof(VT)), bar, policy);
      }
      return;
    }
    const int64_t e = cx.E0 + (int64_t)t * TILE;
    unsigned char* st_base = stage_ptr(s);
    int cnt4 = TILE;
    if (t == ntiles - 1) {  // the last tile of the range may be short; < 4 elements at the very end of the arrays: ordinary loads
      const int cnt = cx.len - t * TILE;
      cnt4 = cnt & ~3;
      if (lane < cnt - cnt4) {
        reinterpret_cast<VT*>(st_base + SM::kIdx)[cnt4 + lane] = val[e + cnt4 + lane];
        if (FMT == 0) reinterpret_cast<int32_t*>(st_base)[cnt4 + lane] = idx[e + cnt4 + lane];
      }
    }
    __syncwarp();
    if (elect_one()) {
      if (refill) fence_proxy_async();
      const uint32_t bv = (uint32_t)cnt4 * (uint32_t)sizeof(VT);
      const uint32_t bi = (FMT == 0) ? (uint32_t)cnt4 * 4u : crec;
      if (bv + bi > 0) {
        mbar_arrive_expect_tx(my_bar + s, bv + bi);
        if (bi) bulk_g2s(st_base, (FMT == 0) ? (const void*)(idx + e) : (const void*)csrc, bi, my_bar + s, policy);
        if (bv) bulk_g2s(st_base + SM::kIdx, val + e, bv, my_bar + s, policy);
      } else {
        mbar_arrive(my_bar + s);
      }
    }
  };
  for (int t = 0; t < NS && t < ntiles; ++t) issue_tile(t, false);

  WSweep<MODE> st;
  st.acc.zero(); st.nsq.zero();
  st.yold = 0.0; st.h_val = make_double2(0.0, 0.0); st.h_state = 0; st.np = 0;
  st.wbase = cx.R0;
  st.S = win_load(cx, cx.R0);
  st.S2 = win_load(cx, cx.R0 + 32);

  // ---- everything below reads what the previous kernel of the iteration wrote (scalars, x, y) ----
  grid_dependency_wait();
  double c = 0.0, sx = 1.0, sy = 1.0;
  bool skip = false;
  if (OP != OP_PLAIN) {
    if (sc->stop) skip = true;
    else if (OP == OP_K2 && sc->beta_zero) {  // beta = 0: the A^T pass is skipped, the scalar step still runs
      if (blockIdx.x == 0 && threadIdx.x == 0) tail_k2(sc, 0.0);
      skip = true;
    }
    else if (OP == OP_K2S && sc->beta_zero) skip = true;  // the combine kernel runs the scalar step
    if (OP == OP_K1 || OP == OP_K1S) { c = -sc->alpha; sy = sc->rbeta; }
    if (OP == OP_K2) { c = -sc->beta; sx = sc->rbeta; }
    if (OP == OP_K2_INIT || OP == OP_K2S) { sx = sc->rbeta; }
  }
  if (skip) {  // drain the copies already requested (shared memory must not be written after the CTA exits)
    for (int t = 0; t < NS && t < ntiles; ++t) mbar_wait(my_bar + (t % NS), 0);
    return;
  }
  cx.c = c; cx.sy = sy;

  CtaRec rec;
  rec.head = make_double2(0.0, 0.0); rec.tail = make_double2(0.0, 0.0);
  rec.head_state = 0; rec.tail_state = 0; rec.tail_row = -1; rec.pad = 0;

  if (cx.len > 0) {
    const int first = __shfl_sync(0xffffffffu, st.S, 0);  // start of row R0 (>= len if no row starts in the range)
    if (first > 0) { st.cur = cx.R0 - 1; st.started = false; st.next_b = first; }
    else {
      st.cur = cx.R0; st.started = true; st.next_b = __shfl_sync(0xffffffffu, st.S, 1);
      if (NEEDS_Y && lane == 0) st.yold = y[row_number(cx, st.cur)];
    }
    const int nr = (cx.len + 255) >> 8;
    // gather for round r: the round's indices from the ring, the eight loads of x issued at once
    auto gather = [&](int r, double (&xx)[8]) {
      const int t = r / RPT, rr = r % RPT, s = t % NS;
      if (rr == 0) mbar_wait_a(bar_a + 8u * (uint32_t)s, (uint32_t)(t / NS) & 1u);
      const unsigned char* sb = stage_ptr(s);
      const int pos0 = r << 8;
      const bool full = pos0 + 256 <= cx.len;
      uint32_t cc[8];
      if (FMT == 0) {
        const uint32_t* si = reinterpret_cast<const uint32_t*>(sb) + rr * 256 + lane;
#pragma unroll
        for (int u = 0; u < 8; ++u) cc[u] = si[32 * u];
      } else {
        // run-compressed index (compress.cuh): H = head bits of the step; my run's head is the last head at or below
        // my lane: index = heads[heads before the step + popc(H & lanes <= mine) - 1] - 32 + lane (the heads are
        // stored biased by 32 - position, the lane's part of the sum sits in the gather base xl)
        const uint32_t* hw = reinterpret_cast<const uint32_t*>(sb) + rr * 8;
        const uint32_t* hp = reinterpret_cast<const uint32_t*>(sb + TILE / 8) - 1;  // -1: popc counts my own head
        const uint32_t le = 0xffffffffu >> (31 - lane);
        for (int q = 0; q < rr * 8; ++q) hp += __popc(hw[q - rr * 8]);  // heads in the earlier rounds of the tile
#pragma unroll
        for (int u = 0; u < 8; ++u) {
          const uint32_t H = hw[u];
          cc[u] = hp[__popc(H & le)];
          hp += __popc(H);
        }
      }
      const double* xg = (FMT == 0) ? x : x + lane - 32;  // FMT 1: biased heads
      if (full) {
#pragma unroll
        for (int u = 0; u < 8; ++u) xx[u] = __ldg(xg + cc[u]);
      } else {
#pragma unroll
        for (int u = 0; u < 8; ++u) xx[u] = (pos0 + 32 * u + lane < cx.len) ? __ldg(xg + cc[u]) : 0.0;
      }
    };
    // round r with its gathers in xc; the gathers of round r + 1 go to xn meanwhile
    auto body = [&](int r, double (&xc)[8], double (&xn)[8]) {
      if (r + 1 < nr) gather(r + 1, xn);
      const int t = r / RPT, rr = r % RPT;
      const VT* sv = reinterpret_cast<const VT*>(stage_ptr(t % NS) + SM::kIdx) + rr * 256 + lane;
      const int pos0 = r << 8;
      double vv[8];
      if (pos0 + 256 <= cx.len) {
#pragma unroll
        for (int u = 0; u < 8; ++u) vv[u] = (double)sv[32 * u];
      } else {
#pragma unroll
        for (int u = 0; u < 8; ++u) vv[u] = (pos0 + 32 * u + lane < cx.len) ? (double)sv[32 * u] : 0.0;
      }
      if (rr == RPT - 1 && t + NS < ntiles) issue_tile(t + NS, true);  // the tile is in registers: its stage is refilled
      consume_round<MODE, OP, SCALE_X>(st, cx, vv, xc, pos0, sx);
    };
    // a full round that lies inside the open row (P0), straight-line: gathers of the next round, values, refill, mac8
    auto straight = [&](int r, double (&xc)[8], double (&xn)[8]) {
      gather(r + 1, xn);
      const int t = r / RPT, rr = r % RPT;
      const VT* sv = reinterpret_cast<const VT*>(stage_ptr(t % NS) + SM::kIdx) + rr * 256 + lane;
      double vv[8];
#pragma unroll
      for (int u = 0; u < 8; ++u) vv[u] = (double)sv[32 * u];
      if (rr == RPT - 1 && t + NS < ntiles) issue_tile(t + NS, true);
      if (SCALE_X) {
#pragma unroll
        for (int u = 0; u < 8; ++u) xc[u] = xc[u] * sx;
      }
      st.acc.mac8(vv, xc);
    };
    double xa[8], xb[8];
    gather(0, xa);
    int r = 0;
#pragma unroll 1
    while (r < nr) {
      // pairs of rounds inside the open row: only the straight-line part exists twice in the code, the two gather
      // register sets swap roles and nothing is copied
#pragma unroll 1
      while (FMT == 0 && r + 2 < nr && st.next_b > ((r + 2) << 8)) {  // (FMT 1: the decode makes the copy too large for the instruction cache)
        straight(r, xa, xb);
        straight(r + 1, xb, xa);
        r += 2;
      }
      // any round (ONE copy of the general code: unrolling all of it twice, or moving the general row shape out of
      // line, measured slower — instruction cache / call overhead); the gathers move over
      body(r, xa, xb);
#pragma unroll
      for (int u = 0; u < 8; ++u) xa[u] = xb[u];
      ++r;
    }
    rec.head = st.h_val; rec.head_state = st.h_state;
  }
  // The row still open at the end of the range continues in the next range.  The last row that starts in the
  // range is R1 - 1 (or, if none starts, the row that was open at the range start); it ends at ptr[R1] >= E1 and
  // is open iff ptr[R1] > E1.
  if (st.np > 0) flush_rows<MODE, OP>(st, cx);  // finished rows still waiting for their reduction
  if (cx.len > 0) {
    const bool open = ptr[cx.R1] > E1;
    if (open) {
      lanes_reduce<32, MODE>(st.acc);
      if (cx.R1 > cx.R0) { rec.tail = st.acc.pack(); rec.tail_state = 1; rec.tail_row = cx.R1 - 1; }
      else { rec.head = st.acc.pack(); rec.head_state = 1; }
    }
  }

  // ---- rows without elements: y_r = c * y_r (K1 / K2) or 0 ----
  if (n_empty > 0) {
    Acc<MODE> z;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n_empty; i += gridDim.x * blockDim.x) {
      z.zero();
      const int64_t r = erows[i];
      const double yo = NEEDS_Y ? y[r] : 0.0;
      finish_row_with<MODE, OP>(z, yo, y, r, c, sy, st.nsq);
    }
  }

  // ---- chain of the CTA's W warp records (warp 0), CTA record, per-CTA partial ----
  if (lane == 0) s_rec[warp] = rec;
  __syncthreads();
  if (warp == 0) {
    double2 hv = make_double2(0.0, 0.0), tv = make_double2(0.0, 0.0);
    int hs = 0, ts = 0, trow = -1;
    if (lane < W) { hv = s_rec[lane].head; tv = s_rec[lane].tail; hs = s_rec[lane].head_state; ts = s_rec[lane].tail_state; trow = s_rec[lane].tail_row; }
    Acc<MODE> carry;
    carry.zero();
    int carry_row = -1;  // -1: no open row; -2: the row that entered the CTA's range from the previous CTA
    {
      const int64_t cE0 = wE[blockIdx.x * W], cE1 = wE[blockIdx.x * W + W];
      if (cE0 < cE1 && ptr[wR[blockIdx.x * W]] > cE0) carry_row = -2;
    }
    bool emit;
    Acc<MODE> e_sum;
    int e_row;
    chain_scan<MODE>(hs, ts, acc_of<MODE>(hv), acc_of<MODE>(tv), trow, carry, carry_row, emit, e_sum, e_row);
    CtaRec my;
    my.head = make_double2(0.0, 0.0); my.tail = make_double2(0.0, 0.0);
    my.head_state = 0; my.tail_state = 0; my.tail_row = -1;
    // the row that entered the CTA from the left ends here: its sum goes to the CTA record
    const unsigned hb = __ballot_sync(0xffffffffu, emit && e_row == -2);
    if (hb) { const int src = __ffs((int)hb) - 1; my.head = acc_bcast<MODE>(e_sum, src).pack(); my.head_state = 2; }
    if (emit && e_row >= 0) {
      const int64_t rn = row_number(cx, e_row);
      const double yo = NEEDS_Y ? y[rn] : 0.0;
      finish_row_with<MODE, OP>(e_sum, yo, y, rn, c, sy, st.nsq);
    }
    if (carry_row != -1) {
      if (carry_row == -2) { my.head = carry.pack(); my.head_state = 1; }
      else { my.tail = carry.pack(); my.tail_state = 1; my.tail_row = carry_row; }
    }
    my.pad = (int)((clock64() - t_start) >> 4);
    if (lane == 0) cta_rec[blockIdx.x] = my;
  }
  lanes_reduce<32, MODE>(st.nsq);
  if (lane == 0) s_slots[warp] = st.nsq.pack();
  __syncthreads();
  grid_launch_dependents();  // the next kernel's prologue may start while the tail below runs
  if (threadIdx.x == 0) {
    Acc<MODE> tot = acc_of<MODE>(s_slots[0]);
    for (int i = 1; i < W; ++i) tot.merge(acc_of<MODE>(s_slots[i]));
    __stcg(partials + blockIdx.x, tot.pack());
    __threadfence();
    const unsigned int t = atomicAdd(&sc->ticket[0], 1u);
    *s_flag = (t == gridDim.x - 1) ? 1 : 0;
  }
  __syncthreads();
  if (*s_flag == 0) return;
  __threadfence();
  // ---- last CTA: chain the pieces of rows that cross CTA boundaries (warp 0), fixed-order sum of partials ----
  Acc<MODE> extra;
  extra.zero();
  if (warp == 0) {
    const int G = (int)gridDim.x;
    Acc<MODE> carry;
    carry.zero();
    int carry_row = -1;
    auto load_rec = [&](int base, double2& hv, double2& tv, int& hs, int& ts, int& trow) {
      hv = make_double2(0.0, 0.0); tv = make_double2(0.0, 0.0);
      hs = 0; ts = 0; trow = -1;
      if (base + lane < G) {
        const CtaRec* g = cta_rec + base + lane;
        hv = __ldcg(&g->head); tv = __ldcg(&g->tail);
        hs = __ldcg(&g->head_state); ts = __ldcg(&g->tail_state); trow = __ldcg(&g->tail_row);
      }
    };
    double2 hv, tv, hv_n, tv_n;
    int hs, ts, trow, hs_n, ts_n, trow_n;
    load_rec(0, hv, tv, hs, ts, trow);
    for (int base = 0; base < G; base += 32) {
      load_rec(base + 32, hv_n, tv_n, hs_n, ts_n, trow_n);
      bool emit;
      Acc<MODE> e_sum;
      int e_row;
      chain_scan<MODE>(hs, ts, acc_of<MODE>(hv), acc_of<MODE>(tv), trow, carry, carry_row, emit, e_sum, e_row);
      if (emit && e_row >= 0) {
        const int64_t rn = row_number(cx, e_row);
        const double yo = NEEDS_Y ? y[rn] : 0.0;
        finish_row_with<MODE, OP>(e_sum, yo, y, rn, c, sy, extra);
      }
      hv = hv_n; tv = tv_n; hs = hs_n; ts = ts_n; trow = trow_n;
    }
    lanes_reduce<32, MODE>(extra);
  }
  if (OP == OP_PLAIN || OP == OP_K2S) {
    if (threadIdx.x == 0) sc->ticket[0] = 0u;
    return;
  }
  Acc<MODE> a;
  a.zero();
  for (int i = threadIdx.x; i < (int)gridDim.x; i += blockDim.x) a.merge(acc_of<MODE>(__ldcg(partials + i)));
  if (threadIdx.x == 0) a.merge(extra);
  lanes_reduce<32, MODE>(a);
  __syncthreads();
  if (lane == 0) s_slots[warp] = a.pack();
  __syncthreads();
  if (threadIdx.x == 0) {
    Acc<MODE> tot = acc_of<MODE>(s_slots[0]);
    for (int i = 1; i < W; ++i) tot.merge(acc_of<MODE>(s_slots[i]));
    if (OP == OP_K1S) partials[gridDim.x] = tot.pack();  // this row block's ||u^_p||^2, unrounded: summed over blocks after the exchange
    const double total = tot.value();
    if (OP == OP_K1) tail_k1(sc, total);
    if (OP == OP_K2) tail_k2(sc, total);
    if (OP == OP_K2_INIT) tail_init_v(sc, total);
    sc->ticket[0] = 0u;
  }
}

// Element split points of `parts` ranges: cost(e) = e + c0 * (rows that start before e) is cut into equal
// parts; split points are rounded down to multiples of `align` elements.  partR[b] = first row with
// ptr[row] >= partE[b].
__global__ void k_stream_partition(const int64_t* __restrict__ ptr, int64_t nrows, int64_t nnz, int parts, int c0, int align,
                                   int64_t* partE, int32_t* partR) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b > parts) return;
  int64_t E;
  if (b == 0) E = 0;
  else if (b == parts) E = nnz;
  else {
    const double total = (double)nnz + (double)c0 * (double)nrows;
    const double target = total * ((double)b / (double)parts);
    int64_t lo = 0, hi = nrows;  // largest row i with F(i) = ptr[i] + c0*i <= target
    while (lo < hi) {
      const int64_t mid = (lo + hi + 1) >> 1;
      const double f = (double)ptr[mid] + (double)c0 * (double)mid;
      if (f <= target) lo = mid; else hi = mid - 1;
    }
    const double f = (double)ptr[lo] + (double)c0 * (double)lo;
    int64_t e = ptr[lo] + (int64_t)(target - f);
    const int64_t cap = (lo < nrows) ? ptr[lo + 1] : nnz;
    if (e > cap) e = cap;
    E = (e / align) * align;
  }
  partE[b] = E;
  if (b == parts) { partR[b] = (int32_t)nrows; return; }
  int64_t lo = 0, hi = nrows;  // first row with ptr[row] >= E  (nrows if none)
  while (lo < hi) {
    const int64_t mid = (lo + hi) >> 1;
    if (ptr[mid] >= E) hi = mid; else lo = mid + 1;
  }
  partR[b] = (int32_t)lo;
}

// ---- rows without elements: counted, listed, and compacted away (create) -----------------------------
__global__ void k_count_empty(const int64_t* __restrict__ ptr, int64_t nrows, int* count) {
  int local = 0;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < nrows; i += (int64_t)gridDim.x * blockDim.x)
    if (ptr[i + 1] == ptr[i]) ++local;
  if (local) atomicAdd(count, local);
}
__global__ void k_flag_nonempty(const int64_t* __restrict__ ptr, int64_t nrows, int64_t* flag) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < nrows; i += (int64_t)gridDim.x * blockDim.x)
    flag[i] = (ptr[i + 1] > ptr[i]) ? 1 : 0;
}
// pos = exclusive scan of flag: non-empty row i is the pos[i]-th entry of (cptr, rid); empty row i the (i - pos[i])-th of erows
__global__ void k_compact_rows(const int64_t* __restrict__ ptr, int64_t nrows, const int64_t* __restrict__ pos,
                               int64_t* cptr, int32_t* rid, int32_t* erows) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i <= nrows; i += (int64_t)gridDim.x * blockDim.x) {
    if (i == nrows) { cptr[pos[nrows]] = ptr[nrows]; continue; }
    if (ptr[i + 1] > ptr[i]) { cptr[pos[i]] = ptr[i]; rid[pos[i]] = (int32_t)i; }
    else erows[i - pos[i]] = (int32_t)i;
  }
}

}  // namespace tomo
