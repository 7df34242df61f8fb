// wspmm.cuh — the multi-right-hand-side sparse products (BASELINE configs[3]) on the skeleton of
// wstream.cuh: eight independent LSQR / LSMR recurrences SHARE every pass over A and A^T.  Vectors are row-major
// blocks (len x 8); one element of the matrix is read once and multiplied with a 64-byte row of the gathered block.
//
//   * Same work split and the same matrix stream as the single-side kernel: every warp owns one contiguous element
//     range (the split points of wstream.cuh are reused) and pulls it through its own TMA ring; nothing is read
//     from HBM through the L1, so the whole L1 is left to the 64-byte gathers.
//   * Lane layout: lane = 4 * es + j.  A step is 8 consecutive elements (es = 0..7); the four lanes of an element
//     each gather 16 bytes (sides 2j, 2j + 1) of its row of the block, so a warp load touches 8 rows.  A round is
//     8 steps (64 elements): its 8 gathers per lane are in flight while the previous round is summed.
//   * Two accumulators per lane (sides 2j, 2j + 1) live across rounds and tiles; where a row ends they are summed
//     over the eight element slots (3 shuffle steps) and lanes 0..3 finish the row for their two sides (fused
//     axpy term, 16-byte store, ||.||^2).  Rows that end inside a step are closed one after the other.
//   * Rows cut by a range boundary leave one record per warp with eight partial sums per piece; the chains over
//     warps and over CTAs (chain_scan of wstream.cuh) run once per side.
//   * Every side has its own Scalars; a stopped side keeps its old column (nothing is written for it).
#pragma once
#include "wstream.cuh"

namespace tomo {

constexpr int kR = 8;             // right-hand sides per pass

struct CtaRec8 {       // CtaRec for eight sides
  double2 head[kR], tail[kR];
  int head_state, tail_state, tail_row, pad;
};

template <typename CFG, typename VT>
struct MSmem {
  static constexpr size_t kIdx = sizeof(int32_t) * CFG::TILE;
  static constexpr size_t kVal = sizeof(VT) * CFG::TILE;
  static constexpr size_t kStage = kIdx + kVal;
  static constexpr size_t kWarp = kStage * CFG::NS;
  static constexpr size_t kBars = 8 * CFG::NS * CFG::W;
  static constexpr size_t kRec = sizeof(CtaRec8) * CFG::W;
  static constexpr size_t kSlots = sizeof(double2) * kR * (CFG::W + 1) + 64;
  static constexpr size_t kTotal = kWarp * CFG::W + kBars + kRec + kSlots;
};

template <int MODE>
struct MSweep {
  Acc<MODE> a0, a1;      // per-lane partials of the open row, sides 2j and 2j + 1
  Acc<MODE> n0, n1;      // ||y_k||^2 partials of those sides (lanes 0..3 only)
  double2 h0, h1;        // head record values of those sides (lanes 0..3); fast mode only: in dd mode they go straight
                         // to the warp's record in shared memory (registers: measured +12 % there, -6 % in fast mode)
  int h_state;           // head record state
  int cur, next_b, wbase, S, S2;
  bool started;
};

struct MCtx {            // per-lane constants of the two sides a lane serves
  double c0, c1, sy0, sy1;
  bool skip0, skip1;
  double* Y;
  CtaRec8* rec;          // the warp's record (shared memory)
};

template <int MODE>
__device__ __forceinline__ Acc<MODE> acc_xor(const Acc<MODE>& a, int off) {
  Acc<MODE> r;
  double2 p = a.pack();
  p.x = __shfl_xor_sync(0xffffffffu, p.x, off);
  p.y = __shfl_xor_sync(0xffffffffu, p.y, off);
  r.unpack(p);
  return r;
}
// sum over the eight element slots (lane bits 2..4); every lane of a side pair ends with the same bits
template <int MODE>
__device__ __forceinline__ void slots_reduce(Acc<MODE>& a0, Acc<MODE>& a1) {
  const int lane = threadIdx.x & 31;
#pragma unroll
  for (int off = 16; off >= 4; off >>= 1) {
    Acc<MODE> o0 = acc_xor<MODE>(a0, off), o1 = acc_xor<MODE>(a1, off);
    if (lane & off) { o0.merge(a0); a0 = o0; o1.merge(a1); a1 = o1; } else { a0.merge(o0); a1.merge(o1); }
  }
}

// lanes 0..3: y[r][2j], y[r][2j+1] <- sums + c * (old * sy), ||.||^2; a stopped side keeps its old value
template <int MODE, int OP>
__device__ __forceinline__ void finish_row8(Acc<MODE> s0, Acc<MODE> s1, int64_t r, const MCtx& mc, Acc<MODE>& n0, Acc<MODE>& n1) {
  constexpr bool NEEDS_Y = (OP == OP_K1 || OP == OP_K2);
  const int j = threadIdx.x & 3;
  double2* yp = reinterpret_cast<double2*>(mc.Y + (size_t)r * kR) + j;
  double2 yo = make_double2(0.0, 0.0);
  if (NEEDS_Y || mc.skip0 || mc.skip1) yo = *yp;
  double yn0, yn1;
  if (NEEDS_Y) {
    double y0 = yo.x, y1 = yo.y;
    if (OP == OP_K1) { y0 = y0 * mc.sy0; y1 = y1 * mc.sy1; }
    if (MODE == 0) { yn0 = fma(mc.c0, y0, s0.value()); yn1 = fma(mc.c1, y1, s1.value()); }
    else { s0.mac(mc.c0, y0); yn0 = s0.value(); s1.mac(mc.c1, y1); yn1 = s1.value(); }
  } else {
    yn0 = s0.value(); yn1 = s1.value();
  }
  if (mc.skip0) yn0 = yo.x;
  if (mc.skip1) yn1 = yo.y;
  *yp = make_double2(yn0, yn1);
  if (OP != OP_PLAIN) {
    if (!mc.skip0) n0.mac(yn0, yn0);
    if (!mc.skip1) n1.mac(yn1, yn1);
  }
}

// One 8-element step [base, base + 8) in which the open row ends (base < next_b <= base + 8): close it, then the rows
// that start and end inside the step one after the other; the last one becomes the open row if it runs on.
template <int MODE, int OP>
__device__ __forceinline__ void slow_step8(MSweep<MODE>& st, const WCtx& cx, const MCtx& mc, double v, double x0, double x1, int base) {
  const int lane = threadIdx.x & 31, es = lane >> 2;
  const int hi = min(base + 8, cx.len);
  const int pos = base + es;
  int lo = base;
  while (true) {
    // the open row's piece [lo, min(next_b, hi))
    const int e1 = min(st.next_b, hi);
    const bool mine = pos >= lo && pos < e1;
    st.a0.mac(mine ? v : 0.0, mine ? x0 : 0.0);
    st.a1.mac(mine ? v : 0.0, mine ? x1 : 0.0);
    if (st.next_b > hi) return;  // it runs on behind the step
    slots_reduce<MODE>(st.a0, st.a1);
    if (lane < 4) {
      if (st.started) finish_row8<MODE, OP>(st.a0, st.a1, row_number(cx, st.cur), mc, st.n0, st.n1);
      else if (MODE == 0) { st.h0 = st.a0.pack(); st.h1 = st.a1.pack(); }
      else { const int j = lane & 3; mc.rec->head[2 * j] = st.a0.pack(); mc.rec->head[2 * j + 1] = st.a1.pack(); }
    }
    if (!st.started) st.h_state = 2;
    st.a0.zero(); st.a1.zero();
    lo = st.next_b;
    st.started = true;
    if (lo >= cx.len) { st.next_b = kBig; return; }  // the range ends with this row
    st.cur = st.cur + 1;
    win_advance(st, cx);
    st.next_b = win_get(st, st.cur + 1);
    if (lo >= hi) return;  // the next row opens exactly at the end of the step
  }
}

// the products of one round (8 steps of 8 elements at relative offset pos0) go to the rows they belong to
template <int MODE, int OP, bool SCALE_X>
__device__ __forceinline__ void consume_round8(MSweep<MODE>& st, const WCtx& cx, const MCtx& mc, double (&vv)[8], double2 (&xx)[8],
                                               int pos0, double sx0, double sx1) {
  double x0[8], x1[8];
#pragma unroll
  for (int u = 0; u < 8; ++u) {
    x0[u] = SCALE_X ? xx[u].x * sx0 : xx[u].x;
    x1[u] = SCALE_X ? xx[u].y * sx1 : xx[u].y;
  }
  if (st.next_b > pos0 + 64) {  // the round lies inside the open row (lanes behind the range hold zeros)
    if (MODE == 1) {  // dd: two interleaved chains of plain mac()s; the TwoSum tree of mac8 costs registers here (measured +10 %)
#pragma unroll
      for (int u = 0; u < 8; ++u) { st.a0.mac(vv[u], x0[u]); st.a1.mac(vv[u], x1[u]); }
      return;
    }
    st.a0.mac8(vv, x0);
    st.a1.mac8(vv, x1);
    return;
  }
  // (fast mode only: measured -7 % there, +11 % in dd mode, where the extra accumulator pair costs registers)
  if (MODE == 0 && pos0 + 64 <= cx.len && st.started) {
    const int nb2 = win_get(st, st.cur + 2);  // end of the row that starts where the open one ends
    if (st.next_b == pos0 + 64 || nb2 > pos0 + 64) {
      // exactly one row ends inside the round and the next one runs on behind it: per-step sums to two accumulator
      // pairs (no register selects), one reduction over the element slots, the row is finished by lanes 0..3
      const int pe = st.next_b;             // pos0 < pe <= pos0 + 64
      const int us = (pe - pos0) >> 3;      // step that holds the row end (8: the round ends with the row)
      const bool first = pos0 + 8 * us + (int)((threadIdx.x & 31) >> 2) < pe;
      Acc<MODE> b0, b1;
      b0.zero(); b1.zero();
#pragma unroll
      for (int u = 0; u < 8; ++u) {
        if (u < us) { st.a0.mac(vv[u], x0[u]); st.a1.mac(vv[u], x1[u]); }
        else if (u > us) { b0.mac(vv[u], x0[u]); b1.mac(vv[u], x1[u]); }
        else {
          const double va = first ? vv[u] : 0.0, vb = first ? 0.0 : vv[u];
          st.a0.mac(va, x0[u]); st.a1.mac(va, x1[u]);
          b0.mac(vb, x0[u]); b1.mac(vb, x1[u]);
        }
      }
      slots_reduce<MODE>(st.a0, st.a1);
      if ((threadIdx.x & 31) < 4) finish_row8<MODE, OP>(st.a0, st.a1, row_number(cx, st.cur), mc, st.n0, st.n1);
      st.a0 = b0; st.a1 = b1;
      if (pe >= cx.len) { st.next_b = kBig; return; }  // the range ends with this row
      st.cur = st.cur + 1;
      st.next_b = nb2;
      win_advance(st, cx);
      return;
    }
  }
#pragma unroll 1
  for (int u = 0; u < 8; ++u) {
    const int base = pos0 + 8 * u;
    if (base >= cx.len) break;
    double v = vv[0], p0 = x0[0], p1 = x1[0];
#pragma unroll
    for (int k = 1; k < 8; ++k) { v = (u == k) ? vv[k] : v; p0 = (u == k) ? x0[k] : p0; p1 = (u == k) ? x1[k] : p1; }
    if (st.next_b > base + 8) { st.a0.mac(v, p0); st.a1.mac(v, p1); }
    else slow_step8<MODE, OP>(st, cx, mc, v, p0, p1, base);
  }
}

// Y[r][k] <- sum_j a_rj X[j][k] (+ c_k * Y[r][k] * sy_k), ||Y[:,k]||^2, for k = 0..7.  Arguments as k_wstream
// (FMT 0); X, Y row-major len x 8; sc[8]; partials: double2[gridDim.x][8].
template <typename CFG, int MODE, typename VT, int OP>
__global__ void __launch_bounds__(CFG::THREADS, 1)
k_wspmm8(const int64_t* __restrict__ ptr, const int32_t* __restrict__ rid, const int32_t* __restrict__ idx,
         const VT* __restrict__ val, int64_t nnz, int nrows, const int32_t* __restrict__ erows, int n_empty,
         const double* __restrict__ X, double* __restrict__ Y, const int64_t* __restrict__ wE, const int32_t* __restrict__ wR,
         CtaRec8* __restrict__ cta_rec, Scalars* sc, double2* partials) {
  constexpr int TILE = CFG::TILE, NS = CFG::NS, W = CFG::W, RPT = TILE / 64;
  using SM = MSmem<CFG, VT>;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  constexpr bool NEEDS_Y = (OP == OP_K1 || OP == OP_K2);
  constexpr bool SCALE_X = (OP == OP_K2 || OP == OP_K2_INIT);

  const int lane = threadIdx.x & 31, warp = uni((int)(threadIdx.x >> 5)), es = lane >> 2, j = lane & 3;
  unsigned char* my_ring = smem_raw + (size_t)warp * SM::kWarp;
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem_raw + SM::kWarp * W);
  uint64_t* my_bar = bars + warp * NS;
  CtaRec8* s_rec = reinterpret_cast<CtaRec8*>(smem_raw + SM::kWarp * W + SM::kBars);
  double2* s_slots = reinterpret_cast<double2*>(smem_raw + SM::kWarp * W + SM::kBars + SM::kRec);  // [W + 1][8]
  int* s_flag = reinterpret_cast<int*>(s_slots + kR * (W + 1));

  if (lane == 0) {
    for (int s = 0; s < NS; ++s) mbar_init(my_bar + s, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    fence_proxy_async();
  }
  __syncwarp();
  const int gw = blockIdx.x * W + warp;
  WCtx cx;
  cx.ptr = ptr; cx.rid = rid; cx.y = Y;
  cx.E0 = uni(wE[gw]);
  const int64_t E1 = uni(wE[gw + 1]);
  cx.R0 = uni(wR[gw]); cx.R1 = uni(wR[gw + 1]);
  cx.len = (int)(E1 - cx.E0);
  cx.c = 0.0; cx.sy = 1.0;
  const int ntiles = (cx.len + TILE - 1) / TILE;
  const uint64_t policy = l2_evict_first_policy();
  const uint32_t ring_a = smem_u32(my_ring), bar_a = smem_u32(my_bar);
  const VT* val0 = val + cx.E0;
  const int32_t* idx0 = idx + cx.E0;
  auto stage_ptr = [&](int s) { return my_ring + (size_t)s * SM::kStage; };
  auto issue_tile = [&](int t, bool refill) {
    const int s = t % NS;
    const uint32_t dst = ring_a + (uint32_t)s * (uint32_t)SM::kStage, bar = bar_a + 8u * (uint32_t)s;
    int cnt4 = TILE;
    if (t == ntiles - 1) {  // the last tile of the range may be short; < 4 elements at the very end of the arrays: ordinary loads
      const int cnt = cx.len - t * TILE;
      cnt4 = cnt & ~3;
      if (lane < cnt - cnt4) {
        reinterpret_cast<VT*>(stage_ptr(s) + SM::kIdx)[cnt4 + lane] = val0[(size_t)t * TILE + cnt4 + lane];
        reinterpret_cast<int32_t*>(stage_ptr(s))[cnt4 + lane] = idx0[(size_t)t * TILE + cnt4 + lane];
      }
      __syncwarp();
    }
    if (elect_one()) {
      if (refill) fence_proxy_async();
      if (cnt4 > 0) {
        mbar_arrive_expect_tx_a(bar, (uint32_t)cnt4 * (uint32_t)(4 + sizeof(VT)));
        bulk_g2s_a(dst, idx0 + (size_t)t * TILE, (uint32_t)cnt4 * 4u, bar, policy);
        bulk_g2s_a(dst + (uint32_t)SM::kIdx, val0 + (size_t)t * TILE, (uint32_t)cnt4 * (uint32_t)sizeof(VT), bar, policy);
      } else {
        mbar_arrive(my_bar + s);
      }
    }
  };
  for (int t = 0; t < NS && t < ntiles; ++t) issue_tile(t, false);

  MSweep<MODE> st;
  st.a0.zero(); st.a1.zero(); st.n0.zero(); st.n1.zero();
  st.h0 = make_double2(0.0, 0.0); st.h1 = make_double2(0.0, 0.0); st.h_state = 0;
  st.cur = cx.R0; st.next_b = kBig; st.started = true;
  st.wbase = cx.R0;
  st.S = win_load(cx, cx.R0);
  st.S2 = win_load(cx, cx.R0 + 32);

  // ---- everything below reads what the previous kernel of the iteration wrote ----
  grid_dependency_wait();
  MCtx mc;
  mc.Y = Y;
  mc.rec = s_rec + warp;
  if (lane < 4) { mc.rec->head[2 * j] = make_double2(0.0, 0.0); mc.rec->head[2 * j + 1] = make_double2(0.0, 0.0); }
  double sx0, sx1;
  {
    const Scalars* s0 = sc + 2 * j;
    const Scalars* s1 = s0 + 1;
    mc.skip0 = s0->stop || (OP == OP_K2 && s0->beta_zero);
    mc.skip1 = s1->stop || (OP == OP_K2 && s1->beta_zero);
    mc.c0 = (OP == OP_K1) ? -s0->alpha : (OP == OP_K2 ? -s0->beta : 0.0);
    mc.c1 = (OP == OP_K1) ? -s1->alpha : (OP == OP_K2 ? -s1->beta : 0.0);
    sx0 = SCALE_X ? s0->rbeta : 1.0; sx1 = SCALE_X ? s1->rbeta : 1.0;
    mc.sy0 = (OP == OP_K1) ? s0->rbeta : 1.0; mc.sy1 = (OP == OP_K1) ? s1->rbeta : 1.0;
  }
  if (OP != OP_PLAIN) {
    const unsigned active = __ballot_sync(0xffffffffu, !sc[lane & 7].stop);
    if (!active) {  // every side has stopped: nothing changes any more (drain the copies already requested)
      for (int t = 0; t < NS && t < ntiles; ++t) mbar_wait_a(bar_a + 8u * (uint32_t)(t % NS), 0);
      return;
    }
  }

  const double2* X2 = reinterpret_cast<const double2*>(X) + j;
  if (cx.len > 0) {
    const int first = __shfl_sync(0xffffffffu, st.S, 0);  // start of row R0 (>= len if no row starts in the range)
    if (first > 0) { st.cur = cx.R0 - 1; st.started = false; st.next_b = first; }
    else { st.cur = cx.R0; st.started = true; st.next_b = __shfl_sync(0xffffffffu, st.S, 1); }
    const int nr = (cx.len + 63) >> 6;
    // gather for round r: the indices of my element slot from the ring, my 16 bytes of each of the 8 rows of X
    auto gather = [&](int r, double2 (&xx)[8]) {
      const int t = r / RPT, rr = r % RPT, s = t % NS;
      if (rr == 0) mbar_wait_a(bar_a + 8u * (uint32_t)s, (uint32_t)(t / NS) & 1u);
      const uint32_t* si = reinterpret_cast<const uint32_t*>(stage_ptr(s)) + rr * 64 + es;
      const int pos0 = r << 6;
      if (pos0 + 64 <= cx.len) {
        uint32_t cc[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) cc[u] = si[8 * u];
#pragma unroll
        for (int u = 0; u < 8; ++u) xx[u] = __ldg(X2 + (size_t)cc[u] * (kR / 2));
      } else {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
          xx[u] = make_double2(0.0, 0.0);
          if (pos0 + 8 * u + es < cx.len) xx[u] = __ldg(X2 + (size_t)si[8 * u] * (kR / 2));
        }
      }
    };
    // round r with the gathers in xc; the gathers of round r + 1 go to xn meanwhile
    auto body = [&](int r, double2 (&xc)[8], double2 (&xn)[8]) {
      if (r + 1 < nr) gather(r + 1, xn);
      const int t = r / RPT, rr = r % RPT;
      const VT* sv = reinterpret_cast<const VT*>(stage_ptr(t % NS) + SM::kIdx) + rr * 64 + es;
      const int pos0 = r << 6;
      double vv[8];
      if (pos0 + 64 <= cx.len) {
#pragma unroll
        for (int u = 0; u < 8; ++u) vv[u] = (double)sv[8 * u];
      } else {
#pragma unroll
        for (int u = 0; u < 8; ++u) vv[u] = (pos0 + 8 * u + es < cx.len) ? (double)sv[8 * u] : 0.0;
      }
      if (rr == RPT - 1 && t + NS < ntiles) { __syncwarp(); issue_tile(t + NS, true); }  // the tile is in registers: refill its stage
      consume_round8<MODE, OP, SCALE_X>(st, cx, mc, vv, xc, pos0, sx0, sx1);
    };
    double2 xa[8], xb[8];
    gather(0, xa);
#pragma unroll 1
    for (int r = 0; r < nr; r += 2) {  // unrolled twice: the two gather register sets swap roles (measured: +17 % over copying)
      body(r, xa, xb);
      if (r + 1 < nr) body(r + 1, xb, xa);
    }

  }
  // ---- the warp's record: the row open at the range start (head) and the one open at its end (tail / head) ----
  CtaRec8* rec = s_rec + warp;
  if (lane < 4) {
    if (MODE == 0) { rec->head[2 * j] = st.h0; rec->head[2 * j + 1] = st.h1; }
    rec->tail[2 * j] = make_double2(0.0, 0.0); rec->tail[2 * j + 1] = make_double2(0.0, 0.0);
  }
  int r_hs = st.h_state, r_ts = 0, r_trow = -1;
  if (cx.len > 0 && ptr[cx.R1] > E1) {  // the last row of the range runs on behind it (see k_wstream)
    slots_reduce<MODE>(st.a0, st.a1);
    if (cx.R1 > cx.R0) {
      r_ts = 1; r_trow = cx.R1 - 1;
      if (lane < 4) { rec->tail[2 * j] = st.a0.pack(); rec->tail[2 * j + 1] = st.a1.pack(); }
    } else {
      r_hs = 1;
      if (lane < 4) { rec->head[2 * j] = st.a0.pack(); rec->head[2 * j + 1] = st.a1.pack(); }
    }
  }
  if (lane == 0) { rec->head_state = r_hs; rec->tail_state = r_ts; rec->tail_row = r_trow; rec->pad = 0; }

  // ---- rows without elements: y_r = c * y_r (K1 / K2) or 0; item = (row, side pair), the pair is the lane's own ----
  if (n_empty > 0) {
    Acc<MODE> z0, z1;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < (int64_t)n_empty * 4; i += (int64_t)gridDim.x * blockDim.x) {
      z0.zero(); z1.zero();
      finish_row8<MODE, OP>(z0, z1, erows[i >> 2], mc, st.n0, st.n1);
    }
  }
  __syncthreads();

  // ---- chain of the CTA's W warp records, once per side (warp 0); CTA record; per-CTA partials ----
  double2* s_extra = s_slots + kR * W;  // [8]: ||.||^2 of the rows finished by the chains
  if (warp == 0) {
    int hs = 0, ts = 0, trow = -1;
    if (lane < W) { hs = s_rec[lane].head_state; ts = s_rec[lane].tail_state; trow = s_rec[lane].tail_row; }
    int crow0 = -1;  // -2: a row enters the CTA's range from the previous CTA
    {
      const int64_t cE0 = wE[blockIdx.x * W], cE1 = wE[blockIdx.x * W + W];
      if (cE0 < cE1 && ptr[wR[blockIdx.x * W]] > cE0) crow0 = -2;
    }
    int my_hs = 0, my_ts = 0, my_trow = -1;
#pragma unroll 1
    for (int k = 0; k < kR; ++k) {
      double2 hv = make_double2(0.0, 0.0), tv = make_double2(0.0, 0.0);
      if (lane < W) { hv = s_rec[lane].head[k]; tv = s_rec[lane].tail[k]; }
      Acc<MODE> carry;
      carry.zero();
      int carry_row = crow0;
      bool emit;
      Acc<MODE> e_sum;
      int e_row;
      chain_scan<MODE>(hs, ts, acc_of<MODE>(hv), acc_of<MODE>(tv), trow, carry, carry_row, emit, e_sum, e_row);
      double2 o_head = make_double2(0.0, 0.0), o_tail = make_double2(0.0, 0.0);
      my_hs = 0; my_ts = 0; my_trow = -1;
      const unsigned hb = __ballot_sync(0xffffffffu, emit && e_row == -2);
      if (hb) { const int src = __ffs((int)hb) - 1; o_head = acc_bcast<MODE>(e_sum, src).pack(); my_hs = 2; }
      Acc<MODE> ex;
      ex.zero();
      const Scalars* sk = sc + k;
      const bool skip = sk->stop || (OP == OP_K2 && sk->beta_zero);
      if (emit && e_row >= 0 && !skip) {
        const double ck = (OP == OP_K1) ? -sk->alpha : (OP == OP_K2 ? -sk->beta : 0.0);
        const double syk = (OP == OP_K1) ? sk->rbeta : 1.0;
        const int64_t rn = row_number(cx, e_row);
        const double yo = NEEDS_Y ? Y[rn * kR + k] : 0.0;
        finish_row_with<MODE, OP>(e_sum, yo, Y + k, rn * kR, ck, syk, ex);
      }
      if (carry_row != -1) {
        if (carry_row == -2) { o_head = carry.pack(); my_hs = 1; }
        else { o_tail = carry.pack(); my_ts = 1; my_trow = carry_row; }
      }
      lanes_reduce<32, MODE>(ex);
      if (lane == 0) { cta_rec[blockIdx.x].head[k] = o_head; cta_rec[blockIdx.x].tail[k] = o_tail; s_extra[k] = ex.pack(); }
    }
    if (lane == 0) { cta_rec[blockIdx.x].head_state = my_hs; cta_rec[blockIdx.x].tail_state = my_ts; cta_rec[blockIdx.x].tail_row = my_trow; }
  }
  slots_reduce<MODE>(st.n0, st.n1);
  if (lane < 4) { s_slots[warp * kR + 2 * j] = st.n0.pack(); s_slots[warp * kR + 2 * j + 1] = st.n1.pack(); }
  __syncthreads();
  grid_launch_dependents();
  if (threadIdx.x < kR) {
    Acc<MODE> tot = acc_of<MODE>(s_slots[threadIdx.x]);
    for (int w = 1; w < W; ++w) tot.merge(acc_of<MODE>(s_slots[w * kR + threadIdx.x]));
    tot.merge(acc_of<MODE>(s_extra[threadIdx.x]));
    __stcg(partials + (size_t)blockIdx.x * kR + threadIdx.x, tot.pack());
  }
  __threadfence();
  __syncthreads();
  if (threadIdx.x == 0) {
    const unsigned int t = atomicAdd(&sc->ticket[0], 1u);
    *s_flag = (t == gridDim.x - 1) ? 1 : 0;
  }
  __syncthreads();
  if (*s_flag == 0) return;
  __threadfence();
  // ---- last CTA: chain the pieces of rows that cross CTA boundaries (warp 0, once per side), column sums, tails ----
  if (warp == 0) {
    const int G = (int)gridDim.x;
#pragma unroll 1
    for (int k = 0; k < kR; ++k) {
      const Scalars* sk = sc + k;
      const bool skip = sk->stop || (OP == OP_K2 && sk->beta_zero);
      const double ck = (OP == OP_K1) ? -sk->alpha : (OP == OP_K2 ? -sk->beta : 0.0);
      const double syk = (OP == OP_K1) ? sk->rbeta : 1.0;
      Acc<MODE> carry, ex;
      carry.zero(); ex.zero();
      int carry_row = -1;
      for (int base = 0; base < G; base += 32) {
        double2 hv = make_double2(0.0, 0.0), tv = make_double2(0.0, 0.0);
        int hs = 0, ts = 0, trow = -1;
        if (base + lane < G) {
          const CtaRec8* g = cta_rec + base + lane;
          hv = __ldcg(&g->head[k]); tv = __ldcg(&g->tail[k]);
          hs = __ldcg(&g->head_state); ts = __ldcg(&g->tail_state); trow = __ldcg(&g->tail_row);
        }
        bool emit;
        Acc<MODE> e_sum;
        int e_row;
        chain_scan<MODE>(hs, ts, acc_of<MODE>(hv), acc_of<MODE>(tv), trow, carry, carry_row, emit, e_sum, e_row);
        if (emit && e_row >= 0 && !skip) {
          const int64_t rn = row_number(cx, e_row);
          const double yo = NEEDS_Y ? Y[rn * kR + k] : 0.0;
          finish_row_with<MODE, OP>(e_sum, yo, Y + k, rn * kR, ck, syk, ex);
        }
      }
      lanes_reduce<32, MODE>(ex);
      if (lane == 0) s_extra[k] = ex.pack();
    }
  }
  __syncthreads();
  if (OP == OP_PLAIN) {
    if (threadIdx.x == 0) sc->ticket[0] = 0u;
    return;
  }
  if (threadIdx.x < kR) {
    Acc<MODE> a;
    a.zero();
    for (int b = 0; b < (int)gridDim.x; ++b) a.merge(acc_of<MODE>(__ldcg(partials + (size_t)b * kR + threadIdx.x)));
    a.merge(acc_of<MODE>(s_extra[threadIdx.x]));
    const double total = a.value();
    Scalars* s = sc + threadIdx.x;
    if (!s->stop) {
      const bool skipped = (OP == OP_K2 && s->beta_zero);
      if (OP == OP_K1) tail_k1(s, total);
      if (OP == OP_K2) tail_k2(s, skipped ? 0.0 : total);
      if (OP == OP_K2_INIT) tail_init_v(s, total);
    }
  }
  __syncthreads();
  if (threadIdx.x == 0) sc->ticket[0] = 0u;
}

}  // namespace tomo
