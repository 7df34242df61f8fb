// stream.cuh — the streaming SpMV kernel of the LSQR hot path:
//     K1  u^ <- A v - alpha u     + ||u^||^2 -> tail: beta, 1/beta, anorm           (over the caller's CSR)
//     K2  v^ <- A^T u - beta v    + ||v^||^2 -> tail: alpha, rotations, estimates   (over the CSC copy)
// "sparse matrix-vector multiplications and vector norm calculations" are what the paper's GPU solver
// offloads; here both are one kernel, with the axpy and the norm fused in.
//
// Design (B200: 148 SMs, HBM3e-bound, TMA engine, 227 KB shared memory per SM):
//   * One persistent CTA per SM.  CTA b owns the ELEMENT range [E_b, E_{b+1}) of the matrix arrays
//     (cost-balanced split at multiples of 4 elements, not aligned to rows) and therefore streams one
//     contiguous piece of `idx` and `val` from HBM exactly once.
//   * Warp 0, the producer, cuts the range into chunks of <= CH elements, lists the rows that start
//     inside each chunk (local offsets in shared memory, row pointers fetched one chunk ahead) and moves
//     the chunk's `idx` and `val` with two cp.async.bulk copies (TMA engine, L2 evict-first) into an
//     S-stage shared-memory ring, completion signalled on an mbarrier.  Memory-level parallelism does
//     not depend on registers or occupancy.
//   * Warps 2..W+1 are consumers: each sweeps a fixed slice of every chunk in rounds of 256 elements.
//     A round is first moved to registers (32 consecutive elements per load: conflict-free) with all
//     eight gathers of x issued at once; then the products are added to a per-lane accumulator, and the
//     row structure only decides where sums are closed (three shapes: inside one row / one row end /
//     general, the last with a segmented warp reduction whose cost does not depend on the number of
//     rows).  Rows that start and end inside a slice are finished by the consumer (axpy term, store,
//     ||.||^2); pieces of rows that cross a slice boundary go to a small per-slice record.
//   * Warp 1, the resolver, chains the records of a chunk with a log-step warp scan (fixed tree order:
//     deterministic), hands the stage back to the producer and finishes the rows that ended, one chunk
//     behind.  Pieces of rows that cross a CTA boundary are chained the same way by the last-arriving
//     CTA of the launch, which also sums the per-CTA ||.||^2 partials in index order and runs the scalar
//     step of the iteration (tails.cuh).
// Every assignment (CTA ranges, chunks, slices, reduction trees) is static, so results are bitwise
// reproducible in both accumulation modes.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "accum.cuh"
#include "state.cuh"
#include "tails.cuh"

namespace tomo {

// ---- shapes -------------------------------------------------------------------------------------
template <int CH_, int W_, int S_, int PF_ = 4>
struct StreamCfg {
  static constexpr int PF = PF_;          // L2 prefetch distance in chunks (0: off)
  static constexpr int CH = CH_;          // elements per chunk (multiple of 32*W)
  static constexpr int W = W_;            // consumer warps
  static constexpr int S = S_;            // ring stages
  static constexpr int SL = CH_ / W_;     // elements per consumer slice
  static constexpr int MAXR = CH_ / 4;    // rows listed per chunk (a chunk is cut short beyond that)
  static constexpr int THREADS = 32 * (W_ + 2);   // producer warp, resolver warp, W consumer warps
};

struct SliceRec {      // what a consumer leaves for the resolver's chain, per slice and chunk
  double2 head;        // partial sum of the row that was open at the slice start
  double2 tail;        // partial sum of the row that started in the slice and continues behind it
  int head_state;      // 0 none, 1 row continues behind the slice, 2 row ended inside the slice
  int tail_state;      // 0 none, 1 present
  int tail_k;          // index of that row in the chunk's row list
  int pad;
};

struct CtaRec {        // the same, per CTA, for the last-arriving CTA's chain (global memory)
  double2 head, tail;
  int head_state, tail_state, tail_row, pad;
};

struct StageHdr {
  int L;               // elements in the chunk
  int nr;              // rows that start in the chunk: rs[0..nr), rs[nr] = start of the next row
  int r_first;         // global row id of rs[0]
  int skew;            // element offset of the chunk inside the staged copy (source aligned to 16 B)
  int last;            // 1: the CTA's final chunk
  int pad[3];
};

template <typename CFG, typename VT>
struct StreamSmem {
  static constexpr size_t kIdx = sizeof(int32_t) * (CFG::CH + 8);
  static constexpr size_t kVal = sizeof(VT) * (CFG::CH + 8);
  static constexpr size_t kRs = sizeof(int32_t) * (CFG::MAXR + 8);
  static constexpr size_t kRec = sizeof(SliceRec) * CFG::W;
  static constexpr size_t kStage = ((kIdx + kVal + kRs + kRec + sizeof(StageHdr)) + 127) / 128 * 128;
  static constexpr size_t kBars = 256;  // full[S], done[S], freed[S]
  static constexpr size_t kSlots = sizeof(double2) * (CFG::W + 2) + 16;
  static constexpr size_t kTotal = kStage * CFG::S + kBars + kSlots;
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

// HBM -> L2 bulk prefetch (TMA engine, no shared memory): keeps the stream several chunks ahead of the ring
__device__ __forceinline__ void bulk_prefetch_l2(const void* src, uint32_t bytes) {
  asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src), "r"(bytes) : "memory");
}

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
  double yn;
  if (OP == OP_K1 || OP == OP_K2) {
    if (OP == OP_K1) yo = yo * sy;
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
template <int MODE, int OP>
__device__ __forceinline__ void finish_row(Acc<MODE> sum, double* __restrict__ y, int64_t r, double c, double sy,
                                           Acc<MODE>& nsq) {
  double yo = 0.0;
  if (OP == OP_K1 || OP == OP_K2) yo = y[r];
  finish_row_with<MODE, OP>(sum, yo, y, r, c, sy, nsq);
}
__device__ __forceinline__ void prefetch_l1(const void* p) { asm volatile("prefetch.global.L1 [%0];" ::"l"(p)); }

// The chain over records as a warp scan.  Lane l holds the record of slice (or CTA) l: an optional head
// piece (state 1: its row continues, 2: its row ends here) followed by an optional tail piece (a row that
// starts here and continues).  Each record is a map on the carry (partial sum and id of the open row):
//   tail present -> carry := tail ;  head ends -> carry := none ;  else carry := carry + head
// Maps compose associatively, so all carries come out of a 5-step Kogge-Stone scan in a fixed tree
// order (deterministic) instead of a serial walk.  Returns, per lane, the row that ends in this record
// (emit_row >= 0, or -2: the row that entered the CTA from the left) with its complete sum.
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

// ---- consumer state of one slice sweep ---------------------------------------------------------------
template <int MODE>
struct Sweep {
  Acc<MODE> acc;     // per-lane partial of the open row
  double yold;       // lane 0: old y of the open row (fetched when the row starts inside the slice)
  double2 h_val;     // lane 0: head record value
  int cur;           // index of the open row in the chunk's row list (-1: the row open at the chunk start)
  int next_b;        // chunk-local offset where the open row ends
  int h_state;       // lane 0: head record state
  bool started;      // the open row starts inside this slice
  bool dirty;        // acc holds contributions
};

struct SweepCtx {    // uniform, read-only
  const int32_t* rs; int nr; int r_first; int a; int b; int has_empty; double c; double sy; double* y;
};

// One 32-element step [base, base+32) of a slice that contains a row end (or starts at one): the lanes'
// products v * x go to the rows they belong to; rows that end are reduced and finished (or recorded).
// Shared by all unrolled steps of the sweep, hence not inlined.
template <int MODE, int OP>
__device__ __forceinline__ void sweep_slow_step(Sweep<MODE>& st, const SweepCtx& cx, Acc<MODE>& nsq, double v, double x,
                                             int base) {
  constexpr bool NEEDS_Y = (OP == OP_K1 || OP == OP_K2);
  const int lane = threadIdx.x & 31;
  const int32_t* rs = cx.rs;
  const int hi = min(base + 32, cx.b);
  const int pos = base + lane;
  int lo = base;
  while (true) {
    if (!st.dirty && st.next_b < hi && st.cur + 2 <= cx.nr && rs[st.cur + 2] <= hi) {
      // ---- segmented: two or more rows end inside [lo, hi) ----
      const bool valid = pos >= lo && pos < hi;
      int k = 0x7fffffff;
      Acc<MODE> t;
      t.zero();
      if (!cx.has_empty) {  // starts of the following rows as a bit mask over the step
        const int j = st.cur + 1 + lane;
        const int sj = (j <= cx.nr) ? rs[j] : 0x7fffffff;
        const unsigned bit = (sj < base + 32) ? (1u << (sj - base)) : 0u;
        const unsigned M = __reduce_or_sync(0xffffffffu, bit);
        if (valid) k = st.cur + __popc(M & ((2u << lane) - 1u));
      } else if (valid) {
        int l2 = st.cur + 1, h2 = cx.nr;
        while (l2 < h2) { const int mid = (l2 + h2) >> 1; if (rs[mid] <= pos) l2 = mid + 1; else h2 = mid; }
        k = l2 - 1;
      }
      if (valid) t.mac(v, x);
      const int kprev = __shfl_up_sync(0xffffffffu, k, 1);
      const bool head = valid && (pos == lo || kprev != k);
      const int kend = valid ? rs[k + 1] : 0;
      const bool fin = head && kend <= hi;
      const bool fin_direct = fin && (k > st.cur || st.started);
      double yo = 0.0;
      if (NEEDS_Y && fin_direct) yo = cx.y[(int64_t)cx.r_first + k];
#pragma unroll
      for (int d = 1; d < 32; d <<= 1) {
        Acc<MODE> o = t.down(d);
        const int kk = __shfl_down_sync(0xffffffffu, k, d);
        if (lane + d < 32 && kk == k) t.merge(o);
      }
      if (fin) {
        if (fin_direct) finish_row_with<MODE, OP>(t, yo, cx.y, (int64_t)cx.r_first + k, cx.c, cx.sy, nsq);
        else { st.h_val = t.pack(); st.h_state = 2; }
      }
      const int klast = __shfl_sync(0xffffffffu, k, hi - 1 - base);
      const unsigned hb = __ballot_sync(0xffffffffu, head);
      const int lhead = 31 - __clz((int)hb);
      const int klast_end = rs[klast + 1];
      if (klast_end > hi) {  // the last row of the step continues: it becomes the open row
        Acc<MODE> hv = acc_bcast<MODE>(t, lhead);
        st.acc.zero();
        if (lane == 0) st.acc = hv;
        st.dirty = true;
        const bool newrow = klast > st.cur;
        st.started = st.started || newrow;
        st.cur = klast;
        st.next_b = klast_end;
        if (NEEDS_Y && newrow && lane == 0) st.yold = cx.y[(int64_t)cx.r_first + st.cur];
      } else {
        st.acc.zero();
        st.dirty = false;
        if (hi < cx.b) {
          if (cx.has_empty) { int l2 = 0, h2 = cx.nr; while (l2 < h2) { const int mid = (l2 + h2) >> 1; if (rs[mid] <= hi) l2 = mid + 1; else h2 = mid; } st.cur = l2 - 1; }
          else st.cur = klast + 1;
          st.started = true;
          st.next_b = rs[st.cur + 1];
          if (NEEDS_Y && lane == 0) st.yold = cx.y[(int64_t)cx.r_first + st.cur];
        } else st.next_b = hi;
      }
      return;
    }
    const int seg_end = min(st.next_b, hi);
    if (lo < seg_end) {
      const bool mine = pos >= lo && pos < seg_end;
      st.acc.mac(mine ? v : 0.0, mine ? x : 0.0);  // other lanes add an exact zero
      st.dirty = true;
    }
    if (st.next_b > hi) return;  // the open row continues behind the step
    // the open row ends at next_b <= hi
    lanes_reduce<32, MODE>(st.acc);
    if (lane == 0) {
      if (st.started) finish_row_with<MODE, OP>(st.acc, st.yold, cx.y, (int64_t)cx.r_first + st.cur, cx.c, cx.sy, nsq);
      else { st.h_val = st.acc.pack(); st.h_state = 2; }
    }
    st.acc.zero();
    st.dirty = false;
    lo = st.next_b;
    if (lo >= cx.b) return;  // slice finished exactly at a row end (next_b == b marks "nothing open")
    if (cx.has_empty) { int l2 = 0, h2 = cx.nr; while (l2 < h2) { const int mid = (l2 + h2) >> 1; if (rs[mid] <= lo) l2 = mid + 1; else h2 = mid; } st.cur = l2 - 1; }
    else st.cur = st.cur + 1;
    st.started = true;
    st.next_b = rs[st.cur + 1];
    if (NEEDS_Y && lane == 0) st.yold = cx.y[(int64_t)cx.r_first + st.cur];
    if (lo >= hi) return;
  }
}

// ---- the kernel -----------------------------------------------------------------------------------
// ptr/idx/val: CSR-like triple with `nrows` rows and `nnz` elements (K1: the CSR of A; K2: the CSC copy,
// i.e. the CSR of A^T).  partE[b], partR[b] (b = 0..G): element split points (multiples of 4, partE[G] =
// nnz) and the first row with ptr[row] >= partE[b] (partR[G] = nrows).
template <typename CFG, int MODE, typename VT, int OP>
__global__ void __launch_bounds__(CFG::THREADS, 1)
k_stream(const int64_t* __restrict__ ptr, const int32_t* __restrict__ idx, const VT* __restrict__ val, int64_t nnz,
         int nrows, int has_empty, const double* __restrict__ x, double* __restrict__ y,
         const int64_t* __restrict__ partE, const int32_t* __restrict__ partR, CtaRec* __restrict__ cta_rec, Scalars* sc,
         double2* partials) {
  constexpr int CH = CFG::CH, W = CFG::W, S = CFG::S, SL = CFG::SL, MAXR = CFG::MAXR, PF = CFG::PF;
  using SM = StreamSmem<CFG, VT>;
  extern __shared__ __align__(128) unsigned char smem_raw[];

  double c = 0.0, sx = 1.0, sy = 1.0;
  if (OP != OP_PLAIN) {
    if (sc->stop) return;
    if (OP == OP_K2 && sc->beta_zero) {  // beta = 0: the A^T pass is skipped, the scalar step still runs
      if (blockIdx.x == 0 && threadIdx.x == 0) tail_k2(sc, 0.0);
      return;
    }
    if (OP == OP_K1) { c = -sc->alpha; sy = sc->rbeta; }
    if (OP == OP_K2) { c = -sc->beta; sx = sc->rbeta; }
    if (OP == OP_K2_INIT) { sx = sc->rbeta; }
  }
  constexpr bool SCALE_X = (OP == OP_K2 || OP == OP_K2_INIT);

  auto stage_base = [&](int s) { return smem_raw + (size_t)s * SM::kStage; };
  auto st_idx = [&](int s) { return reinterpret_cast<int32_t*>(stage_base(s)); };
  auto st_val = [&](int s) { return reinterpret_cast<VT*>(stage_base(s) + SM::kIdx); };
  auto st_rs = [&](int s) { return reinterpret_cast<int32_t*>(stage_base(s) + SM::kIdx + SM::kVal); };
  auto st_rec = [&](int s) { return reinterpret_cast<SliceRec*>(stage_base(s) + SM::kIdx + SM::kVal + SM::kRs); };
  auto st_hdr = [&](int s) { return reinterpret_cast<StageHdr*>(stage_base(s) + SM::kIdx + SM::kVal + SM::kRs + SM::kRec); };
  uint64_t* bar_full = reinterpret_cast<uint64_t*>(smem_raw + SM::kStage * S);
  uint64_t* bar_done = bar_full + S;
  uint64_t* bar_freed = bar_done + S;
  double2* s_slots = reinterpret_cast<double2*>(smem_raw + SM::kStage * S + SM::kBars);
  int* s_flag = reinterpret_cast<int*>(s_slots + (W + 2));

  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const long long t_start = clock64();
  if (threadIdx.x == 0) {
    for (int s = 0; s < S; ++s) { mbar_init(bar_full + s, 1); mbar_init(bar_done + s, W); mbar_init(bar_freed + s, 1); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  __syncthreads();

  const int64_t E0 = partE[blockIdx.x], E1 = partE[blockIdx.x + 1];
  const int R0 = partR[blockIdx.x], R1 = partR[blockIdx.x + 1];
  const bool has_work = (E0 < E1) || (R0 < R1);
  Acc<MODE> nsq;
  nsq.zero();

  if (warp == 0) {
    // ============================== producer: row lists + bulk copies ==============================
    // Nothing in this loop waits on a global load issued in the same iteration: the row pointers of the
    // next chunk are fetched one iteration ahead, the chain and the epilogues belong to warp 1.
    if (has_work) {
      const uint64_t policy = l2_evict_first_policy();
      int64_t e = E0;
      int r = R0;
      int cidx = 0;
      bool more = true;
      // ptr[r + lane] for the next 32 rows (row R1 included: it delimits the last owned row)
      int64_t pcur = (r + lane <= R1) ? ptr[r + lane] : (int64_t)-1;
      while (more) {
        const int s = cidx % S;
        if (cidx >= S) mbar_wait(bar_freed + s, ((cidx / S) - 1) & 1);  // stage released by consumers and resolver
        int L = (int)min((int64_t)CH, E1 - e);
        const bool to_end = (e + L == E1);  // rows starting exactly at the range end belong to the next CTA, except trailing rows
        int32_t* rs = st_rs(s);
        int nr = 0;
        bool cut = false;
        // rows are taken 32 at a time from a window of rowptr entries; after the first block (fetched one
        // chunk ahead) the window is refilled two blocks at a time (more unrolling costs more in code size than it saves), so that a chunk full of short rows
        // costs a few global round trips, not one per 32 rows
        constexpr int NB = 2;
        int64_t pw[NB];
        pw[0] = pcur;
        int have = 1;
        int64_t pnext = -1;
        bool done = false;
        while (!done) {
#pragma unroll
          for (int j = 0; j < NB; ++j) {
            if (j < have && !done) {
              const int64_t p = pw[j];
              const int row = r + nr + lane;
              const bool in = (row < R1) && (p < e + L || to_end);
              const unsigned bal = __ballot_sync(0xffffffffu, in);
              if (in) rs[nr + lane] = (int)(p - e);
              const int cnt = __popc(bal);
              if (cnt < 32) { pnext = __shfl_sync(0xffffffffu, p, cnt); nr += cnt; done = true; }  // lane cnt holds ptr[r + nr + cnt]
              else {
                nr += cnt;
                if (nr >= MAXR) { cut = (r + nr < R1); pnext = ptr[r + nr]; done = true; }
              }
            }
          }
          if (!done) {
#pragma unroll
            for (int j = 0; j < NB; ++j) {
              const int row = r + nr + 32 * j + lane;
              pw[j] = (row <= R1) ? ptr[row] : (int64_t)-1;
            }
            have = NB;
          }
        }
        if (cut && pnext < e + L) L = (int)(pnext - e);  // more than MAXR rows: the chunk ends where row r+nr starts
        const int64_t sent = pnext - e;
        const int skew = (int)(e & 3);
        // ---- move the chunk: source rounded out to 16-byte boundaries, clipped at the array end ----
        const int64_t src0 = e - skew;
        int cnt4 = (skew + L + 3) & ~3;
        int manual = 0;
        if (src0 + cnt4 > nnz) { const int avail = (int)(nnz - src0); manual = avail & 3; cnt4 = avail & ~3; }
        if (manual) {  // < 4 elements at the very end of the arrays: ordinary loads
          if (lane < manual) {
            st_idx(s)[cnt4 + lane] = idx[src0 + cnt4 + lane];
            st_val(s)[cnt4 + lane] = val[src0 + cnt4 + lane];
          }
        }
        e += L;
        r += nr;
        more = (e < E1) || (r < R1);
        if (lane == 0) {
          rs[nr] = (int)min(sent, (int64_t)0x3fffffff);
          StageHdr* h = st_hdr(s);
          h->L = L; h->nr = nr; h->r_first = r - nr; h->skew = skew; h->last = more ? 0 : 1;
        }
        __syncwarp();
        if (lane == 0) {
          if (L > 0 && cnt4 > 0) {
            const uint32_t bi = (uint32_t)cnt4 * 4u, bv = (uint32_t)cnt4 * (uint32_t)sizeof(VT);
            mbar_arrive_expect_tx(bar_full + s, bi + bv);
            bulk_g2s(st_idx(s), idx + src0, bi, bar_full + s, policy);
            bulk_g2s(st_val(s), val + src0, bv, bar_full + s, policy);
          } else {
            mbar_arrive(bar_full + s);
          }
          const int64_t pf0 = ((e + (int64_t)(PF - 1) * CH) + 3) & ~(int64_t)3;
          const int64_t pf1 = min(pf0 + CH, E1 & ~(int64_t)3);
          if (PF > 0 && pf1 > pf0) {
            bulk_prefetch_l2(idx + pf0, (uint32_t)(pf1 - pf0) * 4u);
            bulk_prefetch_l2(val + pf0, (uint32_t)(pf1 - pf0) * (uint32_t)sizeof(VT));
          }
        }
        ++cidx;
        pcur = (more && r + lane <= R1) ? ptr[r + lane] : (int64_t)-1;
      }
    }
  } else if (warp == 1) {
    // ============================== resolver: chain of slice records + epilogues ==============================
    CtaRec my_rec;
    my_rec.head = make_double2(0.0, 0.0); my_rec.tail = make_double2(0.0, 0.0);
    my_rec.head_state = 0; my_rec.tail_state = 0; my_rec.tail_row = -1; my_rec.pad = 0;
    Acc<MODE> carry;
    carry.zero();
    int carry_row = -1;  // -1: no open row; -2: the row that entered the range from the previous CTA
    if (has_work && E0 < E1 && ptr[R0] > E0) carry_row = -2;
    constexpr bool NEEDS_Y = (OP == OP_K1 || OP == OP_K2);
    int pend_row = -1;
    Acc<MODE> pend_sum;
    pend_sum.zero();
    double pend_yo = 0.0;
    int n = 0;
    bool go = has_work;
    while (go) {
      const int s = n % S;
      mbar_wait(bar_done + s, (n / S) & 1);
      const SliceRec* rec = st_rec(s);
      const int r_first = st_hdr(s)->r_first;
      go = (st_hdr(s)->last == 0);
      // lane w holds the record of slice w; the stage is handed back before anything slow happens
      double2 l_head = make_double2(0.0, 0.0), l_tail = make_double2(0.0, 0.0);
      int l_hs = 0, l_ts = 0, l_tk = 0;
      if (lane < W) { l_head = rec[lane].head; l_tail = rec[lane].tail; l_hs = rec[lane].head_state; l_ts = rec[lane].tail_state; l_tk = rec[lane].tail_k; }
      __syncwarp();
      if (lane == 0) mbar_arrive(bar_freed + s);
      bool emit;
      Acc<MODE> e_sum;
      int e_row;
      chain_scan<MODE>(l_hs, l_ts, acc_of<MODE>(l_head), acc_of<MODE>(l_tail), r_first + l_tk, carry, carry_row, emit, e_sum, e_row);
      // the row that entered the CTA from the left ends here: its sum goes to the CTA record
      const unsigned hb = __ballot_sync(0xffffffffu, emit && e_row == -2);
      if (hb) { const int src = __ffs((int)hb) - 1; my_rec.head = acc_bcast<MODE>(e_sum, src).pack(); my_rec.head_state = 2; }
      // epilogue, one chunk behind: the old y of this chunk's rows is requested now and used next time
      const int new_row = (emit && e_row >= 0) ? e_row : -1;
      double new_yo = 0.0;
      if (NEEDS_Y && new_row >= 0) new_yo = y[new_row];
      if (pend_row >= 0) finish_row_with<MODE, OP>(pend_sum, pend_yo, y, pend_row, c, sy, nsq);
      pend_row = new_row; pend_sum = e_sum; pend_yo = new_yo;
      ++n;
    }
    if (pend_row >= 0) finish_row_with<MODE, OP>(pend_sum, pend_yo, y, pend_row, c, sy, nsq);
    // the row still open at the end of the range continues in the next CTA
    if (carry_row != -1) {
      if (carry_row == -2) { my_rec.head = carry.pack(); my_rec.head_state = 1; }
      else { my_rec.tail = carry.pack(); my_rec.tail_state = 1; my_rec.tail_row = carry_row; }
    }
    my_rec.pad = (int)((clock64() - t_start) >> 4);  // busy time of this CTA in 16-cycle units (load-balance read-out)
    if (lane == 0) cta_rec[blockIdx.x] = my_rec;
  } else if (has_work) {
    // ============================== consumers ==============================
    const int w = warp - 2;
    int cidx = 0;
    while (true) {
      const int s = cidx % S;
      mbar_wait(bar_full + s, (cidx / S) & 1);
      const StageHdr* h = st_hdr(s);
      const int L = h->L, nr = h->nr, r_first = h->r_first, last = h->last;
      const int32_t* rs = st_rs(s);
      const int32_t* si = st_idx(s) + h->skew;
      const VT* sv = st_val(s) + h->skew;
      const int a = w * SL, bfull = a + SL, b = min(bfull, L);
      // number of listed rows with start <= pos (uniform binary search in shared memory)
      auto ub = [&](int pos) {
        if (nr <= 32) {  // the usual case (long rows): one shared-memory read and a vote
          const int v = (lane < nr) ? rs[lane] : 0x7fffffff;
          return __popc(__ballot_sync(0xffffffffu, v <= pos));
        }
        int lo = 0, hi = nr;
        while (lo < hi) { const int mid = (lo + hi) >> 1; if (rs[mid] <= pos) lo = mid + 1; else hi = mid; }
        return lo;
      };
      int h_state = 0, t_state = 0, t_k = 0;
      double2 h_val = make_double2(0.0, 0.0), t_val = make_double2(0.0, 0.0);
      constexpr bool NEEDS_Y = (OP == OP_K1 || OP == OP_K2);
      constexpr int NSTEP = 8, SUB = 32 * NSTEP;  // a slice is swept in rounds of 256 elements
      static_assert(SL % SUB == 0, "slice length must be a multiple of 256");
      if (a < b) {
        Sweep<MODE> st;
        st.acc.zero();
        st.dirty = false;
        st.h_state = 0;
        st.h_val = make_double2(0.0, 0.0);
        st.cur = ub(a) - 1;                                      // row containing element a (-1: open at the chunk start)
        st.started = (st.cur >= 0) && (rs[st.cur] == a);          // ... and whether it starts exactly here
        st.next_b = rs[st.cur + 1];                               // where it ends
        st.yold = 0.0;
        SweepCtx cx;
        cx.rs = rs; cx.nr = nr; cx.r_first = r_first; cx.a = a; cx.b = b; cx.has_empty = has_empty; cx.c = c; cx.sy = sy; cx.y = y;
        if (NEEDS_Y && nr > 2 * W) {  // many rows per slice: pull the old y of the slice's rows into L1
          const int k0 = st.started ? st.cur : st.cur + 1;
          const int64_t r0 = (int64_t)r_first + k0;
          const int span = min(nr - k0, SL);
          for (int t = lane * 16; t < span; t += 32 * 16) prefetch_l1(y + r0 + t);
        }
        if (NEEDS_Y && st.started && lane == 0) st.yold = y[(int64_t)r_first + st.cur];
#pragma unroll 1
        for (int ar = a; ar < b; ar += SUB) {
        const int br = min(ar + SUB, b);
        // ---- phase A: the round's matrix entries to registers, all gathers of x in flight at once ----
        double vv[NSTEP], xx[NSTEP];
        if (br == ar + SUB) {  // full round: no predicates
          int32_t cc[NSTEP];
#pragma unroll
          for (int u = 0; u < NSTEP; ++u) { cc[u] = si[ar + 32 * u + lane]; vv[u] = (double)sv[ar + 32 * u + lane]; }
#pragma unroll
          for (int u = 0; u < NSTEP; ++u) xx[u] = __ldg(x + cc[u]);
        } else {
          int32_t cc[NSTEP];
#pragma unroll
          for (int u = 0; u < NSTEP; ++u) {
            const int p0 = ar + 32 * u + lane;
            const bool ok = p0 < br;
            cc[u] = ok ? si[p0] : -1;
            vv[u] = ok ? (double)sv[p0] : 0.0;
          }
#pragma unroll
          for (int u = 0; u < NSTEP; ++u) xx[u] = (cc[u] >= 0) ? __ldg(x + cc[u]) : 0.0;
        }
        if (SCALE_X) {
#pragma unroll
          for (int u = 0; u < NSTEP; ++u) xx[u] = xx[u] * sx;
        }
        // Three shapes of a slice.  P0: it lies inside the open row (long rows: the common case).
        // P1: exactly one row ends inside it and the next one runs on to the slice end or beyond.
        // P2: anything else (short rows), step by step through one shared copy of the general code.
        if (st.next_b >= br) {
          st.acc.mac8(vv, xx);
          st.dirty = true;
        } else if (!has_empty && rs[st.cur + 2] >= br) {
          const int pe = st.next_b;  // ar <= pe < br
          Acc<MODE> accB;
          accB.zero();
          double yold_new = 0.0;
          if (NEEDS_Y && lane == 0) yold_new = y[(int64_t)r_first + st.cur + 1];
#pragma unroll
          for (int u = 0; u < NSTEP; ++u) {
            const int base = ar + 32 * u;
            if (base + 32 <= pe) st.acc.mac(vv[u], xx[u]);
            else if (base >= pe) accB.mac(vv[u], xx[u]);
            else {
              const bool first = base + lane < pe;
              st.acc.mac(first ? vv[u] : 0.0, first ? xx[u] : 0.0);
              accB.mac(first ? 0.0 : vv[u], first ? 0.0 : xx[u]);
            }
          }
          lanes_reduce<32, MODE>(st.acc);
          if (lane == 0) {
            if (st.started) finish_row_with<MODE, OP>(st.acc, st.yold, y, (int64_t)r_first + st.cur, c, sy, nsq);
            else { st.h_val = st.acc.pack(); st.h_state = 2; }
          }
          st.acc = accB;
          st.dirty = true;
          st.cur = st.cur + 1;
          st.started = true;
          st.next_b = rs[st.cur + 1];
          st.yold = yold_new;
        } else {
#pragma unroll 1
          for (int u = 0; u < NSTEP; ++u) {
            const int base = ar + 32 * u;
            if (base >= br) break;
            const int p0 = base + lane;
            const double vs = (p0 < br) ? (double)sv[p0] : 0.0;
            double xs = xx[0];
#pragma unroll
            for (int k = 1; k < NSTEP; ++k) xs = (u == k) ? xx[k] : xs;
            if (st.next_b >= base + 32 && base + 32 <= b) {  // the step lies inside the open row
              st.acc.mac(vs, xs);
              st.dirty = true;
            } else {
              sweep_slow_step<MODE, OP>(st, cx, nsq, vs, xs, base);
            }
          }
        }
        }  // rounds
        if (st.next_b == b && st.dirty) {  // the open row ends exactly at the slice end
          lanes_reduce<32, MODE>(st.acc);
          if (lane == 0) {
            if (st.started) finish_row_with<MODE, OP>(st.acc, st.yold, y, (int64_t)r_first + st.cur, c, sy, nsq);
            else { st.h_val = st.acc.pack(); st.h_state = 2; }
          }
        } else if (st.next_b > b) {  // the open row continues behind the slice
          lanes_reduce<32, MODE>(st.acc);
          if (st.started) { t_val = st.acc.pack(); t_state = 1; t_k = st.cur; }
          else { st.h_val = st.acc.pack(); st.h_state = 1; }
        }
        h_val = st.h_val;
        h_state = st.h_state;
      }
      if (has_empty) {  // rows without elements: y_r = c * y_r
        const bool owns_end = (L == 0) ? (w == 0) : (a < L && L <= bfull);
        if (a < L || owns_end) {
          auto lb = [&](int pos) {  // listed rows with start < pos
            int lo = 0, hi = nr;
            while (lo < hi) { const int mid = (lo + hi) >> 1; if (rs[mid] < pos) lo = mid + 1; else hi = mid; }
            return lo;
          };
          const int klo = lb(a), khi = owns_end ? nr : lb(b);
          for (int k = klo + lane; k < khi; k += 32) {
            if (rs[k + 1] == rs[k]) {
              Acc<MODE> z;
              z.zero();
              finish_row<MODE, OP>(z, y, (int64_t)r_first + k, c, sy, nsq);
            }
          }
        }
      }
      if (lane == 0) {
        SliceRec* rc = st_rec(s) + w;
        rc->head = h_val; rc->tail = t_val; rc->head_state = h_state; rc->tail_state = t_state; rc->tail_k = t_k;
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(bar_done + s);
      ++cidx;
      if (last) break;
    }
  }

  // ============================== per-CTA partial, last-CTA tail ==============================
  lanes_reduce<32, MODE>(nsq);
  if (lane == 0) s_slots[warp] = nsq.pack();
  __syncthreads();
  if (threadIdx.x == 0) {
    Acc<MODE> tot = acc_of<MODE>(s_slots[0]);
    for (int i = 1; i < W + 2; ++i) tot.merge(acc_of<MODE>(s_slots[i]));
    __stcg(partials + blockIdx.x, tot.pack());
    __threadfence();
    const unsigned int t = atomicAdd(&sc->ticket[0], 1u);
    *s_flag = (t == gridDim.x - 1) ? 1 : 0;
  }
  __syncthreads();
  if (*s_flag == 0) return;
  __threadfence();
  // chain the pieces of rows that cross CTA boundaries (warp 0), then the fixed-order sum of partials
  Acc<MODE> extra;
  extra.zero();
  if (warp == 0) {
    const int G = (int)gridDim.x;
    Acc<MODE> carry;
    carry.zero();
    int carry_row = -1;
    // 32 CTA records per scan; the records of the next batch are requested before this one is scanned
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
      if (emit && e_row >= 0) finish_row<MODE, OP>(e_sum, y, e_row, c, sy, extra);
      hv = hv_n; tv = tv_n; hs = hs_n; ts = ts_n; trow = trow_n;
    }
    lanes_reduce<32, MODE>(extra);
  }
  if (OP == OP_PLAIN) {
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
    for (int i = 1; i < W + 2; ++i) tot.merge(acc_of<MODE>(s_slots[i]));
    const double total = tot.value();
    if (OP == OP_K1) tail_k1(sc, total);
    if (OP == OP_K2) tail_k2(sc, total);
    if (OP == OP_K2_INIT) tail_init_v(sc, total);
    sc->ticket[0] = 0u;
  }
}

// Element split points of the G persistent CTAs: cost(e) = e + c0 * (rows that start before e) is
// cut into G equal parts; split points are rounded down to multiples of 4 elements.
__global__ void k_stream_partition(const int64_t* __restrict__ ptr, int64_t nrows, int64_t nnz, int G, int c0,
                                   int64_t* partE, int32_t* partR) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b > G) return;
  int64_t E;
  if (b == 0) E = 0;
  else if (b == G) E = nnz;
  else {
    const double total = (double)nnz + (double)c0 * (double)nrows;
    const double target = total * ((double)b / (double)G);
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
    E = e & ~(int64_t)3;
  }
  partE[b] = E;
  if (b == G) { partR[b] = (int32_t)nrows; return; }
  int64_t lo = 0, hi = nrows;  // first row with ptr[row] >= E  (nrows if none)
  while (lo < hi) {
    const int64_t mid = (lo + hi) >> 1;
    if (ptr[mid] >= E) hi = mid; else lo = mid + 1;
  }
  partR[b] = (int32_t)lo;
}

__global__ void k_count_empty(const int64_t* __restrict__ ptr, int64_t nrows, int* count) {
  int local = 0;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < nrows; i += (int64_t)gridDim.x * blockDim.x)
    if (ptr[i + 1] == ptr[i]) ++local;
  if (local) atomicAdd(count, local);
}

}  // namespace tomo
