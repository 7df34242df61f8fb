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
//   * Warp 0 is the producer: it cuts the range into chunks of <= CH elements, lists the rows that
//     start inside each chunk (local offsets in shared memory), and moves the chunk's `idx` and `val`
//     with two cp.async.bulk copies (TMA engine, L2 evict-first) into an S-stage shared-memory ring,
//     completion signalled on an mbarrier.  S-1 chunks are always in flight: memory-level parallelism
//     does not depend on registers or occupancy.
//   * Warps 1..W are consumers: each sweeps a fixed slice of every chunk, 32 consecutive elements per
//     step (conflict-free shared-memory reads), gathers x through L1/L2 and accumulates per-lane sums
//     that are reduced once per row.  Rows that start and end inside a slice are finished by the
//     consumer (axpy term, store, ||.||^2); pieces of rows that cross a slice boundary go to a small
//     per-slice record, which the producer chains in slice order after the chunk is done
//     (deterministic), finishing those rows.  Pieces of rows that cross a CTA boundary are chained by
//     the last-arriving CTA of the launch, which also sums the per-CTA ||.||^2 partials in index order
//     and runs the scalar step of the iteration (tails.cuh).
//   * Short rows (two or more row ends inside one 32-element step, e.g. the 4-7 entry smoothing
//     rows) take a segmented-reduction path: cost per step independent of the number of rows.
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
template <int CH_, int W_, int S_>
struct StreamCfg {
  static constexpr int CH = CH_;          // elements per chunk (multiple of 32*W)
  static constexpr int W = W_;            // consumer warps
  static constexpr int S = S_;            // ring stages
  static constexpr int SL = CH_ / W_;     // elements per consumer slice
  static constexpr int MAXR = CH_ / 4;    // rows listed per chunk (a chunk is cut short beyond that)
  static constexpr int THREADS = 32 * (W_ + 1);
};

struct SliceRec {      // what a consumer leaves for the producer's chain, per slice and chunk
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
  static constexpr size_t kBars = 128;  // full[S], done[S]
  static constexpr size_t kSlots = sizeof(double2) * (CFG::W + 1) + 16;
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
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
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

// The chain over slice (or CTA) records, executed uniformly by all lanes of a warp: rows whose last
// piece has been seen are handed to lane `n_emit` for the global-memory epilogue.
template <int MODE>
struct Chain {
  Acc<MODE> carry;
  int carry_row;       // global row id of the open row, -1: none
  bool carry_is_head;  // the open row started before this CTA: its sum belongs to the CTA record
  __device__ __forceinline__ void reset() { carry.zero(); carry_row = -1; carry_is_head = false; }
};

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
  constexpr int CH = CFG::CH, W = CFG::W, S = CFG::S, SL = CFG::SL, MAXR = CFG::MAXR;
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
  double2* s_slots = reinterpret_cast<double2*>(smem_raw + SM::kStage * S + SM::kBars);
  int* s_flag = reinterpret_cast<int*>(s_slots + (W + 1));

  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (threadIdx.x == 0) {
    for (int s = 0; s < S; ++s) { mbar_init(bar_full + s, 1); mbar_init(bar_done + s, W); }
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
    // ============================== producer + chain ==============================
    const uint64_t policy = l2_evict_first_policy();
    Chain<MODE> ch;
    ch.reset();
    CtaRec my_rec;
    my_rec.head = make_double2(0.0, 0.0); my_rec.tail = make_double2(0.0, 0.0);
    my_rec.head_state = 0; my_rec.tail_state = 0; my_rec.tail_row = -1; my_rec.pad = 0;
    int64_t e = E0;
    int r = R0;
    if (has_work && E0 < E1 && ptr[R0] > E0) {  // the range starts inside row R0-1
      ch.carry_row = R0 - 1;
      ch.carry_is_head = true;
    }
    int cidx = 0;           // chunks issued
    int n_resolved = 0;     // chunks whose records have been chained
    bool more = has_work;
    // chain the records of the chunk in stage s; returns this lane's row to finish (or -1) and its sum
    auto resolve = [&](int s, int& my_row, Acc<MODE>& my_sum) {
      const SliceRec* rec = st_rec(s);
      const int r_first = st_hdr(s)->r_first;
      int n_emit = 0;
      my_row = -1;
      my_sum.zero();
#pragma unroll 1
      for (int w = 0; w < W; ++w) {
        const int hs = rec[w].head_state, ts = rec[w].tail_state;
        if (hs) {
          ch.carry.merge(acc_of<MODE>(rec[w].head));
          if (hs == 2) {
            if (ch.carry_is_head) {
              my_rec.head = ch.carry.pack();
              my_rec.head_state = 2;
            } else {
              if (lane == n_emit) { my_row = ch.carry_row; my_sum = ch.carry; }
              ++n_emit;
            }
            ch.reset();
          }
        }
        if (ts) {
          ch.carry = acc_of<MODE>(rec[w].tail);
          ch.carry_row = r_first + rec[w].tail_k;
          ch.carry_is_head = false;
        }
      }
    };
    constexpr bool NEEDS_Y = (OP == OP_K1 || OP == OP_K2);
    // rowptr entries of the next 32 rows, fetched one chunk ahead so that their latency overlaps the wait
    int64_t pcur = (has_work && r + lane < R1) ? ptr[r + lane] : (int64_t)-1;
    while (more || n_resolved < cidx) {
      int my_row = -1;
      Acc<MODE> my_sum;
      my_sum.zero();
      const int s = cidx % S;
      if (more) {
        if (cidx >= S) {  // the stage is still occupied by chunk cidx - S: wait for its consumers, chain it
          mbar_wait(bar_done + s, ((cidx / S) - 1) & 1);
          resolve(s, my_row, my_sum);
          ++n_resolved;
        }
        // ---- describe chunk `cidx`: extent and the rows starting inside it ----
        int L = (int)min((int64_t)CH, E1 - e);
        const bool to_end = (e + L == E1);  // rows starting exactly at the range end belong to the next CTA, except trailing rows
        int32_t* rs = st_rs(s);
        int nr = 0;
        bool cut = false;
        int64_t p = pcur;
        while (true) {
          const int row = r + nr + lane;
          const bool in = (row < R1) && (p < e + L || to_end);
          const unsigned bal = __ballot_sync(0xffffffffu, in);
          if (in) rs[nr + lane] = (int)(p - e);
          const int cnt = __popc(bal);
          nr += cnt;
          if (cnt < 32) break;
          if (nr >= MAXR) { cut = (r + nr < R1); break; }
          p = (r + nr + lane < R1) ? ptr[r + nr + lane] : (int64_t)-1;
        }
        int64_t pnext = ptr[r + nr];  // start of the first row not listed (r + nr <= nrows)
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
        }
        ++cidx;
      } else {  // drain: chain the chunks still in the ring, oldest first
        const int sd = n_resolved % S;
        mbar_wait(bar_done + sd, (n_resolved / S) & 1);
        resolve(sd, my_row, my_sum);
        ++n_resolved;
      }
      // both loads are issued before either is used: the row pointers of the next chunk and the old y
      double yo = 0.0;
      if (NEEDS_Y && my_row >= 0) yo = y[my_row];
      pcur = (more && r + lane < R1) ? ptr[r + lane] : (int64_t)-1;
      if (my_row >= 0) finish_row_with<MODE, OP>(my_sum, yo, y, my_row, c, sy, nsq);
    }
    // the row still open at the end of the range continues in the next CTA
    if (ch.carry_row >= 0) {
      if (ch.carry_is_head) { my_rec.head = ch.carry.pack(); my_rec.head_state = 1; }
      else { my_rec.tail = ch.carry.pack(); my_rec.tail_state = 1; my_rec.tail_row = ch.carry_row; }
    }
    if (lane == 0) cta_rec[blockIdx.x] = my_rec;
  } else if (has_work) {
    // ============================== consumers ==============================
    const int w = warp - 1;
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
        int lo = 0, hi = nr;
        while (lo < hi) { const int mid = (lo + hi) >> 1; if (rs[mid] <= pos) lo = mid + 1; else hi = mid; }
        return lo;
      };
      int h_state = 0, t_state = 0, t_k = 0;
      double2 h_val = make_double2(0.0, 0.0), t_val = make_double2(0.0, 0.0);
      constexpr bool NEEDS_Y = (OP == OP_K1 || OP == OP_K2);
      if (a < b) {
        int q = a;
        int cur = ub(a) - 1;                             // row containing element a (-1: open at the chunk start)
        bool started = (cur >= 0) && (rs[cur] == a);      // ... and whether it starts exactly here
        int next_b = rs[cur + 1];                         // where it ends
        if (NEEDS_Y && nr > 2 * W) {  // many rows per slice: pull the old y of the slice's rows into L1
          const int k0 = started ? cur : cur + 1;
          const int64_t r0 = (int64_t)r_first + k0;
          const int span = min(nr - k0, SL);  // at most SL rows can start inside the slice (without empty rows)
          for (int t = lane * 16; t < span; t += 32 * 16) prefetch_l1(y + r0 + t);
        }
        Acc<MODE> acc;
        acc.zero();
        bool dirty = false;
        double yold = 0.0;  // lane 0: old y of the open row, fetched when the row starts
        if (NEEDS_Y && started && lane == 0) yold = y[(int64_t)r_first + cur];
        while (q < b) {
          const int qe = min(q + 32, b);
          if (!dirty && next_b < qe && cur + 2 <= nr && rs[cur + 2] <= qe) {
            // ---- segmented step: two or more rows end inside [q, qe) ----
            const int pos = q + lane;
            const bool valid = pos < qe;
            int k = 0x7fffffff;
            Acc<MODE> t;
            t.zero();
            if (!has_empty) {  // starts of the following rows as a bit mask over the step: k = cur + #starts <= pos
              const int j = cur + 1 + lane;
              const int sj = (j <= nr) ? rs[j] : 0x7fffffff;
              const unsigned bit = (sj < q + 32) ? (1u << (sj - q)) : 0u;
              const unsigned M = __reduce_or_sync(0xffffffffu, bit);
              if (valid) k = cur + __popc(M & ((2u << lane) - 1u));
            } else if (valid) {
              int lo = cur + 1, hi = nr;  // rs[cur] <= q <= pos
              while (lo < hi) { const int mid = (lo + hi) >> 1; if (rs[mid] <= pos) lo = mid + 1; else hi = mid; }
              k = lo - 1;
            }
            if (valid) {
              const int32_t col = si[pos];
              double xv = __ldg(x + col);
              if (SCALE_X) xv = xv * sx;
              t.mac((double)sv[pos], xv);
            }
            const int kprev = __shfl_up_sync(0xffffffffu, k, 1);
            const bool head = valid && (lane == 0 || kprev != k);
            const int kend = valid ? rs[k + 1] : 0;
            const bool fin = head && kend <= qe;            // the whole rest of row k is in this step
            const bool fin_direct = fin && (k > cur || started);
            double yo = 0.0;
            if (NEEDS_Y && fin_direct) yo = y[(int64_t)r_first + k];
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
              Acc<MODE> o = t.down(d);
              const int kk = __shfl_down_sync(0xffffffffu, k, d);
              if (lane + d < 32 && kk == k) t.merge(o);
            }
            if (fin) {
              if (fin_direct) finish_row_with<MODE, OP>(t, yo, y, (int64_t)r_first + k, c, sy, nsq);
              else { h_val = t.pack(); h_state = 2; }  // lane 0: the row open at the slice start ends here
            }
            const int nvalid = qe - q;
            const int klast = __shfl_sync(0xffffffffu, k, nvalid - 1);
            const unsigned hb = __ballot_sync(0xffffffffu, head);
            const int lhead = 31 - __clz((int)hb);
            const int klast_end = rs[klast + 1];
            if (klast_end > qe) {  // the last row of the step continues: it becomes the open row
              Acc<MODE> hv = acc_bcast<MODE>(t, lhead);
              acc.zero();
              if (lane == 0) acc = hv;
              dirty = true;
              const bool newrow = klast > cur;
              started = started || newrow;
              cur = klast;
              next_b = klast_end;
              if (NEEDS_Y && newrow && lane == 0) yold = y[(int64_t)r_first + cur];
            } else {
              acc.zero();
              dirty = false;
              if (qe < b) {
                cur = has_empty ? ub(qe) - 1 : klast + 1;
                started = true;
                next_b = rs[cur + 1];
                if (NEEDS_Y && lane == 0) yold = y[(int64_t)r_first + cur];
              } else next_b = qe;
            }
            q = qe;
          } else {
            // ---- plain steps: the rest of row `cur` inside the slice ----
            const int seg_end = min(next_b, b);
            for (; q + 256 <= seg_end; q += 256) {
              const int p0 = q + lane;
              int32_t cc[8];
              double vv[8], xx[8];
#pragma unroll
              for (int u = 0; u < 8; ++u) { cc[u] = si[p0 + 32 * u]; vv[u] = (double)sv[p0 + 32 * u]; }
#pragma unroll
              for (int u = 0; u < 8; ++u) xx[u] = __ldg(x + cc[u]);
#pragma unroll
              for (int u = 0; u < 8; ++u) { if (SCALE_X) xx[u] = xx[u] * sx; acc.mac(vv[u], xx[u]); }
            }
            if (q + 128 <= seg_end) {
              const int p0 = q + lane;
              const int32_t c0 = si[p0], c1 = si[p0 + 32], c2 = si[p0 + 64], c3 = si[p0 + 96];
              const double v0 = (double)sv[p0], v1 = (double)sv[p0 + 32], v2 = (double)sv[p0 + 64], v3 = (double)sv[p0 + 96];
              double x0 = __ldg(x + c0), x1 = __ldg(x + c1), x2 = __ldg(x + c2), x3 = __ldg(x + c3);
              if (SCALE_X) { x0 = x0 * sx; x1 = x1 * sx; x2 = x2 * sx; x3 = x3 * sx; }
              acc.mac(v0, x0); acc.mac(v1, x1); acc.mac(v2, x2); acc.mac(v3, x3);
              q += 128;
            }
            {  // up to four more steps, the last one possibly partial: all gathers issued together
              const int p0 = q + lane;
              int32_t cc[4];
              double vv[4], xx[4];
#pragma unroll
              for (int u = 0; u < 4; ++u) {
                const bool ok = p0 + 32 * u < seg_end;
                cc[u] = ok ? si[p0 + 32 * u] : 0;
                vv[u] = ok ? (double)sv[p0 + 32 * u] : 0.0;
              }
#pragma unroll
              for (int u = 0; u < 4; ++u) xx[u] = (p0 + 32 * u < seg_end) ? __ldg(x + cc[u]) : 0.0;
#pragma unroll
              for (int u = 0; u < 4; ++u) {
                if (q + 32 * u < seg_end) {  // uniform
                  if (SCALE_X) xx[u] = xx[u] * sx;
                  acc.mac(vv[u], xx[u]);     // masked lanes add an exact zero
                }
              }
              q = seg_end;
            }
            dirty = true;
            if (q == next_b) {  // the row ends here
              lanes_reduce<32, MODE>(acc);
              if (lane == 0) {
                if (started) finish_row_with<MODE, OP>(acc, yold, y, (int64_t)r_first + cur, c, sy, nsq);
                else { h_val = acc.pack(); h_state = 2; }
              }
              acc.zero();
              dirty = false;
              if (q < b) {
                cur = has_empty ? ub(q) - 1 : cur + 1;
                started = true;
                next_b = rs[cur + 1];
                if (NEEDS_Y && lane == 0) yold = y[(int64_t)r_first + cur];
              }
            }
          }
        }
        if (next_b > b) {  // the open row continues behind the slice
          lanes_reduce<32, MODE>(acc);
          if (started) { t_val = acc.pack(); t_state = 1; t_k = cur; }
          else { h_val = acc.pack(); h_state = 1; }
        }
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
    for (int i = 1; i <= W; ++i) tot.merge(acc_of<MODE>(s_slots[i]));
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
    Chain<MODE> ch;
    ch.reset();
    const int G = (int)gridDim.x;
    int n_emit = 0, my_row = -1;
    Acc<MODE> my_sum;
    my_sum.zero();
    for (int base = 0; base < G; base += 32) {
      CtaRec rc;
      rc.head_state = 0; rc.tail_state = 0; rc.tail_row = -1;
      rc.head = make_double2(0.0, 0.0); rc.tail = make_double2(0.0, 0.0);
      if (base + lane < G) {
        const CtaRec* g = cta_rec + base + lane;
        rc.head = __ldcg(&g->head); rc.tail = __ldcg(&g->tail);
        rc.head_state = __ldcg(&g->head_state); rc.tail_state = __ldcg(&g->tail_state); rc.tail_row = __ldcg(&g->tail_row);
      }
      const int cntb = min(32, G - base);
      for (int i = 0; i < cntb; ++i) {
        const int hs = __shfl_sync(0xffffffffu, rc.head_state, i), ts = __shfl_sync(0xffffffffu, rc.tail_state, i);
        if (hs) {
          double2 hv;
          hv.x = __shfl_sync(0xffffffffu, rc.head.x, i); hv.y = __shfl_sync(0xffffffffu, rc.head.y, i);
          ch.carry.merge(acc_of<MODE>(hv));
          if (hs == 2) {
            if (ch.carry_row >= 0) {
              if (lane == n_emit) { my_row = ch.carry_row; my_sum = ch.carry; }
              ++n_emit;
            }
            ch.reset();
          }
        }
        if (ts) {
          double2 tv;
          tv.x = __shfl_sync(0xffffffffu, rc.tail.x, i); tv.y = __shfl_sync(0xffffffffu, rc.tail.y, i);
          ch.carry = acc_of<MODE>(tv);
          ch.carry_row = __shfl_sync(0xffffffffu, rc.tail_row, i);
        }
        if (n_emit == 32 || (base + i == G - 1)) {
          if (my_row >= 0) finish_row<MODE, OP>(my_sum, y, my_row, c, sy, extra);
          n_emit = 0; my_row = -1;
        }
      }
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
    for (int i = 1; i <= W; ++i) tot.merge(acc_of<MODE>(s_slots[i]));
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
