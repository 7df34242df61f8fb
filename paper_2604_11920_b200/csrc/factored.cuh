// factored.cuh — the sensitivity block of A in the factored form of PAPER.md Eq. 5 with the depth-fastest
// unknown ordering of Eq. 7: SURVEY.md §8(f) NEXT-2, second form.
//
//   A = [ A_data ; A_extra ],   A_data[(q, p), (k, j)] = fl( W[q, k] * g_p[j - j0_p] )   for j0_p <= j < j0_p + klen,
//
// q = station pair (ray), p = period, k = lateral node, j = layer; row q * nper + p, column k * nz + j.  W (npairs x
// nnodes, the ray's lateral footprint) is a small CSR matrix, g_p the depth kernel of period p on its window of klen
// layers; A_extra (the smoothing rows) is an ordinary CSR block.  Nothing of A_data is stored per nonzero: a lateral
// entry (12 bytes) stands for nper * klen nonzeros of the CSR form (12 bytes each), so the operator lives in L2 and the
// products are bound by arithmetic, not by HBM.  Every product  fl(W g) * x  is formed from the ROUNDED value
// fl(W g), i.e. from exactly the number the CSR form stores, so in dd mode (order-independent sums, accum.cuh) the
// results are bit for bit those of the CSR path on the expanded matrix.
//
// Lane layout of both kernels: 32 lanes = G groups of nper lanes (G = 32 / nper; the 32 - G * nper last lanes idle).
// Lane (g, p) keeps the klen kernel values of ITS period in registers and walks the lateral entries g, g + G, ...
//   k_fac_rows (A x):   one accumulator per lane (row (q, p)); per entry klen gathers of x[k * nz + j0_p + t].
//   k_fac_cols (A^T x): klen accumulators per lane (layers j0_p .. j0_p + klen - 1 of node k); per entry ONE gather
//                       x[q * nper + p]; the layer sums of a node are put together through shared memory.
// Warps own static ranges (pairs balanced by entry count; lateral-CSC entries split evenly, a node cut by a range
// boundary leaves unrounded (hi, lo) partials and the last warp to arrive closes the node in slot order), so both
// modes are deterministic.
#pragma once
#include "accum.cuh"
#include "state.cuh"
#include "tails.cuh"

namespace tomo {

constexpr int kFacWarps = 16;
constexpr int kFacThreads = kFacWarps * 32;

struct FacSeg {        // one piece of a node's lateral-CSC entry list, owned by one warp
  int64_t e0, e1;      // entries [e0, e1) of the lateral CSC
  int32_t node;
  int32_t nsegs;       // pieces of this node (1: the warp closes the node from its registers)
  int32_t slot;        // nsegs > 1: where this piece's nz partial pairs go (seg_part + slot * nz); slot0 = slot - rank
  int32_t rank;        // index of the piece inside its node
};

struct FacDesc {       // uniform kernel argument
  int32_t nper, nz, klen, G;
  int32_t nodal, pad_;     // 1: kj0 / kern hold a table per lateral node ([nnodes * nper], [nnodes * nper * klen]); two-stage kernels only
  int64_t npairs, nnodes, mdata, ms;
  const int64_t* lptr; const int32_t* lnode; const double* lw;       // W as CSR (pairs x nodes)
  const int64_t* cptr; const int32_t* cpair; const double* cw;       // W as CSC (pairs ascending inside a node)
  const int32_t* kj0; const double* kern;                            // [nper], [nper * klen]
  const int64_t* sptr; const int32_t* sidx; const double* sval;      // A_extra as CSR (ms x n); NULL if ms == 0
  const int64_t* scptr; const int32_t* srow; const double* scval;    // A_extra as CSC; NULL if it has no entries
  const int32_t* pw;       // k_fac_rows: warp w walks the pairs pq[pw[w]] .. pq[pw[w + 1] - 1] (ascending)
  const int32_t* pq;
  const int32_t* wseg;     // k_fac_cols: first piece of every warp [NW + 1]
  const FacSeg* seg;
  double2* seg_part;       // unrounded partial layer sums of the pieces of cut nodes (slot stride nz; two-stage: pstride)
  int64_t pstride;         // max(nz, nper): slot stride of the two-stage kernels (they publish nper values per piece)
  unsigned int* node_cnt;  // arrivals per cut node; zero between launches
  long long* busy;         // per warp: cycles of its share of the most recent product launch (load balance read-out)
  double2* node_nsq;       // per node: sum of the squares of its nz results (unrounded pair), summed in node order by the last CTA
};

template <int MODE>
__device__ __forceinline__ Acc<MODE> fac_acc_of(double2 p) { Acc<MODE> r; r.unpack(p); return r; }

// y_r <- sum + c * yo  (+ running ||y||^2): the fused axpy + norm of K1 / K2 (as finish_row_with in wstream.cuh)
template <int MODE, bool AXPY, bool NORM>
__device__ __forceinline__ double fac_finish(Acc<MODE> sum, double c, double yo, Acc<MODE>& nsq) {
  double yn;
  if (AXPY) {
    if (MODE == 0) yn = fma(c, yo, sum.value());
    else { sum.mac(c, yo); yn = sum.value(); }
  } else {
    yn = sum.value();
  }
  if (NORM) nsq.mac(yn, yn);
  return yn;
}

// the block's partial of the squared norm -> partials[blockIdx.x]; the last CTA returns true
__device__ __forceinline__ bool fac_ticket(Scalars* sc, int* s_flag) {
  if (threadIdx.x == 0) {
    __threadfence();
    const unsigned int t = atomicAdd(&sc->ticket[0], 1u);
    *s_flag = (t == gridDim.x - 1) ? 1 : 0;
  }
  __syncthreads();
  const bool last = *s_flag != 0;
  if (last) __threadfence();
  return last;
}

// ------------------------------------------------------------------------------------------------------------------
// A x over the pairs:  OP_PLAIN  y = A x ;  OP_K1  u^ = A v - alpha u (u = u^ * rbeta applied where read), ||u^||^2, tail
// ------------------------------------------------------------------------------------------------------------------
template <int MODE, int OP, int KLP, bool GUARD>
__global__ void __launch_bounds__(GUARD ? kFacThreads / 2 : kFacThreads, 1)
k_fac_rows(const FacDesc d, const double* __restrict__ x, double* __restrict__ y, Scalars* sc, double2* partials) {
  __shared__ double2 s_slots[kFacWarps];
  __shared__ int s_flag;
  constexpr bool K1 = (OP == OP_K1);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int nwarp = blockDim.x >> 5;   // 16, or 8 in the general-window shape (twice the CTAs, same warp numbering)
  const int gw = blockIdx.x * nwarp + warp, NW = gridDim.x * nwarp;
  const int nper = d.nper, G = d.G, klen = GUARD ? d.klen : KLP;
  const int p = lane % nper, g = lane / nper;
  const bool active = g < G;

  // ---- prologue: nothing the previous kernel writes ----
  double kr[KLP];
#pragma unroll
  for (int t = 0; t < KLP; ++t) kr[t] = (!GUARD || t < klen) ? d.kern[(size_t)p * klen + t] : 0.0;
  const int j0 = d.kj0[p];
  constexpr bool VEC2 = (MODE == 0) && !GUARD && (KLP % 2 == 0);
  const bool vec2 = ((d.nz & 1) == 0) && ((reinterpret_cast<uintptr_t>(x) & 15u) == 0);   // pairs of layers are 16-byte aligned
  const int jodd = j0 & 1;
  const int q0 = d.pw[gw], q1 = d.pw[gw + 1];
  const int64_t x0 = d.ms * gw / NW, x1 = d.ms * (int64_t)(gw + 1) / NW;  // this warp's share of the extra rows

  grid_dependency_wait();
  const long long t_start = clock64();
  double c = 0.0, sy = 1.0;
  if (K1) {
    if (sc->stop) return;
    c = -sc->alpha; sy = sc->rbeta;
  }
  Acc<MODE> nsq;
  nsq.zero();

  int q_next = (q0 < q1) ? d.pq[q0] : 0;
  for (int i = q0; i < q1; ++i) {
    const int q = q_next;
    if (i + 1 < q1) q_next = d.pq[i + 1];
    const int64_t e0 = d.lptr[q], e1 = d.lptr[q + 1];
    Acc<MODE> a0, a1;
    a0.zero(); a1.zero();
    if (active) {
      int64_t e = e0 + g;
      bool has = e < e1;
      int k = has ? d.lnode[e] : 0;
      double w = has ? d.lw[e] : 0.0;
      while (has) {
        const double* xp = x + (int64_t)k * d.nz + j0;
        double xv[KLP];
        if (VEC2 && vec2) {
          // fast mode is bound by L1 wavefronts (one 8-byte gather per product): fetch the window as 16-byte pairs
          // from the even layer at or below j0_p and pick the lane's klen values out of them
          const double2* xq = reinterpret_cast<const double2*>(xp - jodd);
          double fl[KLP + 2];
#pragma unroll
          for (int i = 0; i < KLP / 2; ++i) { const double2 v2 = xq[i]; fl[2 * i] = v2.x; fl[2 * i + 1] = v2.y; }
          fl[KLP] = jodd ? xp[KLP - 1] : 0.0;   // an odd window ends one layer past the last pair
#pragma unroll
          for (int t = 0; t < KLP; ++t) xv[t] = jodd ? fl[t + 1] : fl[t];
        } else {
#pragma unroll
          for (int t = 0; t < KLP; ++t) xv[t] = (!GUARD || t < klen) ? xp[t] : 0.0;
        }
        const double wc = w;
        e += G;
        has = e < e1;
        if (has) { k = d.lnode[e]; w = d.lw[e]; }   // the next entry is on its way while this one is summed
#pragma unroll
        for (int t = 0; t < KLP; t += 2) {
          if (!GUARD || t < klen) a0.mac(wc * kr[t], xv[t]);
          if (t + 1 < KLP && (!GUARD || t + 1 < klen)) a1.mac(wc * kr[t + 1], xv[t + 1]);
        }
      }
    }
    a0.merge(a1);
    for (int gg = 1; gg < G; ++gg) {      // groups in index order (fixed): lane p collects lanes p + gg * nper
      const Acc<MODE> o = a0.down(gg * nper);
      if (g == 0) a0.merge(o);
    }
    if (lane < nper) {
      const int64_t r = (int64_t)q * nper + lane;
      const double yo = K1 ? y[r] * sy : 0.0;
      y[r] = fac_finish<MODE, K1, K1>(a0, c, yo, nsq);
    }
  }
  // the extra (smoothing) rows: one lane per row, entries in order
  for (int64_t r = x0 + lane; r < x1; r += 32) {
    Acc<MODE> a;
    a.zero();
    for (int64_t e = d.sptr[r]; e < d.sptr[r + 1]; ++e) a.mac(d.sval[e], x[d.sidx[e]]);
    const int64_t ro = d.mdata + r;
    const double yo = K1 ? y[ro] * sy : 0.0;
    y[ro] = fac_finish<MODE, K1, K1>(a, c, yo, nsq);
  }
  if (lane == 0) d.busy[gw] = clock64() - t_start;
  if (!K1) return;

  lanes_reduce<32, MODE>(nsq);
  if (lane == 0) s_slots[warp] = nsq.pack();
  __syncthreads();
  grid_launch_dependents();
  if (threadIdx.x == 0) {
    Acc<MODE> tot = fac_acc_of<MODE>(s_slots[0]);
    for (int i = 1; i < nwarp; ++i) tot.merge(fac_acc_of<MODE>(s_slots[i]));
    __stcg(partials + blockIdx.x, tot.pack());
  }
  if (!fac_ticket(sc, &s_flag)) return;
  const double total = final_sum<MODE>(partials, (int)gridDim.x, s_slots);
  if (threadIdx.x == 0) {
    tail_k1(sc, total);
    sc->ticket[0] = 0u;
  }
}

// ------------------------------------------------------------------------------------------------------------------
// A^T x over the lateral CSC:  OP_PLAIN  y = A^T x ;  OP_K2  v^ = A^T u - beta v, ||v^||^2, tail ;  OP_K2_INIT (no axpy)
// ------------------------------------------------------------------------------------------------------------------
template <int MODE, int OP, int KLP, bool GUARD>
__global__ void __launch_bounds__(GUARD ? kFacThreads / 2 : kFacThreads, 1)
k_fac_cols(const FacDesc d, const double* __restrict__ x, double* __restrict__ y, Scalars* sc, double2* partials) {
  extern __shared__ __align__(16) unsigned char fac_smem[];
  __shared__ double2 s_slots[kFacWarps];
  __shared__ int s_kj0[32];
  __shared__ int s_flag;
  constexpr bool NORM = (OP != OP_PLAIN), AXPY = (OP == OP_K2), SCALE = (OP != OP_PLAIN);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int gw = blockIdx.x * (blockDim.x >> 5) + warp;
  const int nper = d.nper, G = d.G, nz = d.nz, klen = GUARD ? d.klen : KLP;
  const int p = lane % nper, g = lane / nper;
  const bool active = g < G;
  double2* my = reinterpret_cast<double2*>(fac_smem) + (size_t)warp * 32 * KLP;   // [t][lane]

  double kr[KLP];
#pragma unroll
  for (int t = 0; t < KLP; ++t) kr[t] = (!GUARD || t < klen) ? d.kern[(size_t)p * klen + t] : 0.0;
  if (threadIdx.x < 32) s_kj0[threadIdx.x] = (threadIdx.x < nper) ? d.kj0[threadIdx.x] : 0;
  const int s0 = d.wseg[gw], s1 = d.wseg[gw + 1];
  __syncthreads();

  grid_dependency_wait();
  double c = 0.0, sx = 1.0;
  if (OP != OP_PLAIN) {
    if (sc->stop) return;
    if (OP == OP_K2 && sc->beta_zero) {   // beta = 0: the A^T pass is skipped, the scalar step still runs
      if (blockIdx.x == 0 && threadIdx.x == 0) tail_k2(sc, 0.0);
      return;
    }
    if (OP == OP_K2) c = -sc->beta;
    sx = sc->rbeta;
  }
  const long long t_start = clock64();

  FacSeg sg_next = {};
  if (s0 < s1) sg_next = d.seg[s0];
  for (int s = s0; s < s1; ++s) {
    const FacSeg sg = sg_next;
    if (s + 1 < s1) sg_next = d.seg[s + 1];   // the next piece's descriptor is on its way
    // the range of the extra block's column this lane will close (layer = lane): on its way during the sums
    int64_t xc0 = 0, xc1 = 0;
    if (d.scptr && lane < nz) { const int64_t colp = (int64_t)sg.node * nz + lane; xc0 = d.scptr[colp]; xc1 = d.scptr[colp + 1]; }
    Acc<MODE> acc[KLP];
#pragma unroll
    for (int t = 0; t < KLP; ++t) acc[t].zero();
    // The piece's entries go by in batches of SB steps (SB * G <= 32 entries): lane l loads entry l of the batch
    // (coalesced, one batch ahead), the lanes of group g pick entry step * G + g up by shuffle, and the gathers of U
    // steps are in flight before their sums start (the pair number no longer sits between two dependent loads).
    if (MODE == 0) {
      constexpr int U = 5;
      const int SB = 32 / G, BE = SB * G;
      int64_t eb = sg.e0;
      int qreg = 0;
      double wreg = 0.0;
      if (lane < BE && eb + lane < sg.e1) { qreg = d.cpair[eb + lane]; wreg = d.cw[eb + lane]; }
      while (eb < sg.e1) {
        const int nb = (int)((sg.e1 - eb < (int64_t)BE) ? (sg.e1 - eb) : (int64_t)BE);
        const int64_t en = eb + BE;
        int qn = 0;
        double wn = 0.0;
        if (lane < BE && en + lane < sg.e1) { qn = d.cpair[en + lane]; wn = d.cw[en + lane]; }
        for (int st = 0; st * G < nb; st += U) {
          double xs[U], ws[U];
          bool ok[U];
#pragma unroll
          for (int u = 0; u < U; ++u) {
            const int src = (st + u) * G + g;
            ok[u] = active && src < nb;
            const int q = __shfl_sync(0xffffffffu, qreg, src & 31);
            ws[u] = __shfl_sync(0xffffffffu, wreg, src & 31);
            xs[u] = ok[u] ? x[(int64_t)q * nper + p] : 0.0;
          }
#pragma unroll
          for (int u = 0; u < U; ++u) {
            if (ok[u]) {
              const double us = SCALE ? xs[u] * sx : xs[u];
#pragma unroll
              for (int t = 0; t < KLP; ++t)
                if (!GUARD || t < klen) acc[t].mac(ws[u] * kr[t], us);
            }
          }
        }
        qreg = qn; wreg = wn; eb = en;
      }
    } else if (active) {
      // dd mode: 11 fp64 instructions per product keep the pipe busy; one entry ahead is enough
      int64_t e = sg.e0 + g;
      bool has = e < sg.e1;
      int q = has ? d.cpair[e] : 0;
      double w = has ? d.cw[e] : 0.0;
      double xs = has ? x[(int64_t)q * nper + p] : 0.0;
      while (has) {
        const double wc = w;
        const double us = SCALE ? xs * sx : xs;
        e += G;
        has = e < sg.e1;
        if (has) { q = d.cpair[e]; w = d.cw[e]; xs = x[(int64_t)q * nper + p]; }
#pragma unroll
        for (int t = 0; t < KLP; ++t)
          if (!GUARD || t < klen) acc[t].mac(wc * kr[t], us);
      }
    }
    const bool none = sg.e0 == sg.e1;   // a node no ray touches: closed from the extra block alone
    if (!none) {
#pragma unroll
      for (int t = 0; t < KLP; ++t) my[t * 32 + lane] = acc[t].pack();
    }
    __syncwarp();
    const int node = sg.node;
    const bool whole = sg.nsegs == 1;
    Acc<MODE> nsq;
    nsq.zero();
    // the closing of layer j of this node: the extra rows' column, the axpy, the rounding, the norm
    auto close = [&](int j, Acc<MODE> S) {
      const int64_t col = (int64_t)node * nz + j;
      const double yo = AXPY ? y[col] : 0.0;
      if (d.scptr) {   // eight entries at a time: the loads of one level are all in flight before the next level starts
        const int64_t c0 = (j == lane) ? xc0 : d.scptr[col], c1 = (j == lane) ? xc1 : d.scptr[col + 1];
        for (int64_t base = c0; base < c1; base += 8) {
          int32_t rr[8];
          double vv[8], xe[8];
#pragma unroll
          for (int i = 0; i < 8; ++i) {
            const bool in = base + i < c1;
            rr[i] = in ? d.srow[base + i] : 0;
            vv[i] = in ? d.scval[base + i] : 0.0;
          }
#pragma unroll
          for (int i = 0; i < 8; ++i) xe[i] = (base + i < c1) ? x[d.mdata + rr[i]] : 0.0;
#pragma unroll
          for (int i = 0; i < 8; ++i)
            if (base + i < c1) S.mac(vv[i], SCALE ? xe[i] * sx : xe[i]);
        }
      }
      y[col] = fac_finish<MODE, AXPY, NORM>(S, c, yo, nsq);
    };
    for (int j = lane; j < nz; j += 32) {   // layer sums over periods (ascending) and groups (ascending): fixed order
      Acc<MODE> S;
      S.zero();
      if (!none) {
        for (int pp = 0; pp < nper; ++pp) {
          const int t = j - s_kj0[pp];
          if (t >= 0 && t < klen)
            for (int gg = 0; gg < G; ++gg) S.merge(fac_acc_of<MODE>(my[t * 32 + gg * nper + pp]));
        }
      }
      if (whole) close(j, S);
      else __stcg(d.seg_part + (size_t)sg.slot * nz + j, S.pack());
    }
    bool closer = whole;
    if (!whole) {
      __threadfence();
      __syncwarp();
      unsigned int old = 0;
      if (lane == 0) old = atomicAdd(d.node_cnt + node, 1u);
      old = __shfl_sync(0xffffffffu, old, 0);
      if (old == (unsigned int)(sg.nsegs - 1)) {    // every other piece of the node has been published
        __threadfence();
        closer = true;
        if (lane == 0) d.node_cnt[node] = 0u;
        const double2* base = d.seg_part + (size_t)(sg.slot - sg.rank) * nz;
        for (int j = lane; j < nz; j += 32) {
          Acc<MODE> S = fac_acc_of<MODE>(__ldcg(base + j));
          for (int r = 1; r < sg.nsegs; ++r) S.merge(fac_acc_of<MODE>(__ldcg(base + (size_t)r * nz + j)));
          close(j, S);
        }
      }
    }
    if (NORM && closer) {
      lanes_reduce<32, MODE>(nsq);
      if (lane == 0) __stcg(d.node_nsq + node, nsq.pack());
    }
    __syncwarp();
  }
  if (lane == 0) d.busy[gw] = clock64() - t_start;
  if (!NORM) return;

  __threadfence();   // the per-node norm pairs this warp wrote, before the CTA takes its ticket
  __syncthreads();
  grid_launch_dependents();
  if (!fac_ticket(sc, &s_flag)) return;
  const double total = final_sum<MODE>(d.node_nsq, (int)d.nnodes, s_slots);
  if (threadIdx.x == 0) {
    if (OP == OP_K2) tail_k2(sc, total);
    if (OP == OP_K2_INIT) tail_init_v(sc, total);
    sc->ticket[0] = 0u;
  }
}

// validation of the depth-kernel table: windows inside [0, nz), finite values
__global__ void k_fac_validate_kern(int64_t nper, int nz, int klen, const int32_t* __restrict__ kj0, const double* __restrict__ kern,
                                    int* flags) {   // nper: number of windows (periods, or nodes * periods of a nodal table)
  int bad = 0;
  const int64_t i0 = (int64_t)blockIdx.x * blockDim.x + threadIdx.x, stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t i = i0; i < nper; i += stride)
    if (kj0[i] < 0 || kj0[i] + klen > nz) bad = 1;
  for (int64_t i = i0; i < nper * klen; i += stride)
    if (!(fabs(kern[i]) <= 1.79769313486231570815e308)) bad = 1;
  if (bad) atomicOr(flags, 1);
}

}  // namespace tomo

namespace tomo {

// ------------------------------------------------------------------------------------------------------------------
// On-device assembly of G (Eq. 5, Eq. 7): the factored description
// multiplied out into the canonical CSR arrays the general path takes.  One warp per station pair: the pair's
// nper rows are cnt * klen elements each and contiguous, so the stores are coalesced; W is read through L1.
// value = fl(W[q, k] * g_p[t]) (one rounding), column = k * nz + j0_p + t.  HBM-bound: 12 bytes written per nonzero.
// ------------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_fac_assemble(int64_t npairs, int nper, int nz, int klen, int nodal, const int64_t* __restrict__ lptr,
                                                      const int32_t* __restrict__ lnode, const double* __restrict__ lw,
                                                      const int32_t* __restrict__ kj0, const double* __restrict__ kern, int64_t ms,
                                                      const int64_t* __restrict__ sptr, const int32_t* __restrict__ sidx,
                                                      const double* __restrict__ sval, int64_t* __restrict__ rowptr,
                                                      int32_t* __restrict__ colind, double* __restrict__ vals) {
  const int lane = threadIdx.x & 31;
  const int64_t warp = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int64_t nwarps = ((int64_t)gridDim.x * blockDim.x) >> 5;
  const int64_t per_entry = (int64_t)nper * klen;
  const int di = 32 / klen, dt = 32 - di * klen;
  for (int64_t q = warp; q < npairs; q += nwarps) {
    const int64_t e0 = lptr[q], e1 = lptr[q + 1];
    const int64_t cnt = e1 - e0, rowlen = cnt * klen, base = e0 * per_entry;
    if (lane < nper) rowptr[q * nper + lane] = base + (int64_t)lane * rowlen;
    for (int p = 0; p < nper; ++p) {
      const int j0 = kj0[p];
      const double* kp = kern + (size_t)p * klen;
      const int64_t out = base + (int64_t)p * rowlen;
      // element idx = i * klen + t of the row; the lane steps by 32 elements: (i, t) advance without a division
      int64_t i = lane / klen;
      int t = lane - (int)i * klen;
      for (int64_t idx = lane; idx < rowlen; idx += 32) {
        const int node = lnode[e0 + i];
        if (nodal) {   // the node's own table (kj0[k * nper + p], kern[(k * nper + p) * klen + t])
          const int64_t tab = (int64_t)node * nper + p;
          colind[out + idx] = node * nz + kj0[tab] + t;
          vals[out + idx] = lw[e0 + i] * kern[tab * klen + t];
        } else {
          colind[out + idx] = node * nz + j0 + t;
          vals[out + idx] = lw[e0 + i] * kp[t];
        }
        i += di; t += dt;
        if (t >= klen) { t -= klen; ++i; }
      }
    }
  }
  // the extra block, appended unchanged
  const int64_t nnz_data = lptr[npairs] * per_entry, mdata = npairs * nper;
  const int64_t tid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x, nthreads = (int64_t)gridDim.x * blockDim.x;
  if (ms > 0) {
    const int64_t snnz = sptr[ms];
    for (int64_t r = tid; r <= ms; r += nthreads) rowptr[mdata + r] = nnz_data + sptr[r];
    for (int64_t e = tid; e < snnz; e += nthreads) { colind[nnz_data + e] = sidx[e]; vals[nnz_data + e] = sval[e]; }
  } else if (tid == 0) {
    rowptr[mdata] = nnz_data;
  }
}

}  // namespace tomo

namespace tomo {

// ------------------------------------------------------------------------------------------------------------------
// Fast mode, two-stage contraction (option "two_stage", default on; accumulate = 0 only).  In exact arithmetic
//     (A_data x)[q, p] = sum_k W[q, k] * S[k, p],        S[k, p] = sum_t g_p[t] * x[k * nz + j0_p + t]
//     (A_data^T u)[k, j] = sum_p g_p[j - j0_p] * T[k, p],  T[k, p] = sum_q W[q, k] * u[q * nper + p]
// i.e. the depth contraction is done once per node instead of once per ray entry: klen times fewer products.  The
// operator applied is W (x) g with UNROUNDED entries; it differs from the stored-CSR operator (entries fl(W g)) by
// one rounding per entry, which is inside what "fast" claims (plain fp64 sums, any association; DESIGN.md F-fac2).
// dd mode never takes this path: its bit-for-bit contract is on the rounded entries.
// ------------------------------------------------------------------------------------------------------------------
template <int MODE> struct Fac2S { using type = double; };
template <> struct Fac2S<1> { using type = double2; };   // dd: S[k, p] and T[k, p] stay unrounded (hi, lo) pairs

template <int MODE>
__global__ void __launch_bounds__(256) k_fac2_stage(const FacDesc d, const double* __restrict__ x, typename Fac2S<MODE>::type* __restrict__ S,
                                                    const Scalars* sc, int check_stop) {
  grid_dependency_wait();
  if (check_stop && sc->stop) return;
  const int64_t total = d.nnodes * d.nper;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) {
    const int64_t k = i / d.nper;
    const int p = (int)(i - k * d.nper);
    const int64_t tab = d.nodal ? i : (int64_t)p;   // the node's own table, or the one all nodes share
    const double* xp = x + k * d.nz + d.kj0[tab];
    const double* kp = d.kern + (size_t)tab * d.klen;
    Acc<MODE> s;
    s.zero();
    for (int t = 0; t < d.klen; ++t) s.mac(kp[t], xp[t]);
    if constexpr (MODE == 0) S[i] = s.value(); else S[i] = s.pack();
  }
  grid_launch_dependents();
}

// Entries [e0, e1) of a CSR / CSC list of W, for lane (g, p) the entries g, g + G, ... in order: use(weight, gather(index)).
// The entries go by in coalesced batches of SB = 32 / G steps (lane l loads entry l of the batch, one batch ahead; the
// groups pick theirs up by shuffle), the gathers of U steps are in flight before they are used.  (Issuing the next
// batch's gathers before the current batch is consumed was measured slower: 9.0 k -> 7.6 k it/s at config 1.)
template <int U, typename VT, typename GATHER, typename USE>
__device__ __forceinline__ void fac2_walk(const int32_t* __restrict__ idx, const double* __restrict__ val, int64_t e0, int64_t e1, int G, int g,
                                          bool active, int lane, GATHER gather, USE use) {
  const int SB = 32 / G, BE = SB * G;
  int64_t eb = e0;
  int ireg = 0;
  double wreg = 0.0;
  if (lane < BE && eb + lane < e1) { ireg = idx[eb + lane]; wreg = val[eb + lane]; }
  while (eb < e1) {
    const int nb = (int)((e1 - eb < (int64_t)BE) ? (e1 - eb) : (int64_t)BE);
    const int64_t en = eb + BE;
    int in = 0;
    double wn = 0.0;
    if (lane < BE && en + lane < e1) { in = idx[en + lane]; wn = val[en + lane]; }
    for (int st = 0; st * G < nb; st += U) {
      // no branch per step: a step beyond the batch takes weight 0 and entry 0 (its product adds an exact zero); the
      // idle lanes behind the last group sum into accumulators nobody reads
      VT xs[U];
      double ws[U];
#pragma unroll
      for (int u = 0; u < U; ++u) {
        const int src = (st + u) * G + g;
        const bool in = src < nb;
        const int i = __shfl_sync(0xffffffffu, ireg, src & 31);
        const double w = __shfl_sync(0xffffffffu, wreg, src & 31);
        ws[u] = in ? w : 0.0;
        xs[u] = gather(in ? i : 0);
      }
#pragma unroll
      for (int u = 0; u < U; ++u) use(ws[u], xs[u]);
    }
    ireg = in; wreg = wn; eb = en;
  }
}

template <int MODE, int OP>   // OP_PLAIN, OP_K1
__global__ void __launch_bounds__(kFacThreads, 1)
k_fac2_rows(const FacDesc d, const typename Fac2S<MODE>::type* __restrict__ S, const double* __restrict__ x, double* __restrict__ y, Scalars* sc, double2* partials) {
  __shared__ double2 s_slots[kFacWarps];
  __shared__ int s_flag;
  constexpr bool K1 = (OP == OP_K1);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
  const int gw = blockIdx.x * nwarp + warp, NW = gridDim.x * nwarp;
  const int nper = d.nper, G = d.G;
  const int p = lane % nper, g = lane / nper;
  const bool active = g < G;
  const int q0 = d.pw[gw], q1 = d.pw[gw + 1];
  const int64_t x0 = d.ms * gw / NW, x1 = d.ms * (int64_t)(gw + 1) / NW;
  grid_dependency_wait();
  const long long t_start = clock64();
  double c = 0.0, sy = 1.0;
  if (K1) {
    if (sc->stop) return;
    c = -sc->alpha; sy = sc->rbeta;
  }
  Acc<MODE> nsq;
  nsq.zero();
  int q_next = (q0 < q1) ? d.pq[q0] : 0;
  int64_t en0 = 0, en1 = 0;
  if (q0 < q1) { en0 = d.lptr[q_next]; en1 = d.lptr[q_next + 1]; }
  int q_next2 = (q0 + 1 < q1) ? d.pq[q0 + 1] : 0;
  for (int i = q0; i < q1; ++i) {
    const int q = q_next;
    const int64_t pe0 = en0, pe1 = en1;
    q_next = q_next2;
    if (i + 1 < q1) { en0 = d.lptr[q_next]; en1 = d.lptr[q_next + 1]; }   // the next pair's range and the pair after it
    if (i + 2 < q1) q_next2 = d.pq[i + 2];
    const int64_t r = (int64_t)q * nper + lane;
    const double yo = (K1 && lane < nper) ? y[r] * sy : 0.0;
    Acc<MODE> a;
    a.zero();
    using SV = typename Fac2S<MODE>::type;
    fac2_walk<10, SV>(d.lnode, d.lw, pe0, pe1, G, g, active, lane,
                      [&](int k) { return S[(int64_t)k * nper + p]; },
                      [&](double w, SV sv) {
                        if constexpr (MODE == 0) a.mac(w, sv);
                        else {   // w * (hi + lo): TwoProd of the high word, the low word's product joins its error term
                          const double pr = w * sv.x;
                          const double er = fma(w, sv.y, fma(w, sv.x, -pr));
                          double sm, qq;
                          two_sum(a.v.hi, pr, sm, qq);
                          a.v.hi = sm;
                          a.v.lo = a.v.lo + (qq + er);
                        }
                      });
    for (int gg = 1; gg < G; ++gg) {
      const Acc<MODE> o = a.down(gg * nper);
      if (g == 0) a.merge(o);
    }
    if (lane < nper) y[r] = fac_finish<MODE, K1, K1>(a, c, yo, nsq);
  }
  for (int64_t r = x0 + lane; r < x1; r += 32) {
    Acc<MODE> a;
    a.zero();
    for (int64_t e = d.sptr[r]; e < d.sptr[r + 1]; ++e) a.mac(d.sval[e], x[d.sidx[e]]);
    const int64_t ro = d.mdata + r;
    const double yo = K1 ? y[ro] * sy : 0.0;
    y[ro] = fac_finish<MODE, K1, K1>(a, c, yo, nsq);
  }
  if (lane == 0) d.busy[gw] = clock64() - t_start;
  if (!K1) return;
  lanes_reduce<32, MODE>(nsq);
  if (lane == 0) s_slots[warp] = nsq.pack();
  __syncthreads();
  grid_launch_dependents();
  if (threadIdx.x == 0) {
    Acc<MODE> tot = fac_acc_of<MODE>(s_slots[0]);
    for (int i = 1; i < nwarp; ++i) tot.merge(fac_acc_of<MODE>(s_slots[i]));
    __stcg(partials + blockIdx.x, tot.pack());
  }
  if (!fac_ticket(sc, &s_flag)) return;
  const double total = final_sum<MODE>(partials, (int)gridDim.x, s_slots);
  if (threadIdx.x == 0) {
    tail_k1(sc, total);
    sc->ticket[0] = 0u;
  }
}

template <int MODE, int OP>   // OP_PLAIN, OP_K2, OP_K2_INIT
__global__ void __launch_bounds__(kFacThreads, 1)
k_fac2_cols(const FacDesc d, const double* __restrict__ x, double* __restrict__ y, Scalars* sc, double2* partials) {
  __shared__ double2 s_T[kFacWarps][32];   // per warp: the node's T[p] (dd: unrounded pairs)
  __shared__ double2 s_slots[kFacWarps];
  __shared__ int s_kj0[32];
  __shared__ int s_flag;
  constexpr bool NORM = (OP != OP_PLAIN), AXPY = (OP == OP_K2), SCALE = (OP != OP_PLAIN);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int gw = blockIdx.x * (blockDim.x >> 5) + warp;
  const int nper = d.nper, G = d.G, nz = d.nz, klen = d.klen;
  const int p = lane % nper, g = lane / nper;
  const bool active = g < G;
  double2* my = s_T[warp];
  if (threadIdx.x < 32) s_kj0[threadIdx.x] = (threadIdx.x < nper) ? d.kj0[threadIdx.x] : 0;
  const int s0 = d.wseg[gw], s1 = d.wseg[gw + 1];
  __syncthreads();
  grid_dependency_wait();
  double c = 0.0, sx = 1.0;
  if (OP != OP_PLAIN) {
    if (sc->stop) return;
    if (OP == OP_K2 && sc->beta_zero) {
      if (blockIdx.x == 0 && threadIdx.x == 0) tail_k2(sc, 0.0);
      return;
    }
    if (OP == OP_K2) c = -sc->beta;
    sx = sc->rbeta;
  }
  const long long t_start = clock64();
  FacSeg sg_next = {};
  if (s0 < s1) sg_next = d.seg[s0];
  for (int s = s0; s < s1; ++s) {
    const FacSeg sg = sg_next;
    if (s + 1 < s1) sg_next = d.seg[s + 1];
    const int node = sg.node;
    int64_t xc0 = 0, xc1 = 0;
    if (d.scptr && lane < nz) { const int64_t colp = (int64_t)node * nz + lane; xc0 = d.scptr[colp]; xc1 = d.scptr[colp + 1]; }
    Acc<MODE> a;
    a.zero();
    fac2_walk<10, double>(d.cpair, d.cw, sg.e0, sg.e1, G, g, active, lane,
                 [&](int q) { const double xe = x[(int64_t)q * nper + p]; return SCALE ? xe * sx : xe; },
                 [&](double w, double us) { a.mac(w, us); });
    for (int gg = 1; gg < G; ++gg) {     // T[p] of this piece in lanes 0 .. nper-1 (groups in index order)
      const Acc<MODE> o = a.down(gg * nper);
      if (g == 0) a.merge(o);
    }
    bool closer = sg.nsegs == 1;
    if (!closer) {    // a cut node: publish this piece's T, the last piece to arrive adds them in slot order
      if (lane < nper) __stcg(d.seg_part + (size_t)sg.slot * d.pstride + lane, a.pack());
      __threadfence();
      __syncwarp();
      unsigned int old = 0;
      if (lane == 0) old = atomicAdd(d.node_cnt + node, 1u);
      old = __shfl_sync(0xffffffffu, old, 0);
      if (old == (unsigned int)(sg.nsegs - 1)) {
        __threadfence();
        closer = true;
        if (lane == 0) d.node_cnt[node] = 0u;
        if (lane < nper) {
          const double2* base = d.seg_part + (size_t)(sg.slot - sg.rank) * d.pstride + lane;
          a.unpack(__ldcg(base));
          for (int r = 1; r < sg.nsegs; ++r) a.merge(fac_acc_of<MODE>(__ldcg(base + (size_t)r * d.pstride)));
        }
      }
    }
    if (closer) {
      if (lane < nper) my[lane] = a.pack();
      __syncwarp();
      Acc<MODE> nsq;
      nsq.zero();
      for (int j = lane; j < nz; j += 32) {
        const int64_t col = (int64_t)node * nz + j;
        const double yo = AXPY ? y[col] : 0.0;
        Acc<MODE> S;
        S.zero();
        for (int pp = 0; pp < nper; ++pp) {     // the depth contraction: periods ascending
          const int64_t tab = d.nodal ? (int64_t)node * nper + pp : (int64_t)pp;
          const int t = j - (d.nodal ? d.kj0[tab] : s_kj0[pp]);
          if (t >= 0 && t < klen) {
            const double gk = d.kern[(size_t)tab * klen + t];
            const double2 Tp = my[pp];
            S.mac(gk, Tp.x);
            if (MODE == 1) S.mac(gk, Tp.y);   // g * (hi + lo): both words as exact products
          }
        }
        if (d.scptr) {
          const int64_t c0 = (j == lane) ? xc0 : d.scptr[col], c1 = (j == lane) ? xc1 : d.scptr[col + 1];
          for (int64_t base = c0; base < c1; base += 8) {
            int32_t rr[8];
            double vv[8], xe[8];
#pragma unroll
            for (int i = 0; i < 8; ++i) {
              const bool in = base + i < c1;
              rr[i] = in ? d.srow[base + i] : 0;
              vv[i] = in ? d.scval[base + i] : 0.0;
            }
#pragma unroll
            for (int i = 0; i < 8; ++i) xe[i] = (base + i < c1) ? x[d.mdata + rr[i]] : 0.0;
#pragma unroll
            for (int i = 0; i < 8; ++i)
              if (base + i < c1) S.mac(vv[i], SCALE ? xe[i] * sx : xe[i]);
          }
        }
        y[col] = fac_finish<MODE, AXPY, NORM>(S, c, yo, nsq);
      }
      if (NORM) {
        lanes_reduce<32, MODE>(nsq);
        if (lane == 0) __stcg(d.node_nsq + node, nsq.pack());
      }
    }
    __syncwarp();
  }
  if (lane == 0) d.busy[gw] = clock64() - t_start;
  if (!NORM) return;
  __threadfence();
  __syncthreads();
  grid_launch_dependents();
  if (!fac_ticket(sc, &s_flag)) return;
  const double total = final_sum<MODE>(d.node_nsq, (int)d.nnodes, s_slots);
  if (threadIdx.x == 0) {
    if (OP == OP_K2) tail_k2(sc, total);
    if (OP == OP_K2_INIT) tail_init_v(sc, total);
    sc->ticket[0] = 0u;
  }
}

}  // namespace tomo
