// tomo_lsqr.cu — host side of libtomolsqr.so: the C ABI of include/tomo_lsqr.h, handle lifetime,
// the create pipeline (validate -> transpose -> partitions), the solve driver (init kernels, CUDA-graph
// replay of `check_every` iterations, one host poll per replay) and the inspection hooks.
// All arithmetic of the method is in the kernels (kernels.cuh, tails.cuh); this file only launches.
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "../../include/tomo_lsqr.h"
#include "build.cuh"
#include "kernels.cuh"
#include "wstream.cuh"
#include "compress.cuh"
#include "shard.cuh"
#include "multi.cuh"
#include "factored.cuh"

using namespace tomo;

namespace {

thread_local char g_cuda_msg[256] = "no CUDA error recorded";
thread_local char g_noalloc_msg[256] = "tomo_lsqr_spmv_noalloc: beyond the static scratch array (TOMO_NOALLOC_MAX_ROWS / TOMO_NOALLOC_MAX_SMS)";

tomo_status_t cuda_fail(cudaError_t e, const char* what) {
  snprintf(g_cuda_msg, sizeof(g_cuda_msg), "CUDA error in %s: %s", what, cudaGetErrorString(e));
  cudaGetLastError();  // clear the sticky-less error state
  return e == cudaErrorMemoryAllocation ? TOMO_ERR_OOM : TOMO_ERR_CUDA;
}

#define CK(call)                                             \
  do {                                                       \
    cudaError_t e__ = (call);                                \
    if (e__ != cudaSuccess) return cuda_fail(e__, #call);    \
  } while (0)

bool is_device_ptr(const void* p) {
  if (!p) return false;
  cudaPointerAttributes a;
  if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
  return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

struct PollWord { int32_t itn, istop, stop; };

constexpr int kMaxProfileIters = 1 << 16;

}  // namespace

// one direction of the sparse product as the streaming kernel sees it (wstream.cuh): 0 = A over the caller's CSR,
// 1 = A^T over the CSC copy
struct Dir {
  const int64_t* ptr = nullptr;   // starts of the non-empty rows (alias of the CSR / CSC pointer array if no row is empty)
  int64_t* ptr_own = nullptr;     // ... owned copy when rows had to be compacted away
  int32_t* rid = nullptr;         // row numbers of the non-empty rows (NULL: identity)
  int32_t* erows = nullptr;       // rows without elements
  int nrows = 0, n_empty = 0;     // nrows: non-empty rows
  const int32_t* idx = nullptr; const void* val = nullptr;
  int64_t* wE = nullptr; int32_t* wR = nullptr;   // split points of the sms * W warp ranges
  unsigned char* cidx = nullptr; int64_t* coff = nullptr; int64_t cbytes = 0, heads = 0;  // run-compressed index (FMT 1)
};

// the factored sensitivity block (factored.cuh; tomo_lsqr_create_factored): what the handle owns of it
struct FacState {
  FacDesc d = {};                 // the kernel argument (borrowed W / A_extra CSR arrays, owned rest)
  FacDesc dm[4];                  // ... per mode (0 fast, 1 dd, 2 fast two-stage, 3 dd two-stage): the A^T x work split differs (wseg, seg)
  double2* S2 = nullptr;          // two-stage contraction: S[k, p], the depth contraction of x per node and period (fast: doubles, dd: pairs)
  int64_t E = 0, snnz = 0;        // lateral entries, entries of the extra rows
  int klp = 0; bool guard = false;  // kernel shape: window length as a template constant (8, 12, 16) or the general one (32, guarded)
  int nsegs = 0, nslots = 0;
  int64_t* cptr = nullptr; int32_t* cpair = nullptr; double* cw = nullptr;
  int32_t* kj0 = nullptr; double* kern = nullptr;
  int32_t* kj0n = nullptr; double* kernn = nullptr;   // nodal tables (tomo_lsqr_set_nodal_kernels)
  int64_t* scptr = nullptr; int32_t* srow = nullptr; double* scval = nullptr;
  int32_t* pw = nullptr; int32_t* pq = nullptr; int32_t* pw2 = nullptr; int32_t* pq2 = nullptr; int32_t* wseg[4] = {nullptr, nullptr, nullptr, nullptr}; FacSeg* seg[4] = {nullptr, nullptr, nullptr, nullptr};
  double2* seg_part = nullptr; unsigned int* node_cnt = nullptr; double2* node_nsq = nullptr; long long* busy = nullptr;
};

struct tomo_lsqr_s {
  int64_t m = 0, n = 0, nnz = 0;
  FacState* fac = nullptr;               // non-NULL: A is held in factored form, the CSR / CSC members below are unused
  int device = 0;                        // the device the handle was created on; every call checks it is current
  tomo_valtype_t vt = TOMO_VAL_F64;
  // borrowed CSR
  const int64_t* rowptr = nullptr; const int32_t* colind = nullptr; const void* vals = nullptr;
  // owned CSC (= CSR of A^T)
  int64_t* colptr = nullptr; int32_t* rowind = nullptr; void* cvals = nullptr;
  // element split points of the persistent CTAs, per direction
  bool part_dirty = true;
  Dir dir[2];
  CtaRec* cta_rec = nullptr; int SG = 0;
  // work vectors and device state
  double *u = nullptr, *v = nullptr, *w = nullptr, *x = nullptr, *hbar = nullptr;  // w doubles as LSMR's h
  int solver = 0;  // 0 LSQR, 1 LSMR (set per solve)
  // shared-pass multi-RHS state (multi.cuh): len x 8 blocks, eight Scalars, static row partitions
  double *mU = nullptr, *mV = nullptr, *mW = nullptr, *mX = nullptr, *mH = nullptr; Scalars* msc = nullptr; Scalars* h_msc = nullptr;
  CtaRec8* cta_rec8 = nullptr; double2* mpartials = nullptr; int MG = 0, multi_shared = 1;
  bool multi_ready = false;              // every m* allocation succeeded and the partitions were computed
  PollWord* h_mpoll = nullptr;           // pinned: two slots of eight {itn, istop, stop} words
  cudaGraphExec_t mgexec = nullptr; int mgraph_k = 0, mgraph_mode = -1;
  Scalars* sc = nullptr; double2* part_spmv = nullptr; double2* part_vec = nullptr; int part_cap = 0;
  double *hist_r2 = nullptr, *hist_ar = nullptr; int32_t hist_cap = 0;
  double *bh = nullptr, *xh = nullptr;   // device staging for solve_host
  Scalars* h_sc = nullptr; PollWord* h_poll = nullptr;  // pinned
  cudaEvent_t ev_poll[2] = {nullptr, nullptr};
  cudaStream_t cap_stream = nullptr;
  cudaGraphExec_t gexec = nullptr; int graph_k = 0, graph_mode = -1, graph_G = 0;
  // options
  int check_every = 10, accumulate = 1, use_graph = 1, profile = 0, row_cost = 320, pdl = 1, compress = 0, two_stage = 1;
  // info
  int sms = 0; double create_ms = 0, transpose_ms = 0, transpose_kernels_ms = 0, update_ms = 0, scratch_bytes = 0;
  double2* sh_send = nullptr; double2* sh_recv = nullptr; int64_t sh_send_cap = 0, sh_recv_cap = 0;  // exchange buffers of the sharded solve
  void* pos = nullptr; bool pos_wide = false;   // CSR element -> CSC slot (built by the first tomo_lsqr_update_values)
  double k1_ms = 0, k2_ms = 0, k4_ms = 0, k_launches = 0;
  double kernels_enqueued = 0;  // cumulative count of this library's kernel launches (graph nodes included)
  std::vector<cudaEvent_t> prof_ev;
};

namespace {

int vec_blocks(const tomo_lsqr_s* h, int64_t len) {
  int64_t b = (len + kThreads - 1) / kThreads;
  return (int)std::max<int64_t>(1, std::min<int64_t>(b, (int64_t)h->sms * 16));
}

// Kernel shapes <elements per tile, ring stages per warp, warps per CTA> (wstream.cuh), per direction (measured on
// B200, config 1).  Every warp streams its own contiguous element range through its own ring.  A over the CSR
// gathers v^ (n doubles, runs of consecutive columns): a 3-stage ring (144 KB) keeps two tiles per warp in
// flight.  A^T over the CSC gathers u^ (m doubles, short runs): the 2-stage ring (96 KB) leaves ~130 KB of L1 to
// the gather, which is worth more there than the deeper ring.
#ifndef TOMO_TILE
#define TOMO_TILE 256
#endif
#ifndef TOMO_NS
#define TOMO_NS 3
#endif
#ifndef TOMO_NS_T
#define TOMO_NS_T 2
#endif
#ifndef TOMO_W
#define TOMO_W 16
#endif
using WC = WCfg<TOMO_TILE, TOMO_NS, TOMO_W>;      // A over the CSR
using WCT = WCfg<TOMO_TILE, TOMO_NS_T, TOMO_W>;   // A^T over the CSC copy (same tile and warp count: same kind of split points)
template <bool TR> struct WCOf { using type = WC; };
template <> struct WCOf<true> { using type = WCT; };

template <int MODE, typename VT, int OP, int FMT, bool TR>
cudaError_t launch_wstream_t(const tomo_lsqr_s* h, const double* x, double* y, cudaStream_t st, Scalars* sc_shared = nullptr) {
  using C = typename WCOf<TR>::type;
  const Dir& d = h->dir[TR ? 1 : 0];
  auto kern = k_wstream<C, MODE, VT, OP, FMT>;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)h->SG); cfg.blockDim = dim3(C::THREADS);
  cfg.dynamicSmemBytes = WSmem<C, VT, FMT>::kTotal; cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at; cfg.numAttrs = (h->pdl && OP != OP_PLAIN && OP != OP_K1S && OP != OP_K2S) ? 1 : 0;
  return cudaLaunchKernelEx(&cfg, kern, d.ptr, (const int32_t*)d.rid, d.idx, (const VT*)d.val, (const unsigned char*)d.cidx,
                            (const int64_t*)d.coff, h->nnz, d.nrows, (const int32_t*)d.erows, d.n_empty, x, y,
                            (const int64_t*)d.wE, (const int32_t*)d.wR, h->cta_rec, sc_shared ? sc_shared : h->sc, h->part_spmv);
}

// The > 48 KB dynamic shared memory opt-in of every k_wstream instantiation, on the CURRENT device (function
// attributes are per device): called by create, so that a handle on a second GPU works and a refusal is
// reported at create rather than as an opaque launch error inside a stream capture.
template <typename C, int MODE, typename VT, int OP, int FMT>
cudaError_t stream_attr_one() {
  return cudaFuncSetAttribute(k_wstream<C, MODE, VT, OP, FMT>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                              (int)WSmem<C, VT, FMT>::kTotal);
}
template <int MODE, typename VT, int FMT>
cudaError_t stream_attr_ops() {
  cudaError_t e;
  if ((e = stream_attr_one<WC, MODE, VT, OP_PLAIN, FMT>()) != cudaSuccess) return e;
  if ((e = stream_attr_one<WC, MODE, VT, OP_K1, FMT>()) != cudaSuccess) return e;
  if ((e = stream_attr_one<WCT, MODE, VT, OP_PLAIN, FMT>()) != cudaSuccess) return e;
  if ((e = stream_attr_one<WCT, MODE, VT, OP_K2, FMT>()) != cudaSuccess) return e;
  if (FMT == 0) {  // the row-sharded solve runs on the int32 index
    if ((e = stream_attr_one<WC, MODE, VT, OP_K1S, 0>()) != cudaSuccess) return e;
    if ((e = stream_attr_one<WCT, MODE, VT, OP_K2S, 0>()) != cudaSuccess) return e;
  }
  return stream_attr_one<WCT, MODE, VT, OP_K2_INIT, FMT>();
}
template <typename VT>
cudaError_t stream_attr_vt() {
  cudaError_t e;
  if ((e = stream_attr_ops<0, VT, 0>()) != cudaSuccess) return e;
  if ((e = stream_attr_ops<1, VT, 0>()) != cudaSuccess) return e;
  if ((e = stream_attr_ops<0, VT, 1>()) != cudaSuccess) return e;
  return stream_attr_ops<1, VT, 1>();
}
cudaError_t set_kernel_attributes(tomo_valtype_t vt) {
  return vt == TOMO_VAL_F64 ? stream_attr_vt<double>() : stream_attr_vt<float>();
}

template <int MODE, typename VT, int OP, int FMT>
void launch_wstream_dir(const tomo_lsqr_s* h, bool transpose, const double* x, double* y, cudaStream_t st) {
  // K1 runs over the CSR only, K2 / K2_INIT over the CSC only; the plain product runs over either
  if (OP == OP_K1) launch_wstream_t<MODE, VT, OP_K1, FMT, false>(h, x, y, st);
  else if (OP == OP_K2) launch_wstream_t<MODE, VT, OP_K2, FMT, true>(h, x, y, st);
  else if (OP == OP_K2_INIT) launch_wstream_t<MODE, VT, OP_K2_INIT, FMT, true>(h, x, y, st);
  else if (transpose) launch_wstream_t<MODE, VT, OP_PLAIN, FMT, true>(h, x, y, st);
  else launch_wstream_t<MODE, VT, OP_PLAIN, FMT, false>(h, x, y, st);
}

// ---- factored operator (factored.cuh): launch shapes ----
template <int KLP, bool GUARD> constexpr size_t fac_cols_smem() { return (size_t)(GUARD ? kFacWarps / 2 : kFacWarps) * 32 * KLP * sizeof(double2); }

template <int MODE, int OP, int KLP, bool GUARD>
cudaError_t launch_fac_one(const tomo_lsqr_s* h, bool cols, const double* x, double* y, cudaStream_t st) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)(GUARD ? 2 * h->sms : h->sms));
  cfg.blockDim = dim3(GUARD ? kFacThreads / 2 : kFacThreads);
  cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at; cfg.numAttrs = (h->pdl && OP != OP_PLAIN) ? 1 : 0;
  if (cols) {
    if constexpr (OP == OP_PLAIN || OP == OP_K2 || OP == OP_K2_INIT) {
      cfg.dynamicSmemBytes = fac_cols_smem<KLP, GUARD>();
      return cudaLaunchKernelEx(&cfg, k_fac_cols<MODE, OP, KLP, GUARD>, h->fac->dm[MODE], x, y, h->sc, h->part_spmv);
    }
  } else {
    if constexpr (OP == OP_PLAIN || OP == OP_K1) {
      cfg.dynamicSmemBytes = 0;
      return cudaLaunchKernelEx(&cfg, k_fac_rows<MODE, OP, KLP, GUARD>, h->fac->dm[MODE], x, y, h->sc, h->part_spmv);
    }
  }
  return cudaErrorInvalidValue;
}
template <int MODE, int OP>
cudaError_t launch_fac_mode(const tomo_lsqr_s* h, bool cols, const double* x, double* y, cudaStream_t st) {
  switch (h->fac->klp) {
    case 8: return launch_fac_one<MODE, OP, 8, false>(h, cols, x, y, st);
    case 12: return launch_fac_one<MODE, OP, 12, false>(h, cols, x, y, st);
    case 16: return launch_fac_one<MODE, OP, 16, false>(h, cols, x, y, st);
    default: return launch_fac_one<MODE, OP, 32, true>(h, cols, x, y, st);
  }
}
// two-stage contraction (k_fac2_*): the depth contraction once per node, then W.  Fast mode by default; dd mode with
// option "two_stage" = 2 (exact entries W*g, reading F-fac3)
template <int MODE, int OP>
cudaError_t launch_fac2(const tomo_lsqr_s* h, bool cols, const double* x, double* y, cudaStream_t st) {
  const FacState* f = h->fac;
  using SV = typename Fac2S<MODE>::type;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cudaLaunchConfig_t cfg = {};
  cfg.stream = st; cfg.attrs = at; cfg.numAttrs = (h->pdl && OP != OP_PLAIN) ? 1 : 0;
  cfg.blockDim = dim3(kFacThreads); cfg.gridDim = dim3((unsigned)h->sms);
  if (cols) {
    if constexpr (OP == OP_PLAIN || OP == OP_K2 || OP == OP_K2_INIT)
      return cudaLaunchKernelEx(&cfg, k_fac2_cols<MODE, OP>, f->dm[MODE ? 3 : 2], x, y, h->sc, h->part_spmv);
  } else {
    if constexpr (OP == OP_PLAIN || OP == OP_K1) {
      cudaLaunchConfig_t c1 = cfg;
      c1.blockDim = dim3(256);
      c1.gridDim = dim3((unsigned)std::max<int64_t>(1, std::min<int64_t>((f->d.nnodes * f->d.nper + 255) / 256, (int64_t)h->sms * 8)));
      cudaError_t e = cudaLaunchKernelEx(&c1, k_fac2_stage<MODE>, f->dm[MODE ? 3 : 2], x, (SV*)f->S2, (const Scalars*)h->sc, OP == OP_K1 ? 1 : 0);
      if (e != cudaSuccess) return e;
      return cudaLaunchKernelEx(&cfg, k_fac2_rows<MODE, OP>, f->dm[MODE ? 3 : 2], (const SV*)f->S2, x, y, h->sc, h->part_spmv);
    }
  }
  return cudaErrorInvalidValue;
}
template <int OP>
void launch_fac(const tomo_lsqr_s* h, bool transpose, const double* x, double* y, cudaStream_t st) {
  if (h->fac->d.nodal) { if (h->accumulate) launch_fac2<1, OP>(h, transpose, x, y, st); else launch_fac2<0, OP>(h, transpose, x, y, st); return; }
  if (h->accumulate) { if (h->two_stage == 2) launch_fac2<1, OP>(h, transpose, x, y, st); else launch_fac_mode<1, OP>(h, transpose, x, y, st); }
  else if (h->two_stage) launch_fac2<0, OP>(h, transpose, x, y, st);
  else launch_fac_mode<0, OP>(h, transpose, x, y, st);
}
// the > 48 KB dynamic shared memory opt-in of the k_fac_cols instantiations on the current device
template <int MODE, int KLP, bool GUARD>
cudaError_t fac_attr_one() {
  cudaError_t e;
  const int b = (int)fac_cols_smem<KLP, GUARD>();
  if ((e = cudaFuncSetAttribute(k_fac_cols<MODE, OP_PLAIN, KLP, GUARD>, cudaFuncAttributeMaxDynamicSharedMemorySize, b)) != cudaSuccess) return e;
  if ((e = cudaFuncSetAttribute(k_fac_cols<MODE, OP_K2, KLP, GUARD>, cudaFuncAttributeMaxDynamicSharedMemorySize, b)) != cudaSuccess) return e;
  return cudaFuncSetAttribute(k_fac_cols<MODE, OP_K2_INIT, KLP, GUARD>, cudaFuncAttributeMaxDynamicSharedMemorySize, b);
}
cudaError_t set_fac_attributes(int klp) {
  cudaError_t e;
  switch (klp) {
    case 8: if ((e = fac_attr_one<0, 8, false>()) != cudaSuccess) return e; return fac_attr_one<1, 8, false>();
    case 12: if ((e = fac_attr_one<0, 12, false>()) != cudaSuccess) return e; return fac_attr_one<1, 12, false>();
    case 16: if ((e = fac_attr_one<0, 16, false>()) != cudaSuccess) return e; return fac_attr_one<1, 16, false>();
    default: if ((e = fac_attr_one<0, 32, true>()) != cudaSuccess) return e; return fac_attr_one<1, 32, true>();
  }
}

template <int OP>
void launch_spmv(const tomo_lsqr_s* h, bool transpose, const double* x, double* y, cudaStream_t st) {
  if (h->fac) { launch_fac<OP>(h, transpose, x, y, st); return; }
  const bool cz = h->compress && h->dir[transpose ? 1 : 0].cidx;
  if (h->vt == TOMO_VAL_F64) {
    if (h->accumulate) { if (cz) launch_wstream_dir<1, double, OP, 1>(h, transpose, x, y, st); else launch_wstream_dir<1, double, OP, 0>(h, transpose, x, y, st); }
    else { if (cz) launch_wstream_dir<0, double, OP, 1>(h, transpose, x, y, st); else launch_wstream_dir<0, double, OP, 0>(h, transpose, x, y, st); }
  } else {
    if (h->accumulate) { if (cz) launch_wstream_dir<1, float, OP, 1>(h, transpose, x, y, st); else launch_wstream_dir<1, float, OP, 0>(h, transpose, x, y, st); }
    else { if (cz) launch_wstream_dir<0, float, OP, 1>(h, transpose, x, y, st); else launch_wstream_dir<0, float, OP, 0>(h, transpose, x, y, st); }
  }
}

template <int VOP>
void launch_vec(const tomo_lsqr_s* h, const double* in0, double* a0, double* a1, double* a2, int64_t len, cudaStream_t st,
                double* a3 = nullptr) {
  const int g = vec_blocks(h, len);
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)g); cfg.blockDim = dim3(kThreads); cfg.dynamicSmemBytes = 0; cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at; cfg.numAttrs = (h->pdl && (VOP == VOP_K4 || VOP == VOP_K4_LSMR)) ? 1 : 0;
  if (h->accumulate) cudaLaunchKernelEx(&cfg, k_vec<1, VOP>, in0, a0, a1, a2, a3, len, h->sc, h->part_vec);
  else cudaLaunchKernelEx(&cfg, k_vec<0, VOP>, in0, a0, a1, a2, a3, len, h->sc, h->part_vec);
}

// the vector update that closes an iteration: LSQR's x / w step or LSMR's hbar / x / h step
void launch_k4(const tomo_lsqr_s* h, cudaStream_t st) {
  if (h->solver == 1) launch_vec<VOP_K4_LSMR>(h, nullptr, h->v, h->w, h->x, h->n, st, h->hbar);
  else launch_vec<VOP_K4>(h, nullptr, h->v, h->w, h->x, h->n, st);
}

tomo_status_t rebuild_partitions(tomo_lsqr_s* h, cudaStream_t st) {
  if (h->fac) { h->part_dirty = false; return TOMO_OK; }   // a factored handle has its own static splits (built at create)
  if (!h->part_dirty) return TOMO_OK;
  const int tb = 128;
  // one persistent CTA per SM, W warp ranges each: cost-balanced element split points at multiples of the tile size
  // (fewer CTAs for small systems were measured slower: config 0 35 instead of 26 us per launch — the launch is
  // bound by the serial tiles of a warp, not by the chain over CTA records)
  h->SG = h->sms;
  const int parts = h->SG * WC::W;
  const int gs = (parts + 1 + tb - 1) / tb;
  for (int d = 0; d < 2; ++d)
    k_stream_partition<<<gs, tb, 0, st>>>(h->dir[d].ptr, h->dir[d].nrows, h->nnz, parts, h->row_cost, WC::TILE, h->dir[d].wE, h->dir[d].wR);
  CK(cudaGetLastError());
  h->part_dirty = false;
  return TOMO_OK;
}

// Rows (d = 0) or columns (d = 1) without elements are compacted away for the streaming kernel and listed.
tomo_status_t build_dir(tomo_lsqr_s* h, int d, const int64_t* ptr, int64_t nrows, const int32_t* idx, const void* val,
                        cudaStream_t st) {
  Dir& D = h->dir[d];
  D.idx = idx; D.val = val; D.ptr = ptr; D.nrows = (int)nrows; D.n_empty = 0;
  int* d_cnt = nullptr;
  CK(cudaMalloc(&d_cnt, sizeof(int)));
  cudaMemsetAsync(d_cnt, 0, sizeof(int), st);
  k_count_empty<<<h->sms * 4, 256, 0, st>>>(ptr, nrows, d_cnt);
  int cnt = 0;
  cudaError_t e = cudaMemcpyAsync(&cnt, d_cnt, sizeof(int), cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  cudaFree(d_cnt);
  if (e != cudaSuccess) return cuda_fail(e, "count empty rows");
  if (cnt > 0) {
    int64_t *flag = nullptr, *pos = nullptr;
    const int64_t ne = nrows - cnt;
    e = cudaMalloc(&flag, sizeof(int64_t) * (nrows + 1));
    if (e == cudaSuccess) e = cudaMalloc(&pos, sizeof(int64_t) * (nrows + 1));
    if (e == cudaSuccess) e = cudaMalloc(&D.ptr_own, sizeof(int64_t) * (ne + 1));
    if (e == cudaSuccess) e = cudaMalloc(&D.rid, sizeof(int32_t) * std::max<int64_t>(ne, 1));
    if (e == cudaSuccess) e = cudaMalloc(&D.erows, sizeof(int32_t) * cnt);
    if (e == cudaSuccess) {
      k_flag_nonempty<<<h->sms * 4, 256, 0, st>>>(ptr, nrows, flag);
      k_exscan<<<1, 1024, 0, st>>>(flag, nrows, pos);
      k_compact_rows<<<h->sms * 4, 256, 0, st>>>(ptr, nrows, pos, D.ptr_own, D.rid, D.erows);
      e = cudaGetLastError();
      if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    }
    cudaFree(flag); cudaFree(pos);
    if (e != cudaSuccess) return cuda_fail(e, "compact empty rows");
    D.ptr = D.ptr_own; D.nrows = (int)ne; D.n_empty = cnt;
  }
  const int parts = h->sms * WC::W;
  CK(cudaMalloc(&D.wE, sizeof(int64_t) * (parts + 1)));
  CK(cudaMalloc(&D.wR, sizeof(int32_t) * (parts + 1)));
  return TOMO_OK;
}

}  // namespace

namespace {
// NEXT-2: the run-compressed index of direction d (compress.cuh), built on first use of option "compress".
tomo_status_t build_compressed(tomo_lsqr_s* h, int d, cudaStream_t st) {
  Dir& D = h->dir[d];
  if (D.cidx || h->nnz == 0) return TOMO_OK;
  const int64_t ntiles = (h->nnz + WC::TILE - 1) / WC::TILE;
  int64_t* size = nullptr; int64_t* coff = nullptr; unsigned char* out = nullptr;
  cudaError_t e = cudaMalloc(&size, sizeof(int64_t) * ntiles);
  if (e == cudaSuccess) e = cudaMalloc(&coff, sizeof(int64_t) * (ntiles + 1));
  int64_t total = 0;
  if (e == cudaSuccess) {
    k_cz_size<WC::TILE><<<h->sms * 8, 256, 0, st>>>(D.idx, h->nnz, ntiles, size);
    k_exscan<<<1, 1024, 0, st>>>(size, ntiles, coff);
    e = cudaMemcpyAsync(&total, coff + ntiles, sizeof(int64_t), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  }
  if (e == cudaSuccess) e = cudaMalloc(&out, (size_t)total + 16);
  if (e == cudaSuccess) e = cudaMemsetAsync(out, 0, (size_t)total + 16, st);
  if (e == cudaSuccess) {
    k_cz_fill<WC::TILE><<<h->sms * 8, 256, 0, st>>>(D.idx, h->nnz, ntiles, coff, out);
    e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  }
  cudaFree(size);
  if (e != cudaSuccess) { cudaFree(coff); cudaFree(out); return cuda_fail(e, "build the run-compressed index"); }
  D.cidx = out; D.coff = coff; D.cbytes = total;
  D.heads = (total - ntiles * (WC::TILE / 8)) / 4;  // upper bound (includes the 16-byte padding)
  return TOMO_OK;
}
}  // namespace

// ------------------------------------------------------------------------------------------------
// create / destroy
// ------------------------------------------------------------------------------------------------
namespace {

// The transpose passes (build.cuh).  only_pos = false: allocate and fill the CSC copy (create).  only_pos = true:
// the CSC copy exists; replay the passes to record the permutation pos[q] = CSC slot of CSR element q
// (uint32 when nnz < 2^32, else int64) that tomo_lsqr_update_values needs; built on its first call.
template <typename VT>
tomo_status_t build_csc(tomo_lsqr_s* h, cudaStream_t st, bool only_pos) {
  const int64_t m = h->m, n = h->n, nnz = h->nnz;
  if (!only_pos) {
    CK(cudaMalloc(&h->colptr, sizeof(int64_t) * (n + 1)));
    CK(cudaMalloc(&h->rowind, sizeof(int32_t) * std::max<int64_t>(nnz, 1)));
    CK(cudaMalloc(&h->cvals, sizeof(VT) * std::max<int64_t>(nnz, 1)));
  } else {
    h->pos_wide = nnz >= ((int64_t)1 << 32);
    CK(cudaMalloc(&h->pos, (h->pos_wide ? sizeof(int64_t) : sizeof(uint32_t)) * std::max<int64_t>(nnz, 1)));
  }
  // number of row chunks (= warps): bounded by the scratch budget T*n*4 bytes <= 4 GB
  int64_t T = std::min<int64_t>((int64_t)h->sms * 16, std::max<int64_t>(32, (int64_t)(4.0e9 / (4.0 * (double)n))));
  T = std::max<int64_t>(1, std::min<int64_t>(T, m));
  int32_t* chunk = nullptr; uint32_t* cnt = nullptr; int64_t* coltotal = nullptr;
  auto drop_pos = [&]() { if (only_pos) { cudaFree(h->pos); h->pos = nullptr; } };  // a half-built permutation must not survive
  cudaError_t e = cudaMalloc(&chunk, sizeof(int32_t) * (T + 1));
  if (e != cudaSuccess) { drop_pos(); return cuda_fail(e, "cudaMalloc(transpose chunks)"); }
  e = cudaMalloc(&cnt, sizeof(uint32_t) * T * n);
  if (e != cudaSuccess) { cudaFree(chunk); drop_pos(); return cuda_fail(e, "cudaMalloc(transpose scratch)"); }
  e = cudaMalloc(&coltotal, sizeof(int64_t) * n);
  if (e != cudaSuccess) { cudaFree(chunk); cudaFree(cnt); drop_pos(); return cuda_fail(e, "cudaMalloc(coltotal)"); }
  h->scratch_bytes = (double)(sizeof(uint32_t) * T * n + sizeof(int64_t) * n + sizeof(int32_t) * (T + 1));
  tomo_status_t rc = TOMO_OK;
  cudaEvent_t k0 = nullptr, k1 = nullptr;
  cudaEventCreate(&k0); cudaEventCreate(&k1);
  do {
    const int tb = 128;
    cudaEventRecord(k0, st);
    k_partition<<<(int)((T + 1 + tb - 1) / tb), tb, 0, st>>>(h->rowptr, m, (int)T, 1, 1, chunk);
    k_partition_fix<<<1, 32, 0, st>>>((int)T, chunk);
    if ((e = cudaMemsetAsync(cnt, 0, sizeof(uint32_t) * T * n, st)) != cudaSuccess) break;
    const int wb = (int)((T + kWarps - 1) / kWarps);
    k_tr_count<<<wb, kThreads, 0, st>>>(h->rowptr, h->colind, chunk, (int)T, n, cnt);
    k_tr_colscan<<<(int)((n + 255) / 256), 256, 0, st>>>((int)T, n, cnt, coltotal);
    if (!only_pos) {
      k_exscan<<<1, 1024, 0, st>>>(coltotal, n, h->colptr);
      k_tr_scatter<VT, uint32_t><<<wb, kThreads, 0, st>>>(h->rowptr, h->colind, (const VT*)h->vals, chunk, (int)T, n, cnt,
                                                         h->colptr, h->rowind, (VT*)h->cvals, (uint32_t*)nullptr);
    } else if (h->pos_wide) {
      k_tr_scatter<VT, int64_t><<<wb, kThreads, 0, st>>>(h->rowptr, h->colind, (const VT*)h->vals, chunk, (int)T, n, cnt,
                                                        h->colptr, (int32_t*)nullptr, (VT*)nullptr, (int64_t*)h->pos);
    } else {
      k_tr_scatter<VT, uint32_t><<<wb, kThreads, 0, st>>>(h->rowptr, h->colind, (const VT*)h->vals, chunk, (int)T, n, cnt,
                                                         h->colptr, (int32_t*)nullptr, (VT*)nullptr, (uint32_t*)h->pos);
    }
    cudaEventRecord(k1, st);
    if ((e = cudaGetLastError()) != cudaSuccess) break;
    e = cudaStreamSynchronize(st);
    float ms = 0;
    if (e == cudaSuccess && !only_pos && cudaEventElapsedTime(&ms, k0, k1) == cudaSuccess) h->transpose_kernels_ms = ms;
  } while (0);
  if (k0) cudaEventDestroy(k0);
  if (k1) cudaEventDestroy(k1);
  if (e != cudaSuccess) rc = cuda_fail(e, "CSR->CSC transpose");
  cudaFree(chunk); cudaFree(cnt); cudaFree(coltotal);
  if (rc != TOMO_OK && only_pos) { cudaFree(h->pos); h->pos = nullptr; }
  return rc;
}

void free_handle(tomo_lsqr_s* h) {
  if (!h) return;
  if (h->gexec) cudaGraphExecDestroy(h->gexec);
  if (h->cap_stream) cudaStreamDestroy(h->cap_stream);
  for (int i = 0; i < 2; ++i) if (h->ev_poll[i]) cudaEventDestroy(h->ev_poll[i]);
  for (cudaEvent_t e : h->prof_ev) cudaEventDestroy(e);
  cudaFree(h->colptr); cudaFree(h->rowind); cudaFree(h->cvals); cudaFree(h->pos); cudaFree(h->sh_send); cudaFree(h->sh_recv);
  cudaFree(h->mU); cudaFree(h->mV); cudaFree(h->mW); cudaFree(h->mX); cudaFree(h->mH); cudaFree(h->msc); cudaFree(h->cta_rec8);
  cudaFree(h->mpartials); if (h->h_msc) cudaFreeHost(h->h_msc); if (h->h_mpoll) cudaFreeHost(h->h_mpoll); if (h->mgexec) cudaGraphExecDestroy(h->mgexec);
  for (Dir& D : h->dir) { cudaFree(D.ptr_own); cudaFree(D.rid); cudaFree(D.erows); cudaFree(D.wE); cudaFree(D.wR); cudaFree(D.cidx); cudaFree(D.coff); }
  if (FacState* f = h->fac) {
    cudaFree(f->cptr); cudaFree(f->cpair); cudaFree(f->cw); cudaFree(f->kj0); cudaFree(f->kern); cudaFree(f->kj0n); cudaFree(f->kernn);
    cudaFree(f->scptr); cudaFree(f->srow); cudaFree(f->scval); cudaFree(f->pw); cudaFree(f->pq); cudaFree(f->pw2); cudaFree(f->pq2); cudaFree(f->S2); for (int i = 0; i < 4; ++i) { cudaFree(f->wseg[i]); cudaFree(f->seg[i]); }
    cudaFree(f->seg_part); cudaFree(f->node_cnt); cudaFree(f->node_nsq); cudaFree(f->busy);
    delete f;
  }
  cudaFree(h->cta_rec);
  cudaFree(h->u); cudaFree(h->v); cudaFree(h->w); cudaFree(h->x); cudaFree(h->hbar);
  cudaFree(h->sc); cudaFree(h->part_spmv); cudaFree(h->part_vec);
  cudaFree(h->hist_r2); cudaFree(h->hist_ar); cudaFree(h->bh); cudaFree(h->xh);
  if (h->h_sc) cudaFreeHost(h->h_sc);
  if (h->h_poll) cudaFreeHost(h->h_poll);
  cudaGetLastError();
  delete h;
}

}  // namespace

extern "C" tomo_status_t tomo_lsqr_create(tomo_lsqr_t* out, int64_t m, int64_t n, int64_t nnz, const int64_t* d_rowptr,
                                          const int32_t* d_colind, const void* d_vals, tomo_valtype_t vt,
                                          void* cuda_stream) {
  if (!out) return TOMO_ERR_INVALID_ARG;
  *out = nullptr;
  if (vt != TOMO_VAL_F64 && vt != TOMO_VAL_F32) return TOMO_ERR_INVALID_ARG;
  if (m < 1 || n < 1 || nnz < 0) return TOMO_ERR_INVALID_ARG;
  if (m >= (int64_t)INT32_MAX || n >= (int64_t)INT32_MAX || nnz >= ((int64_t)1 << 40)) return TOMO_ERR_RANGE;  // warp ranges hold 32-bit relative offsets
  if (!d_rowptr || (nnz > 0 && (!d_colind || !d_vals))) return TOMO_ERR_INVALID_ARG;
  int dev = 0, major = 0, sms = 0;
  CK(cudaGetDevice(&dev));
  CK(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
  CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  if (major != 10) return TOMO_ERR_UNSUPPORTED_ARCH;
  if (!is_device_ptr(d_rowptr) || (nnz > 0 && (!is_device_ptr(d_colind) || !is_device_ptr(d_vals))))
    return TOMO_ERR_NOT_DEVICE_PTR;
  if (((uintptr_t)d_colind & 15u) || ((uintptr_t)d_vals & 15u) || ((uintptr_t)d_rowptr & 7u)) return TOMO_ERR_INVALID_ARG;
  cudaStream_t st = (cudaStream_t)cuda_stream;

  tomo_lsqr_s* h = new (std::nothrow) tomo_lsqr_s();
  if (!h) return TOMO_ERR_OOM;
  h->m = m; h->n = n; h->nnz = nnz; h->vt = vt; h->sms = sms; h->device = dev;
  { cudaError_t ea = set_kernel_attributes(vt); if (ea != cudaSuccess) { delete h; return cuda_fail(ea, "cudaFuncSetAttribute(shared memory opt-in)"); } }
  h->rowptr = d_rowptr; h->colind = d_colind; h->vals = d_vals;

  cudaEvent_t e0 = nullptr, e1 = nullptr, e2 = nullptr;
  tomo_status_t rc = TOMO_OK;
  int* d_flags = nullptr;
  do {
    cudaError_t e;
    if ((e = cudaEventCreate(&e0)) != cudaSuccess || (e = cudaEventCreate(&e1)) != cudaSuccess ||
        (e = cudaEventCreate(&e2)) != cudaSuccess) { rc = cuda_fail(e, "cudaEventCreate"); break; }
    cudaEventRecord(e0, st);
    // --- validation (one device pass, one sync) ---
    if ((e = cudaMalloc(&d_flags, sizeof(int))) != cudaSuccess) { rc = cuda_fail(e, "cudaMalloc"); break; }
    cudaMemsetAsync(d_flags, 0, sizeof(int), st);
    if (vt == TOMO_VAL_F64) k_validate<double><<<sms * 8, kThreads, 0, st>>>(m, n, nnz, d_rowptr, d_colind, (const double*)d_vals, d_flags);
    else k_validate<float><<<sms * 8, kThreads, 0, st>>>(m, n, nnz, d_rowptr, d_colind, (const float*)d_vals, d_flags);
    int flags = 0;
    if ((e = cudaMemcpyAsync(&flags, d_flags, sizeof(int), cudaMemcpyDeviceToHost, st)) != cudaSuccess ||
        (e = cudaStreamSynchronize(st)) != cudaSuccess) { rc = cuda_fail(e, "CSR validation"); break; }
    if (flags) { rc = TOMO_ERR_BAD_CSR; break; }
    // --- transpose ---
    cudaEventRecord(e1, st);
    rc = (vt == TOMO_VAL_F64) ? build_csc<double>(h, st, false) : build_csc<float>(h, st, false);
    if (rc != TOMO_OK) break;
    cudaEventRecord(e2, st);
    // --- work space ---
    h->part_cap = sms * 32 + 2;  // >= the largest grid of any kernel that publishes partials
#define ALLOC(p, bytes) if ((e = cudaMalloc(&(p), (bytes))) != cudaSuccess) { rc = cuda_fail(e, "cudaMalloc(work)"); break; }
    ALLOC(h->cta_rec, sizeof(CtaRec) * sms);
    ALLOC(h->u, sizeof(double) * m); ALLOC(h->v, sizeof(double) * n);
    ALLOC(h->w, sizeof(double) * n); ALLOC(h->x, sizeof(double) * n);
    ALLOC(h->sc, sizeof(Scalars));
    ALLOC(h->part_spmv, sizeof(double2) * h->part_cap);
    ALLOC(h->part_vec, sizeof(double2) * h->part_cap);
#undef ALLOC
    if ((e = cudaMemsetAsync(h->sc, 0, sizeof(Scalars), st)) != cudaSuccess) { rc = cuda_fail(e, "memset"); break; }
    // the two directions of the product as the streaming kernel sees them (rows / columns without entries are
    // compacted away and listed)
    if ((rc = build_dir(h, 0, h->rowptr, m, h->colind, h->vals, st)) != TOMO_OK) break;
    if ((rc = build_dir(h, 1, h->colptr, n, h->rowind, h->cvals, st)) != TOMO_OK) break;
    if ((e = cudaMallocHost(&h->h_sc, sizeof(Scalars))) != cudaSuccess ||
        (e = cudaMallocHost(&h->h_poll, 2 * sizeof(PollWord))) != cudaSuccess) { rc = cuda_fail(e, "cudaMallocHost"); break; }
    for (int i = 0; i < 2; ++i)
      if ((e = cudaEventCreateWithFlags(&h->ev_poll[i], cudaEventDisableTiming)) != cudaSuccess) break;
    if (e != cudaSuccess) { rc = cuda_fail(e, "cudaEventCreate"); break; }
    if ((e = cudaStreamCreateWithFlags(&h->cap_stream, cudaStreamNonBlocking)) != cudaSuccess) { rc = cuda_fail(e, "cudaStreamCreate"); break; }
    rc = rebuild_partitions(h, st);
    if (rc != TOMO_OK) break;
    if ((e = cudaStreamSynchronize(st)) != cudaSuccess) { rc = cuda_fail(e, "create"); break; }
    float ms = 0;
    cudaEventElapsedTime(&ms, e1, e2); h->transpose_ms = ms;
    cudaEventRecord(e1, st); cudaEventSynchronize(e1);
    cudaEventElapsedTime(&ms, e0, e1); h->create_ms = ms;
  } while (0);
  if (d_flags) cudaFree(d_flags);
  if (e0) cudaEventDestroy(e0);
  if (e1) cudaEventDestroy(e1);
  if (e2) cudaEventDestroy(e2);
  if (rc != TOMO_OK) { free_handle(h); return rc; }
  *out = h;
  return TOMO_OK;
}

// ------------------------------------------------------------------------------------------------
// NEXT-2, factored form (factored.cuh): create
// ------------------------------------------------------------------------------------------------
namespace {

// CSR -> CSC of a small block with the transpose passes of build.cuh (a temporary handle carries the arguments)
tomo_status_t transpose_block(int sms, int64_t m, int64_t n, int64_t nnz, const int64_t* ptr, const int32_t* idx, const double* val,
                              cudaStream_t st, int64_t** cptr, int32_t** cidx, double** cval) {
  tomo_lsqr_s t;
  t.m = m; t.n = n; t.nnz = nnz; t.sms = sms; t.rowptr = ptr; t.colind = idx; t.vals = val;
  tomo_status_t rc = build_csc<double>(&t, st, false);
  if (rc != TOMO_OK) { cudaFree(t.colptr); cudaFree(t.rowind); cudaFree(t.cvals); return rc; }
  *cptr = t.colptr; *cidx = t.rowind; *cval = (double*)t.cvals;
  return TOMO_OK;
}

}  // namespace

extern "C" tomo_status_t tomo_lsqr_create_factored(tomo_lsqr_t* out, int64_t npairs, int32_t nper, int64_t nnodes, int32_t nz,
                                                   const int64_t* d_lptr, const int32_t* d_lnode, const double* d_lw,
                                                   int32_t klen, const int32_t* d_kj0, const double* d_kern, int64_t ms,
                                                   int64_t snnz, const int64_t* d_sptr, const int32_t* d_sidx,
                                                   const double* d_svals, void* cuda_stream) {
  if (!out) return TOMO_ERR_INVALID_ARG;
  *out = nullptr;
  if (npairs < 1 || nnodes < 1 || nz < 1 || nper < 1 || klen < 1 || ms < 0 || snnz < 0) return TOMO_ERR_INVALID_ARG;
  if (nper > 32 || klen > 32 || klen > nz) return TOMO_ERR_RANGE;
  if ((double)npairs * nper + (double)ms >= (double)INT32_MAX || (double)nnodes * nz >= (double)INT32_MAX) return TOMO_ERR_RANGE;
  if (!d_lptr || !d_kj0 || !d_kern || (ms > 0 && !d_sptr) || (snnz > 0 && (!d_sidx || !d_svals || ms == 0))) return TOMO_ERR_INVALID_ARG;
  int dev = 0, major = 0, sms = 0;
  CK(cudaGetDevice(&dev));
  CK(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
  CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  if (major != 10) return TOMO_ERR_UNSUPPORTED_ARCH;
  if (!is_device_ptr(d_lptr) || !is_device_ptr(d_kj0) || !is_device_ptr(d_kern) || (ms > 0 && !is_device_ptr(d_sptr)) ||
      (snnz > 0 && (!is_device_ptr(d_sidx) || !is_device_ptr(d_svals))))
    return TOMO_ERR_NOT_DEVICE_PTR;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const int64_t m = npairs * nper + ms, n = nnodes * nz;

  // the pair pointer array on the host: the number of lateral entries and the warps' pair ranges come from it
  std::vector<int64_t> lptr((size_t)npairs + 1);
  CK(cudaMemcpyAsync(lptr.data(), d_lptr, sizeof(int64_t) * (npairs + 1), cudaMemcpyDeviceToHost, st));
  CK(cudaStreamSynchronize(st));
  const int64_t E = lptr[npairs];
  if (lptr[0] != 0 || E < 0 || E >= ((int64_t)1 << 40)) return TOMO_ERR_BAD_CSR;
  for (int64_t q = 0; q < npairs; ++q) if (lptr[q] > lptr[q + 1]) return TOMO_ERR_BAD_CSR;
  if (E > 0 && (!d_lnode || !d_lw)) return TOMO_ERR_INVALID_ARG;
  if (E > 0 && (!is_device_ptr(d_lnode) || !is_device_ptr(d_lw))) return TOMO_ERR_NOT_DEVICE_PTR;

  tomo_lsqr_s* h = new (std::nothrow) tomo_lsqr_s();
  FacState* f = new (std::nothrow) FacState();
  if (!h || !f) { delete h; delete f; return TOMO_ERR_OOM; }
  h->fac = f;
  h->m = m; h->n = n; h->nnz = E * nper * klen + snnz; h->vt = TOMO_VAL_F64; h->sms = sms; h->device = dev;
  h->SG = sms; h->part_dirty = false;
  f->E = E; f->snnz = snnz;
  f->klp = (klen == 8 || klen == 12 || klen == 16) ? klen : 32;
  f->guard = f->klp == 32;
  const int NW = sms * kFacWarps;

  cudaEvent_t e0 = nullptr, e1 = nullptr;
  tomo_status_t rc = TOMO_OK;
  int* d_flags = nullptr;
  do {
    cudaError_t e;
    if ((e = set_fac_attributes(f->klp)) != cudaSuccess) { rc = cuda_fail(e, "cudaFuncSetAttribute(shared memory opt-in)"); break; }
    if ((e = cudaEventCreate(&e0)) != cudaSuccess || (e = cudaEventCreate(&e1)) != cudaSuccess) { rc = cuda_fail(e, "cudaEventCreate"); break; }
    cudaEventRecord(e0, st);
    // --- validation: W and A_extra as canonical CSR blocks, the kernel table ---
    if ((e = cudaMalloc(&d_flags, sizeof(int))) != cudaSuccess) { rc = cuda_fail(e, "cudaMalloc"); break; }
    cudaMemsetAsync(d_flags, 0, sizeof(int), st);
    k_validate<double><<<sms * 8, kThreads, 0, st>>>(npairs, nnodes, E, d_lptr, d_lnode, d_lw, d_flags);
    if (ms > 0) k_validate<double><<<sms * 8, kThreads, 0, st>>>(ms, n, snnz, d_sptr, d_sidx, d_svals, d_flags);
    k_fac_validate_kern<<<1, 256, 0, st>>>((int64_t)nper, nz, klen, d_kj0, d_kern, d_flags);
    int flags = 0;
    if ((e = cudaMemcpyAsync(&flags, d_flags, sizeof(int), cudaMemcpyDeviceToHost, st)) != cudaSuccess ||
        (e = cudaStreamSynchronize(st)) != cudaSuccess) { rc = cuda_fail(e, "validation of the factored operator"); break; }
    if (flags) { rc = TOMO_ERR_BAD_CSR; break; }
    // --- the transposes: W by node, A_extra by column ---
    if ((rc = transpose_block(sms, npairs, nnodes, E, d_lptr, d_lnode, d_lw, st, &f->cptr, &f->cpair, &f->cw)) != TOMO_OK) break;
    if (snnz > 0 && (rc = transpose_block(sms, ms, n, snnz, d_sptr, d_sidx, d_svals, st, &f->scptr, &f->srow, &f->scval)) != TOMO_OK) break;
#define ALLOC(p, bytes) if ((e = cudaMalloc(&(p), (bytes))) != cudaSuccess) { rc = cuda_fail(e, "cudaMalloc(factored)"); break; }
    ALLOC(f->kj0, sizeof(int32_t) * nper); ALLOC(f->kern, sizeof(double) * nper * klen);
    if ((e = cudaMemcpyAsync(f->kj0, d_kj0, sizeof(int32_t) * nper, cudaMemcpyDeviceToDevice, st)) != cudaSuccess ||
        (e = cudaMemcpyAsync(f->kern, d_kern, sizeof(double) * nper * klen, cudaMemcpyDeviceToDevice, st)) != cudaSuccess) { rc = cuda_fail(e, "copy of the kernel table"); break; }
    // --- static work split (host): pairs by entry count for A x; lateral-CSC entries cut evenly for A^T x ---
    const int G = 32 / nper;
    std::vector<int32_t> pw_k[2], pq_k[2];
    for (int kind = 0; kind < 2; ++kind) {   // 0: per-entry kernels, 1: two-stage kernels (a pair's fixed cost weighs 3 steps there)
      std::vector<int32_t>& pw = pw_k[kind];
      std::vector<int32_t>& pq = pq_k[kind];
      pw.assign((size_t)NW + 1, 0); pq.assign((size_t)npairs, 0);
      const double kPair = kind ? 3.0 : 0.3;
      // cost of a pair in lane steps: ceil(entries / G) + 0.3 (group combine, row stores; fitted to the per-warp busy
      // cycles on B200: 245 cycles per pair against 918 per step in dd mode, 104 against 512 in fast mode).
      // A CTA takes a contiguous run of pairs (equal cost); inside the CTA the pairs are dealt to the warps longest
      // first, each to the least loaded warp (a contiguous split at pair granularity left +-18 % between warps);
      // a warp walks its pairs in ascending order.
      auto cost = [&](int64_t q) { return (double)((lptr[q + 1] - lptr[q] + G - 1) / G) + kPair; };
      std::vector<double> pre((size_t)npairs + 1, 0.0);
      for (int64_t q = 0; q < npairs; ++q) pre[q + 1] = pre[q] + cost(q);
      std::vector<int64_t> pc((size_t)sms + 1, 0);
      int64_t q = 0;
      for (int c = 1; c < sms; ++c) {
        const double target = pre[npairs] * (double)c / (double)sms;
        while (q < npairs && 0.5 * (pre[q] + pre[q + 1]) < target) ++q;
        pc[c] = q;
      }
      pc[sms] = npairs;
      std::vector<int64_t> items;
      std::vector<std::vector<int32_t>> bins(kFacWarps);
      size_t outp = 0;
      for (int c = 0; c < sms; ++c) {
        items.clear();
        for (int64_t i = pc[c]; i < pc[c + 1]; ++i) items.push_back(i);
        std::stable_sort(items.begin(), items.end(), [&](int64_t a2, int64_t b2) { return cost(a2) > cost(b2); });
        double load[kFacWarps] = {};
        for (auto& bn : bins) bn.clear();
        for (int64_t i : items) {
          int best = 0;
          for (int w = 1; w < kFacWarps; ++w) if (load[w] < load[best]) best = w;
          bins[best].push_back((int32_t)i); load[best] += cost(i);
        }
        for (int w = 0; w < kFacWarps; ++w) {
          std::sort(bins[w].begin(), bins[w].end());
          pw[(size_t)c * kFacWarps + w] = (int32_t)outp;
          for (int32_t i : bins[w]) pq[outp++] = i;
        }
      }
      pw[NW] = (int32_t)outp;
    }
    std::vector<int64_t> cptr((size_t)nnodes + 1);
    if ((e = cudaMemcpyAsync(cptr.data(), f->cptr, sizeof(int64_t) * (nnodes + 1), cudaMemcpyDeviceToHost, st)) != cudaSuccess ||
        (e = cudaStreamSynchronize(st)) != cudaSuccess) { rc = cuda_fail(e, "copy of the node pointers"); break; }
    std::vector<FacSeg> segs_m[4];
    std::vector<int32_t> wseg_m[4];
    int nslots_max = 0;
    for (int mode = 0; mode < 4; ++mode) {
      std::vector<FacSeg>& segs = segs_m[mode];
      std::vector<int32_t>& wseg = wseg_m[mode];
      std::vector<int32_t> owner;
      wseg.assign((size_t)NW + 1, 0);
      // Cost axis: a node costs a closing overhead (in entry units: the layer sums through shared memory, the extra
      // block's column, the stores) followed by one unit per entry; the warps own equal stretches of that axis.  A
      // node whose entries straddle a boundary is cut there (pieces of at least kMinPiece entries).
      // measured on B200 (per-warp busy cycles): closing a node is a chain of dependent loads worth ~5 k cycles,
      // i.e. the time of ~26 entries in dd mode and ~55 in fast mode, hence one split per mode
      // (two-stage fast mode: an entry is one FMA, the closing is the same chain: ~250 entries)
      const double kCloseM[4] = {55.0, 26.0, 330.0, 160.0};
      const double kClose = kCloseM[mode], kCloseEmpty = 0.5 * kCloseM[mode];
      const int64_t kMinPiece = 8;
      int64_t empty = 0;
      for (int64_t k = 0; k < nnodes; ++k) empty += cptr[k] == cptr[k + 1];
      const double C = (double)E + kClose * (double)(nnodes - empty) + kCloseEmpty * (double)empty;
      auto bound = [&](int w) { return C * (double)w / (double)NW; };   // start of warp w's stretch
      int w = 0, nslots = 0;
      double cum = 0.0;
      for (int64_t k = 0; k < nnodes; ++k) {
        const int64_t lo = cptr[k], hi = cptr[k + 1];
        const size_t first = segs.size();
        while (w + 1 < NW && bound(w + 1) <= cum) ++w;
        if (lo == hi) {
          segs.push_back(FacSeg{lo, lo, (int32_t)k, 1, 0, 0}); owner.push_back(w);
          cum += kCloseEmpty;
        } else {
          const double ent0 = cum + kClose;   // cost position of the node's first entry
          int64_t a = lo;
          while (a < hi) {
            int64_t b2 = hi;
            if (w + 1 < NW) {
              const double room = bound(w + 1) - ent0;   // entries of this node that fit before the boundary
              int64_t lim = lo + (room > 0.0 ? (int64_t)room : 0);
              lim = std::max(lim, a + std::min<int64_t>(kMinPiece, hi - a));
              b2 = (hi - lim < kMinPiece) ? hi : std::min(lim, hi);
            }
            segs.push_back(FacSeg{a, b2, (int32_t)k, 1, 0, 0}); owner.push_back(w);
            a = b2;
            if (a < hi) { const double pos = ent0 + (double)(a - lo); while (w + 1 < NW && bound(w + 1) <= pos) ++w; }
          }
          cum = ent0 + (double)(hi - lo);
        }
        const int cnt = (int)(segs.size() - first);
        if (cnt > 1) {
          for (int r = 0; r < cnt; ++r) { segs[first + r].nsegs = cnt; segs[first + r].rank = r; segs[first + r].slot = nslots + r; }
          nslots += cnt;
        }
      }
      for (size_t i = 0; i < segs.size(); ++i) wseg[(size_t)owner[i] + 1] += 1;
      for (int i = 0; i < NW; ++i) wseg[i + 1] += wseg[i];
      f->nsegs = (int)segs.size(); f->nslots = nslots;
      nslots_max = std::max(nslots_max, nslots);
    }
    ALLOC(f->pw, sizeof(int32_t) * (NW + 1)); ALLOC(f->pq, sizeof(int32_t) * npairs);
    ALLOC(f->pw2, sizeof(int32_t) * (NW + 1)); ALLOC(f->pq2, sizeof(int32_t) * npairs);
    if ((e = cudaMemcpyAsync(f->pq, pq_k[0].data(), sizeof(int32_t) * npairs, cudaMemcpyHostToDevice, st)) != cudaSuccess ||
        (e = cudaMemcpyAsync(f->pq2, pq_k[1].data(), sizeof(int32_t) * npairs, cudaMemcpyHostToDevice, st)) != cudaSuccess ||
        (e = cudaMemcpyAsync(f->pw2, pw_k[1].data(), sizeof(int32_t) * (NW + 1), cudaMemcpyHostToDevice, st)) != cudaSuccess) { rc = cuda_fail(e, "upload of the pair lists"); break; }
    for (int mode = 0; mode < 4 && rc == TOMO_OK; ++mode) {
      if ((e = cudaMalloc(&f->wseg[mode], sizeof(int32_t) * (NW + 1))) != cudaSuccess ||
          (e = cudaMalloc(&f->seg[mode], sizeof(FacSeg) * std::max<size_t>(segs_m[mode].size(), 1))) != cudaSuccess ||
          (e = cudaMemcpyAsync(f->wseg[mode], wseg_m[mode].data(), sizeof(int32_t) * (NW + 1), cudaMemcpyHostToDevice, st)) != cudaSuccess ||
          (e = cudaMemcpyAsync(f->seg[mode], segs_m[mode].data(), sizeof(FacSeg) * segs_m[mode].size(), cudaMemcpyHostToDevice, st)) != cudaSuccess)
        rc = cuda_fail(e, "upload of the A^T x work split");
    }
    if (rc != TOMO_OK) break;
    ALLOC(f->seg_part, sizeof(double2) * (size_t)std::max(nslots_max, 1) * std::max<int>(nz, nper));
    ALLOC(f->S2, sizeof(double2) * nnodes * nper);
    ALLOC(f->node_cnt, sizeof(unsigned int) * nnodes); ALLOC(f->node_nsq, sizeof(double2) * nnodes);
    ALLOC(f->busy, sizeof(long long) * NW);
    if ((e = cudaMemsetAsync(f->busy, 0, sizeof(long long) * NW, st)) != cudaSuccess) { rc = cuda_fail(e, "memset"); break; }
    if ((e = cudaMemcpyAsync(f->pw, pw_k[0].data(), sizeof(int32_t) * (NW + 1), cudaMemcpyHostToDevice, st)) != cudaSuccess ||
        (e = cudaMemsetAsync(f->node_cnt, 0, sizeof(unsigned int) * nnodes, st)) != cudaSuccess ||
        (e = cudaMemsetAsync(f->node_nsq, 0, sizeof(double2) * nnodes, st)) != cudaSuccess ||
        (e = cudaStreamSynchronize(st)) != cudaSuccess) { rc = cuda_fail(e, "upload of the work split"); break; }
    // --- work space (as tomo_lsqr_create) ---
    h->part_cap = sms * 32 + 2;
    ALLOC(h->u, sizeof(double) * m); ALLOC(h->v, sizeof(double) * n);
    ALLOC(h->w, sizeof(double) * n); ALLOC(h->x, sizeof(double) * n);
    ALLOC(h->sc, sizeof(Scalars));
    ALLOC(h->part_spmv, sizeof(double2) * h->part_cap);
    ALLOC(h->part_vec, sizeof(double2) * h->part_cap);
#undef ALLOC
    if ((e = cudaMemsetAsync(h->sc, 0, sizeof(Scalars), st)) != cudaSuccess) { rc = cuda_fail(e, "memset"); break; }
    if ((e = cudaMallocHost(&h->h_sc, sizeof(Scalars))) != cudaSuccess ||
        (e = cudaMallocHost(&h->h_poll, 2 * sizeof(PollWord))) != cudaSuccess) { rc = cuda_fail(e, "cudaMallocHost"); break; }
    for (int i = 0; i < 2; ++i)
      if ((e = cudaEventCreateWithFlags(&h->ev_poll[i], cudaEventDisableTiming)) != cudaSuccess) break;
    if (e != cudaSuccess) { rc = cuda_fail(e, "cudaEventCreate"); break; }
    if ((e = cudaStreamCreateWithFlags(&h->cap_stream, cudaStreamNonBlocking)) != cudaSuccess) { rc = cuda_fail(e, "cudaStreamCreate"); break; }
    FacDesc& d = f->d;
    d.nper = nper; d.nz = nz; d.klen = klen; d.G = G;
    d.npairs = npairs; d.nnodes = nnodes; d.mdata = npairs * nper; d.ms = ms;
    d.lptr = d_lptr; d.lnode = d_lnode; d.lw = d_lw;
    d.cptr = f->cptr; d.cpair = f->cpair; d.cw = f->cw;
    d.kj0 = f->kj0; d.kern = f->kern;
    d.sptr = d_sptr; d.sidx = d_sidx; d.sval = d_svals;
    d.scptr = f->scptr; d.srow = f->srow; d.scval = f->scval;
    d.pw = f->pw; d.pq = f->pq; d.wseg = f->wseg[1]; d.seg = f->seg[1];
    d.seg_part = f->seg_part; d.node_cnt = f->node_cnt; d.node_nsq = f->node_nsq; d.busy = f->busy;
    d.pstride = std::max<int>(nz, nper);
    for (int mode = 0; mode < 4; ++mode) {
      f->dm[mode] = d; f->dm[mode].wseg = f->wseg[mode]; f->dm[mode].seg = f->seg[mode];
      if (mode >= 2) { f->dm[mode].pw = f->pw2; f->dm[mode].pq = f->pq2; }
    }
    cudaEventRecord(e1, st);
    if ((e = cudaEventSynchronize(e1)) != cudaSuccess) { rc = cuda_fail(e, "create_factored"); break; }
    float msf = 0;
    cudaEventElapsedTime(&msf, e0, e1); h->create_ms = msf;
  } while (0);
  if (d_flags) cudaFree(d_flags);
  if (e0) cudaEventDestroy(e0);
  if (e1) cudaEventDestroy(e1);
  if (rc != TOMO_OK) { free_handle(h); return rc; }
  *out = h;
  return TOMO_OK;
}

// NEXT-4: on-device assembly of G from its factored description (k_fac_assemble)
extern "C" tomo_status_t tomo_lsqr_assemble_csr(int64_t npairs, int32_t nper, int64_t nnodes, int32_t nz, const int64_t* d_lptr,
                                                const int32_t* d_lnode, const double* d_lw, int32_t klen, const int32_t* d_kj0,
                                                const double* d_kern, int64_t ms, int64_t snnz, const int64_t* d_sptr,
                                                const int32_t* d_sidx, const double* d_svals, int64_t nnz, int64_t* d_rowptr,
                                                int32_t* d_colind, double* d_vals, int32_t nodal, void* cuda_stream) {
  if (nodal != 0 && nodal != 1) return TOMO_ERR_INVALID_ARG;
  if (npairs < 1 || nnodes < 1 || nz < 1 || nper < 1 || klen < 1 || ms < 0 || snnz < 0 || nnz < 0) return TOMO_ERR_INVALID_ARG;
  if (nper > 32 || klen > 32 || klen > nz) return TOMO_ERR_RANGE;
  if ((double)npairs * nper + (double)ms >= (double)INT32_MAX || (double)nnodes * nz >= (double)INT32_MAX) return TOMO_ERR_RANGE;
  if (!d_lptr || !d_kj0 || !d_kern || !d_rowptr || (ms > 0 && !d_sptr) || (snnz > 0 && (!d_sidx || !d_svals || ms == 0)) ||
      (nnz > 0 && (!d_colind || !d_vals)))
    return TOMO_ERR_INVALID_ARG;
  int dev = 0, major = 0, sms = 0;
  CK(cudaGetDevice(&dev));
  CK(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
  CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  if (major != 10) return TOMO_ERR_UNSUPPORTED_ARCH;
  if (!is_device_ptr(d_lptr) || !is_device_ptr(d_kj0) || !is_device_ptr(d_kern) || !is_device_ptr(d_rowptr) ||
      (ms > 0 && !is_device_ptr(d_sptr)) || (snnz > 0 && (!is_device_ptr(d_sidx) || !is_device_ptr(d_svals))) ||
      (nnz > 0 && (!is_device_ptr(d_colind) || !is_device_ptr(d_vals))))
    return TOMO_ERR_NOT_DEVICE_PTR;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  // the caller's nnz must be the size of the assembled matrix: entries of W x nper x klen + the extra block
  int64_t E = 0, sn = 0;
  CK(cudaMemcpyAsync(&E, d_lptr + npairs, sizeof(int64_t), cudaMemcpyDeviceToHost, st));
  if (ms > 0) CK(cudaMemcpyAsync(&sn, d_sptr + ms, sizeof(int64_t), cudaMemcpyDeviceToHost, st));
  CK(cudaStreamSynchronize(st));
  if (E < 0 || sn != snnz || E * (int64_t)nper * klen + snnz != nnz) return TOMO_ERR_INVALID_ARG;
  if (E > 0 && (!d_lnode || !d_lw)) return TOMO_ERR_INVALID_ARG;
  if (E > 0 && (!is_device_ptr(d_lnode) || !is_device_ptr(d_lw))) return TOMO_ERR_NOT_DEVICE_PTR;
  k_fac_assemble<<<sms * 8, 256, 0, st>>>(npairs, nper, nz, klen, (int)nodal, d_lptr, d_lnode, d_lw, d_kj0, d_kern, ms, d_sptr, d_sidx, d_svals,
                                         d_rowptr, d_colind, d_vals);
  CK(cudaGetLastError());
  CK(cudaStreamSynchronize(st));
  return TOMO_OK;
}

extern "C" void tomo_lsqr_destroy(tomo_lsqr_t h) { free_handle(h); }

// ------------------------------------------------------------------------------------------------
// solve
// ------------------------------------------------------------------------------------------------
namespace {

// one LSQR iteration = three launches (kernels.cuh)
void enqueue_iteration(const tomo_lsqr_s* h, cudaStream_t st) {
  launch_spmv<OP_K1>(h, false, h->v, h->u, st);
  launch_spmv<OP_K2>(h, true, h->u, h->v, st);
  launch_k4(h, st);
}

tomo_status_t ensure_graph(tomo_lsqr_s* h) {
  const int gkey = h->accumulate + 2 * h->solver + 4 * h->two_stage;
  if (h->gexec && h->graph_k == h->check_every && h->graph_mode == gkey && h->graph_G == h->SG) return TOMO_OK;
  if (h->gexec) { cudaGraphExecDestroy(h->gexec); h->gexec = nullptr; }
  cudaGraph_t g = nullptr;
  CK(cudaStreamBeginCapture(h->cap_stream, cudaStreamCaptureModeRelaxed));
  for (int i = 0; i < h->check_every; ++i) enqueue_iteration(h, h->cap_stream);
  cudaError_t e = cudaStreamEndCapture(h->cap_stream, &g);
  if (e != cudaSuccess) return cuda_fail(e, "cudaStreamEndCapture");
  e = cudaGraphInstantiate(&h->gexec, g, 0);
  cudaGraphDestroy(g);
  if (e != cudaSuccess) { h->gexec = nullptr; return cuda_fail(e, "cudaGraphInstantiate"); }
  h->graph_k = h->check_every; h->graph_mode = gkey; h->graph_G = h->SG;
  return TOMO_OK;
}

tomo_status_t ensure_history(tomo_lsqr_s* h, int32_t cap) {
  if (cap <= h->hist_cap) return TOMO_OK;
  cudaFree(h->hist_r2); cudaFree(h->hist_ar);
  h->hist_r2 = h->hist_ar = nullptr; h->hist_cap = 0;
  CK(cudaMalloc(&h->hist_r2, sizeof(double) * cap));
  CK(cudaMalloc(&h->hist_ar, sizeof(double) * cap));
  h->hist_cap = cap;
  return TOMO_OK;
}

bool bad_param(double v) { return !(v >= 0.0) || !(v <= 1.79769313486231570815e308); }

// the body shared by solve and solve_host; d_b, d_x are device pointers
tomo_status_t solve_device(tomo_lsqr_s* h, const double* d_b, double damp, double atol, double btol, int32_t max_iters,
                           double* d_x, tomo_lsqr_result_t* res, double* h_r2, double* h_ar, cudaStream_t st) {
  const bool want_hist = (h_r2 || h_ar) && max_iters > 0;
  if (want_hist) { tomo_status_t rc = ensure_history(h, max_iters); if (rc != TOMO_OK) return rc; }
  if (h->solver == 1 && !h->hbar) CK(cudaMalloc(&h->hbar, sizeof(double) * h->n));
  { tomo_status_t rc = rebuild_partitions(h, st); if (rc != TOMO_OK) return rc; }
  const bool profile = h->profile != 0;
  const bool graph = h->use_graph && !profile;
  if (graph) { tomo_status_t rc = ensure_graph(h); if (rc != TOMO_OK) return rc; }

  // fresh device state: parameters + zeroed recurrences (cs2 = -1 as in Paige & Saunders)
  Scalars* hs = h->h_sc;
  memset(hs, 0, sizeof(Scalars));
  hs->damp = damp; hs->atol = atol; hs->btol = btol; hs->max_iters = max_iters;
  hs->cs2 = -1.0;
  hs->solver = h->solver;
  hs->hist_r2 = want_hist ? h->hist_r2 : nullptr;
  hs->hist_ar = want_hist ? h->hist_ar : nullptr;
  hs->hist_cap = want_hist ? h->hist_cap : 0;
  CK(cudaMemcpyAsync(h->sc, hs, sizeof(Scalars), cudaMemcpyHostToDevice, st));
  CK(cudaMemsetAsync(h->x, 0, sizeof(double) * h->n, st));
  if (h->solver == 1) CK(cudaMemsetAsync(h->hbar, 0, sizeof(double) * h->n, st));
  // a1: beta_1 = ||b||, u^ = b, v^ = A^T u, alpha_1, w = v
  launch_vec<VOP_INIT_U>(h, d_b, h->u, nullptr, nullptr, h->m, st);
  launch_spmv<OP_K2_INIT>(h, true, h->u, h->v, st);
  launch_vec<VOP_INIT_VW>(h, nullptr, h->v, h->w, nullptr, h->n, st);
  CK(cudaGetLastError());
  h->kernels_enqueued += 3;

  const int k = h->check_every;
  const int chunks = max_iters > 0 ? (max_iters + k - 1) / k : 0;
  if (profile) {
    const size_t need = (size_t)std::min((int64_t)chunks * k, (int64_t)kMaxProfileIters) * 4;
    while (h->prof_ev.size() < need) {
      cudaEvent_t e; CK(cudaEventCreate(&e)); h->prof_ev.push_back(e);
    }
  }
  int it_enq = 0;
  bool stopped = false;
  for (int c = 0; c < chunks && !stopped; ++c) {
    const int slot = c & 1;
    if (graph) {
      CK(cudaGraphLaunch(h->gexec, st));
    } else {
      for (int i = 0; i < k; ++i, ++it_enq) {
        const bool pe = profile && it_enq < kMaxProfileIters;
        if (pe) cudaEventRecord(h->prof_ev[4 * it_enq + 0], st);
        launch_spmv<OP_K1>(h, false, h->v, h->u, st);
        if (pe) cudaEventRecord(h->prof_ev[4 * it_enq + 1], st);
        launch_spmv<OP_K2>(h, true, h->u, h->v, st);
        if (pe) cudaEventRecord(h->prof_ev[4 * it_enq + 2], st);
        launch_k4(h, st);
        if (pe) cudaEventRecord(h->prof_ev[4 * it_enq + 3], st);
      }
      CK(cudaGetLastError());
    }
    h->kernels_enqueued += (h->fac && (h->fac->d.nodal || (h->accumulate ? h->two_stage == 2 : h->two_stage != 0)) ? 4.0 : 3.0) * k;   // the two-stage A x is two launches
    // host poll: {itn, istop, stop}.  The next replay is enqueued before this one is inspected, so the
    // device never idles on the host; kernels after a stop return at once and leave x frozen.
    CK(cudaMemcpyAsync(&h->h_poll[slot], &h->sc->itn, sizeof(PollWord), cudaMemcpyDeviceToHost, st));
    CK(cudaEventRecord(h->ev_poll[slot], st));
    if (c >= 1) {
      CK(cudaEventSynchronize(h->ev_poll[slot ^ 1]));
      if (h->h_poll[slot ^ 1].stop) stopped = true;
    }
  }
  CK(cudaMemcpyAsync(d_x, h->x, sizeof(double) * h->n, cudaMemcpyDeviceToDevice, st));
  CK(cudaMemcpyAsync(hs, h->sc, sizeof(Scalars), cudaMemcpyDeviceToHost, st));
  CK(cudaStreamSynchronize(st));
  if (res) {
    res->itn = hs->itn; res->istop = hs->istop;
    res->r1norm = hs->r1norm; res->r2norm = hs->r2norm; res->arnorm = hs->arnorm;
    res->anorm = hs->anorm; res->acond = hs->acond; res->xnorm = hs->xnorm;
  }
  if (want_hist && hs->itn > 0) {
    if (h_r2) CK(cudaMemcpy(h_r2, h->hist_r2, sizeof(double) * hs->itn, cudaMemcpyDeviceToHost));
    if (h_ar) CK(cudaMemcpy(h_ar, h->hist_ar, sizeof(double) * hs->itn, cudaMemcpyDeviceToHost));
  }
  if (profile) {
    h->k1_ms = h->k2_ms = h->k4_ms = 0; h->k_launches = 0;
    const int cnt = std::min<int>(std::min<int>(hs->itn, it_enq), kMaxProfileIters);
    for (int i = 0; i < cnt; ++i) {
      float a = 0, b = 0, c4 = 0;
      cudaEventElapsedTime(&a, h->prof_ev[4 * i], h->prof_ev[4 * i + 1]);
      cudaEventElapsedTime(&b, h->prof_ev[4 * i + 1], h->prof_ev[4 * i + 2]);
      cudaEventElapsedTime(&c4, h->prof_ev[4 * i + 2], h->prof_ev[4 * i + 3]);
      h->k1_ms += a; h->k2_ms += b; h->k4_ms += c4;
    }
    h->k_launches = cnt;
  }
  return TOMO_OK;
}

// a handle lives on the device it was created on: that device must be the current one
tomo_status_t check_device(const tomo_lsqr_s* h) {
  if (!h) return TOMO_ERR_INVALID_ARG;
  int dev = -1;
  CK(cudaGetDevice(&dev));
  return dev == h->device ? TOMO_OK : TOMO_ERR_INVALID_ARG;
}

tomo_status_t check_solve_args(tomo_lsqr_s* h, double damp, double atol, double btol, int32_t max_iters) {
  if (!h) return TOMO_ERR_INVALID_ARG;
  { tomo_status_t rc = check_device(h); if (rc != TOMO_OK) return rc; }
  if (bad_param(damp) || bad_param(atol) || bad_param(btol) || max_iters < 0) return TOMO_ERR_INVALID_ARG;
  return TOMO_OK;
}

}  // namespace

extern "C" tomo_status_t tomo_lsqr_solve(tomo_lsqr_t h, const double* d_b, double damp, double atol, double btol,
                                         int32_t max_iters, double* d_x, tomo_lsqr_result_t* res, double* h_r2norm_hist,
                                         double* h_arnorm_hist, void* cuda_stream) {
  tomo_status_t rc = check_solve_args(h, damp, atol, btol, max_iters);
  if (rc != TOMO_OK) return rc;
  if (!d_b || !d_x) return TOMO_ERR_INVALID_ARG;
  if (!is_device_ptr(d_b) || !is_device_ptr(d_x)) return TOMO_ERR_NOT_DEVICE_PTR;
  h->solver = 0;
  return solve_device(h, d_b, damp, atol, btol, max_iters, d_x, res, h_r2norm_hist, h_arnorm_hist, (cudaStream_t)cuda_stream);
}

extern "C" tomo_status_t tomo_lsmr_solve(tomo_lsqr_t h, const double* d_b, double damp, double atol, double btol,
                                         int32_t max_iters, double* d_x, tomo_lsqr_result_t* res, double* h_normr_hist,
                                         double* h_normar_hist, void* cuda_stream) {
  tomo_status_t rc = check_solve_args(h, damp, atol, btol, max_iters);
  if (rc != TOMO_OK) return rc;
  if (!d_b || !d_x) return TOMO_ERR_INVALID_ARG;
  if (!is_device_ptr(d_b) || !is_device_ptr(d_x)) return TOMO_ERR_NOT_DEVICE_PTR;
  h->solver = 1;
  rc = solve_device(h, d_b, damp, atol, btol, max_iters, d_x, res, h_normr_hist, h_normar_hist, (cudaStream_t)cuda_stream);
  h->solver = 0;
  return rc;
}

namespace {
tomo_status_t solve_host_any(tomo_lsqr_s* h, int solver, const double* h_b, double damp, double atol, double btol,
                             int32_t max_iters, double* h_x, tomo_lsqr_result_t* res, cudaStream_t st) {
  tomo_status_t rc = check_solve_args(h, damp, atol, btol, max_iters);
  if (rc != TOMO_OK) return rc;
  if (!h_b || !h_x) return TOMO_ERR_INVALID_ARG;
  if (!h->bh) CK(cudaMalloc(&h->bh, sizeof(double) * h->m));
  if (!h->xh) CK(cudaMalloc(&h->xh, sizeof(double) * h->n));
  CK(cudaMemcpyAsync(h->bh, h_b, sizeof(double) * h->m, cudaMemcpyHostToDevice, st));
  h->solver = solver;
  rc = solve_device(h, h->bh, damp, atol, btol, max_iters, h->xh, res, nullptr, nullptr, st);
  h->solver = 0;
  if (rc != TOMO_OK) return rc;
  CK(cudaMemcpyAsync(h_x, h->xh, sizeof(double) * h->n, cudaMemcpyDeviceToHost, st));
  CK(cudaStreamSynchronize(st));
  return TOMO_OK;
}
}  // namespace

extern "C" tomo_status_t tomo_lsqr_solve_host(tomo_lsqr_t h, const double* h_b, double damp, double atol, double btol,
                                              int32_t max_iters, double* h_x, tomo_lsqr_result_t* res, void* cuda_stream) {
  return solve_host_any(h, 0, h_b, damp, atol, btol, max_iters, h_x, res, (cudaStream_t)cuda_stream);
}

extern "C" tomo_status_t tomo_lsmr_solve_host(tomo_lsqr_t h, const double* h_b, double damp, double atol, double btol,
                                              int32_t max_iters, double* h_x, tomo_lsqr_result_t* res, void* cuda_stream) {
  return solve_host_any(h, 1, h_b, damp, atol, btol, max_iters, h_x, res, (cudaStream_t)cuda_stream);
}

// ------------------------------------------------------------------------------------------------
// multi-RHS, SpMV hook, inspection, options
// ------------------------------------------------------------------------------------------------
namespace {

// column r of a row-major len x nrhs block <-> contiguous vector
__global__ void k_col_gather(const double* __restrict__ B, int nrhs, int r, int64_t len, double* __restrict__ out) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < len; i += (int64_t)gridDim.x * blockDim.x)
    out[i] = B[i * nrhs + r];
}
__global__ void k_col_scatter(const double* __restrict__ in, int nrhs, int r, int64_t len, double* __restrict__ X) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < len; i += (int64_t)gridDim.x * blockDim.x)
    X[i * nrhs + r] = in[i];
}

}  // namespace

namespace {

// block products (wspmm.cuh): same split points as the single-side kernel of the direction, a 2-stage ring per warp
// (96 KB of shared memory: the rest of the SM's 228 KB is L1 for the 64-byte gathers)
using WM = WCfg<TOMO_TILE, 2, TOMO_W>;

template <int MODE, typename VT, int OP>
void launch_spmm_t(const tomo_lsqr_s* h, bool transpose, const double* X, double* Y, cudaStream_t st) {
  const Dir& d = h->dir[transpose ? 1 : 0];
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)h->SG); cfg.blockDim = dim3(WM::THREADS);
  cfg.dynamicSmemBytes = MSmem<WM, VT>::kTotal; cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at; cfg.numAttrs = h->pdl ? 1 : 0;
  cudaLaunchKernelEx(&cfg, k_wspmm8<WM, MODE, VT, OP>, d.ptr, (const int32_t*)d.rid, d.idx, (const VT*)d.val, h->nnz, d.nrows,
                     (const int32_t*)d.erows, d.n_empty, X, Y, (const int64_t*)d.wE, (const int32_t*)d.wR, h->cta_rec8, h->msc,
                     h->mpartials);
}

template <int OP>
void launch_spmm(const tomo_lsqr_s* h, bool transpose, const double* X, double* Y, cudaStream_t st) {
  if (h->vt == TOMO_VAL_F64) {
    if (h->accumulate) launch_spmm_t<1, double, OP>(h, transpose, X, Y, st); else launch_spmm_t<0, double, OP>(h, transpose, X, Y, st);
  } else {
    if (h->accumulate) launch_spmm_t<1, float, OP>(h, transpose, X, Y, st); else launch_spmm_t<0, float, OP>(h, transpose, X, Y, st);
  }
}

template <int MODE, typename VT>
cudaError_t spmm_attr_ops() {
  cudaError_t e;
  const int smem = (int)MSmem<WM, VT>::kTotal;
  if ((e = cudaFuncSetAttribute(k_wspmm8<WM, MODE, VT, OP_K1>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem)) != cudaSuccess) return e;
  if ((e = cudaFuncSetAttribute(k_wspmm8<WM, MODE, VT, OP_K2>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem)) != cudaSuccess) return e;
  return cudaFuncSetAttribute(k_wspmm8<WM, MODE, VT, OP_K2_INIT>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
}
cudaError_t set_multi_attributes(tomo_valtype_t vt) {
  cudaError_t e;
  if (vt == TOMO_VAL_F64) { if ((e = spmm_attr_ops<0, double>()) != cudaSuccess) return e; return spmm_attr_ops<1, double>(); }
  if ((e = spmm_attr_ops<0, float>()) != cudaSuccess) return e;
  return spmm_attr_ops<1, float>();
}

template <int VOP>
void launch_vec8(const tomo_lsqr_s* h, const double* in0, int nrhs, double* a0, double* a1, double* a2, int64_t len, cudaStream_t st,
                 double* a3 = nullptr) {
  const int g = (int)std::max<int64_t>(1, std::min<int64_t>((len * kR + kMThreads - 1) / kMThreads, (int64_t)h->MG));
  if (h->accumulate) k_vec8<1, VOP><<<g, kMThreads, 0, st>>>(in0, nrhs, a0, a1, a2, len, h->msc, h->mpartials, a3);
  else k_vec8<0, VOP><<<g, kMThreads, 0, st>>>(in0, nrhs, a0, a1, a2, len, h->msc, h->mpartials, a3);
}

void enqueue_multi_iteration(const tomo_lsqr_s* h, cudaStream_t st) {
  launch_spmm<OP_K1>(h, false, h->mV, h->mU, st);
  launch_spmm<OP_K2>(h, true, h->mU, h->mV, st);
  if (h->solver == 1) launch_vec8<VOP_K4_LSMR>(h, nullptr, kR, h->mV, h->mW, h->mX, h->n, st, h->mH);
  else launch_vec8<VOP_K4>(h, nullptr, kR, h->mV, h->mW, h->mX, h->n, st);
}

// Work space of the block solve, allocated on first use.  All-or-nothing: the pointers are committed to the
// handle only after every allocation and the partition kernels have succeeded, so a transient out-of-memory
// leaves the handle as it was.
tomo_status_t ensure_multi(tomo_lsqr_s* h, cudaStream_t st) {
  if (h->multi_ready) return TOMO_OK;
  const int64_t m = h->m, n = h->n;
  const int MG = h->sms * 8;
  double *mU = nullptr, *mV = nullptr, *mW = nullptr, *mX = nullptr, *mH = nullptr;
  Scalars *msc = nullptr, *h_msc = nullptr; PollWord* h_mpoll = nullptr;
  CtaRec8* cr = nullptr; double2* mp = nullptr;
  cudaError_t e = cudaSuccess;
  do {
    if ((e = cudaMalloc(&mU, sizeof(double) * m * kR)) != cudaSuccess) break;
    if ((e = cudaMalloc(&mV, sizeof(double) * n * kR)) != cudaSuccess) break;
    if ((e = cudaMalloc(&mW, sizeof(double) * n * kR)) != cudaSuccess) break;
    if ((e = cudaMalloc(&mX, sizeof(double) * n * kR)) != cudaSuccess) break;
    if ((e = cudaMalloc(&mH, sizeof(double) * n * kR)) != cudaSuccess) break;
    if ((e = cudaMalloc(&msc, sizeof(Scalars) * kR)) != cudaSuccess) break;
    if ((e = cudaMallocHost(&h_msc, sizeof(Scalars) * kR)) != cudaSuccess) break;
    if ((e = cudaMallocHost(&h_mpoll, sizeof(PollWord) * kR * 2)) != cudaSuccess) break;
    if ((e = cudaMalloc(&cr, sizeof(CtaRec8) * h->sms)) != cudaSuccess) break;
    if ((e = cudaMalloc(&mp, sizeof(double2) * kR * MG)) != cudaSuccess) break;
    e = set_multi_attributes(h->vt);
  } while (0);
  if (e != cudaSuccess) {
    cudaFree(mU); cudaFree(mV); cudaFree(mW); cudaFree(mX); cudaFree(mH); cudaFree(msc); cudaFree(cr); cudaFree(mp);
    if (h_msc) cudaFreeHost(h_msc);
    if (h_mpoll) cudaFreeHost(h_mpoll);
    return cuda_fail(e, "block-solve work space");
  }
  h->mU = mU; h->mV = mV; h->mW = mW; h->mX = mX; h->mH = mH; h->msc = msc; h->h_msc = h_msc; h->h_mpoll = h_mpoll;
  h->cta_rec8 = cr; h->mpartials = mp; h->MG = MG;
  h->multi_ready = true;
  return TOMO_OK;
}

// Eight recurrences sharing every pass over A and A^T (multi.cuh).  nrhs < 8 is padded with zero columns.
// solver: 0 LSQR, 1 LSMR (per-side scalars either way).
tomo_status_t solve_multi_shared(tomo_lsqr_s* h, int solver, int32_t nrhs, const double* d_B, double damp, double atol, double btol,
                                 int32_t max_iters, double* d_X, tomo_lsqr_result_t* res, cudaStream_t st) {
  const int64_t m = h->m, n = h->n;
  { tomo_status_t rc = ensure_multi(h, st); if (rc != TOMO_OK) return rc; }
  { tomo_status_t rc = rebuild_partitions(h, st); if (rc != TOMO_OK) return rc; }
  h->solver = solver;
  const int k = h->check_every;
  const int gkey = h->accumulate + 2 * solver;
  if (h->use_graph && !(h->mgexec && h->mgraph_k == k && h->mgraph_mode == gkey)) {
    if (h->mgexec) { cudaGraphExecDestroy(h->mgexec); h->mgexec = nullptr; }
    cudaGraph_t g = nullptr;
    CK(cudaStreamBeginCapture(h->cap_stream, cudaStreamCaptureModeRelaxed));
    for (int i = 0; i < k; ++i) enqueue_multi_iteration(h, h->cap_stream);
    cudaError_t e = cudaStreamEndCapture(h->cap_stream, &g);
    if (e != cudaSuccess) return cuda_fail(e, "cudaStreamEndCapture");
    e = cudaGraphInstantiate(&h->mgexec, g, 0);
    cudaGraphDestroy(g);
    if (e != cudaSuccess) { h->mgexec = nullptr; return cuda_fail(e, "cudaGraphInstantiate"); }
    h->mgraph_k = k; h->mgraph_mode = gkey;
  }
  Scalars* hs = h->h_msc;
  memset(hs, 0, sizeof(Scalars) * kR);
  for (int r = 0; r < kR; ++r) {
    hs[r].damp = damp; hs[r].atol = atol; hs[r].btol = btol; hs[r].max_iters = max_iters; hs[r].cs2 = -1.0; hs[r].solver = solver;
  }
  CK(cudaMemcpyAsync(h->msc, hs, sizeof(Scalars) * kR, cudaMemcpyHostToDevice, st));
  CK(cudaMemsetAsync(h->mX, 0, sizeof(double) * n * kR, st));
  CK(cudaMemsetAsync(h->mV, 0, sizeof(double) * n * kR, st));
  CK(cudaMemsetAsync(h->mW, 0, sizeof(double) * n * kR, st));
  if (solver == 1) CK(cudaMemsetAsync(h->mH, 0, sizeof(double) * n * kR, st));
  launch_vec8<VOP_INIT_U>(h, d_B, nrhs, h->mU, nullptr, nullptr, m, st);
  launch_spmm<OP_K2_INIT>(h, true, h->mU, h->mV, st);
  launch_vec8<VOP_INIT_VW>(h, nullptr, kR, h->mV, h->mW, nullptr, n, st);
  CK(cudaGetLastError());
  h->kernels_enqueued += 3;
  const bool profile = h->profile != 0;
  const bool graph = h->use_graph && !profile;
  const int chunks = max_iters > 0 ? (max_iters + k - 1) / k : 0;
  if (profile) {
    const size_t need = (size_t)std::min((int64_t)chunks * k, (int64_t)kMaxProfileIters) * 4;
    while (h->prof_ev.size() < need) { cudaEvent_t e; CK(cudaEventCreate(&e)); h->prof_ev.push_back(e); }
  }
  int it_enq = 0;
  bool stopped = false;
  for (int c = 0; c < chunks && !stopped; ++c) {
    const int slot = c & 1;
    if (graph) CK(cudaGraphLaunch(h->mgexec, st));
    else {
      for (int i = 0; i < k; ++i, ++it_enq) {
        const bool pe = profile && it_enq < kMaxProfileIters;
        if (pe) cudaEventRecord(h->prof_ev[4 * it_enq + 0], st);
        launch_spmm<OP_K1>(h, false, h->mV, h->mU, st);
        if (pe) cudaEventRecord(h->prof_ev[4 * it_enq + 1], st);
        launch_spmm<OP_K2>(h, true, h->mU, h->mV, st);
        if (pe) cudaEventRecord(h->prof_ev[4 * it_enq + 2], st);
        if (solver == 1) launch_vec8<VOP_K4_LSMR>(h, nullptr, kR, h->mV, h->mW, h->mX, h->n, st, h->mH);
        else launch_vec8<VOP_K4>(h, nullptr, kR, h->mV, h->mW, h->mX, h->n, st);
        if (pe) cudaEventRecord(h->prof_ev[4 * it_enq + 3], st);
      }
      CK(cudaGetLastError());
    }
    h->kernels_enqueued += 3.0 * k;
    // poll the eight {itn, istop, stop} words one replay behind the one being enqueued (as solve_device does):
    // the device never idles on the host; replays after every side has stopped are empty launches
    CK(cudaMemcpy2DAsync(h->h_mpoll + (size_t)slot * kR, sizeof(PollWord), &h->msc->itn, sizeof(Scalars), sizeof(PollWord), kR,
                         cudaMemcpyDeviceToHost, st));
    CK(cudaEventRecord(h->ev_poll[slot], st));
    if (c >= 1) {
      CK(cudaEventSynchronize(h->ev_poll[slot ^ 1]));
      bool all = true;
      for (int r = 0; r < kR; ++r) all = all && (h->h_mpoll[(size_t)(slot ^ 1) * kR + r].stop != 0);
      if (all) stopped = true;
    }
  }
  CK(cudaMemcpyAsync(h->h_msc, h->msc, sizeof(Scalars) * kR, cudaMemcpyDeviceToHost, st));
  CK(cudaMemcpy2DAsync(d_X, sizeof(double) * nrhs, h->mX, sizeof(double) * kR, sizeof(double) * nrhs, n, cudaMemcpyDeviceToDevice, st));
  CK(cudaStreamSynchronize(st));
  if (res)
    for (int r = 0; r < nrhs; ++r) {
      const Scalars& q = h->h_msc[r];
      res[r].itn = q.itn; res[r].istop = q.istop; res[r].r1norm = q.r1norm; res[r].r2norm = q.r2norm;
      res[r].arnorm = q.arnorm; res[r].anorm = q.anorm; res[r].acond = q.acond; res[r].xnorm = q.xnorm;
    }
  if (profile) {
    h->k1_ms = h->k2_ms = h->k4_ms = 0; h->k_launches = 0;
    int itn_max = 0;
    for (int r = 0; r < kR; ++r) itn_max = std::max(itn_max, (int)h->h_msc[r].itn);
    const int cnt = std::min<int>(std::min<int>(itn_max, it_enq), kMaxProfileIters);
    for (int i = 0; i < cnt; ++i) {
      float a = 0, b = 0, c4 = 0;
      cudaEventElapsedTime(&a, h->prof_ev[4 * i], h->prof_ev[4 * i + 1]);
      cudaEventElapsedTime(&b, h->prof_ev[4 * i + 1], h->prof_ev[4 * i + 2]);
      cudaEventElapsedTime(&c4, h->prof_ev[4 * i + 2], h->prof_ev[4 * i + 3]);
      h->k1_ms += a; h->k2_ms += b; h->k4_ms += c4;
    }
    h->k_launches = cnt;
  }
  return TOMO_OK;
}

tomo_status_t solve_multi_any(tomo_lsqr_s* h, int solver, int32_t nrhs, const double* d_B, double damp, double atol, double btol,
                              int32_t max_iters, double* d_X, tomo_lsqr_result_t* res, cudaStream_t st) {
  tomo_status_t rc = check_solve_args(h, damp, atol, btol, max_iters);
  if (rc != TOMO_OK) return rc;
  if (nrhs < 1 || nrhs > 8 || !d_B || !d_X) return TOMO_ERR_INVALID_ARG;
  if (!is_device_ptr(d_B) || !is_device_ptr(d_X)) return TOMO_ERR_NOT_DEVICE_PTR;
  if (h->multi_shared && !h->fac) {   // a factored handle runs the sides one after the other (no block kernel for it)
    rc = solve_multi_shared(h, solver, nrhs, d_B, damp, atol, btol, max_iters, d_X, res, st);
    h->solver = 0;
    return rc;
  }
  if (!h->bh) CK(cudaMalloc(&h->bh, sizeof(double) * h->m));
  if (!h->xh) CK(cudaMalloc(&h->xh, sizeof(double) * h->n));
  for (int r = 0; r < nrhs; ++r) {
    k_col_gather<<<vec_blocks(h, h->m), kThreads, 0, st>>>(d_B, nrhs, r, h->m, h->bh);
    h->solver = solver;
    rc = solve_device(h, h->bh, damp, atol, btol, max_iters, h->xh, res ? res + r : nullptr, nullptr, nullptr, st);
    h->solver = 0;
    if (rc != TOMO_OK) return rc;
    k_col_scatter<<<vec_blocks(h, h->n), kThreads, 0, st>>>(h->xh, nrhs, r, h->n, d_X);
  }
  CK(cudaGetLastError());
  CK(cudaStreamSynchronize(st));
  return TOMO_OK;
}

}  // namespace

extern "C" tomo_status_t tomo_lsqr_solve_multi(tomo_lsqr_t h, int32_t nrhs, const double* d_B, double damp, double atol,
                                               double btol, int32_t max_iters, double* d_X, tomo_lsqr_result_t* res,
                                               void* cuda_stream) {
  return solve_multi_any(h, 0, nrhs, d_B, damp, atol, btol, max_iters, d_X, res, (cudaStream_t)cuda_stream);
}

extern "C" tomo_status_t tomo_lsmr_solve_multi(tomo_lsqr_t h, int32_t nrhs, const double* d_B, double damp, double atol,
                                               double btol, int32_t max_iters, double* d_X, tomo_lsqr_result_t* res,
                                               void* cuda_stream) {
  return solve_multi_any(h, 1, nrhs, d_B, damp, atol, btol, max_iters, d_X, res, (cudaStream_t)cuda_stream);
}

namespace {
template <typename VT>
tomo_status_t update_values_t(tomo_lsqr_s* h, const VT* d_vals, cudaStream_t st) {
  int* d_flag = nullptr;
  CK(cudaMalloc(&d_flag, sizeof(int)));
  cudaMemsetAsync(d_flag, 0, sizeof(int), st);
  k_values_finite<VT><<<h->sms * 8, 256, 0, st>>>(d_vals, h->nnz, d_flag);
  int flag = 0;
  cudaError_t e = cudaMemcpyAsync(&flag, d_flag, sizeof(int), cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  cudaFree(d_flag);
  if (e != cudaSuccess) return cuda_fail(e, "value check");
  if (flag) return TOMO_ERR_BAD_CSR;  // nothing has been touched yet
  if (!h->pos && h->nnz > 0) { tomo_status_t rc = build_csc<VT>(h, st, true); if (rc != TOMO_OK) return rc; }
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  cudaEventRecord(e0, st);
  if (h->nnz > 0) {
    if (h->pos_wide) k_update_values<VT, int64_t><<<h->sms * 16, 256, 0, st>>>(d_vals, (const int64_t*)h->pos, h->nnz, (VT*)h->cvals);
    else k_update_values<VT, uint32_t><<<h->sms * 16, 256, 0, st>>>(d_vals, (const uint32_t*)h->pos, h->nnz, (VT*)h->cvals);
  }
  cudaEventRecord(e1, st);
  e = cudaGetLastError();
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  float ms = 0;
  if (e == cudaSuccess && cudaEventElapsedTime(&ms, e0, e1) == cudaSuccess) h->update_ms = ms;
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  if (e != cudaSuccess) return cuda_fail(e, "value refresh");
  if (h->vals != (const void*)d_vals) {  // the captured graphs hold the old pointer as a kernel argument
    if (h->gexec) { cudaGraphExecDestroy(h->gexec); h->gexec = nullptr; }
    if (h->mgexec) { cudaGraphExecDestroy(h->mgexec); h->mgexec = nullptr; }
  }
  h->vals = d_vals;
  h->dir[0].val = d_vals;
  return TOMO_OK;
}
}  // namespace

// NEXT-4 for the factored form: new depth kernels on the same rays
// a kernel table per lateral node (the paper's Theta_k): the handle applies it through the two-stage kernels
extern "C" tomo_status_t tomo_lsqr_set_nodal_kernels(tomo_lsqr_t h, const int32_t* d_kj0, const double* d_kern, void* cuda_stream) {
  if (!h || !h->fac || !d_kj0 || !d_kern) return TOMO_ERR_INVALID_ARG;
  { tomo_status_t rc = check_device(h); if (rc != TOMO_OK) return rc; }
  if (!is_device_ptr(d_kj0) || !is_device_ptr(d_kern)) return TOMO_ERR_NOT_DEVICE_PTR;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  FacState* f = h->fac;
  const int64_t ntab = f->d.nnodes * f->d.nper;
  const int klen = f->d.klen, nz = f->d.nz;
  int* d_flags = nullptr;
  CK(cudaMalloc(&d_flags, sizeof(int)));
  cudaMemsetAsync(d_flags, 0, sizeof(int), st);
  k_fac_validate_kern<<<h->sms * 4, 256, 0, st>>>(ntab, nz, klen, d_kj0, d_kern, d_flags);
  int flags = 0;
  cudaError_t e = cudaMemcpyAsync(&flags, d_flags, sizeof(int), cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  cudaFree(d_flags);
  if (e != cudaSuccess) return cuda_fail(e, "validation of the nodal kernel table");
  if (flags) return TOMO_ERR_BAD_CSR;   // nothing has been touched
  if (!f->kj0n) {
    int32_t* a = nullptr; double* b2 = nullptr;
    if ((e = cudaMalloc(&a, sizeof(int32_t) * ntab)) != cudaSuccess) return cuda_fail(e, "cudaMalloc(nodal windows)");
    if ((e = cudaMalloc(&b2, sizeof(double) * ntab * klen)) != cudaSuccess) { cudaFree(a); return cuda_fail(e, "cudaMalloc(nodal kernels)"); }
    f->kj0n = a; f->kernn = b2;
  }
  CK(cudaMemcpyAsync(f->kj0n, d_kj0, sizeof(int32_t) * ntab, cudaMemcpyDeviceToDevice, st));
  CK(cudaMemcpyAsync(f->kernn, d_kern, sizeof(double) * ntab * klen, cudaMemcpyDeviceToDevice, st));
  CK(cudaStreamSynchronize(st));
  if (!f->d.nodal) {   // the kernel argument changes: captured graphs hold the old one
    if (h->gexec) { cudaGraphExecDestroy(h->gexec); h->gexec = nullptr; }
    f->d.nodal = 1; f->d.kj0 = f->kj0n; f->d.kern = f->kernn;
    for (int mode = 0; mode < 4; ++mode) { f->dm[mode].nodal = 1; f->dm[mode].kj0 = f->kj0n; f->dm[mode].kern = f->kernn; }
  }
  return TOMO_OK;
}

extern "C" tomo_status_t tomo_lsqr_update_kernels(tomo_lsqr_t h, const int32_t* d_kj0, const double* d_kern, void* cuda_stream) {
  if (!h || !h->fac || h->fac->d.nodal || !d_kj0 || !d_kern) return TOMO_ERR_INVALID_ARG;
  { tomo_status_t rc = check_device(h); if (rc != TOMO_OK) return rc; }
  if (!is_device_ptr(d_kj0) || !is_device_ptr(d_kern)) return TOMO_ERR_NOT_DEVICE_PTR;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  FacState* f = h->fac;
  const int nper = f->d.nper, klen = f->d.klen, nz = f->d.nz;
  int* d_flags = nullptr;
  CK(cudaMalloc(&d_flags, sizeof(int)));
  cudaMemsetAsync(d_flags, 0, sizeof(int), st);
  k_fac_validate_kern<<<1, 256, 0, st>>>((int64_t)nper, nz, klen, d_kj0, d_kern, d_flags);
  int flags = 0;
  cudaError_t e = cudaMemcpyAsync(&flags, d_flags, sizeof(int), cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  cudaFree(d_flags);
  if (e != cudaSuccess) return cuda_fail(e, "validation of the kernel table");
  if (flags) return TOMO_ERR_BAD_CSR;   // nothing has been touched
  // the handle's own copies are overwritten in place: captured graphs keep pointing at them
  CK(cudaMemcpyAsync(f->kj0, d_kj0, sizeof(int32_t) * nper, cudaMemcpyDeviceToDevice, st));
  CK(cudaMemcpyAsync(f->kern, d_kern, sizeof(double) * nper * klen, cudaMemcpyDeviceToDevice, st));
  CK(cudaStreamSynchronize(st));
  return TOMO_OK;
}

extern "C" tomo_status_t tomo_lsqr_update_values(tomo_lsqr_t h, const void* d_vals, void* cuda_stream) {
  if (!h || h->fac || (h->nnz > 0 && !d_vals)) return TOMO_ERR_INVALID_ARG;  // a factored handle stores no value per nonzero
  { tomo_status_t rc = check_device(h); if (rc != TOMO_OK) return rc; }
  if (h->nnz > 0 && !is_device_ptr(d_vals)) return TOMO_ERR_NOT_DEVICE_PTR;
  if ((uintptr_t)d_vals & 15u) return TOMO_ERR_INVALID_ARG;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  return h->vt == TOMO_VAL_F64 ? update_values_t<double>(h, (const double*)d_vals, st) : update_values_t<float>(h, (const float*)d_vals, st);
}

// ------------------------------------------------------------------------------------------------
// NEXT-3: row-sharded LSQR (shard.cuh)
// ------------------------------------------------------------------------------------------------
namespace {

template <int MODE, typename VT>
tomo_status_t solve_sharded_t(tomo_lsqr_s* const* sh, int nlocal, int rank, int nranks, tomo_allgather_fn allgather, void* ctx,
                              const double* const* d_b, double damp, double atol, double btol, int32_t max_iters, double* d_x,
                              tomo_lsqr_result_t* res, cudaStream_t st) {
  tomo_lsqr_s* h0 = sh[0];
  const int64_t n = h0->n;
  const int P = nlocal * nranks;
  // exchange buffers: per block one norm pair followed by n column pairs; send = my nlocal blocks, recv = all P blocks
  const int64_t per = n + 1;
  if (h0->sh_send_cap < per * nlocal) {
    cudaFree(h0->sh_send); h0->sh_send = nullptr; h0->sh_send_cap = 0;
    CK(cudaMalloc(&h0->sh_send, sizeof(double2) * per * nlocal));
    h0->sh_send_cap = per * nlocal;
  }
  if (nranks > 1 && h0->sh_recv_cap < per * P) {
    cudaFree(h0->sh_recv); h0->sh_recv = nullptr; h0->sh_recv_cap = 0;
    CK(cudaMalloc(&h0->sh_recv, sizeof(double2) * per * P));
    h0->sh_recv_cap = per * P;
  }
  // layout: norms [blocks], then column pairs [blocks][n]; with one rank the send buffer is the gathered buffer
  double2* norm_send = h0->sh_send;
  double2* t_send = h0->sh_send + nlocal;
  double2* norm_all = nranks > 1 ? h0->sh_recv : norm_send;
  double2* t_all = nranks > 1 ? h0->sh_recv + P : t_send;
  auto exchange = [&](double2* send, double2* recv, int64_t pairs_per_rank) -> tomo_status_t {
    if (nranks == 1) return TOMO_OK;
    if (allgather(ctx, send, recv, (size_t)pairs_per_rank * sizeof(double2), (void*)st) != 0) return TOMO_ERR_CUDA;
    return TOMO_OK;
  };
  for (int l = 0; l < nlocal; ++l) { tomo_status_t rc = rebuild_partitions(sh[l], st); if (rc != TOMO_OK) return rc; }

  Scalars* hs = h0->h_sc;
  memset(hs, 0, sizeof(Scalars));
  hs->damp = damp; hs->atol = atol; hs->btol = btol; hs->max_iters = max_iters; hs->cs2 = -1.0; hs->solver = 0;
  CK(cudaMemcpyAsync(h0->sc, hs, sizeof(Scalars), cudaMemcpyHostToDevice, st));
  CK(cudaMemsetAsync(h0->x, 0, sizeof(double) * n, st));
  Scalars* sc = h0->sc;
  const int gv = vec_blocks(h0, n);
  auto k1s = [&](int l) { launch_wstream_t<MODE, VT, OP_K1S, 0, false>(sh[l], h0->v, sh[l]->u, st, sc);
                          cudaMemcpyAsync(norm_send + l, sh[l]->part_spmv + sh[l]->SG, sizeof(double2), cudaMemcpyDeviceToDevice, st); };
  auto k2s = [&](int l) { launch_wstream_t<MODE, VT, OP_K2S, 0, true>(sh[l], sh[l]->u, reinterpret_cast<double*>(t_send + (int64_t)l * n), st, sc); };
  // a1: beta_1 = ||b||, u^ = b, v^ = A^T u, alpha_1, w = v
  for (int l = 0; l < nlocal; ++l)
    k_vec<MODE, VOP_INIT_US><<<vec_blocks(sh[l], sh[l]->m), kThreads, 0, st>>>(d_b[l], sh[l]->u, nullptr, nullptr,
                                                                             reinterpret_cast<double*>(norm_send + l), sh[l]->m, sc, sh[l]->part_vec);
  { tomo_status_t rc = exchange(norm_send, norm_all, nlocal); if (rc != TOMO_OK) return rc; }
  k_shard_norm<MODE, 0><<<1, 32, 0, st>>>(norm_all, P, sc);
  for (int l = 0; l < nlocal; ++l) k2s(l);
  { tomo_status_t rc = exchange(t_send, t_all, (int64_t)nlocal * n); if (rc != TOMO_OK) return rc; }
  k_shard_combine<MODE, true><<<gv, 256, 0, st>>>(t_all, P, n, h0->v, sc, h0->part_vec);
  k_vec<MODE, VOP_INIT_VW><<<gv, kThreads, 0, st>>>(nullptr, h0->v, h0->w, nullptr, nullptr, n, sc, h0->part_vec);
  CK(cudaGetLastError());
  double launches = 4.0 + 2.0 * nlocal;
  const int k = h0->check_every;
  bool stopped = false;
  for (int it = 0; it < max_iters && !stopped; ++it) {
    for (int l = 0; l < nlocal; ++l) k1s(l);
    { tomo_status_t rc = exchange(norm_send, norm_all, nlocal); if (rc != TOMO_OK) return rc; }
    k_shard_norm<MODE, 1><<<1, 32, 0, st>>>(norm_all, P, sc);
    for (int l = 0; l < nlocal; ++l) k2s(l);
    { tomo_status_t rc = exchange(t_send, t_all, (int64_t)nlocal * n); if (rc != TOMO_OK) return rc; }
    k_shard_combine<MODE, false><<<gv, 256, 0, st>>>(t_all, P, n, h0->v, sc, h0->part_vec);
    k_vec<MODE, VOP_K4><<<gv, kThreads, 0, st>>>(nullptr, h0->v, h0->w, h0->x, nullptr, n, sc, h0->part_vec);
    launches += 3.0 + 2.0 * nlocal;
    if ((it + 1) % k == 0 || it + 1 == max_iters) {  // host poll (every rank sees the same replicated stop flag)
      CK(cudaGetLastError());
      CK(cudaMemcpyAsync(&h0->h_poll[0], &sc->itn, sizeof(PollWord), cudaMemcpyDeviceToHost, st));
      CK(cudaStreamSynchronize(st));
      if (h0->h_poll[0].stop) stopped = true;
    }
  }
  h0->kernels_enqueued += launches;
  CK(cudaMemcpyAsync(d_x, h0->x, sizeof(double) * n, cudaMemcpyDeviceToDevice, st));
  CK(cudaMemcpyAsync(hs, sc, sizeof(Scalars), cudaMemcpyDeviceToHost, st));
  CK(cudaStreamSynchronize(st));
  if (res) {
    res->itn = hs->itn; res->istop = hs->istop;
    res->r1norm = hs->r1norm; res->r2norm = hs->r2norm; res->arnorm = hs->arnorm;
    res->anorm = hs->anorm; res->acond = hs->acond; res->xnorm = hs->xnorm;
  }
  return TOMO_OK;
}

}  // namespace

extern "C" tomo_status_t tomo_lsqr_solve_sharded(const tomo_lsqr_t* shards, int32_t nlocal, int32_t rank, int32_t nranks,
                                                 tomo_allgather_fn allgather, void* ctx, const double* const* d_b, double damp,
                                                 double atol, double btol, int32_t max_iters, double* d_x, tomo_lsqr_result_t* res,
                                                 void* cuda_stream) {
  if (!shards || nlocal < 1 || nlocal > 64 || nranks < 1 || rank < 0 || rank >= nranks || !d_b || !d_x) return TOMO_ERR_INVALID_ARG;
  if (nranks > 1 && !allgather) return TOMO_ERR_INVALID_ARG;
  tomo_lsqr_s* h0 = shards[0];
  tomo_status_t rc = check_solve_args(h0, damp, atol, btol, max_iters);
  if (rc != TOMO_OK) return rc;
  if (!is_device_ptr(d_x)) return TOMO_ERR_NOT_DEVICE_PTR;
  for (int l = 0; l < nlocal; ++l) {
    const tomo_lsqr_s* h = shards[l];
    if (!h || h->fac || h->n != h0->n || h->vt != h0->vt || h->device != h0->device) return TOMO_ERR_INVALID_ARG;
    if (!d_b[l]) return TOMO_ERR_INVALID_ARG;
    if (!is_device_ptr(d_b[l])) return TOMO_ERR_NOT_DEVICE_PTR;
  }
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (h0->vt == TOMO_VAL_F64)
    return h0->accumulate ? solve_sharded_t<1, double>(shards, nlocal, rank, nranks, allgather, ctx, d_b, damp, atol, btol, max_iters, d_x, res, st)
                          : solve_sharded_t<0, double>(shards, nlocal, rank, nranks, allgather, ctx, d_b, damp, atol, btol, max_iters, d_x, res, st);
  return h0->accumulate ? solve_sharded_t<1, float>(shards, nlocal, rank, nranks, allgather, ctx, d_b, damp, atol, btol, max_iters, d_x, res, st)
                        : solve_sharded_t<0, float>(shards, nlocal, rank, nranks, allgather, ctx, d_b, damp, atol, btol, max_iters, d_x, res, st);
}

extern "C" tomo_status_t tomo_lsqr_spmv(tomo_lsqr_t h, int transpose, const double* d_in, double* d_out, void* cuda_stream) {
  if (!h || !d_in || !d_out || (transpose != 0 && transpose != 1)) return TOMO_ERR_INVALID_ARG;
  if (!is_device_ptr(d_in) || !is_device_ptr(d_out)) return TOMO_ERR_NOT_DEVICE_PTR;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  tomo_status_t rc = check_device(h);
  if (rc != TOMO_OK) return rc;
  rc = rebuild_partitions(h, st);
  if (rc != TOMO_OK) return rc;
  launch_spmv<OP_PLAIN>(h, transpose != 0, d_in, d_out, st);
  CK(cudaGetLastError());
  CK(cudaStreamSynchronize(st));
  return TOMO_OK;
}

extern "C" tomo_status_t tomo_lsqr_get_csc(tomo_lsqr_t h, int64_t* d_colptr, int32_t* d_rowind, void* d_cvals, void* cuda_stream) {
  if (!h || h->fac) return TOMO_ERR_INVALID_ARG;
  { tomo_status_t rc = check_device(h); if (rc != TOMO_OK) return rc; }
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const size_t vb = h->vt == TOMO_VAL_F64 ? sizeof(double) : sizeof(float);
  if (d_colptr) CK(cudaMemcpyAsync(d_colptr, h->colptr, sizeof(int64_t) * (h->n + 1), cudaMemcpyDeviceToDevice, st));
  if (d_rowind && h->nnz) CK(cudaMemcpyAsync(d_rowind, h->rowind, sizeof(int32_t) * h->nnz, cudaMemcpyDeviceToDevice, st));
  if (d_cvals && h->nnz) CK(cudaMemcpyAsync(d_cvals, h->cvals, vb * h->nnz, cudaMemcpyDeviceToDevice, st));
  CK(cudaStreamSynchronize(st));
  return TOMO_OK;
}

extern "C" tomo_status_t tomo_lsqr_set_option(tomo_lsqr_t h, const char* key, int64_t value) {
  if (!h || !key) return TOMO_ERR_INVALID_ARG;
  const std::string k(key);
  if (k == "check_every") { if (value < 1 || value > 100000) return TOMO_ERR_INVALID_ARG; h->check_every = (int)value; }
  else if (k == "accumulate") { if (value != 0 && value != 1) return TOMO_ERR_INVALID_ARG; h->accumulate = (int)value; }
  else if (k == "graph") { if (value != 0 && value != 1) return TOMO_ERR_INVALID_ARG; h->use_graph = (int)value; }
  else if (k == "profile") { if (value != 0 && value != 1) return TOMO_ERR_INVALID_ARG; h->profile = (int)value; }
  else if (k == "two_stage") { if (value < 0 || value > 2) return TOMO_ERR_INVALID_ARG; h->two_stage = (int)value; }
  else if (k == "multi_shared") { if (value != 0 && value != 1) return TOMO_ERR_INVALID_ARG; h->multi_shared = (int)value; }
  else if (k == "compress") {
    if (value != 0 && value != 1) return TOMO_ERR_INVALID_ARG;
    if (h->fac) return value == 0 ? TOMO_OK : TOMO_ERR_INVALID_ARG;
    { tomo_status_t rc = check_device(h); if (rc != TOMO_OK) return rc; }
    if (value == 1) for (int d = 0; d < 2; ++d) { tomo_status_t rc = build_compressed(h, d, nullptr); if (rc != TOMO_OK) return rc; }
    if (h->compress != (int)value && h->gexec) { cudaGraphExecDestroy(h->gexec); h->gexec = nullptr; }
    h->compress = (int)value;
  }
  else if (k == "pdl") { if (value != 0 && value != 1) return TOMO_ERR_INVALID_ARG; if (h->pdl != (int)value && h->gexec) { cudaGraphExecDestroy(h->gexec); h->gexec = nullptr; } h->pdl = (int)value; }
  else if (k == "row_cost") { if (value < 0 || value > 4096) return TOMO_ERR_INVALID_ARG; if (h->row_cost != (int)value) h->part_dirty = true; h->row_cost = (int)value; }
  else return TOMO_ERR_INVALID_ARG;
  return TOMO_OK;
}

extern "C" tomo_status_t tomo_lsqr_get_info(tomo_lsqr_t h, const char* key, double* out) {
  if (!h || !key || !out) return TOMO_ERR_INVALID_ARG;
  const std::string k(key);
  const double vb = h->vt == TOMO_VAL_F64 ? 8.0 : 4.0;
  if (k == "create_ms") *out = h->create_ms;
  else if (k == "factored") *out = h->fac ? 1.0 : 0.0;
  else if (k == "nodal_kernels") *out = (h->fac && h->fac->d.nodal) ? 1.0 : 0.0;
  else if (k == "lateral_entries") *out = h->fac ? (double)h->fac->E : 0.0;
  else if (k == "cut_nodes_pieces") *out = h->fac ? (double)h->fac->nslots : 0.0;
  else if (k == "operator_bytes")   // what a product has to read of the operator itself
    *out = h->fac ? 12.0 * (double)h->fac->E + 8.0 * (double)(h->fac->d.npairs + 1) + 12.0 * (double)h->fac->snnz + 8.0 * (double)(h->fac->d.ms + 1)
                  : (double)h->nnz * (4.0 + vb) + 8.0 * (double)(h->m + 1);
  else if (h->fac && (k == "warp_busy_min" || k == "warp_busy_mean" || k == "warp_busy_max" || k == "warp_busy_argmax")) {
    // busy cycles of the warps in the most recent product launch on the factored operator (balance of the static split)
    const int NW = h->sms * kFacWarps;
    std::vector<long long> b((size_t)NW);
    CK(cudaMemcpy(b.data(), h->fac->busy, sizeof(long long) * NW, cudaMemcpyDeviceToHost));
    double mn = 1e300, mx = -1, sum = 0; int arg = 0;
    for (int i = 0; i < NW; ++i) { const double c = (double)b[i]; mn = std::min(mn, c); if (c > mx) { mx = c; arg = i; } sum += c; }
    *out = k == "warp_busy_min" ? mn : k == "warp_busy_max" ? mx : k == "warp_busy_argmax" ? (double)arg : sum / NW;
  }
  else if (h->fac && k.rfind("warp_busy@", 0) == 0) {   // one warp's figure
    const int i = atoi(k.c_str() + 10);
    if (i < 0 || i >= h->sms * kFacWarps) return TOMO_ERR_INVALID_ARG;
    long long b = 0;
    CK(cudaMemcpy(&b, h->fac->busy + i, sizeof(long long), cudaMemcpyDeviceToHost));
    *out = (double)b;
  }
  else if (h->fac && (k == "csc_bytes" || k.rfind("compress_bytes", 0) == 0 || k.rfind("cta_busy", 0) == 0)) return TOMO_ERR_INVALID_ARG;
  else if (k == "transpose_ms") *out = h->transpose_ms;
  else if (k == "transpose_kernels_ms") *out = h->transpose_kernels_ms;
  else if (k == "update_ms") *out = h->update_ms;
  else if (k == "csc_bytes") *out = (double)h->nnz * (4.0 + vb) + 8.0 * (double)(h->n + 1);
  else if (k == "scratch_bytes") *out = h->scratch_bytes;
  else if (k == "compress_bytes_rows") *out = (double)h->dir[0].cbytes + 8.0 * (double)((h->nnz + WC::TILE - 1) / WC::TILE + 1);
  else if (k == "compress_bytes_cols") *out = (double)h->dir[1].cbytes + 8.0 * (double)((h->nnz + WC::TILE - 1) / WC::TILE + 1);
  else if (k == "blocks_rows" || k == "blocks_cols") *out = (double)h->SG;
  else if (k == "k1_ms") *out = h->k1_ms;
  else if (k == "k2_ms") *out = h->k2_ms;
  else if (k == "k4_ms") *out = h->k4_ms;
  else if (k == "k_launches") *out = h->k_launches;
  else if (k == "kernels_enqueued") *out = h->kernels_enqueued;
  else if (k == "cta_busy_min" || k == "cta_busy_max" || k == "cta_busy_mean") {
    // busy cycles of the persistent CTAs in the most recent SpMV launch (load balance of the static split)
    std::vector<CtaRec> rec(h->SG);
    CK(cudaMemcpy(rec.data(), h->cta_rec, sizeof(CtaRec) * h->SG, cudaMemcpyDeviceToHost));
    double mn = 1e300, mx = 0, sum = 0;
    for (const CtaRec& r : rec) { const double c = 16.0 * (double)r.pad; mn = std::min(mn, c); mx = std::max(mx, c); sum += c; }
    *out = k == "cta_busy_min" ? mn : k == "cta_busy_max" ? mx : sum / std::max(1, h->SG);
  }
  else return TOMO_ERR_INVALID_ARG;
  return TOMO_OK;
}

// ------------------------------------------------------------------------------------------------
// tomo_lsqr_spmv_noalloc: the plain product over the caller's CSR for callers that cannot allocate.  The scratch of the
// streaming kernel (and of the compaction of rows without entries) lives in one file-scope device array.
// ------------------------------------------------------------------------------------------------
namespace {

// layout of the static scratch array; every member starts at a multiple of 256 bytes
struct NoAllocScratch {
  alignas(256) unsigned char sc[4096];                                          // Scalars (only the ticket words are used)
  alignas(256) int cnt[64];                                                     // number of rows without entries
  alignas(256) CtaRec rec[TOMO_NOALLOC_MAX_SMS];                                // one record per persistent CTA
  alignas(256) double2 part[TOMO_NOALLOC_MAX_SMS + 2];                          // per-CTA ||.||^2 partials (unused by the plain product, still written)
  alignas(256) int64_t wE[TOMO_NOALLOC_MAX_SMS * WC::W + 1];                    // element split points of the warp ranges
  alignas(256) int32_t wR[TOMO_NOALLOC_MAX_SMS * WC::W + 1];                    // ... and their first rows
  alignas(256) int64_t pos[TOMO_NOALLOC_MAX_ROWS + 1];                          // exclusive scan of the non-empty flags
  alignas(256) int64_t cptr[TOMO_NOALLOC_MAX_ROWS + 1];                         // non-empty flags, then the compacted row pointers
  alignas(256) int32_t rid[TOMO_NOALLOC_MAX_ROWS];                              // row numbers of the non-empty rows
  alignas(256) int32_t erows[TOMO_NOALLOC_MAX_ROWS];                            // rows without entries
};
static_assert(sizeof(Scalars) <= 4096, "Scalars outgrew its slot of the static scratch");
static_assert(sizeof(NoAllocScratch) <= TOMO_NOALLOC_SCRATCH_BYTES, "TOMO_NOALLOC_SCRATCH_BYTES is too small for the layout");

}  // namespace

// The name below is a HOST-side stand-in in host code, not a device address: the address a kernel can use comes
// from cudaGetSymbolAddress, once per device, with that device current (noalloc_setup).
static __device__ __align__(256) unsigned char g_noalloc_scratch[TOMO_NOALLOC_SCRATCH_BYTES];

namespace {

constexpr int kNoAllocMaxDevices = 64;
std::mutex g_noalloc_mu;
NoAllocScratch* g_noalloc_ptr[kNoAllocMaxDevices] = {};   // device address of the array on device d (NULL: not set up yet)

// once per device (the device is current): address of the device's copy of the array, shared-memory opt-in of the
// four instantiations the entry launches
tomo_status_t noalloc_setup(int dev, NoAllocScratch** out) {
  std::lock_guard<std::mutex> lock(g_noalloc_mu);
  if (!g_noalloc_ptr[dev]) {
    void* p = nullptr;
    cudaError_t e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
    if (e != cudaSuccess) return cuda_fail(e, "cudaGetSymbolAddress(static scratch)");
    if (!p || ((uintptr_t)p & 255u)) { snprintf(g_cuda_msg, sizeof(g_cuda_msg), "static scratch: bad device address"); return TOMO_ERR_CUDA; }
    if ((e = stream_attr_one<WC, 0, double, OP_PLAIN, 0>()) != cudaSuccess || (e = stream_attr_one<WC, 1, double, OP_PLAIN, 0>()) != cudaSuccess ||
        (e = stream_attr_one<WC, 0, float, OP_PLAIN, 0>()) != cudaSuccess || (e = stream_attr_one<WC, 1, float, OP_PLAIN, 0>()) != cudaSuccess)
      return cuda_fail(e, "cudaFuncSetAttribute(shared memory opt-in)");
    g_noalloc_ptr[dev] = static_cast<NoAllocScratch*>(p);
  }
  *out = g_noalloc_ptr[dev];
  return TOMO_OK;
}

template <int MODE, typename VT>
cudaError_t noalloc_launch(int sms, const int64_t* ptr, const int32_t* rid, const int32_t* idx, const VT* val, int64_t nnz, int nrows,
                           const int32_t* erows, int n_empty, const double* x, double* y, NoAllocScratch* S, cudaStream_t st) {
  k_wstream<WC, MODE, VT, OP_PLAIN, 0><<<sms, WC::THREADS, WSmem<WC, VT, 0>::kTotal, st>>>(
      ptr, rid, idx, val, nullptr, nullptr, nnz, nrows, erows, n_empty, x, y, S->wE, S->wR, S->rec, reinterpret_cast<Scalars*>(S->sc), S->part);
  return cudaGetLastError();
}

}  // namespace

extern "C" tomo_status_t tomo_lsqr_spmv_noalloc(int64_t m, int64_t n, int64_t nnz, const int64_t* d_rowptr, const int32_t* d_colind,
                                           const void* d_vals, tomo_valtype_t vt, int accumulate, const double* d_x, double* d_y,
                                           void* cuda_stream) {
  if (vt != TOMO_VAL_F64 && vt != TOMO_VAL_F32) return TOMO_ERR_INVALID_ARG;
  if (accumulate != 0 && accumulate != 1) return TOMO_ERR_INVALID_ARG;
  if (m < 1 || n < 1 || nnz < 0 || !d_x || !d_y) return TOMO_ERR_INVALID_ARG;
  if (m >= (int64_t)INT32_MAX || n >= (int64_t)INT32_MAX || nnz >= ((int64_t)1 << 40)) return TOMO_ERR_RANGE;
  if (!d_rowptr || (nnz > 0 && (!d_colind || !d_vals))) return TOMO_ERR_INVALID_ARG;
  int dev = 0, major = 0, sms = 0;
  CK(cudaGetDevice(&dev));
  CK(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
  CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  if (major != 10) return TOMO_ERR_UNSUPPORTED_ARCH;
  if (m > (int64_t)TOMO_NOALLOC_MAX_ROWS) {
    snprintf(g_noalloc_msg, sizeof(g_noalloc_msg), "tomo_lsqr_spmv_noalloc: m = %lld rows exceeds TOMO_NOALLOC_MAX_ROWS = %d (the static scratch array); use a handle (tomo_lsqr_create + tomo_lsqr_spmv)",
             (long long)m, (int)TOMO_NOALLOC_MAX_ROWS);
    return TOMO_ERR_NOALLOC_LIMIT;
  }
  if (sms > TOMO_NOALLOC_MAX_SMS || dev >= kNoAllocMaxDevices) {
    snprintf(g_noalloc_msg, sizeof(g_noalloc_msg), "tomo_lsqr_spmv_noalloc: device %d with %d multiprocessors is beyond TOMO_NOALLOC_MAX_SMS = %d / %d devices (the static scratch array)",
             dev, sms, (int)TOMO_NOALLOC_MAX_SMS, kNoAllocMaxDevices);
    return TOMO_ERR_NOALLOC_LIMIT;
  }
  if (!is_device_ptr(d_rowptr) || !is_device_ptr(d_x) || !is_device_ptr(d_y) || (nnz > 0 && (!is_device_ptr(d_colind) || !is_device_ptr(d_vals))))
    return TOMO_ERR_NOT_DEVICE_PTR;
  if (((uintptr_t)d_colind & 15u) || ((uintptr_t)d_vals & 15u) || ((uintptr_t)d_rowptr & 7u)) return TOMO_ERR_INVALID_ARG;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  NoAllocScratch* S = nullptr;
  { tomo_status_t rc = noalloc_setup(dev, &S); if (rc != TOMO_OK) return rc; }

  // the array keeps the last call's contents: the ticket words and the counter must start at zero
  CK(cudaMemsetAsync(S->sc, 0, sizeof(Scalars), st));
  CK(cudaMemsetAsync(S->cnt, 0, sizeof(int), st));
  k_count_empty<<<sms * 4, 256, 0, st>>>(d_rowptr, m, S->cnt);
  CK(cudaGetLastError());
  int cnt = 0;
  CK(cudaMemcpyAsync(&cnt, S->cnt, sizeof(int), cudaMemcpyDeviceToHost, st));
  CK(cudaStreamSynchronize(st));
  const int64_t* ptr = d_rowptr; const int32_t* rid = nullptr; const int32_t* erows = nullptr;
  int nrows = (int)m;
  if (cnt > 0) {  // rows without entries never enter the stream (build_dir): compact them away, into the static array
    k_flag_nonempty<<<sms * 4, 256, 0, st>>>(d_rowptr, m, S->cptr);
    k_exscan<<<1, 1024, 0, st>>>(S->cptr, m, S->pos);
    k_compact_rows<<<sms * 4, 256, 0, st>>>(d_rowptr, m, S->pos, S->cptr, S->rid, S->erows);
    CK(cudaGetLastError());
    ptr = S->cptr; rid = S->rid; erows = S->erows; nrows = (int)(m - cnt);
  }
  const int parts = sms * WC::W;  // the split a handle with default options uses (row_cost 320): same summation order
  k_stream_partition<<<(parts + 1 + 127) / 128, 128, 0, st>>>(ptr, nrows, nnz, parts, 320, WC::TILE, S->wE, S->wR);
  CK(cudaGetLastError());
  cudaError_t e;
  if (vt == TOMO_VAL_F64)
    e = accumulate ? noalloc_launch<1, double>(sms, ptr, rid, d_colind, (const double*)d_vals, nnz, nrows, erows, cnt, d_x, d_y, S, st)
                   : noalloc_launch<0, double>(sms, ptr, rid, d_colind, (const double*)d_vals, nnz, nrows, erows, cnt, d_x, d_y, S, st);
  else
    e = accumulate ? noalloc_launch<1, float>(sms, ptr, rid, d_colind, (const float*)d_vals, nnz, nrows, erows, cnt, d_x, d_y, S, st)
                   : noalloc_launch<0, float>(sms, ptr, rid, d_colind, (const float*)d_vals, nnz, nrows, erows, cnt, d_x, d_y, S, st);
  if (e != cudaSuccess) return cuda_fail(e, "k_wstream (no-alloc product)");
  CK(cudaStreamSynchronize(st));
  return TOMO_OK;
}

extern "C" const char* tomo_status_string(tomo_status_t s) {
  switch (s) {
    case TOMO_OK: return "ok";
    case TOMO_ERR_INVALID_ARG: return "invalid argument";
    case TOMO_ERR_BAD_CSR: return "CSR arrays are not canonical (rowptr order, column range/order, or non-finite value)";
    case TOMO_ERR_NOT_DEVICE_PTR: return "a device pointer was expected";
    case TOMO_ERR_OOM: return "out of device or pinned memory";
    case TOMO_ERR_CUDA: return g_cuda_msg;
    case TOMO_ERR_UNSUPPORTED_ARCH: return "device is not compute capability 10.x (sm_100a build, no fallback)";
    case TOMO_ERR_RANGE: return "m, n or nnz out of range";
    case TOMO_ERR_NOALLOC_LIMIT: return g_noalloc_msg;
  }
  return "unknown status";
}
