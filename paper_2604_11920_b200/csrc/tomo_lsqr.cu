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
#include <new>
#include <string>
#include <vector>

#include "../../include/tomo_lsqr.h"
#include "build.cuh"
#include "kernels.cuh"
#include "stream.cuh"
#include "multi.cuh"

using namespace tomo;

namespace {

thread_local char g_cuda_msg[256] = "no CUDA error recorded";

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

struct tomo_lsqr_s {
  int64_t m = 0, n = 0, nnz = 0;
  tomo_valtype_t vt = TOMO_VAL_F64;
  // borrowed CSR
  const int64_t* rowptr = nullptr; const int32_t* colind = nullptr; const void* vals = nullptr;
  // owned CSC (= CSR of A^T)
  int64_t* colptr = nullptr; int32_t* rowind = nullptr; void* cvals = nullptr;
  // element split points of the persistent CTAs, per direction
  bool part_dirty = true;
  int64_t* sE_r = nullptr; int64_t* sE_c = nullptr; int32_t* sR_r = nullptr; int32_t* sR_c = nullptr;
  CtaRec* cta_rec = nullptr; int SG = 0; int empty_rows = 0, empty_cols = 0;
  // work vectors and device state
  double *u = nullptr, *v = nullptr, *w = nullptr, *x = nullptr, *hbar = nullptr;  // w doubles as LSMR's h
  int solver = 0;  // 0 LSQR, 1 LSMR (set per solve)
  // shared-pass multi-RHS state (multi.cuh): len x 8 blocks, eight Scalars, static row partitions
  double *mU = nullptr, *mV = nullptr, *mW = nullptr, *mX = nullptr; Scalars* msc = nullptr; Scalars* h_msc = nullptr;
  int32_t *mpart_r = nullptr, *mpart_c = nullptr; double2* mpartials = nullptr; int MG = 0, multi_shared = 1;
  cudaGraphExec_t mgexec = nullptr; int mgraph_k = 0, mgraph_mode = -1;
  Scalars* sc = nullptr; double2* part_spmv = nullptr; double2* part_vec = nullptr; int part_cap = 0;
  double *hist_r2 = nullptr, *hist_ar = nullptr; int32_t hist_cap = 0;
  double *bh = nullptr, *xh = nullptr;   // device staging for solve_host
  Scalars* h_sc = nullptr; PollWord* h_poll = nullptr;  // pinned
  cudaEvent_t ev_poll[2] = {nullptr, nullptr};
  cudaStream_t cap_stream = nullptr;
  cudaGraphExec_t gexec = nullptr; int graph_k = 0, graph_mode = -1, graph_G = 0;
  // options
  int check_every = 10, accumulate = 1, use_graph = 1, profile = 0, row_cost = 96;
  // info
  int sms = 0; double create_ms = 0, transpose_ms = 0, scratch_bytes = 0;
  double k1_ms = 0, k2_ms = 0, k4_ms = 0, k_launches = 0;
  double kernels_enqueued = 0;  // cumulative count of this library's kernel launches (graph nodes included)
  std::vector<cudaEvent_t> prof_ev;
};

namespace {

int vec_blocks(const tomo_lsqr_s* h, int64_t len) {
  int64_t b = (len + kThreads - 1) / kThreads;
  return (int)std::max<int64_t>(1, std::min<int64_t>(b, (int64_t)h->sms * 16));
}

// Kernel shapes <elements per chunk, consumer warps, ring stages, L2 prefetch distance>, per accumulation
// mode (measured on B200, config 1): the double-double sums are instruction-bound, so they take the
// longer slices (two 256-element rounds per slice, half the per-slice bookkeeping); the plain sums are
// bandwidth-bound and take the deeper ring, which also leaves ~60 KB of L1 for the gathered vector.
#ifdef TOMO_CH
using SCfgFast = StreamCfg<TOMO_CH, TOMO_W, TOMO_S, TOMO_PF>;
using SCfgDD = StreamCfg<TOMO_CH, TOMO_W, TOMO_S, TOMO_PF>;
#else
using SCfgFast = StreamCfg<4096, 16, 3, 0>;
using SCfgDD = StreamCfg<8192, 16, 2, 0>;
#endif
template <int MODE> struct SCfgOf { using type = SCfgFast; };
template <> struct SCfgOf<1> { using type = SCfgDD; };

template <int MODE, typename VT, int OP>
void launch_stream_t(const tomo_lsqr_s* h, bool transpose, const double* x, double* y, cudaStream_t st) {
  const int64_t* ptr = transpose ? h->colptr : h->rowptr;
  const int32_t* idx = transpose ? h->rowind : h->colind;
  const VT* val = (const VT*)(transpose ? h->cvals : h->vals);
  const int nrows = (int)(transpose ? h->n : h->m);
  using SCfg = typename SCfgOf<MODE>::type;
  auto kern = k_stream<SCfg, MODE, VT, OP>;
  static bool attr_set = false;  // per instantiation
  constexpr size_t smem = StreamSmem<SCfg, VT>::kTotal;
  if (!attr_set) { cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem); attr_set = true; }
  kern<<<h->SG, SCfg::THREADS, smem, st>>>(ptr, idx, val, h->nnz, nrows, transpose ? h->empty_cols : h->empty_rows, x, y,
                                           transpose ? h->sE_c : h->sE_r, transpose ? h->sR_c : h->sR_r, h->cta_rec, h->sc,
                                           h->part_spmv);
}

template <int OP>
void launch_spmv(const tomo_lsqr_s* h, bool transpose, const double* x, double* y, cudaStream_t st) {
  if (h->vt == TOMO_VAL_F64) {
    if (h->accumulate) launch_stream_t<1, double, OP>(h, transpose, x, y, st);
    else launch_stream_t<0, double, OP>(h, transpose, x, y, st);
  } else {
    if (h->accumulate) launch_stream_t<1, float, OP>(h, transpose, x, y, st);
    else launch_stream_t<0, float, OP>(h, transpose, x, y, st);
  }
}

template <int VOP>
void launch_vec(const tomo_lsqr_s* h, const double* in0, double* a0, double* a1, double* a2, int64_t len, cudaStream_t st,
                double* a3 = nullptr) {
  const int g = vec_blocks(h, len);
  if (h->accumulate) k_vec<1, VOP><<<g, kThreads, 0, st>>>(in0, a0, a1, a2, a3, len, h->sc, h->part_vec);
  else k_vec<0, VOP><<<g, kThreads, 0, st>>>(in0, a0, a1, a2, a3, len, h->sc, h->part_vec);
}

// the vector update that closes an iteration: LSQR's x / w step or LSMR's hbar / x / h step
void launch_k4(const tomo_lsqr_s* h, cudaStream_t st) {
  if (h->solver == 1) launch_vec<VOP_K4_LSMR>(h, nullptr, h->v, h->w, h->x, h->n, st, h->hbar);
  else launch_vec<VOP_K4>(h, nullptr, h->v, h->w, h->x, h->n, st);
}

tomo_status_t rebuild_partitions(tomo_lsqr_s* h, cudaStream_t st) {
  if (!h->part_dirty) return TOMO_OK;
  const int tb = 128;
  // stream kernel: one persistent CTA per SM, cost-balanced element split points
  h->SG = h->sms;
  const int gs = (h->SG + 1 + tb - 1) / tb;
  k_stream_partition<<<gs, tb, 0, st>>>(h->rowptr, h->m, h->nnz, h->SG, h->row_cost, h->sE_r, h->sR_r);
  k_stream_partition<<<gs, tb, 0, st>>>(h->colptr, h->n, h->nnz, h->SG, h->row_cost, h->sE_c, h->sR_c);
  CK(cudaGetLastError());
  h->part_dirty = false;
  return TOMO_OK;
}

}  // namespace

// ------------------------------------------------------------------------------------------------
// create / destroy
// ------------------------------------------------------------------------------------------------
namespace {

template <typename VT>
tomo_status_t build_csc(tomo_lsqr_s* h, cudaStream_t st) {
  const int64_t m = h->m, n = h->n, nnz = h->nnz;
  CK(cudaMalloc(&h->colptr, sizeof(int64_t) * (n + 1)));
  CK(cudaMalloc(&h->rowind, sizeof(int32_t) * std::max<int64_t>(nnz, 1)));
  CK(cudaMalloc(&h->cvals, sizeof(VT) * std::max<int64_t>(nnz, 1)));
  // number of row chunks (= warps): bounded by the scratch budget T*n*4 bytes <= 4 GB
  int64_t T = std::min<int64_t>((int64_t)h->sms * 16, std::max<int64_t>(32, (int64_t)(4.0e9 / (4.0 * (double)n))));
  T = std::max<int64_t>(1, std::min<int64_t>(T, m));
  int32_t* chunk = nullptr; uint32_t* cnt = nullptr; int64_t* coltotal = nullptr;
  CK(cudaMalloc(&chunk, sizeof(int32_t) * (T + 1)));
  cudaError_t e = cudaMalloc(&cnt, sizeof(uint32_t) * T * n);
  if (e != cudaSuccess) { cudaFree(chunk); return cuda_fail(e, "cudaMalloc(transpose scratch)"); }
  e = cudaMalloc(&coltotal, sizeof(int64_t) * n);
  if (e != cudaSuccess) { cudaFree(chunk); cudaFree(cnt); return cuda_fail(e, "cudaMalloc(coltotal)"); }
  h->scratch_bytes = (double)(sizeof(uint32_t) * T * n + sizeof(int64_t) * n + sizeof(int32_t) * (T + 1));
  tomo_status_t rc = TOMO_OK;
  do {
    const int tb = 128;
    k_partition<<<(int)((T + 1 + tb - 1) / tb), tb, 0, st>>>(h->rowptr, m, (int)T, 1, 1, chunk);
    k_partition_fix<<<1, 32, 0, st>>>((int)T, chunk);
    if ((e = cudaMemsetAsync(cnt, 0, sizeof(uint32_t) * T * n, st)) != cudaSuccess) break;
    const int wb = (int)((T + kWarps - 1) / kWarps);
    k_tr_count<<<wb, kThreads, 0, st>>>(h->rowptr, h->colind, chunk, (int)T, n, cnt);
    k_tr_colscan<<<(int)((n + 255) / 256), 256, 0, st>>>((int)T, n, cnt, coltotal);
    k_exscan<<<1, 1024, 0, st>>>(coltotal, n, h->colptr);
    k_tr_scatter<VT><<<wb, kThreads, 0, st>>>(h->rowptr, h->colind, (const VT*)h->vals, chunk, (int)T, n, cnt,
                                             h->colptr, h->rowind, (VT*)h->cvals);
    if ((e = cudaGetLastError()) != cudaSuccess) break;
    e = cudaStreamSynchronize(st);
  } while (0);
  if (e != cudaSuccess) rc = cuda_fail(e, "CSR->CSC transpose");
  cudaFree(chunk); cudaFree(cnt); cudaFree(coltotal);
  return rc;
}

void free_handle(tomo_lsqr_s* h) {
  if (!h) return;
  if (h->gexec) cudaGraphExecDestroy(h->gexec);
  if (h->cap_stream) cudaStreamDestroy(h->cap_stream);
  for (int i = 0; i < 2; ++i) if (h->ev_poll[i]) cudaEventDestroy(h->ev_poll[i]);
  for (cudaEvent_t e : h->prof_ev) cudaEventDestroy(e);
  cudaFree(h->colptr); cudaFree(h->rowind); cudaFree(h->cvals);
  cudaFree(h->mU); cudaFree(h->mV); cudaFree(h->mW); cudaFree(h->mX); cudaFree(h->msc); cudaFree(h->mpart_r); cudaFree(h->mpart_c);
  cudaFree(h->mpartials); if (h->h_msc) cudaFreeHost(h->h_msc); if (h->mgexec) cudaGraphExecDestroy(h->mgexec);
  cudaFree(h->sE_r); cudaFree(h->sE_c); cudaFree(h->sR_r); cudaFree(h->sR_c); cudaFree(h->cta_rec);
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
  if (m >= (int64_t)INT32_MAX || n >= (int64_t)INT32_MAX || nnz >= ((int64_t)1 << 62)) return TOMO_ERR_RANGE;
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
  h->m = m; h->n = n; h->nnz = nnz; h->vt = vt; h->sms = sms;
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
    rc = (vt == TOMO_VAL_F64) ? build_csc<double>(h, st) : build_csc<float>(h, st);
    if (rc != TOMO_OK) break;
    cudaEventRecord(e2, st);
    // --- work space ---
    h->part_cap = sms * 32 + 2;  // >= the largest grid of any kernel that publishes partials
#define ALLOC(p, bytes) if ((e = cudaMalloc(&(p), (bytes))) != cudaSuccess) { rc = cuda_fail(e, "cudaMalloc(work)"); break; }
    ALLOC(h->sE_r, sizeof(int64_t) * (sms + 1)); ALLOC(h->sE_c, sizeof(int64_t) * (sms + 1));
    ALLOC(h->sR_r, sizeof(int32_t) * (sms + 1)); ALLOC(h->sR_c, sizeof(int32_t) * (sms + 1));
    ALLOC(h->cta_rec, sizeof(CtaRec) * sms);
    ALLOC(h->u, sizeof(double) * m); ALLOC(h->v, sizeof(double) * n);
    ALLOC(h->w, sizeof(double) * n); ALLOC(h->x, sizeof(double) * n);
    ALLOC(h->sc, sizeof(Scalars));
    ALLOC(h->part_spmv, sizeof(double2) * h->part_cap);
    ALLOC(h->part_vec, sizeof(double2) * h->part_cap);
#undef ALLOC
    if ((e = cudaMemsetAsync(h->sc, 0, sizeof(Scalars), st)) != cudaSuccess) { rc = cuda_fail(e, "memset"); break; }
    {  // rows / columns without entries need the (rare) empty-row pass of the stream kernel
      int* d_cnt = nullptr;
      if ((e = cudaMalloc(&d_cnt, 2 * sizeof(int))) != cudaSuccess) { rc = cuda_fail(e, "cudaMalloc"); break; }
      cudaMemsetAsync(d_cnt, 0, 2 * sizeof(int), st);
      k_count_empty<<<sms * 4, 256, 0, st>>>(h->rowptr, m, d_cnt);
      k_count_empty<<<sms * 4, 256, 0, st>>>(h->colptr, n, d_cnt + 1);
      int cnt[2] = {0, 0};
      e = cudaMemcpyAsync(cnt, d_cnt, sizeof(cnt), cudaMemcpyDeviceToHost, st);
      if (e == cudaSuccess) e = cudaStreamSynchronize(st);
      cudaFree(d_cnt);
      if (e != cudaSuccess) { rc = cuda_fail(e, "count empty rows"); break; }
      h->empty_rows = cnt[0]; h->empty_cols = cnt[1];
    }
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
  const int gkey = h->accumulate + 2 * h->solver;
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
    const size_t need = (size_t)std::min(max_iters, kMaxProfileIters) * 4;
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
    h->kernels_enqueued += 3.0 * k;
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

tomo_status_t check_solve_args(tomo_lsqr_s* h, double damp, double atol, double btol, int32_t max_iters) {
  if (!h) return TOMO_ERR_INVALID_ARG;
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

extern "C" tomo_status_t tomo_lsqr_solve_host(tomo_lsqr_t h, const double* h_b, double damp, double atol, double btol,
                                              int32_t max_iters, double* h_x, tomo_lsqr_result_t* res, void* cuda_stream) {
  tomo_status_t rc = check_solve_args(h, damp, atol, btol, max_iters);
  if (rc != TOMO_OK) return rc;
  if (!h_b || !h_x) return TOMO_ERR_INVALID_ARG;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (!h->bh) CK(cudaMalloc(&h->bh, sizeof(double) * h->m));
  if (!h->xh) CK(cudaMalloc(&h->xh, sizeof(double) * h->n));
  CK(cudaMemcpyAsync(h->bh, h_b, sizeof(double) * h->m, cudaMemcpyHostToDevice, st));
  h->solver = 0;
  rc = solve_device(h, h->bh, damp, atol, btol, max_iters, h->xh, res, nullptr, nullptr, st);
  if (rc != TOMO_OK) return rc;
  CK(cudaMemcpyAsync(h_x, h->xh, sizeof(double) * h->n, cudaMemcpyDeviceToHost, st));
  CK(cudaStreamSynchronize(st));
  return TOMO_OK;
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

template <int OP>
void launch_spmm(const tomo_lsqr_s* h, bool transpose, const double* X, double* Y, cudaStream_t st) {
  const int64_t* ptr = transpose ? h->colptr : h->rowptr;
  const int32_t* idx = transpose ? h->rowind : h->colind;
  const int32_t* part = transpose ? h->mpart_c : h->mpart_r;
  if (h->vt == TOMO_VAL_F64) {
    const double* val = (const double*)(transpose ? h->cvals : h->vals);
    if (h->accumulate) k_spmm8<1, double, OP><<<h->MG, kMThreads, 0, st>>>(ptr, idx, val, X, Y, part, h->msc, h->mpartials);
    else k_spmm8<0, double, OP><<<h->MG, kMThreads, 0, st>>>(ptr, idx, val, X, Y, part, h->msc, h->mpartials);
  } else {
    const float* val = (const float*)(transpose ? h->cvals : h->vals);
    if (h->accumulate) k_spmm8<1, float, OP><<<h->MG, kMThreads, 0, st>>>(ptr, idx, val, X, Y, part, h->msc, h->mpartials);
    else k_spmm8<0, float, OP><<<h->MG, kMThreads, 0, st>>>(ptr, idx, val, X, Y, part, h->msc, h->mpartials);
  }
}

template <int VOP>
void launch_vec8(const tomo_lsqr_s* h, const double* in0, int nrhs, double* a0, double* a1, double* a2, int64_t len, cudaStream_t st) {
  const int g = (int)std::max<int64_t>(1, std::min<int64_t>((len * kR + kMThreads - 1) / kMThreads, (int64_t)h->MG));
  if (h->accumulate) k_vec8<1, VOP><<<g, kMThreads, 0, st>>>(in0, nrhs, a0, a1, a2, len, h->msc, h->mpartials);
  else k_vec8<0, VOP><<<g, kMThreads, 0, st>>>(in0, nrhs, a0, a1, a2, len, h->msc, h->mpartials);
}

void enqueue_multi_iteration(const tomo_lsqr_s* h, cudaStream_t st) {
  launch_spmm<OP_K1>(h, false, h->mV, h->mU, st);
  launch_spmm<OP_K2>(h, true, h->mU, h->mV, st);
  launch_vec8<VOP_K4>(h, nullptr, kR, h->mV, h->mW, h->mX, h->n, st);
}

// Eight recurrences sharing every pass over A and A^T (multi.cuh).  nrhs < 8 is padded with zero columns.
tomo_status_t solve_multi_shared(tomo_lsqr_s* h, int32_t nrhs, const double* d_B, double damp, double atol, double btol,
                                 int32_t max_iters, double* d_X, tomo_lsqr_result_t* res, cudaStream_t st) {
  const int64_t m = h->m, n = h->n;
  if (!h->mU) {
    CK(cudaMalloc(&h->mU, sizeof(double) * m * kR)); CK(cudaMalloc(&h->mV, sizeof(double) * n * kR));
    CK(cudaMalloc(&h->mW, sizeof(double) * n * kR)); CK(cudaMalloc(&h->mX, sizeof(double) * n * kR));
    CK(cudaMalloc(&h->msc, sizeof(Scalars) * kR)); CK(cudaMallocHost(&h->h_msc, sizeof(Scalars) * kR));
    h->MG = h->sms * 8;
    CK(cudaMalloc(&h->mpart_r, sizeof(int32_t) * (h->MG + 1))); CK(cudaMalloc(&h->mpart_c, sizeof(int32_t) * (h->MG + 1)));
    CK(cudaMalloc(&h->mpartials, sizeof(double2) * kR * h->MG));
    const int tb = 128, gb = (h->MG + 1 + tb - 1) / tb;
    k_partition<<<gb, tb, 0, st>>>(h->rowptr, m, h->MG, 16, 1, h->mpart_r);
    k_partition_fix<<<1, 32, 0, st>>>(h->MG, h->mpart_r);
    k_partition<<<gb, tb, 0, st>>>(h->colptr, n, h->MG, 16, 1, h->mpart_c);
    k_partition_fix<<<1, 32, 0, st>>>(h->MG, h->mpart_c);
    CK(cudaGetLastError());
  }
  const int k = h->check_every;
  if (h->use_graph && !(h->mgexec && h->mgraph_k == k && h->mgraph_mode == h->accumulate)) {
    if (h->mgexec) { cudaGraphExecDestroy(h->mgexec); h->mgexec = nullptr; }
    cudaGraph_t g = nullptr;
    CK(cudaStreamBeginCapture(h->cap_stream, cudaStreamCaptureModeRelaxed));
    for (int i = 0; i < k; ++i) enqueue_multi_iteration(h, h->cap_stream);
    cudaError_t e = cudaStreamEndCapture(h->cap_stream, &g);
    if (e != cudaSuccess) return cuda_fail(e, "cudaStreamEndCapture");
    e = cudaGraphInstantiate(&h->mgexec, g, 0);
    cudaGraphDestroy(g);
    if (e != cudaSuccess) { h->mgexec = nullptr; return cuda_fail(e, "cudaGraphInstantiate"); }
    h->mgraph_k = k; h->mgraph_mode = h->accumulate;
  }
  Scalars* hs = h->h_msc;
  memset(hs, 0, sizeof(Scalars) * kR);
  for (int r = 0; r < kR; ++r) { hs[r].damp = damp; hs[r].atol = atol; hs[r].btol = btol; hs[r].max_iters = max_iters; hs[r].cs2 = -1.0; }
  CK(cudaMemcpyAsync(h->msc, hs, sizeof(Scalars) * kR, cudaMemcpyHostToDevice, st));
  CK(cudaMemsetAsync(h->mX, 0, sizeof(double) * n * kR, st));
  CK(cudaMemsetAsync(h->mV, 0, sizeof(double) * n * kR, st));
  CK(cudaMemsetAsync(h->mW, 0, sizeof(double) * n * kR, st));
  launch_vec8<VOP_INIT_U>(h, d_B, nrhs, h->mU, nullptr, nullptr, m, st);
  launch_spmm<OP_K2_INIT>(h, true, h->mU, h->mV, st);
  launch_vec8<VOP_INIT_VW>(h, nullptr, kR, h->mV, h->mW, nullptr, n, st);
  CK(cudaGetLastError());
  h->kernels_enqueued += 3;
  const int chunks = max_iters > 0 ? (max_iters + k - 1) / k : 0;
  for (int c = 0; c < chunks; ++c) {
    if (h->use_graph) CK(cudaGraphLaunch(h->mgexec, st));
    else { for (int i = 0; i < k; ++i) enqueue_multi_iteration(h, st); CK(cudaGetLastError()); }
    h->kernels_enqueued += 3.0 * k;
    // poll: the eight {itn, istop, stop} words; stop when every side has stopped
    CK(cudaMemcpy2DAsync(h->h_msc, sizeof(Scalars), h->msc, sizeof(Scalars), sizeof(Scalars), kR, cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    bool all = true;
    for (int r = 0; r < kR; ++r) all = all && (h->h_msc[r].stop != 0);
    if (all) break;
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
  return TOMO_OK;
}

}  // namespace

extern "C" tomo_status_t tomo_lsqr_solve_multi(tomo_lsqr_t h, int32_t nrhs, const double* d_B, double damp, double atol,
                                               double btol, int32_t max_iters, double* d_X, tomo_lsqr_result_t* res,
                                               void* cuda_stream) {
  tomo_status_t rc = check_solve_args(h, damp, atol, btol, max_iters);
  if (rc != TOMO_OK) return rc;
  if (nrhs < 1 || nrhs > 8 || !d_B || !d_X) return TOMO_ERR_INVALID_ARG;
  if (!is_device_ptr(d_B) || !is_device_ptr(d_X)) return TOMO_ERR_NOT_DEVICE_PTR;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (h->multi_shared) return solve_multi_shared(h, nrhs, d_B, damp, atol, btol, max_iters, d_X, res, st);
  if (!h->bh) CK(cudaMalloc(&h->bh, sizeof(double) * h->m));
  if (!h->xh) CK(cudaMalloc(&h->xh, sizeof(double) * h->n));
  for (int r = 0; r < nrhs; ++r) {
    k_col_gather<<<vec_blocks(h, h->m), kThreads, 0, st>>>(d_B, nrhs, r, h->m, h->bh);
    h->solver = 0;
    rc = solve_device(h, h->bh, damp, atol, btol, max_iters, h->xh, res ? res + r : nullptr, nullptr, nullptr, st);
    if (rc != TOMO_OK) return rc;
    k_col_scatter<<<vec_blocks(h, h->n), kThreads, 0, st>>>(h->xh, nrhs, r, h->n, d_X);
  }
  CK(cudaGetLastError());
  CK(cudaStreamSynchronize(st));
  return TOMO_OK;
}

extern "C" tomo_status_t tomo_lsqr_spmv(tomo_lsqr_t h, int transpose, const double* d_in, double* d_out, void* cuda_stream) {
  if (!h || !d_in || !d_out || (transpose != 0 && transpose != 1)) return TOMO_ERR_INVALID_ARG;
  if (!is_device_ptr(d_in) || !is_device_ptr(d_out)) return TOMO_ERR_NOT_DEVICE_PTR;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  tomo_status_t rc = rebuild_partitions(h, st);
  if (rc != TOMO_OK) return rc;
  launch_spmv<OP_PLAIN>(h, transpose != 0, d_in, d_out, st);
  CK(cudaGetLastError());
  CK(cudaStreamSynchronize(st));
  return TOMO_OK;
}

extern "C" tomo_status_t tomo_lsqr_get_csc(tomo_lsqr_t h, int64_t* d_colptr, int32_t* d_rowind, void* d_cvals, void* cuda_stream) {
  if (!h) return TOMO_ERR_INVALID_ARG;
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
  else if (k == "accumulate") { if (value != 0 && value != 1) return TOMO_ERR_INVALID_ARG; if (h->accumulate != (int)value) h->part_dirty = true; h->accumulate = (int)value; }
  else if (k == "graph") { if (value != 0 && value != 1) return TOMO_ERR_INVALID_ARG; h->use_graph = (int)value; }
  else if (k == "profile") { if (value != 0 && value != 1) return TOMO_ERR_INVALID_ARG; h->profile = (int)value; }
  else if (k == "multi_shared") { if (value != 0 && value != 1) return TOMO_ERR_INVALID_ARG; h->multi_shared = (int)value; }
  else if (k == "row_cost") { if (value < 0 || value > 4096) return TOMO_ERR_INVALID_ARG; if (h->row_cost != (int)value) h->part_dirty = true; h->row_cost = (int)value; }
  else return TOMO_ERR_INVALID_ARG;
  return TOMO_OK;
}

extern "C" tomo_status_t tomo_lsqr_get_info(tomo_lsqr_t h, const char* key, double* out) {
  if (!h || !key || !out) return TOMO_ERR_INVALID_ARG;
  const std::string k(key);
  const double vb = h->vt == TOMO_VAL_F64 ? 8.0 : 4.0;
  if (k == "create_ms") *out = h->create_ms;
  else if (k == "transpose_ms") *out = h->transpose_ms;
  else if (k == "csc_bytes") *out = (double)h->nnz * (4.0 + vb) + 8.0 * (double)(h->n + 1);
  else if (k == "scratch_bytes") *out = h->scratch_bytes;
  else if (k == "blocks_rows" || k == "blocks_cols") *out = (double)h->SG;
  else if (k == "k1_ms") *out = h->k1_ms;
  else if (k == "k2_ms") *out = h->k2_ms;
  else if (k == "k4_ms") *out = h->k4_ms;
  else if (k == "k_launches") *out = h->k_launches;
  else if (k == "kernels_enqueued") *out = h->kernels_enqueued;
  else if (k.rfind("cta_busy@", 0) == 0) {  // busy cycles of CTA <i> in the most recent sparse-product launch
    const int i = atoi(k.c_str() + 9);
    if (i < 0 || i >= h->SG) return TOMO_ERR_INVALID_ARG;
    CtaRec r;
    CK(cudaMemcpy(&r, h->cta_rec + i, sizeof(CtaRec), cudaMemcpyDeviceToHost));
    *out = 16.0 * (double)r.pad;
  }
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
  }
  return "unknown status";
}
