// build.cuh — one-off device work of tomo_lsqr_create: CSR validation, the stable
// CSR -> CSC transpose, and the nnz-balanced static partitions of rows and columns.  Integer work
// only; nothing here depends on thread timing, so two creates give byte-identical CSC arrays.
//
// Transpose (no sort, no key/value buffers): the rows are cut into T contiguous chunks, one per warp.
//   pass A  cnt[t][j]  = number of entries of chunk t in column j           (integer atomics: exact)
//   pass B  per column j, an exclusive scan of cnt[.][j] over t  (+ the column total)
//   scan    colptr = exclusive scan of the column totals
//   pass C  warp t walks ITS rows in order; inside a row the columns are distinct (canonical CSR), so
//           the lanes bump distinct cursors cnt[t][col] without atomics; rows of a chunk are sequential
//           and chunks are ordered, hence entries land in ascending row order inside every column.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace tomo {

enum : int { BAD_PTR0 = 1, BAD_PTR_END = 2, BAD_PTR_ORDER = 4, BAD_COL_RANGE = 8, BAD_COL_ORDER = 16, BAD_VALUE = 32 };

template <typename VT>
__global__ void k_validate(int64_t m, int64_t n, int64_t nnz, const int64_t* __restrict__ ptr,
                           const int32_t* __restrict__ idx, const VT* __restrict__ val, int* flags) {
  const int lane = threadIdx.x & 31;
  const int64_t warp0 = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int64_t nwarps = ((int64_t)gridDim.x * blockDim.x) >> 5;
  int bad = 0;
  if (warp0 == 0 && lane == 0) {
    if (ptr[0] != 0) bad |= BAD_PTR0;
    if (ptr[m] != nnz) bad |= BAD_PTR_END;
  }
  for (int64_t r = warp0; r < m; r += nwarps) {
    int64_t s = ptr[r], e = ptr[r + 1];
    if (s > e || s < 0 || e > nnz) { bad |= BAD_PTR_ORDER; continue; }
    for (int64_t q = s + lane; q < e; q += 32) {
      int32_t c = idx[q];
      if (c < 0 || (int64_t)c >= n) bad |= BAD_COL_RANGE;
      if (q > s && idx[q - 1] >= c) bad |= BAD_COL_ORDER;
      double v = (double)val[q];
      if (!(fabs(v) <= 1.79769313486231570815e308)) bad |= BAD_VALUE;
    }
  }
  if (bad) atomicOr(flags, bad);
}

// part[b], b = 0..G: first row of block b.  Rows are weighed  len + c0  (c0: fixed per-row overhead in
// nnz units); f(i) = ptr[i] + c0*i is the prefix of that weight, so a split point is a binary search.
__global__ void k_partition(const int64_t* __restrict__ ptr, int64_t nrows, int G, int c0, int align, int32_t* part) {
  int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b > G) return;
  if (b == 0) { part[0] = 0; return; }
  if (b == G) { part[G] = (int32_t)nrows; return; }
  const double total = (double)ptr[nrows] + (double)c0 * (double)nrows;
  const double target = total * ((double)b / (double)G);
  int64_t lo = 0, hi = nrows;  // smallest i with f(i) >= target
  while (lo < hi) {
    int64_t mid = (lo + hi) >> 1;
    double f = (double)ptr[mid] + (double)c0 * (double)mid;
    if (f >= target) hi = mid; else lo = mid + 1;
  }
  int64_t r = (lo / align) * align;
  part[b] = (int32_t)r;
}

// monotone clean-up after alignment (rounding can only move a split down, so order is preserved, but
// make the invariant explicit)
__global__ void k_partition_fix(int G, int32_t* part) {
  if (blockIdx.x == 0 && threadIdx.x == 0)
    for (int b = 1; b <= G; ++b)
      if (part[b] < part[b - 1]) part[b] = part[b - 1];
}

// pass A
__global__ void k_tr_count(const int64_t* __restrict__ ptr, const int32_t* __restrict__ idx,
                           const int32_t* __restrict__ chunk, int T, int64_t n, uint32_t* cnt) {
  const int lane = threadIdx.x & 31;
  const int t = (int)(((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5);
  if (t >= T) return;
  const int64_t s = ptr[chunk[t]], e = ptr[chunk[t + 1]];
  uint32_t* my = cnt + (int64_t)t * n;
  for (int64_t q = s + lane; q < e; q += 32) atomicAdd(my + idx[q], 1u);
}

// pass B: thread j scans cnt[0..T)[j] (eight independent loads in flight); coltotal[j] = column length
__global__ void k_tr_colscan(int T, int64_t n, uint32_t* cnt, int64_t* coltotal) {
  const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= n) return;
  uint32_t run = 0;
  int t = 0;
  for (; t + 8 <= T; t += 8) {
    uint32_t c[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) c[u] = cnt[(int64_t)(t + u) * n + j];
#pragma unroll
    for (int u = 0; u < 8; ++u) { cnt[(int64_t)(t + u) * n + j] = run; run += c[u]; }
  }
  for (; t < T; ++t) {
    const uint32_t c = cnt[(int64_t)t * n + j];
    cnt[(int64_t)t * n + j] = run;
    run += c;
  }
  coltotal[j] = (int64_t)run;
}

// exclusive scan of in[0..len) -> out[0..len], out[len] = total; single block of 1024 threads
__global__ void __launch_bounds__(1024) k_exscan(const int64_t* __restrict__ in, int64_t len, int64_t* out) {
  __shared__ int64_t s_sum[1024];
  const int t = threadIdx.x;
  const int64_t per = (len + 1023) / 1024;
  const int64_t b = min((int64_t)t * per, len), e = min(b + per, len);
  int64_t acc = 0;
  for (int64_t i = b; i < e; ++i) acc += in[i];
  s_sum[t] = acc;
  __syncthreads();
  if (t == 0) {
    int64_t run = 0;
    for (int k = 0; k < 1024; ++k) { int64_t v = s_sum[k]; s_sum[k] = run; run += v; }
    out[len] = run;
  }
  __syncthreads();
  acc = s_sum[t];
  for (int64_t i = b; i < e; ++i) { int64_t v = in[i]; out[i] = acc; acc += v; }
}

// pass C.  pos (optional): pos[q] = CSC slot of CSR element q, the permutation tomo_lsqr_update_values replays;
// rowind / cvals may be NULL when only the permutation is wanted.
template <typename VT, typename PT>
__global__ void k_tr_scatter(const int64_t* __restrict__ ptr, const int32_t* __restrict__ idx,
                             const VT* __restrict__ val, const int32_t* __restrict__ chunk, int T, int64_t n,
                             uint32_t* cnt, const int64_t* __restrict__ colptr, int32_t* rowind, VT* cvals, PT* pos) {
  const int lane = threadIdx.x & 31;
  const int t = (int)(((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5);
  if (t >= T) return;
  uint32_t* my = cnt + (int64_t)t * n;
  for (int r = chunk[t]; r < chunk[t + 1]; ++r) {
    const int64_t s = ptr[r], e = ptr[r + 1];
    for (int64_t q = s + lane; q < e; q += 32) {
      const int32_t c = idx[q];
      const uint32_t k = __ldcg(my + c);
      __stcg(my + c, k + 1u);
      const int64_t d = colptr[c] + (int64_t)k;
      if (rowind) { rowind[d] = r; cvals[d] = val[q]; }
      if (pos) pos[q] = (PT)d;
    }
    __syncwarp();
  }
}

// NEXT-4 (every outer iteration re-evaluates G on the same rays and solves
// again): new values in CSR order go to their CSC slots.  Consecutive rows of one station pair hit adjacent slots
// of the same columns, so the 8-byte scattered writes merge in L2.
template <typename VT, typename PT>
__global__ void k_update_values(const VT* __restrict__ val, const PT* __restrict__ pos, int64_t nnz, VT* __restrict__ cvals) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; q < nnz; q += stride) cvals[pos[q]] = val[q];
}

// all values finite? (the check create makes, for a refreshed value array)
template <typename VT>
__global__ void k_values_finite(const VT* __restrict__ val, int64_t nnz, int* flags) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  int bad = 0;
  for (int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; q < nnz; q += stride)
    if (!(fabs((double)val[q]) <= 1.79769313486231570815e308)) bad = BAD_VALUE;
  if (bad) atomicOr(flags, bad);
}

}  // namespace tomo
