// compress.cuh — the run-compressed index of the structure-exploiting operator.
//
// Where the structure comes from: a data row of the tomography matrix is the sensitivity of one traveltime to the
// model, K_i = sum over ray nodes of lateral weight x depth kernel (Eq. 5), and the unknowns
// are numbered depth-fastest (Eq. 7): the entries of one lateral node are a RUN of consecutive column
// indices (12 at BASELINE configs 1-4).  In the CSC copy the <= nper rows of one station pair are adjacent, so
// row indices inside a column come in (shorter) runs too.  The library does not assume the structure: it
// encodes whatever runs the index array has; an index array without runs is stored at 4.6 B per element
// instead of 4 (and "compress" reports the size it got).
//
// Format, per tile of TILE consecutive elements (tiles are aligned to multiples of TILE, like the warp ranges
// of wstream.cuh), one record at byte offset coff[t] (16-byte aligned):
//     TILE/8 bytes   head bits, one 32-bit word per 32-element step: bit i = "element i starts a run":
//                    i == 0 (a head is forced at every step, so a step decodes without looking back) or
//                    idx[e] != idx[e-1] + 1
//     4 bytes per head: idx[e] - i + 32 for every head, in element order (biased by its position i in the step, so
//                    that the lane adds only its own lane number, and by 32 to stay non-negative); padded to 16 bytes.
// Decoding (k_wstream, FMT 1): r = popc(H & lanes <= mine) counts the heads up to and including mine, the last
// of them is my run's head: index = heads[heads before this step + r - 1] - 32 + lane.  One popc, one shared load.
// Runs may cross row boundaries: row membership comes from the row pointers, not from the index stream.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace tomo {

// one warp per tile: bytes of the tile's record
template <int TILE>
__global__ void k_cz_size(const int32_t* __restrict__ idx, int64_t nnz, int64_t ntiles, int64_t* __restrict__ size) {
  const int lane = threadIdx.x & 31;
  const int64_t warp0 = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int64_t nwarps = ((int64_t)gridDim.x * blockDim.x) >> 5;
  for (int64_t t = warp0; t < ntiles; t += nwarps) {
    int heads = 0;
    for (int s = 0; s < TILE / 32; ++s) {
      const int64_t e = t * TILE + 32 * s + lane;
      bool cont = true;  // elements behind the end of the array: no head
      if (e < nnz) cont = (lane != 0) && (idx[e] == idx[e - 1] + 1);
      heads += __popc(__ballot_sync(0xffffffffu, !cont));
    }
    if (lane == 0) size[t] = (int64_t)((TILE / 8 + 4 * heads + 15) & ~15);
  }
}

// one warp per tile: flags and heads
template <int TILE>
__global__ void k_cz_fill(const int32_t* __restrict__ idx, int64_t nnz, int64_t ntiles, const int64_t* __restrict__ coff,
                          unsigned char* __restrict__ out) {
  const int lane = threadIdx.x & 31;
  const int64_t warp0 = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int64_t nwarps = ((int64_t)gridDim.x * blockDim.x) >> 5;
  for (int64_t t = warp0; t < ntiles; t += nwarps) {
    uint32_t* flags = reinterpret_cast<uint32_t*>(out + coff[t]);
    int32_t* heads = reinterpret_cast<int32_t*>(out + coff[t] + TILE / 8);
    int hb = 0;
    for (int s = 0; s < TILE / 32; ++s) {
      const int64_t e = t * TILE + 32 * s + lane;
      bool cont = true;
      int32_t c = 0;
      if (e < nnz) { c = idx[e]; cont = (lane != 0) && (c == idx[e - 1] + 1); }
      const unsigned H = __ballot_sync(0xffffffffu, !cont);
      if (lane == 0) flags[s] = H;
      if (!cont) heads[hb + __popc(H & ((1u << lane) - 1u))] = c - lane + 32;
      hb += __popc(H);
    }
    // padding words of the record stay unwritten: they are never read (only copied)
  }
}

}  // namespace tomo
