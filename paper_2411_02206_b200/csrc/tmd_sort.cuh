// tmd_sort.cuh -- A2: load-balance ordering of the tracks (north_star: "tracks sorted by cluster
// count for warp load balance").  A counting sort of the tracks by trk_ncl, longest first, so that the 32 tracks of a
// warp of the track-decode kernel run (almost) the same number of serial steps and the long tracks start first.
// The permutation only decides which thread decodes which track: the output order is fixed by C5 and does not depend
// on it (ties inside a length class are placed in arbitrary order).  Integer only.
#pragma once

#include "tmd_common.cuh"
#include "tmd_scan.cuh"

namespace tmd {

// Length classes: exact below 1024 clusters, 64 clusters wide above (format maximum 65535).
constexpr uint32_t LEN_BINS = 2048;
constexpr int SORT_THREADS = 512;
constexpr int SORT_ITEMS = 8;
constexpr int SORT_TILE = SORT_THREADS * SORT_ITEMS;

__device__ __forceinline__ uint32_t len_class(uint32_t ncl) { return ncl < 1024u ? ncl : 1024u + (ncl >> 6); }

// pass 1: len_hist[class] += tracks of the tile in the class (shared-memory histogram, one global atomic per non-empty class)
__global__ void __launch_bounds__(SORT_THREADS) k_len_hist(const uint16_t* __restrict__ trk_ncl, uint32_t n_tracks,
                                                         uint32_t* __restrict__ len_hist) {
  __shared__ uint32_t h[LEN_BINS];
  for (uint32_t b = threadIdx.x; b < LEN_BINS; b += SORT_THREADS) h[b] = 0;
  __syncthreads();
  const uint32_t base = blockIdx.x * SORT_TILE;
#pragma unroll
  for (int k = 0; k < SORT_ITEMS; ++k) {
    const uint32_t t = base + k * SORT_THREADS + threadIdx.x;
    if (t < n_tracks) atomicAdd(&h[len_class(trk_ncl[t])], 1u);
  }
  __syncthreads();
  for (uint32_t b = threadIdx.x; b < LEN_BINS; b += SORT_THREADS)
    if (h[b]) atomicAdd(&len_hist[b], h[b]);
}

// pass 2 (one block): len_base[class] = number of tracks in longer classes (descending order); cursor cleared
__global__ void __launch_bounds__(1024) k_len_scan(const uint32_t* __restrict__ len_hist, uint32_t* __restrict__ len_base,
                                                   uint32_t* __restrict__ len_cursor) {
  __shared__ uint32_t ws[33];
  static_assert(LEN_BINS == 2048, "two classes per thread");
  const uint32_t d0 = threadIdx.x * 2, d1 = d0 + 1;              // position in descending order
  const uint32_t c0 = LEN_BINS - 1 - d0, c1 = LEN_BINS - 1 - d1;  // class
  const uint32_t v0 = len_hist[c0], v1 = len_hist[c1];
  uint32_t total;
  const uint32_t ex = block_excl_scan(v0 + v1, ws, &total);
  len_base[c0] = ex;
  len_base[c1] = ex + v0;
  len_cursor[c0] = 0;
  len_cursor[c1] = 0;
}

// pass 3: perm[slot] = track; slot = len_base[class] + (a range reserved per block and class) + (rank inside the block)
__global__ void __launch_bounds__(SORT_THREADS) k_len_perm(const uint16_t* __restrict__ trk_ncl, uint32_t n_tracks,
                                                         const uint32_t* __restrict__ len_base, uint32_t* __restrict__ len_cursor,
                                                         uint32_t* __restrict__ perm) {
  __shared__ uint32_t h[LEN_BINS];
  for (uint32_t b = threadIdx.x; b < LEN_BINS; b += SORT_THREADS) h[b] = 0;
  __syncthreads();
  const uint32_t base = blockIdx.x * SORT_TILE;
  uint32_t cls[SORT_ITEMS], loc[SORT_ITEMS];
#pragma unroll
  for (int k = 0; k < SORT_ITEMS; ++k) {
    const uint32_t t = base + k * SORT_THREADS + threadIdx.x;
    cls[k] = 0; loc[k] = 0;
    if (t < n_tracks) {
      cls[k] = len_class(trk_ncl[t]);
      loc[k] = atomicAdd(&h[cls[k]], 1u);
    }
  }
  __syncthreads();
  for (uint32_t b = threadIdx.x; b < LEN_BINS; b += SORT_THREADS) {
    const uint32_t c = h[b];
    if (c) h[b] = len_base[b] + atomicAdd(&len_cursor[b], c);
  }
  __syncthreads();
#pragma unroll
  for (int k = 0; k < SORT_ITEMS; ++k) {
    const uint32_t t = base + k * SORT_THREADS + threadIdx.x;
    if (t < n_tracks) perm[h[cls[k]] + loc[k]] = t;
  }
}

}  // namespace tmd
