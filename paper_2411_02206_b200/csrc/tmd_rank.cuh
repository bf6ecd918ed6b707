// tmd_rank.cuh -- A3 (count part): per-chunk histogram over bins and the rank of every attached cluster among the
// clusters of its chunk that fall in the same bin (ascending global attached index g).  Integer only.  The bins come
// from the geometry walk of the track-decode kernel (tmd_decode.cuh), which leaves bin(g) in its intermediate records.
//
// Together with the column scan (tmd_scan.cuh) this yields the canonical position of every attached cluster
// (DESIGN.md §3 reading 11):   position(g) = rel[chunk][bin] + rank16[g].
#pragma once

#include "tmd_common.cuh"
#include "tmd_scan.cuh"

namespace tmd {

struct RankArgs {
  const uint2* inter;           // [n_attached] intermediate records of the track-decode kernel; bin = .y >> 16
  uint16_t* hist;               // [n_chunks][n_bins]
  uint16_t* rank16;             // [n_attached]
  uint32_t n_attached;
};

constexpr int RANK_THREADS = 1024;

// One block per chunk c = the attached clusters g in [c << CHUNK_SHIFT, (c+1) << CHUNK_SHIFT).
// Dynamic shared memory: bin_of[CHUNK_WINDOW] u16, list[CHUNK_WINDOW] u16, cnt[n_bins] u32, start[n_bins] u32.
__global__ void __launch_bounds__(RANK_THREADS, 1) k_rank(DevGeo G, RankArgs A) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  uint16_t* bin_of = reinterpret_cast<uint16_t*>(smem_raw);
  uint16_t* list = bin_of + CHUNK_WINDOW;
  uint32_t* cnt = reinterpret_cast<uint32_t*>(list + CHUNK_WINDOW);
  uint32_t* start = cnt + G.n_bins;
  __shared__ uint32_t ws[33];

  const uint32_t c = blockIdx.x, tid = threadIdx.x, nth = blockDim.x, n_bins = G.n_bins;
  const uint32_t w0 = c << CHUNK_SHIFT;
  const uint32_t w1 = min(w0 + CHUNK_WINDOW, A.n_attached);
  const uint32_t n = w1 - w0;
  for (uint32_t b = tid; b < n_bins; b += nth) cnt[b] = 0;
  // 1. bins of the chunk's clusters in g order (the geometry walk A3 ran inside the track-decode kernel)
  for (uint32_t i = tid; i < n; i += nth) bin_of[i] = (uint16_t)(A.inter[w0 + i].y >> 16);
  __syncthreads();
  // 2. histogram of the chunk
  for (uint32_t i = tid; i < n; i += nth) {
    const uint16_t b = bin_of[i];
    if (b != BIN_INVALID) atomicAdd(&cnt[b], 1u);
  }
  __syncthreads();
  // 3. exclusive scan over bins -> start[b]; cnt[b] becomes the fill cursor; hist row out
  {
    const uint32_t per = (n_bins + nth - 1) / nth;
    const uint32_t b0 = tid * per, b1 = min(b0 + per, n_bins);
    uint32_t s = 0;
    for (uint32_t b = b0; b < b1; ++b) s += cnt[b];
    uint32_t total;
    uint32_t ex = block_excl_scan(s, ws, &total);
    for (uint32_t b = b0; b < b1; ++b) {
      const uint32_t h = cnt[b];
      start[b] = ex;
      cnt[b] = ex;
      ex += h;
    }
    __syncthreads();
    uint16_t* hist_row = A.hist + (size_t)c * n_bins;
    for (uint32_t b = tid; b < n_bins; b += nth) {
      const uint32_t e = (b + 1 < n_bins) ? start[b + 1] : total;
      hist_row[b] = (uint16_t)(e - start[b]);      // <= CHUNK_WINDOW = 32768
    }
  }
  __syncthreads();
  // 4. per-bin lists of local indices (arbitrary order inside a bin)
  for (uint32_t i = tid; i < n; i += nth) {
    const uint16_t b = bin_of[i];
    if (b != BIN_INVALID) list[atomicAdd(&cnt[b], 1u)] = (uint16_t)i;
  }
  __syncthreads();
  // 5. rank inside the bin = number of list entries with a smaller local index.  Short lists: one thread per bin.
  constexpr uint32_t LONG = 48;                  // at most CHUNK_WINDOW / (LONG+1) < 1024 bins are longer
  __shared__ uint16_t long_bins[1024];
  __shared__ uint32_t n_long;
  if (tid == 0) n_long = 0;
  __syncthreads();
  for (uint32_t b = tid; b < n_bins; b += nth) {
    const uint32_t s = start[b], e = cnt[b];
    if (e - s > LONG) {
      long_bins[atomicAdd(&n_long, 1u)] = (uint16_t)b;
      continue;
    }
    for (uint32_t k = s; k < e; ++k) {
      const uint16_t v = list[k];
      uint32_t r = 0;
      for (uint32_t m = s; m < e; ++m) r += (list[m] < v);
      bin_of[v] = (uint16_t)r;   // bin_of[v] is dead once its bin is ranked: reuse as the rank
    }
  }
  __syncthreads();
  // long lists (degenerate inputs): the whole block ranks one bin at a time
  for (uint32_t q = 0; q < n_long; ++q) {
    const uint32_t b = long_bins[q], s = start[b], e = cnt[b];
    for (uint32_t k = s + tid; k < e; k += nth) {
      const uint16_t v = list[k];
      uint32_t r = 0;
      for (uint32_t m = s; m < e; ++m) r += (list[m] < v);
      bin_of[v] = (uint16_t)r;
    }
  }
  __syncthreads();
  // 6. ranks out, coalesced
  for (uint32_t i = tid; i < n; i += nth) A.rank16[w0 + i] = bin_of[i];
}

}  // namespace tmd
