// tmd_sort.cuh -- A2: load-balance ordering of the tracks (north_star: "tracks sorted by cluster
// count for warp load balance").  INSIDE windows of SORT_WINDOW consecutive tracks, tracks are ordered by (phase, length
// class descending): `phase` = (first residual index of the track) mod 16 is where the track's residuals start inside the
// 16-residual groups the decode kernel stages (tmd_decode.cuh).  The 32 tracks of a warp of the track-decode kernel then
// (a) run (almost) the same number of serial steps and (b) cross their group boundaries AT THE SAME STEP, so the refill
// of the staging buffers is one warp-uniform branch every 16 clusters instead of a divergent one on almost every cluster
// (measured: 87 % of the warp-steps executed the refill block before).  The tracks a block works on stay close together
// in the input arrays and in the intermediate records (a window of 8192 tracks spans a few MB of each stream).
// The permutation only decides which thread decodes which track: the output order is fixed by C5 and does not depend
// on it (ties inside a class are placed in arbitrary order).  Integer only.
#pragma once

#include "tmd_common.cuh"
#include "tmd_scan.cuh"

namespace tmd {

// Sort key = phase * LEN_CLASSES + (LEN_CLASSES - 1 - length class): 16 phases x 128 length classes.
// Length classes: exact below 64 clusters, 8 wide below 320, 64 wide below 1344, 4096 wide above (format maximum 65535).
constexpr uint32_t LEN_CLASSES = 128;
constexpr uint32_t LEN_BINS = 16 * LEN_CLASSES;
constexpr int SORT_THREADS = 1024;
constexpr int SORT_ITEMS = 8;

__device__ __forceinline__ uint32_t len_class(uint32_t ncl) {
  if (ncl < 64u) return ncl;
  if (ncl < 320u) return 64u + ((ncl - 64u) >> 3);
  if (ncl < 1344u) return 96u + ((ncl - 320u) >> 6);
  return 112u + min(15u, (ncl - 1344u) >> 12);
}

// A window holds SORT_WINDOW_BLOCKS x SORT_BLOCK_TRACKS consecutive tracks: large enough that each of the 16 phases still
// holds thousands of tracks to order by length (32 tracks of one phase and one narrow length range per warp need
// 16 x 32 x (number of length ranges) tracks).  Three small kernels: per-window key histogram (k_sort_count), its exclusive
// scan (k_sort_scan), placement (k_sort_place: a block reserves its range of every key with one atomic per key; the order
// inside a key is arbitrary).
constexpr uint32_t SORT_BLOCK_TRACKS = SORT_THREADS * SORT_ITEMS;     // 8192
constexpr uint32_t SORT_WINDOW_BLOCKS = 8;
constexpr uint32_t SORT_WINDOW = SORT_BLOCK_TRACKS * SORT_WINDOW_BLOCKS;

__device__ __forceinline__ uint32_t sort_key(const uint32_t* __restrict__ off, const uint16_t* __restrict__ trk_ncl, uint32_t t) {
  const uint32_t phase = (off[t] - t) & 15u;                           // first residual index of the track, mod the group size
  return phase * LEN_CLASSES + (LEN_CLASSES - 1u - len_class(trk_ncl[t]));
}

// ghist[window][key] += tracks of this block with that key   (ghist zeroed before)
template <bool BATCH>
__global__ void __launch_bounds__(SORT_THREADS) k_sort_count(const __grid_constant__ FrameArgs F0, const FrameArgs* __restrict__ table) {
  __shared__ uint32_t h[LEN_BINS];
  static_assert(LEN_BINS == 2 * SORT_THREADS, "two keys per thread");
  const FrameArgs& F = frame_of<BATCH>(F0, table, blockIdx.y);
  const uint32_t n_tracks = F.in.n_tracks, base = blockIdx.x * SORT_BLOCK_TRACKS;
  if (base >= n_tracks) return;
  const uint32_t* __restrict__ off = F.at<uint32_t>(F.W.o_off);
  uint32_t* __restrict__ ghist = F.at<uint32_t>(F.W.o_sort_hist) + (size_t)(blockIdx.x / SORT_WINDOW_BLOCKS) * LEN_BINS;
  h[threadIdx.x] = 0;
  h[threadIdx.x + SORT_THREADS] = 0;
  __syncthreads();
#pragma unroll
  for (int k = 0; k < SORT_ITEMS; ++k) {
    const uint32_t t = base + k * SORT_THREADS + threadIdx.x;
    if (t < n_tracks) atomicAdd(&h[sort_key(off, F.in.trk_ncl, t)], 1u);
  }
  __syncthreads();
#pragma unroll
  for (int k = 0; k < 2; ++k) {
    const uint32_t v = h[threadIdx.x + k * SORT_THREADS];
    if (v) atomicAdd(&ghist[threadIdx.x + k * SORT_THREADS], v);
  }
}

// one block per window: ghist[window][*] <- its exclusive scan (the first slot of every key inside the window)
template <bool BATCH>
__global__ void __launch_bounds__(SORT_THREADS) k_sort_scan(const __grid_constant__ FrameArgs F0, const FrameArgs* __restrict__ table) {
  __shared__ uint32_t ws[33];
  const FrameArgs& F = frame_of<BATCH>(F0, table, blockIdx.y);
  if (blockIdx.x * SORT_WINDOW >= F.in.n_tracks) return;
  uint32_t* __restrict__ g = F.at<uint32_t>(F.W.o_sort_hist) + (size_t)blockIdx.x * LEN_BINS;
  const uint32_t k0 = threadIdx.x * 2, v0 = g[k0], v1 = g[k0 + 1];
  uint32_t total;
  const uint32_t ex = block_excl_scan(v0 + v1, ws, &total);
  g[k0] = ex;
  g[k0 + 1] = ex + v0;
}

// placement: perm[window base + slot] = track
template <bool BATCH>
__global__ void __launch_bounds__(SORT_THREADS) k_sort_place(const __grid_constant__ FrameArgs F0, const FrameArgs* __restrict__ table) {
  __shared__ uint32_t h[LEN_BINS];
  const FrameArgs& F = frame_of<BATCH>(F0, table, blockIdx.y);
  const uint32_t n_tracks = F.in.n_tracks, base = blockIdx.x * SORT_BLOCK_TRACKS;
  if (base >= n_tracks) return;
  const uint32_t* __restrict__ off = F.at<uint32_t>(F.W.o_off);
  const uint32_t window = blockIdx.x / SORT_WINDOW_BLOCKS;
  uint32_t* __restrict__ gcur = F.at<uint32_t>(F.W.o_sort_hist) + (size_t)window * LEN_BINS;
  uint32_t* __restrict__ perm = F.at<uint32_t>(F.W.o_perm) + (size_t)window * SORT_WINDOW;
  h[threadIdx.x] = 0;
  h[threadIdx.x + SORT_THREADS] = 0;
  __syncthreads();
  uint32_t key[SORT_ITEMS], loc[SORT_ITEMS];
#pragma unroll
  for (int k = 0; k < SORT_ITEMS; ++k) {
    const uint32_t t = base + k * SORT_THREADS + threadIdx.x;
    key[k] = 0; loc[k] = 0;
    if (t < n_tracks) {
      key[k] = sort_key(off, F.in.trk_ncl, t);
      loc[k] = atomicAdd(&h[key[k]], 1u);
    }
  }
  __syncthreads();
#pragma unroll
  for (int k = 0; k < 2; ++k) {                         // reserve this block's range of every key it holds
    const uint32_t i = threadIdx.x + k * SORT_THREADS, v = h[i];
    h[i] = v ? atomicAdd(&gcur[i], v) : 0u;
  }
  __syncthreads();
#pragma unroll
  for (int k = 0; k < SORT_ITEMS; ++k) {
    const uint32_t t = base + k * SORT_THREADS + threadIdx.x;
    if (t < n_tracks) perm[h[key[k]] + loc[k]] = t;
  }
}

}  // namespace tmd
