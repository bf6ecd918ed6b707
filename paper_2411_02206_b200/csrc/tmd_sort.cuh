// tmd_sort.cuh -- A2: load-balance ordering of the tracks (north_star: "tracks sorted by cluster
// count for warp load balance").  Tracks are sorted by trk_ncl, longest first, INSIDE windows of SORT_WINDOW consecutive
// tracks: the 32 tracks of a warp of the track-decode kernel then run (almost) the same number of serial steps, while
// the tracks a block works on stay close together in the input arrays and in the intermediate records (a window of 8192
// tracks spans a few MB of each stream), which keeps the working set of pages small.
// The permutation only decides which thread decodes which track: the output order is fixed by C5 and does not depend
// on it (ties inside a length class are placed in arbitrary order).  Integer only.
// The kernel does not write the permutation itself but, in that order, a HEADER RECORD per track with everything the decode
// kernel needs to start it: hdr[p] = {off[t], t, trk_time0[t], trk_ncl[t] | trk_pad0[t] << 16} and
// hdr2[p] = trk_sec0[t] | trk_row0[t] << 8 | (uint8)trk_qpt[t] << 16.  A decode thread then starts with two coalesced loads
// instead of three dependent round trips (perm -> off / sector / row -> pad / time / q/pT, each a scattered sector):
// timestamps showed 10.6 us from block start to the first step of a 129 us block at c3.
#pragma once

#include "tmd_common.cuh"
#include "tmd_scan.cuh"

namespace tmd {

// Length classes: exact below 1024 clusters, 64 clusters wide above (format maximum 65535).
constexpr uint32_t LEN_BINS = 2048;
constexpr int SORT_THREADS = 1024;
constexpr int SORT_ITEMS = 8;
constexpr uint32_t SORT_WINDOW = SORT_THREADS * SORT_ITEMS;

__device__ __forceinline__ uint32_t len_class(uint32_t ncl) { return ncl < 1024u ? ncl : 1024u + (ncl >> 6); }

// One block per window: shared-memory counting sort by length class, descending.
template <bool BATCH>
__global__ void __launch_bounds__(SORT_THREADS) k_len_sort_window(const __grid_constant__ FrameArgs F0, const FrameArgs* __restrict__ table) {
  __shared__ uint32_t h[LEN_BINS];
  __shared__ uint32_t ws[33];
  static_assert(LEN_BINS == 2 * SORT_THREADS, "two classes per thread");
  const FrameArgs& F = frame_of<BATCH>(F0, table, blockIdx.y);
  const uint32_t n_tracks = F.in.n_tracks;
  if (blockIdx.x * SORT_WINDOW >= n_tracks) return;
  const uint16_t* __restrict__ trk_ncl = F.in.trk_ncl;
  uint4* __restrict__ hdr = F.at<uint4>(F.W.o_hdr);
  uint32_t* __restrict__ hdr2 = F.at<uint32_t>(F.W.o_hdr2);
  const uint32_t* __restrict__ off = F.at<uint32_t>(F.W.o_off);
  h[threadIdx.x] = 0;
  h[threadIdx.x + SORT_THREADS] = 0;
  __syncthreads();
  const uint32_t base = blockIdx.x * SORT_WINDOW;
  uint32_t cls[SORT_ITEMS], loc[SORT_ITEMS], ncl[SORT_ITEMS];
#pragma unroll
  for (int k = 0; k < SORT_ITEMS; ++k) {
    const uint32_t t = base + k * SORT_THREADS + threadIdx.x;
    cls[k] = 0; loc[k] = 0; ncl[k] = 0;
    if (t < n_tracks) {
      ncl[k] = trk_ncl[t];
      cls[k] = len_class(ncl[k]);
      loc[k] = atomicAdd(&h[cls[k]], 1u);
    }
  }
  __syncthreads();
  {  // h[class] <- number of tracks of the window in longer classes
    const uint32_t d0 = threadIdx.x * 2, d1 = d0 + 1;              // position in descending order
    const uint32_t c0 = LEN_BINS - 1 - d0, c1 = LEN_BINS - 1 - d1;  // class
    const uint32_t v0 = h[c0], v1 = h[c1];
    uint32_t total;
    const uint32_t ex = block_excl_scan(v0 + v1, ws, &total);
    h[c0] = ex;
    h[c1] = ex + v0;
  }
  __syncthreads();
#pragma unroll
  for (int k = 0; k < SORT_ITEMS; ++k) {
    const uint32_t t = base + k * SORT_THREADS + threadIdx.x;
    if (t < n_tracks) {
      const uint32_t p = base + h[cls[k]] + loc[k];
      hdr[p] = make_uint4(off[t], t, F.in.trk_time0[t], ncl[k] | ((uint32_t)F.in.trk_pad0[t] << 16));
      hdr2[p] = (uint32_t)F.in.trk_sec0[t] | ((uint32_t)F.in.trk_row0[t] << 8) | ((uint32_t)(uint8_t)F.in.trk_qpt[t] << 16);
    }
  }
}

}  // namespace tmd
