// tmd_scan.cuh -- prefix sums of the decoder: track offsets (A1), chunk table, column scan over chunks and bin
// offsets (A4).  Integer only.
#pragma once

#include "tmd_common.cuh"

namespace tmd {

__device__ __forceinline__ uint32_t warp_incl_scan(uint32_t v) {
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    uint32_t n = __shfl_up_sync(0xffffffffu, v, o);
    if (lane_id() >= (uint32_t)o) v += n;
  }
  return v;
}

// Exclusive scan of one value per thread over the block; returns the exclusive prefix, *total = block sum.
// `ws` = 33 words of shared memory.  Contains __syncthreads (all threads must call).
__device__ __forceinline__ uint32_t block_excl_scan(uint32_t v, uint32_t* ws, uint32_t* total) {
  const uint32_t lane = lane_id(), wid = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
  uint32_t inc = warp_incl_scan(v);
  __syncthreads();  // protect ws from a previous call
  if (lane == 31) ws[wid] = inc;
  __syncthreads();
  if (wid == 0) {
    uint32_t s = lane < nw ? ws[lane] : 0;
    uint32_t si = warp_incl_scan(s);
    ws[lane] = si - s;
    if (lane == 31) ws[32] = si;
  }
  __syncthreads();
  *total = ws[32];
  return ws[wid] + inc - v;
}

// The same for TWO values per thread with one set of barriers (the unattached decode scans pad and time sums together).
// `ws` = 66 words of shared memory.
__device__ __forceinline__ void block_excl_scan2(uint32_t a, uint32_t b, uint32_t* ws, uint32_t* ex_a, uint32_t* ex_b, uint32_t* tot_a,
                                                 uint32_t* tot_b) {
  const uint32_t lane = lane_id(), wid = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
  const uint32_t ia = warp_incl_scan(a), ib = warp_incl_scan(b);
  __syncthreads();  // protect ws from a previous call
  if (lane == 31) { ws[wid] = ia; ws[33 + wid] = ib; }
  __syncthreads();
  if (wid == 0) {
    const uint32_t sa = lane < nw ? ws[lane] : 0, sb = lane < nw ? ws[33 + lane] : 0;
    const uint32_t sia = warp_incl_scan(sa), sib = warp_incl_scan(sb);
    ws[lane] = sia - sa; ws[33 + lane] = sib - sb;
    if (lane == 31) { ws[32] = sia; ws[65] = sib; }
  }
  __syncthreads();
  *tot_a = ws[32]; *tot_b = ws[65];
  *ex_a = ws[wid] + ia - a; *ex_b = ws[33 + wid] + ib - b;
}

// ---- A1: off[t] = exclusive prefix sum of trk_ncl (PAPER.md L70 precomputes these indices on the CPU) --------------
constexpr int SCAN_THREADS = 512;
constexpr int SCAN_ITEMS = 8;
constexpr int SCAN_TILE = SCAN_THREADS * SCAN_ITEMS;

template <bool BATCH>
__global__ void __launch_bounds__(SCAN_THREADS) k_track_tile_sums(const __grid_constant__ FrameArgs F0, const FrameArgs* __restrict__ table) {
  __shared__ uint32_t ws[33];
  const FrameArgs& F = frame_of<BATCH>(F0, table, blockIdx.y);
  if (blockIdx.x >= F.W.n_tiles) return;
  const uint16_t* __restrict__ trk_ncl = F.in.trk_ncl;
  const uint32_t n_tracks = F.in.n_tracks;
  uint32_t* __restrict__ tile_sum = F.at<uint32_t>(F.W.o_tile_sum);
  const uint32_t base = blockIdx.x * SCAN_TILE + threadIdx.x * SCAN_ITEMS;
  uint32_t s = 0;
  if (base + SCAN_ITEMS <= n_tracks) {
    uint4 v = *reinterpret_cast<const uint4*>(trk_ncl + base);  // 8 x u16, 16-byte aligned
    s = (v.x & 0xFFFFu) + (v.x >> 16) + (v.y & 0xFFFFu) + (v.y >> 16) + (v.z & 0xFFFFu) + (v.z >> 16) + (v.w & 0xFFFFu) + (v.w >> 16);
  } else {
    for (uint32_t i = base; i < n_tracks && i < base + SCAN_ITEMS; ++i) s += trk_ncl[i];
  }
  uint32_t total;
  block_excl_scan(s, ws, &total);
  if (threadIdx.x == 0) tile_sum[blockIdx.x] = total;
}

// single block: exclusive scan of tile_sum in place; tile_sum[n_tiles] = grand total
template <bool BATCH>
__global__ void __launch_bounds__(1024) k_scan_tile_sums(const __grid_constant__ FrameArgs F0, const FrameArgs* __restrict__ table) {
  __shared__ uint32_t ws[33];
  const FrameArgs& F = frame_of<BATCH>(F0, table, blockIdx.y);
  uint32_t* __restrict__ tile_sum = F.at<uint32_t>(F.W.o_tile_sum);
  const uint32_t n_tiles = F.W.n_tiles;
  if (n_tiles == 0) return;
  uint32_t carry = 0;
  for (uint32_t base = 0; base < n_tiles; base += blockDim.x) {
    uint32_t i = base + threadIdx.x;
    uint32_t v = i < n_tiles ? tile_sum[i] : 0, total;
    uint32_t ex = block_excl_scan(v, ws, &total);
    if (i < n_tiles) tile_sum[i] = carry + ex;
    carry += total;
  }
  if (threadIdx.x == 0) tile_sum[n_tiles] = carry;
}

// off[t] for every track; off[n_tracks] = total
template <bool BATCH>
__global__ void __launch_bounds__(SCAN_THREADS) k_track_offsets(const __grid_constant__ FrameArgs F0, const FrameArgs* __restrict__ table) {
  __shared__ uint32_t ws[33];
  const FrameArgs& F = frame_of<BATCH>(F0, table, blockIdx.y);
  const uint32_t n_tiles = F.W.n_tiles;
  if (blockIdx.x >= n_tiles) return;
  const uint16_t* __restrict__ trk_ncl = F.in.trk_ncl;
  const uint32_t n_tracks = F.in.n_tracks;
  const uint32_t* __restrict__ tile_sum = F.at<uint32_t>(F.W.o_tile_sum);
  uint32_t* __restrict__ off = F.at<uint32_t>(F.W.o_off);
  const uint32_t base = blockIdx.x * SCAN_TILE + threadIdx.x * SCAN_ITEMS;
  uint32_t v[SCAN_ITEMS], s = 0;
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; ++k) {
    v[k] = (base + k < n_tracks) ? trk_ncl[base + k] : 0;
    s += v[k];
  }
  uint32_t total;
  uint32_t run = tile_sum[blockIdx.x] + block_excl_scan(s, ws, &total);
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; ++k) {
    if (base + k < n_tracks) off[base + k] = run;
    run += v[k];
  }
  if (blockIdx.x == n_tiles - 1 && threadIdx.x == 0) off[n_tracks] = tile_sum[n_tiles];
}

// ---- A4 part 1: column sums over groups of chunks ---------------------------------------------------------------------
// hist[c][b] (u16) = attached clusters of chunk c in bin b.   gsum[grp][b] = sum over the group's chunks.
template <bool BATCH>
__global__ void __launch_bounds__(256) k_col_group_sums(uint32_t n_bins, const __grid_constant__ FrameArgs F0, const FrameArgs* __restrict__ table) {
  const FrameArgs& F = frame_of<BATCH>(F0, table, blockIdx.z);
  const uint32_t b = blockIdx.x * blockDim.x + threadIdx.x, grp = blockIdx.y;
  const uint32_t n_chunks = F.W.n_chunks;
  if (b >= n_bins || grp >= F.W.n_groups) return;
  const uint16_t* __restrict__ hist = F.at<uint16_t>(F.W.o_hist);
  uint32_t* __restrict__ gsum = F.at<uint32_t>(F.W.o_gsum);
  const uint32_t c0 = grp * COL_GROUP, c1 = min(c0 + COL_GROUP, n_chunks);
  uint32_t s = 0;
#pragma unroll 8
  for (uint32_t c = c0; c < c1; ++c) s += hist[(size_t)c * n_bins + b];
  gsum[(size_t)grp * n_bins + b] = s;
}

// per bin: exclusive scan of gsum over groups (in place), att_cnt[b] = total
template <bool BATCH>
__global__ void __launch_bounds__(256) k_col_group_scan(uint32_t n_bins, const __grid_constant__ FrameArgs F0, const FrameArgs* __restrict__ table) {
  const FrameArgs& F = frame_of<BATCH>(F0, table, blockIdx.y);
  const uint32_t b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= n_bins) return;
  uint32_t* __restrict__ gsum = F.at<uint32_t>(F.W.o_gsum);
  uint32_t* __restrict__ att_cnt = F.at<uint32_t>(F.W.o_att_cnt);
  const uint32_t n_groups = F.W.n_groups;
  uint32_t run = 0;
  uint32_t g = 0;
  for (; g + 8 <= n_groups; g += 8) {
    uint32_t v[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) v[k] = gsum[(size_t)(g + k) * n_bins + b];
#pragma unroll
    for (int k = 0; k < 8; ++k) {
      gsum[(size_t)(g + k) * n_bins + b] = run;
      run += v[k];
    }
  }
  for (; g < n_groups; ++g) {
    uint32_t v = gsum[(size_t)g * n_bins + b];
    gsum[(size_t)g * n_bins + b] = run;
    run += v;
  }
  att_cnt[b] = run;
}

// single block: bin_offset[b] = exclusive scan of att_cnt[b] + u_cnt[b]; u_start[b] = exclusive scan of u_cnt[b]
// (C5: a bin holds its attached clusters first, then its unattached ones).  totals[0] = sum u_cnt.
template <bool BATCH>
__global__ void __launch_bounds__(1024) k_bin_offsets(uint32_t n_bins, const __grid_constant__ FrameArgs F0, const FrameArgs* __restrict__ table) {
  __shared__ uint32_t ws[33];
  const FrameArgs& F = frame_of<BATCH>(F0, table, blockIdx.y);
  const uint32_t* __restrict__ att_cnt = F.at<uint32_t>(F.W.o_att_cnt);
  const uint32_t* __restrict__ u_cnt = F.in.u_bin_count;
  uint32_t* __restrict__ bin_offset = F.bin_offset;
  uint32_t* __restrict__ u_start = F.at<uint32_t>(F.W.o_u_start);
  const uint32_t per = (n_bins + blockDim.x - 1) / blockDim.x;
  const uint32_t b0 = threadIdx.x * per, b1 = min(b0 + per, n_bins);
  uint32_t sa = 0, su = 0;
  for (uint32_t b = b0; b < b1; ++b) {
    su += u_cnt[b];
    sa += att_cnt[b] + u_cnt[b];
  }
  uint32_t ta, tu;
  uint32_t ea = block_excl_scan(sa, ws, &ta);
  uint32_t eu = block_excl_scan(su, ws, &tu);
  for (uint32_t b = b0; b < b1; ++b) {
    bin_offset[b] = ea;
    u_start[b] = eu;
    eu += u_cnt[b];
    ea += att_cnt[b] + u_cnt[b];
  }
  if (threadIdx.x == 0) {
    bin_offset[n_bins] = ta;
    u_start[n_bins] = tu;
  }
}

// ---- A4 part 2: rel[c][b] = bin_offset[b] + attached clusters of bin b in chunks < c ---------------------------------
template <bool BATCH>
__global__ void __launch_bounds__(256) k_col_apply(uint32_t n_bins, const __grid_constant__ FrameArgs F0, const FrameArgs* __restrict__ table) {
  const FrameArgs& F = frame_of<BATCH>(F0, table, blockIdx.z);
  const uint32_t b = blockIdx.x * blockDim.x + threadIdx.x, grp = blockIdx.y;
  const uint32_t n_chunks = F.W.n_chunks;
  if (b >= n_bins || grp >= F.W.n_groups) return;
  const uint16_t* __restrict__ hist = F.at<uint16_t>(F.W.o_hist);
  const uint32_t* __restrict__ gsum = F.at<uint32_t>(F.W.o_gsum);
  const uint32_t* __restrict__ bin_offset = F.bin_offset;
  uint32_t* __restrict__ rel = F.at<uint32_t>(F.W.o_rel);
  const uint32_t c0 = grp * COL_GROUP, c1 = min(c0 + COL_GROUP, n_chunks);
  uint32_t run = bin_offset[b] + gsum[(size_t)grp * n_bins + b];
#pragma unroll 8
  for (uint32_t c = c0; c < c1; ++c) {
    const uint32_t h = hist[(size_t)c * n_bins + b];
    rel[(size_t)c * n_bins + b] = run;
    run += h;
  }
}

}  // namespace tmd
