// tmd_rank.cuh -- A3 (count part): the per-chunk histogram over bins and the rank of every attached cluster among the
// clusters of its chunk that fall in the same bin (ascending global attached index g).  Integer only.  The bins come from
// the geometry walk of the track-decode kernel (tmd_decode.cuh), which leaves bin(g) in its intermediate records.
//
// Together with the column scan (tmd_scan.cuh) this yields the canonical position of every attached cluster
// (DESIGN.md §3 reading 11):   position(g) = rel[g >> chunk_shift][bin(g)] + rank16[g].
//
// Design: ONE WARP owns one chunk of 2^chunk_shift (32768 for a full time frame) consecutive clusters and goes through it in g order, 32 clusters at a time.
// Because a warp executes in order, the rank is a plain read-increment of a per-warp counter array in shared memory --
// no atomics, no sort, and the result is the sequential one by construction.  The 32 clusters are cut into runs of
// strictly ascending (or descending) bins, inside which all bins differ, so one conflict-free load / store round serves
// a run; consecutive clusters of a track lie on consecutive pad rows, so a round handles ~32 clusters (adversarial
// inputs degrade to one cluster per round, still exact).  The records of the next 16 groups are loaded while the
// current 16 are ranked.
#pragma once

#include "tmd_common.cuh"

namespace tmd {

constexpr int WR_WARPS = 4;                            // warps per block (each with its own chunk and counters)
constexpr int WR_THREADS = WR_WARPS * 32;
constexpr int WR_DEPTH = 16;                           // groups of 32 clusters loaded ahead

struct RankArgs {
  const uint2* inter;           // [n_attached] intermediate records of the track-decode kernel; bin = .y >> 16
  uint16_t* hist;               // [n_chunks][n_bins]
  uint16_t* rank16;             // [n_attached]
  uint16_t* start16;            // [n_chunks][start_stride] exclusive scan of the hist row; entry n_bins = clusters with a bin
  uint32_t n_attached, n_chunks, chunk_shift, start_stride;
};

// row stride (entries) of the start16 table: n_bins + 1 entries, padded to 16 bytes
__host__ __device__ inline uint32_t sc_start_stride(uint32_t n_bins) { return (n_bins + 1 + 7) & ~7u; }

__device__ __forceinline__ RankArgs rank_args(const FrameArgs& F, uint32_t n_bins) {
  RankArgs A;
  A.inter = F.at<uint2>(F.W.o_inter); A.hist = F.at<uint16_t>(F.W.o_hist); A.rank16 = F.at<uint16_t>(F.W.o_rank16);
  A.start16 = F.at<uint16_t>(F.W.o_start16);
  A.n_attached = (uint32_t)F.in.n_attached; A.n_chunks = F.W.n_chunks; A.chunk_shift = F.W.chunk_shift;
  A.start_stride = sc_start_stride(n_bins);
  return A;
}

// bytes of dynamic shared memory per warp: cnt u16[n_bins], padded to 16 bytes
__host__ __device__ inline uint32_t wr_warp_smem(uint32_t n_bins) { return (n_bins * 2 + 15) & ~15u; }

// Rank of 32 consecutive clusters (lane order) with bins b (BIN_INVALID = no output bin) against the warp's counters:
// rank = cnt[b]++ executed in lane order.  The 32 clusters are cut into runs of strictly ascending bins (or strictly
// descending ones, whichever gives fewer runs); inside a run all bins differ, so one load / store round serves it.
// warp_runs computes the run starts (no shared memory: independent between groups, so a batch of groups is done at once);
// warp_rank32 does the rounds, which are the only sequential part.
__device__ __forceinline__ uint32_t warp_runs(uint32_t b, uint32_t lane) {
  const uint32_t prev = __shfl_up_sync(0xffffffffu, b, 1);
  const uint32_t brk_a = __ballot_sync(0xffffffffu, lane == 0 || !(b > prev));
  const uint32_t brk_d = __ballot_sync(0xffffffffu, lane == 0 || !(b < prev));
  return __popc(brk_a) <= __popc(brk_d) ? brk_a : brk_d;          // bit l: lane l starts a run (bit 0 always set)
}

__device__ __forceinline__ uint32_t warp_rank32(uint16_t* cnt, uint32_t b, uint32_t brk, uint32_t lane) {
  uint32_t rank = 0;
  if (brk == 1u) {                                                 // one run: the usual case
    if (b != BIN_INVALID) {
      rank = cnt[b];
      cnt[b] = (uint16_t)(rank + 1);
    }
    __syncwarp();
    return rank;
  }
  while (brk) {
    const uint32_t lo = __ffs(brk) - 1;
    brk &= brk - 1;
    const uint32_t hi = brk ? __ffs(brk) - 1 : 32u;
    if (lane >= lo && lane < hi && b != BIN_INVALID) {
      const uint32_t c = cnt[b];
      rank = c;
      cnt[b] = (uint16_t)(c + 1);
    }
    __syncwarp();                                                  // the next run may touch the same counters
  }
  return rank;
}

template <bool BATCH>
__global__ void __launch_bounds__(WR_THREADS) k_rank(const __grid_constant__ DevGeo G, const __grid_constant__ FrameArgs F0,
                                                     const FrameArgs* __restrict__ table) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const uint32_t lane = lane_id(), wib = threadIdx.x >> 5, n_bins = G.n_bins;
  const RankArgs A = rank_args(frame_of<BATCH>(F0, table, blockIdx.y), n_bins);
  const uint32_t cnt_bytes = wr_warp_smem(n_bins);
  uint16_t* cnt = reinterpret_cast<uint16_t*>(smem_raw + (size_t)wib * cnt_bytes);
  const uint32_t n_warps = gridDim.x * WR_WARPS;
  for (uint32_t c = blockIdx.x * WR_WARPS + wib; c < A.n_chunks; c += n_warps) {
    const uint32_t g0 = c << A.chunk_shift, g1 = min(g0 + (1u << A.chunk_shift), A.n_attached);
    __syncwarp();
    for (uint32_t i = lane; i < cnt_bytes / 16; i += 32) reinterpret_cast<uint4*>(cnt)[i] = make_uint4(0, 0, 0, 0);
    __syncwarp();
    uint32_t cur[WR_DEPTH], nxt[WR_DEPTH];
#pragma unroll
    for (int k = 0; k < WR_DEPTH; ++k) {
      const uint32_t g = g0 + k * 32 + lane;
      cur[k] = g < g1 ? __ldcg(&A.inter[g].y) : 0xFFFFFFFFu;         // raw word: the bin is taken at the use, not here
    }
    for (uint32_t gb = g0; gb < g1; gb += WR_DEPTH * 32) {
      uint32_t runs[WR_DEPTH];
      if (gb + 2 * WR_DEPTH * 32 <= g1) {                           // this batch and the next lie inside the chunk: no guards
        // the batch after the next into the L2: one instruction, lane l takes the l-th 128-byte line of its 4 KB (0.66 -> 0.58 ms at
        // c3: the loads of the next batch then come from the L2; three batches ahead 0.59, four 0.62, six 0.73)
        if (gb + 3 * WR_DEPTH * 32 <= g1) asm volatile("prefetch.global.L2 [%0];" ::"l"(A.inter + gb + 2 * WR_DEPTH * 32 + lane * 16));
        const uint32_t* src = &A.inter[gb + WR_DEPTH * 32 + lane].y;
#pragma unroll
        for (int k = 0; k < WR_DEPTH; ++k) nxt[k] = __ldcg(src + k * 64);   // 32 records of 8 bytes further on
#pragma unroll
        for (int k = 0; k < WR_DEPTH; ++k) runs[k] = warp_runs(cur[k] >> 16, lane);
        uint16_t* dst = A.rank16 + gb + lane;
#pragma unroll
        for (int k = 0; k < WR_DEPTH; ++k) dst[k * 32] = (uint16_t)warp_rank32(cnt, cur[k] >> 16, runs[k], lane);
      } else {
#pragma unroll
        for (int k = 0; k < WR_DEPTH; ++k) {
          const uint32_t g = gb + (WR_DEPTH + k) * 32 + lane;
          nxt[k] = g < g1 ? __ldcg(&A.inter[g].y) : 0xFFFFFFFFu;     // no use of the value before the next batch
        }
#pragma unroll
        for (int k = 0; k < WR_DEPTH; ++k) runs[k] = warp_runs(cur[k] >> 16, lane);
#pragma unroll
        for (int k = 0; k < WR_DEPTH; ++k) {
          const uint32_t g = gb + k * 32 + lane;
          if (gb + k * 32 < g1) {                                   // warp-uniform
            const uint32_t rank = warp_rank32(cnt, cur[k] >> 16, runs[k], lane);
            if (g < g1) A.rank16[g] = (uint16_t)rank;
          }
        }
      }
#pragma unroll
      for (int k = 0; k < WR_DEPTH; ++k) cur[k] = nxt[k];
    }
    __syncwarp();
    uint16_t* hist_row = A.hist + (size_t)c * n_bins;
    for (uint32_t b = lane; b < n_bins; b += 32) hist_row[b] = cnt[b];   // <= 2^CHUNK_SHIFT_MAX = 32768
    // first slot of every bin in the chunk's (bin, rank) order, for the scatter kernel: lane l scans bins [l*per, l*per+per)
    {
      const uint32_t per = (n_bins + 31) / 32, b0 = min(lane * per, n_bins), b1 = min(b0 + per, n_bins);
      uint32_t s = 0;
      for (uint32_t b = b0; b < b1; ++b) s += cnt[b];
      uint32_t inc = s;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const uint32_t p = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= (uint32_t)o) inc += p;
      }
      uint32_t ex = inc - s;
      uint16_t* start_row = A.start16 + (size_t)c * A.start_stride;
      __syncwarp();                                                        // the hist row has been read out of cnt
      for (uint32_t b = b0; b < b1; ++b) {
        const uint32_t h = cnt[b];
        cnt[b] = (uint16_t)ex;
        ex += h;
      }
      __syncwarp();
      for (uint32_t b = lane; b < n_bins; b += 32) start_row[b] = cnt[b];  // coalesced
      if (lane == 31) start_row[n_bins] = (uint16_t)inc;                   // number of clusters of the chunk that have a bin
    }
  }
}

}  // namespace tmd
