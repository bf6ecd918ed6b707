// tmd_common.cuh -- shared definitions of the sm_100a track-model decoder kernels.
//
// Model = SURVEY.md §8(c) C1-C5 (readings listed in DESIGN.md §3); paper passages: PAPER.md L68, L70.
// No code is shared with oracle/ (own structs, constants and helpers).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/tmd.h"

namespace tmd {

// A "chunk" is a window of 2^chunk_shift consecutive attached clusters (in g order).  Chunks are the unit of the
// deterministic scatter: per-chunk histograms over bins, a column scan over chunks, and ranks inside the
// chunk.  The shift is chosen per call from the number of attached clusters (tmd_api.cu): 2^15 for a full time frame,
// smaller for small inputs so that the rank kernel still has a chunk for every resident warp.
constexpr int CHUNK_SHIFT_MAX = 15;     // rank16 and the u16 histograms hold counts <= 2^15
constexpr int CHUNK_SHIFT_MIN = 11;
constexpr uint32_t MAX_BINS = 8192;     // n_sectors_out * n_rows
constexpr uint32_t COL_GROUP = 64;      // chunks per group in the column scan
constexpr uint16_t BIN_INVALID = 0xFFFFu;

struct RowGeo {   // one LDS.128 per step
  float x, padw, inv_padw, half;
};

struct DevGeo {
  uint32_t n_az, n_sides, n_sectors_out, n_rows, n_bins;
  float cos_a, sin_a;
  float qk;             // fmul(0.0625f, fmul(bz_tesla, 0.00299792458f))
  uint32_t rows_magic;  // floor(2^24 / n_rows) + 1:  bin / n_rows == (bin * rows_magic) >> 24  for bin < 8192 (< 2^24 / n_rows)
  uint32_t az_magic;    // floor(2^24 / n_az) + 1, the same for values < 64
  const RowGeo* rows;   // DEVICE [n_rows]
};

// error words in the workspace (TMD_VALIDATE); words 2-3 hold the 64-bit sum of trk_ncl
enum { ERR_TRACK_FIELD = 0, ERR_SECTOR_OUT = 1, ERR_NCL_SUM_LO = 2, ERR_NCL_SUM_HI = 3, ERR_WORDS = 4 };

// Layout of one frame's workspace (byte offsets from its 256-byte aligned base) and the sizes derived from the frame's
// counts.  A pure function of (n_bins, n_tracks, n_attached, SM count): tmd_workspace_bytes and tmd_decode agree.
struct Workspace {
  uint32_t n_tiles, n_chunks, n_groups, chunk_shift;
  size_t o_err, o_tile_sum, o_off, o_hdr, o_hdr2, o_att_cnt, o_u_start, o_gsum, o_hist, o_start16, o_rel, o_rank16, o_inter, o_table, total;
};

// Everything the kernels need to know about ONE time frame.  tmd_decode passes it by value (kernel parameter space);
// tmd_decode_batch keeps one per frame in device memory (frame 0's workspace) and the kernels pick theirs with the
// frame coordinate of the grid, so that many small frames share one launch sequence.
struct FrameArgs {
  tmd_compressed in;         // DEVICE pointers
  uint4* clusters;
  uint32_t* bin_offset;
  uint32_t* probe_state;     // nullable
  uint32_t probe_step;
  uint32_t validate;         // TMD_VALIDATE: report malformed fields in the error words
  unsigned char* ws;         // this frame's workspace
  Workspace W;

  template <typename T>
  __host__ __device__ __forceinline__ T* at(size_t offset) const { return reinterpret_cast<T*>(ws + offset); }
  __host__ __device__ __forceinline__ uint32_t n_res() const { return (uint32_t)in.n_attached - in.n_tracks; }
};

// The frame a block works on: the by-value parameter, or entry `f` of the batch table.
template <bool BATCH>
__device__ __forceinline__ const FrameArgs& frame_of(const FrameArgs& F0, const FrameArgs* __restrict__ table, uint32_t f) {
  return BATCH ? table[f] : F0;
}

// ---- the integer part of one step: leg / row / sector bookkeeping (C3-3, C3-4, C3-5 without the rotation) ----------
struct WalkState {
  uint32_t row, az, side;
  int dir;
};

// v mod m by multiplication (reading 19): magic = floor(2^24 / m) + 1 is exact for v * m < 2^24 (v < 256 here)
__device__ __forceinline__ uint32_t reduce_mod(uint32_t v, uint32_t m, uint32_t magic) { return v - ((v * magic) >> 24) * m; }

// returns the reduced sector step d (0 = same sector); updates row / az / dir
__device__ __forceinline__ uint32_t walk_step(WalkState& w, uint32_t rowdiff, uint32_t secleg, const DevGeo& G) {
  if (secleg & 0x80u) w.dir = -w.dir;
  const uint32_t rd = reduce_mod(rowdiff, G.n_rows, G.rows_magic);
  const uint32_t r = w.row + (w.dir > 0 ? rd : G.n_rows - rd);
  w.row = r >= G.n_rows ? r - G.n_rows : r;
  const uint32_t d = reduce_mod(secleg & 0x3Fu, G.n_az, G.az_magic);
  const uint32_t a = w.az + d;
  w.az = a >= G.n_az ? a - G.n_az : a;
  return d;
}

// cp.async (LDGSTS): 16-byte global -> shared copy past the L1 (.cg: the data is used once; allocating it in the L1 cost the
// decode kernel 13 %); bytes past src_bytes are zero-filled
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src, uint32_t src_bytes) {
  const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(d), "l"(gmem_src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }

__device__ __forceinline__ uint32_t lane_id() { return threadIdx.x & 31u; }

}  // namespace tmd
