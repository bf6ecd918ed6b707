// tmd_encode_unattached.cuh -- track-model ENCODING of the unattached clusters (the synchronous-side step, PAPER.md L68:
// "unassigned clusters are sorted by coordinate position ... stored as differences relative to the preceding cluster").
// per (sector,row) bin, sort ascending by the tuple (time, pad, qtot, qmax, sigpad, sigtime,
// flags), store pad / time as differences to the predecessor (the first of a bin: to (0,0)), copy the rest through.
//
// Steps (integer only):  k_un_count (per-bin histogram) -> k_un_offsets (exclusive scan, tile table) -> k_un_bucket (records
// into their bin's range, in arbitrary order) -> k_un_sort_tiles (bitonic sort of tiles of UN_TILE records in shared memory;
// a tile never straddles a bin) -> k_un_merge x ceil(log2(max tiles per bin)) (pairwise merge of sorted runs inside a bin,
// merge-path partitioned, ping-pong between two buffers) -> k_un_diff (differences + SoA split).
// Records that compare equal on the whole tuple are identical, so the result does not depend on the bucket order.
#pragma once

#include "tmd_common.cuh"
#include "tmd_scan.cuh"

namespace tmd {

constexpr int UN_TILE = 2048;              // records per sorted tile (32 KB of shared memory)
constexpr int UN_THREADS = 256;
constexpr int UN_ITEMS = UN_TILE / UN_THREADS;

struct UnEncodeArgs {
  uint32_t n_un, n_bins, n_rows;
  const uint4* un;          // [n_un] input records, any order
  uint32_t* bin_count;      // [n_bins]  (= out u_bin_count)
  uint32_t* bin_start;      // [n_bins + 1] exclusive scan of bin_count
  uint32_t* tile_start;     // [n_bins + 1] exclusive scan of tiles per bin
  uint32_t* cursor;         // [n_bins] bucket cursors
  uint32_t* max_tiles;      // [1] largest number of tiles in one bin
  uint4* buf_a;             // [n_un]
  uint4* buf_b;             // [n_un]
};

// the sort key of a record: lexicographic (time, pad, qtot, qmax, sigpad, sigtime, flags) as four unsigned words
struct UnKey { uint32_t k0, k1, k2, k3; };
__device__ __forceinline__ UnKey un_key(const uint4& r) {
  UnKey k;
  k.k0 = r.x;                                                          // time
  k.k1 = (r.y << 16) | (r.y >> 16);                                    // pad : qtot
  k.k2 = ((r.z & 0xFFFFu) << 16) | ((r.z >> 8) & 0xFF00u) | (r.z >> 24);   // qmax : sigpad : sigtime
  k.k3 = (r.w << 24) | (r.w >> 8);                                     // flags, then (row, sector, zero): equal inside a bin, and
                                                                       // below the all-ones padding record of a partial tile
  return k;
}
__device__ __forceinline__ bool un_less(const uint4& a, const uint4& b) {
  const UnKey x = un_key(a), y = un_key(b);
  if (x.k0 != y.k0) return x.k0 < y.k0;
  if (x.k1 != y.k1) return x.k1 < y.k1;
  if (x.k2 != y.k2) return x.k2 < y.k2;
  return x.k3 < y.k3;
}
__device__ __forceinline__ uint32_t un_bin(const uint4& r, uint32_t n_rows) { return ((r.w >> 16) & 0xFFu) * n_rows + ((r.w >> 8) & 0xFFu); }

__global__ void __launch_bounds__(256) k_un_count(UnEncodeArgs A, uint32_t* __restrict__ err) {
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < A.n_un; i += gridDim.x * blockDim.x) {
    const uint4 r = A.un[i];
    const uint32_t row = (r.w >> 8) & 0xFFu, b = un_bin(r, A.n_rows);
    if (row >= A.n_rows || b >= A.n_bins) atomicOr(&err[ERR_TRACK_FIELD], 8u);
    else atomicAdd(&A.bin_count[b], 1u);
  }
}

// single block: bin_start = exclusive scan of bin_count, tile_start = exclusive scan of ceil(count / UN_TILE), cursor = bin_start
__global__ void __launch_bounds__(1024) k_un_offsets(UnEncodeArgs A) {
  __shared__ uint32_t ws[33];
  __shared__ uint32_t s_max;
  if (threadIdx.x == 0) s_max = 0;
  const uint32_t per = (A.n_bins + blockDim.x - 1) / blockDim.x;
  const uint32_t b0 = min(threadIdx.x * per, A.n_bins), b1 = min(b0 + per, A.n_bins);
  uint32_t sc = 0, st = 0, mx = 0;
  for (uint32_t b = b0; b < b1; ++b) {
    const uint32_t c = A.bin_count[b], t = (c + UN_TILE - 1) / UN_TILE;
    sc += c; st += t; mx = max(mx, t);
  }
  uint32_t tc, tt;
  uint32_t ec = block_excl_scan(sc, ws, &tc);
  uint32_t et = block_excl_scan(st, ws, &tt);
  atomicMax(&s_max, mx);
  for (uint32_t b = b0; b < b1; ++b) {
    const uint32_t c = A.bin_count[b];
    A.bin_start[b] = ec; A.cursor[b] = ec; A.tile_start[b] = et;
    ec += c; et += (c + UN_TILE - 1) / UN_TILE;
  }
  __syncthreads();
  if (threadIdx.x == 0) { A.bin_start[A.n_bins] = tc; A.tile_start[A.n_bins] = tt; A.max_tiles[0] = s_max; }
}

__global__ void __launch_bounds__(256) k_un_bucket(UnEncodeArgs A) {
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < A.n_un; i += gridDim.x * blockDim.x) {
    const uint4 r = A.un[i];
    const uint32_t b = un_bin(r, A.n_rows);
    if (((r.w >> 8) & 0xFFu) < A.n_rows && b < A.n_bins) A.buf_a[atomicAdd(&A.cursor[b], 1u)] = r;
  }
}

// bin of global tile id `tile`: the last b with tile_start[b] <= tile (bins without tiles share their successor's start)
__device__ __forceinline__ uint32_t un_bin_of_tile(const uint32_t* __restrict__ tile_start, uint32_t n_bins, uint32_t tile) {
  uint32_t lo = 0, hi = n_bins;             // invariant: tile_start[lo] <= tile < tile_start[hi]
  while (hi - lo > 1) {
    const uint32_t mid = (lo + hi) >> 1;
    if (__ldg(tile_start + mid) <= tile) lo = mid; else hi = mid;
  }
  return lo;
}

// One block per tile: bitonic sort of up to UN_TILE records of ONE bin in shared memory (padding = records greater than any).
__global__ void __launch_bounds__(UN_THREADS) k_un_sort_tiles(UnEncodeArgs A) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  uint4* s = reinterpret_cast<uint4*>(smem_raw);
  const uint32_t tile = blockIdx.x;
  if (tile >= A.tile_start[A.n_bins]) return;
  const uint32_t b = un_bin_of_tile(A.tile_start, A.n_bins, tile);
  const uint32_t first = A.bin_start[b] + (tile - A.tile_start[b]) * UN_TILE;
  const uint32_t n = min((uint32_t)UN_TILE, A.bin_start[b + 1] - first);
  for (uint32_t i = threadIdx.x; i < UN_TILE; i += UN_THREADS)
    s[i] = i < n ? A.buf_a[first + i] : make_uint4(0xFFFFFFFFu, 0xFFFFFFFFu, 0xFFFFFFFFu, 0xFFFFFFFFu);
  __syncthreads();
  for (uint32_t k = 2; k <= UN_TILE; k <<= 1) {
    for (uint32_t j = k >> 1; j > 0; j >>= 1) {
      for (uint32_t i = threadIdx.x; i < UN_TILE / 2; i += UN_THREADS) {
        const uint32_t lo = ((i & ~(j - 1)) << 1) | (i & (j - 1)), hi = lo | j;   // lo has bit j clear
        const uint4 x = s[lo], y = s[hi];
        const bool up = (lo & k) == 0;
        if (un_less(y, x) == up) { s[lo] = y; s[hi] = x; }
      }
      __syncthreads();
    }
  }
  for (uint32_t i = threadIdx.x; i < n; i += UN_THREADS) A.buf_a[first + i] = s[i];
}

// merge path: number of elements taken from run a (length na) among the first `diag` outputs of merge(a, b); a wins ties
__device__ __forceinline__ uint32_t un_merge_path(const uint4* a, uint32_t na, const uint4* b, uint32_t nb, uint32_t diag) {
  uint32_t lo = diag > nb ? diag - nb : 0, hi = min(diag, na);
  while (lo < hi) {
    const uint32_t mid = (lo + hi) >> 1;                 // take mid from a, diag - mid from b
    if (un_less(b[diag - 1 - mid], a[mid])) hi = mid; else lo = mid + 1;
  }
  return lo;
}

// One block per output tile.  Pass `p` merges, inside every bin, runs of 2^p tiles pairwise (src -> dst).
__global__ void __launch_bounds__(UN_THREADS) k_un_merge(UnEncodeArgs A, const uint4* __restrict__ src, uint4* __restrict__ dst, uint32_t p) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  uint4* s = reinterpret_cast<uint4*>(smem_raw);
  __shared__ uint32_t s_split[2];
  const uint32_t tile = blockIdx.x;
  if (tile >= A.tile_start[A.n_bins]) return;
  const uint32_t b = un_bin_of_tile(A.tile_start, A.n_bins, tile);
  const uint32_t bin_first = A.bin_start[b], bin_n = A.bin_start[b + 1] - bin_first;
  const uint32_t t_in_bin = tile - A.tile_start[b];
  const uint32_t run = (uint32_t)UN_TILE << p;                            // records per input run
  const uint32_t pair_first = (t_in_bin >> (p + 1)) * 2 * run;            // first record (in the bin) of the pair of runs
  const uint32_t na = min(run, bin_n - pair_first), nb = min(run, bin_n - pair_first - na);
  const uint4* a = src + bin_first + pair_first;
  const uint4* bb = a + na;
  const uint32_t out0 = (t_in_bin * UN_TILE) - pair_first;                // this tile's first output inside the merged pair
  const uint32_t n_out = min((uint32_t)UN_TILE, na + nb - out0);
  if (threadIdx.x < 2) s_split[threadIdx.x] = un_merge_path(a, na, bb, nb, threadIdx.x == 0 ? out0 : out0 + n_out);
  __syncthreads();
  const uint32_t a0 = s_split[0], a1 = s_split[1], b0 = out0 - a0, b1 = out0 + n_out - a1;
  const uint32_t ca = a1 - a0, cb = b1 - b0;                              // ca + cb == n_out
  for (uint32_t i = threadIdx.x; i < n_out; i += UN_THREADS) s[i] = i < ca ? a[a0 + i] : bb[b0 + (i - ca)];
  __syncthreads();
  const uint4* sa = s;
  const uint4* sb = s + ca;
  const uint32_t d0 = min(threadIdx.x * UN_ITEMS, n_out), d1 = min(d0 + UN_ITEMS, n_out);
  uint32_t ia = un_merge_path(sa, ca, sb, cb, d0), ib = d0 - ia;
  uint4 out[UN_ITEMS];
#pragma unroll
  for (int k = 0; k < UN_ITEMS; ++k) {
    if (d0 + k < d1) {
      const bool take_b = ia >= ca || (ib < cb && un_less(sb[ib], sa[ia]));
      out[k] = take_b ? sb[ib] : sa[ia];
      ib += take_b; ia += !take_b;
    }
  }
  uint4* o = dst + bin_first + pair_first + out0;
#pragma unroll
  for (int k = 0; k < UN_ITEMS; ++k)
    if (d0 + k < d1) o[d0 + k] = out[k];
}

struct UnDiffOut {
  uint16_t* u_qtot; uint16_t* u_qmax; uint8_t* u_flags; uint8_t* u_sigpad; uint8_t* u_sigtime; uint16_t* u_paddiff; uint32_t* u_timediff;
};

// differences to the preceding cluster of the bin (the first of a bin: to (0,0)) and the SoA split
__global__ void __launch_bounds__(256) k_un_diff(UnEncodeArgs A, const uint4* __restrict__ sorted, UnDiffOut O) {
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < A.n_un; i += gridDim.x * blockDim.x) {
    const uint4 r = sorted[i];
    uint32_t pp = 0, pt = 0;
    if (i > 0) {
      const uint4 q = sorted[i - 1];
      if (((q.w ^ r.w) & 0x00FFFF00u) == 0) { pp = q.y & 0xFFFFu; pt = q.x; }   // same (row, sector): same bin
    }
    O.u_paddiff[i] = (uint16_t)((r.y & 0xFFFFu) - pp);
    O.u_timediff[i] = r.x - pt;
    O.u_qtot[i] = (uint16_t)(r.y >> 16); O.u_qmax[i] = (uint16_t)(r.z & 0xFFFFu);
    O.u_sigpad[i] = (uint8_t)(r.z >> 16); O.u_sigtime[i] = (uint8_t)(r.z >> 24); O.u_flags[i] = (uint8_t)(r.w & 0xFFu);
  }
}

}  // namespace tmd
