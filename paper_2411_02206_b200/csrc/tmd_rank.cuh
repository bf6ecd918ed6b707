// tmd_rank.cuh -- A3: the geometry walk of the attached clusters as a PARALLEL segmented scan, the per-chunk histogram
// over bins, and the rank of every attached cluster among the clusters of its chunk that fall in the same bin
// (ascending global attached index g).  Integer only; reads a_rowdiff / a_secleg and the per-track first clusters, so it
// does not depend on the floating-point track model and runs concurrently with the track-decode kernel.
//
// Together with the column scan (tmd_scan.cuh) this yields the canonical position of every attached cluster
// (DESIGN.md §3 reading 11):   position(g) = rel[g >> CHUNK_SHIFT][bin(g)] + rank16[g].
//
// The walk (SURVEY.md §8(c) C3-3, C3-4, C3-5 without the rotation) is a prefix "sum" in the group Z2 |x (Z_rows x Z_az):
//   dir_j = dir_0 * prod(-1)^leg_i,   row_j = row_0 + sum dir_i * rd_i (mod n_rows),   az_j = az_0 + sum d_i (mod n_az),
// with a reset at every first cluster of a track.  An element is packed in one word (below) and `walk_combine` is the
// associative operator, so the per-thread serial walk of the paper's kernel becomes: every thread walks 16
// consecutive clusters, a block-wide scan of the 512 aggregates supplies each thread's incoming state, and a second
// walk over the same 16 (kept in registers) emits the bins.
#pragma once

#include "tmd_common.cuh"
#include "tmd_scan.cuh"

namespace tmd {

constexpr int SUB_SHIFT = 13;                         // a block ranks one sub-chunk of 8192 clusters at a time
constexpr uint32_t SUB_WINDOW = 1u << SUB_SHIFT;
constexpr int SUBS_PER_CHUNK = 1 << (CHUNK_SHIFT - SUB_SHIFT);
constexpr int WR_THREADS = 512;
constexpr int WR_ITEMS = SUB_WINDOW / WR_THREADS;     // 16 consecutive clusters per thread
constexpr uint32_t WR_GRANULES = SUB_WINDOW / 16 + 1; // aligned 16-byte granules of residual bytes a sub-chunk can touch
constexpr uint32_t WR_LONG = 48;                      // per-bin lists longer than this are ranked by the whole block
static_assert(WR_ITEMS == 16, "one thread owns half a bitmap word");

struct WalkRankArgs {
  const uint32_t* off;          // [n_tracks+1]
  const uint32_t* sub_first;    // [n_sub+1] first track t with off[t] >= s << SUB_SHIFT; [n_sub] = n_tracks
  const uint8_t* trk_row0; const uint8_t* trk_sec0;
  const uint8_t* a_rowdiff; const uint8_t* a_secleg;
  uint16_t* hist;               // [n_chunks][n_bins]
  uint16_t* rank16;             // [n_attached]
  uint32_t n_tracks, n_attached, n_chunks, chunks_per_block;
};

// ---- walk elements ---------------------------------------------------------------------------------------------------
// bits 0-7: row (absolute) or row shift (relative), 8-13: az or az shift, 14: direction (1 = inward) or leg parity,
// 15: side, 16: absolute (a first cluster lies at or before this element), 17: malformed first cluster (track dropped).
constexpr uint32_t W_DIR = 1u << 14, W_SIDE = 1u << 15, W_ABS = 1u << 16, W_BAD = 1u << 17;

__device__ __forceinline__ uint32_t walk_combine(uint32_t a, uint32_t b, uint32_t n_rows, uint32_t n_az) {
  if (b & W_ABS) return b;
  uint32_t s = (a & 0xFFu) + ((a & W_DIR) ? n_rows - (b & 0xFFu) : (b & 0xFFu));
  if (s >= n_rows) s -= n_rows;
  uint32_t z = ((a >> 8) & 0x3Fu) + ((b >> 8) & 0x3Fu);
  if (z >= n_az) z -= n_az;
  return (a & (W_ABS | W_SIDE | W_BAD)) | ((a ^ b) & W_DIR) | (z << 8) | s;
}

// residual bytes -> relative element (reading 19: both bytes are reduced first)
__device__ __forceinline__ uint32_t walk_elem(uint32_t rowdiff, uint32_t secleg, const DevGeo& G) {
  const uint32_t rd = rowdiff - ((rowdiff * G.rows_magic) >> 24) * G.n_rows;
  const uint32_t d6 = secleg & 0x3Fu;
  const uint32_t d = d6 - ((d6 * G.az_magic) >> 24) * G.n_az;
  const uint32_t leg = secleg >> 7;
  const uint32_t s = (leg && rd) ? G.n_rows - rd : rd;   // the leg flag flips the direction before the row moves
  return (leg ? W_DIR : 0u) | (d << 8) | s;
}

// first cluster of track t -> absolute element
__device__ __forceinline__ uint32_t walk_seed(uint32_t row0, uint32_t sec0, const DevGeo& G) {
  if (row0 >= G.n_rows || sec0 >= G.n_az * G.n_sides) return W_ABS | W_BAD;
  const uint32_t side = sec0 >= G.n_az ? 1u : 0u;
  return W_ABS | (side ? W_SIDE : 0u) | ((sec0 - side * G.n_az) << 8) | row0;
}

__device__ __forceinline__ uint32_t walk_bin(uint32_t w, const DevGeo& G) {
  const uint32_t sec = ((w & W_SIDE) ? G.n_az : 0u) + ((w >> 8) & 0x3Fu);
  return ((w & W_BAD) || sec >= G.n_sectors_out) ? (uint32_t)BIN_INVALID : sec * G.n_rows + (w & 0xFFu);
}

// Block-wide exclusive scan with walk_combine (ordered).  ws = 34 words.  Returns the exclusive prefix, *total = all.
__device__ __forceinline__ uint32_t block_walk_scan(uint32_t v, uint32_t* ws, uint32_t* total, uint32_t n_rows, uint32_t n_az) {
  const uint32_t lane = lane_id(), wid = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
  uint32_t inc = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const uint32_t p = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= (uint32_t)o) inc = walk_combine(p, inc, n_rows, n_az);
  }
  uint32_t ex = __shfl_up_sync(0xffffffffu, inc, 1);
  if (lane == 0) ex = 0;
  __syncthreads();
  if (lane == 31) ws[wid] = inc;
  __syncthreads();
  if (wid == 0) {
    const uint32_t s = lane < nw ? ws[lane] : 0;
    uint32_t si = s;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t p = __shfl_up_sync(0xffffffffu, si, o);
      if (lane >= (uint32_t)o) si = walk_combine(p, si, n_rows, n_az);
    }
    uint32_t se = __shfl_up_sync(0xffffffffu, si, 1);
    if (lane == 0) se = 0;
    ws[lane] = se;
    if (lane == 31) ws[33] = si;
  }
  __syncthreads();
  *total = ws[33];
  return walk_combine(ws[wid], ex, n_rows, n_az);
}

// staged residual bytes: pair e = rowdiff | secleg << 8 of residual (r_base + e) at u16 index e + 2 * (e >> 4)
// (a 4-byte pad after every 16 pairs: threads that are 16 pairs apart read different banks)
__device__ __forceinline__ uint32_t stage_index(uint32_t e) { return e + ((e >> 4) << 1); }

// One persistent block ranks the chunks [c0, c1) in order (contiguous in g), so the walk state of a track that
// straddles a sub-chunk boundary is carried in a register; only the very first one is recomputed from the track start.
// Dynamic shared memory: stage u16[WR_GRANULES*18] (aliased by rank_of u16[SUB_WINDOW]), list u16[SUB_WINDOW],
// cnt u32[n_bins], base u32[n_bins], bitmap u32[256], wprefix u32[256].
__global__ void __launch_bounds__(WR_THREADS, 2) k_walk_rank(DevGeo G, WalkRankArgs A) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  constexpr uint32_t STAGE_U16 = WR_GRANULES * 18;
  uint16_t* stage = reinterpret_cast<uint16_t*>(smem_raw);
  uint16_t* rank_of = stage;                                   // alias: the staged bytes are dead after the first walk
  uint16_t* list = stage + ((STAGE_U16 + 7) & ~7u);
  uint32_t* cnt = reinterpret_cast<uint32_t*>(list + SUB_WINDOW);
  uint32_t* base = cnt + G.n_bins;
  uint32_t* bitmap = base + G.n_bins;
  uint32_t* wprefix = bitmap + SUB_WINDOW / 32;
  __shared__ uint32_t ws[34];
  __shared__ uint16_t long_bins[SUB_WINDOW / (WR_LONG + 1) + 1];
  __shared__ uint32_t n_long;

  const uint32_t tid = threadIdx.x, n_bins = G.n_bins, n_rows = G.n_rows, n_az = G.n_az;
  const uint32_t c0 = blockIdx.x * A.chunks_per_block, c1 = min(c0 + A.chunks_per_block, A.n_chunks);
  if (c0 >= c1) return;

  // ---- walk state at the first cluster of chunk c0 (only if that cluster is not a first cluster of a track)
  uint32_t carry = 0;
  {
    const uint32_t g_lo = c0 << CHUNK_SHIFT;
    const uint32_t tf = A.sub_first[c0 * SUBS_PER_CHUNK];
    if (tf > 0 && (tf >= A.n_tracks || A.off[tf] != g_lo)) {
      const uint32_t ts = tf - 1, o = A.off[ts];
      const uint32_t n_pre = g_lo - o - 1, r0 = o - ts;         // residuals of track ts before g_lo
      const uint32_t per = (n_pre + WR_THREADS - 1) / WR_THREADS;
      const uint32_t e0 = min(tid * per, n_pre), e1 = min(e0 + per, n_pre);
      uint32_t agg = 0;
      for (uint32_t e = e0; e < e1; ++e) agg = walk_combine(agg, walk_elem(A.a_rowdiff[r0 + e], A.a_secleg[r0 + e], G), n_rows, n_az);
      uint32_t total;
      block_walk_scan(agg, ws, &total, n_rows, n_az);
      carry = walk_combine(walk_seed(A.trk_row0[ts], A.trk_sec0[ts], G), total, n_rows, n_az);
    }
  }

  for (uint32_t c = c0; c < c1; ++c) {
    for (uint32_t b = tid; b < n_bins; b += WR_THREADS) base[b] = 0;
    for (uint32_t sub = 0; sub < (uint32_t)SUBS_PER_CHUNK; ++sub) {
      const uint32_t sc = c * SUBS_PER_CHUNK + sub;
      const uint32_t g_lo = sc << SUB_SHIFT;
      if (g_lo >= A.n_attached) break;
      const uint32_t g_hi = min(g_lo + SUB_WINDOW, A.n_attached), n = g_hi - g_lo;
      const uint32_t tf = A.sub_first[sc], tl = A.sub_first[sc + 1];
      const uint32_t r_lo = g_lo - tf, r_hi = g_hi - tl, r_base = r_lo & ~15u;
      // ---- A: clear; stage the residual bytes [r_base, r_hi) as (rowdiff, secleg) pairs
      __syncthreads();                                           // previous sub-chunk done with rank_of / list / cnt
      if (tid < SUB_WINDOW / 32) bitmap[tid] = 0;
      for (uint32_t b = tid; b < n_bins; b += WR_THREADS) cnt[b] = 0;
      if (tid == 0) n_long = 0;
      for (uint32_t gr = tid; r_base + gr * 16 < r_hi; gr += WR_THREADS) {
        const uint32_t r = r_base + gr * 16;
        uint32_t rd[4], sl[4];
        if (r + 16 <= A.n_attached - A.n_tracks) {
          const uint4 a = *reinterpret_cast<const uint4*>(A.a_rowdiff + r);
          const uint4 b = *reinterpret_cast<const uint4*>(A.a_secleg + r);
          rd[0] = a.x; rd[1] = a.y; rd[2] = a.z; rd[3] = a.w;
          sl[0] = b.x; sl[1] = b.y; sl[2] = b.z; sl[3] = b.w;
        } else {                                                 // the last granule of the arrays
#pragma unroll
          for (int q = 0; q < 4; ++q) {
            rd[q] = 0; sl[q] = 0;
            for (int k = 0; k < 4; ++k) {
              const uint32_t rr = r + q * 4 + k;
              if (rr < r_hi) { rd[q] |= (uint32_t)A.a_rowdiff[rr] << (8 * k); sl[q] |= (uint32_t)A.a_secleg[rr] << (8 * k); }
            }
          }
        }
        uint32_t* dst = reinterpret_cast<uint32_t*>(stage + gr * 18);
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          dst[2 * q] = __byte_perm(rd[q], sl[q], 0x5140);        // bytes: rd0 sl0 rd1 sl1
          dst[2 * q + 1] = __byte_perm(rd[q], sl[q], 0x7362);    // bytes: rd2 sl2 rd3 sl3
        }
      }
      __syncthreads();
      // ---- B: first clusters of the tracks that start in this sub-chunk
      for (uint32_t t = tf + tid; t < tl; t += WR_THREADS) {
        const uint32_t li = A.off[t] - g_lo;
        atomicOr(&bitmap[li >> 5], 1u << (li & 31u));
      }
      __syncthreads();
      // ---- C: tracks started before each bitmap word
      {
        const uint32_t pc = tid < SUB_WINDOW / 32 ? __popc(bitmap[tid]) : 0u;
        uint32_t total;
        const uint32_t ex = block_excl_scan(pc, ws, &total);
        if (tid < SUB_WINDOW / 32) wprefix[tid] = ex;
      }
      __syncthreads();
      // ---- walk 1: the thread's 16 elements and their aggregate
      const uint32_t li0 = tid * WR_ITEMS;
      uint32_t e[WR_ITEMS];
      uint32_t agg = 0;
      {
        const uint32_t word = bitmap[tid >> 1], sh = (tid & 1u) * 16u;
        const uint32_t heads = (word >> sh) & 0xFFFFu;
        uint32_t t = tf + wprefix[tid >> 1] + __popc(word & ((1u << sh) - 1u));   // tracks started before li0; current = t - 1
        uint32_t r_run = g_lo + li0 - t;                                          // = g - (t - 1) - 1
#pragma unroll
        for (int k = 0; k < WR_ITEMS; ++k) {
          uint32_t w = 0;
          if (li0 + k < n) {
            if ((heads >> k) & 1u) {
              w = walk_seed(A.trk_row0[t], A.trk_sec0[t], G);
              ++t;                                                                 // r_run is unchanged by a first cluster
            } else {
              const uint32_t pair = stage[stage_index(r_run - r_base)];
              w = walk_elem(pair & 0xFFu, pair >> 8, G);
              ++r_run;
            }
          }
          e[k] = w;
          agg = walk_combine(agg, w, n_rows, n_az);
        }
      }
      uint32_t total;
      uint32_t state = block_walk_scan(agg, ws, &total, n_rows, n_az);   // syncs: every thread is done with `stage`
      state = walk_combine(carry, state, n_rows, n_az);
      carry = walk_combine(carry, total, n_rows, n_az);
      // ---- walk 2: bins; arrival slot inside the bin
      uint32_t bs[WR_ITEMS];                                             // bin | slot << 16
#pragma unroll
      for (int k = 0; k < WR_ITEMS; ++k) {
        state = walk_combine(state, e[k], n_rows, n_az);
        uint32_t v = BIN_INVALID;
        if (li0 + k < n) {
          const uint32_t bin = walk_bin(state, G);
          if (bin != BIN_INVALID) v = bin | (atomicAdd(&cnt[bin], 1u) << 16);
        }
        bs[k] = v;
      }
      __syncthreads();
      // ---- exclusive scan over bins: cnt[b] becomes the start of bin b's list
      uint32_t n_valid;
      {
        const uint32_t per = (n_bins + WR_THREADS - 1) / WR_THREADS;
        const uint32_t b0 = min(tid * per, n_bins), b1 = min(b0 + per, n_bins);
        uint32_t s = 0;
        for (uint32_t b = b0; b < b1; ++b) s += cnt[b];
        uint32_t ex = block_excl_scan(s, ws, &n_valid);
        for (uint32_t b = b0; b < b1; ++b) {
          const uint32_t h = cnt[b];
          cnt[b] = ex;
          ex += h;
        }
      }
      __syncthreads();
      // ---- per-bin lists of local indices (arrival order)
#pragma unroll
      for (int k = 0; k < WR_ITEMS; ++k) {
        const uint32_t bin = bs[k] & 0xFFFFu;
        if (bin != BIN_INVALID) list[cnt[bin] + (bs[k] >> 16)] = (uint16_t)(li0 + k);
        else if (li0 + k < n) rank_of[li0 + k] = 0;
      }
      __syncthreads();
      // ---- rank inside the bin = entries of the list with a smaller local index, on top of the chunk's earlier sub-chunks
      for (uint32_t b = tid; b < n_bins; b += WR_THREADS) {
        const uint32_t s = cnt[b], en = (b + 1 < n_bins) ? cnt[b + 1] : n_valid;
        if (en == s) continue;
        const uint32_t bb = base[b];
        base[b] = bb + (en - s);
        if (en - s > WR_LONG) {
          long_bins[atomicAdd(&n_long, 1u)] = (uint16_t)b;
          continue;
        }
        for (uint32_t k = s; k < en; ++k) {
          const uint32_t v = list[k];
          uint32_t r = bb;
          for (uint32_t m = s; m < en; ++m) r += (list[m] < v);
          rank_of[v] = (uint16_t)r;
        }
      }
      __syncthreads();
      for (uint32_t q = 0; q < n_long; ++q) {     // long lists (degenerate inputs): the whole block ranks one bin at a time
        const uint32_t b = long_bins[q], s = cnt[b], en = (b + 1 < n_bins) ? cnt[b + 1] : n_valid;
        const uint32_t bb = base[b] - (en - s);
        for (uint32_t k = s + tid; k < en; k += WR_THREADS) {
          const uint32_t v = list[k];
          uint32_t r = bb;
          for (uint32_t m = s; m < en; ++m) r += (list[m] < v);
          rank_of[v] = (uint16_t)r;
        }
      }
      __syncthreads();
      // ---- ranks out, coalesced
      {
        const uint32_t* src = reinterpret_cast<const uint32_t*>(rank_of);
        uint32_t* dst = reinterpret_cast<uint32_t*>(A.rank16 + g_lo);    // g_lo is a multiple of 8192
        for (uint32_t p = tid; 2 * p + 1 < n; p += WR_THREADS) dst[p] = src[p];
        if ((n & 1u) && tid == 0) A.rank16[g_lo + n - 1] = rank_of[n - 1];
      }
    }
    __syncthreads();
    uint16_t* hist_row = A.hist + (size_t)c * n_bins;
    for (uint32_t b = tid; b < n_bins; b += WR_THREADS) hist_row[b] = (uint16_t)base[b];   // <= CHUNK_WINDOW = 32768
    __syncthreads();
  }
}

}  // namespace tmd
