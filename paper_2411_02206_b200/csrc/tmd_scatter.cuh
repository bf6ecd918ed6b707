// tmd_scatter.cuh -- A6: copy-through of the charge / width / flag fields and the deterministic scatter of the attached
// clusters into canonical order (DESIGN.md §3 reading 11):
//   position(g) = rel[g >> chunk_shift][bin(g)] + rank16[g]
// with bin(g), T, P from the track-decode kernel's intermediate record, rank16 from the rank kernel (tmd_rank.cuh) and
// rel from the column scan (tmd_scan.cuh).  Integer / byte moves only.
//
// One thread per attached cluster, in g order: every read is coalesced in g; the only irregular accesses are the rel
// lookups (one 22 KB row per chunk: L1 / L2) and the 16-byte stores, which the L2 merges into full sectors because
// neighbouring ranks of a bin are written by neighbouring chunks.
// Measured on B200: what bounds this kernel is the rate of 16-byte stores that are spread over the whole
// output (~72 G stores/s), not the bytes in flight -- with sequential store addresses the same kernel runs at 6.2 TB/s.
// Wider variants (2 or 4 clusters per thread, persistent blocks with register prefetch) widen the window of g that is in
// flight, which makes the stores less local in time, and were slower.
#pragma once

#include "tmd_common.cuh"

namespace tmd {

struct ScatterArgs {
  const uint2* inter;       // [n_attached] {T, P | bin << 16}
  const uint16_t* rank16;   // [n_attached]
  const uint32_t* rel;      // [n_chunks][n_bins]
  const uint16_t* a_qtot; const uint16_t* a_qmax; const uint8_t* a_flags; const uint8_t* a_sigpad; const uint8_t* a_sigtime;
  uint4* clusters;
  uint32_t n_attached, n_clusters_total, chunk_shift;
};

constexpr int SCATTER_THREADS = 256;

__device__ __forceinline__ uint4 pack_cluster(uint32_t T, uint32_t P, uint32_t qtot, uint32_t qmax, uint32_t sigpad, uint32_t sigtime,
                                              uint32_t flags, uint32_t row, uint32_t sec) {
  uint4 v;
  v.x = T;
  v.y = P | (qtot << 16);
  v.z = qmax | (sigpad << 16) | (sigtime << 24);
  v.w = flags | (row << 8) | (sec << 16);
  return v;
}

__global__ void __launch_bounds__(SCATTER_THREADS) k_scatter(DevGeo G, ScatterArgs A) {
  const uint32_t g = blockIdx.x * SCATTER_THREADS + threadIdx.x;
  if (g >= A.n_attached) return;
  const uint2 rec = __ldg(A.inter + g);
  const uint32_t rank = __ldg(A.rank16 + g), qtot = __ldg(A.a_qtot + g), qmax = __ldg(A.a_qmax + g);
  const uint32_t sigpad = __ldg(A.a_sigpad + g), sigtime = __ldg(A.a_sigtime + g), flags = __ldg(A.a_flags + g);
  const uint32_t bin = rec.y >> 16;
  if (bin == BIN_INVALID) return;   // decoded sector has no output bin (reading 20)
  const uint32_t pos = __ldg(A.rel + (size_t)(g >> A.chunk_shift) * G.n_bins + bin) + rank;
  const uint32_t sec = (bin * G.rows_magic) >> 24, row = bin - sec * G.n_rows;
  if (pos < A.n_clusters_total) A.clusters[pos] = pack_cluster(rec.x, rec.y & 0xFFFFu, qtot, qmax, sigpad, sigtime, flags, row, sec);
}

}  // namespace tmd
