// tmd_scatter.cuh -- A6: copy-through of the charge / width / flag fields and the deterministic scatter of the attached
// clusters into canonical order (DESIGN.md §3 reading 11):
//   position(g) = rel[g >> CHUNK_SHIFT][bin(g)] + rank16[g]
// with bin(g), T, P from the track-decode kernel's intermediate record, rank16 from the rank kernel (tmd_rank.cuh) and
// rel from the column scan (tmd_scan.cuh).  Integer / byte moves only.
//
// One thread per SCATTER_VEC = 4 consecutive attached clusters g: every input stream is read with one vector load per
// thread (2 x 16 B of records, 8 B of ranks, 8 + 8 B of charges, 3 x 4 B of widths / flags), all issued before the first
// use, so a warp has ~2.2 KB in flight; the only irregular accesses are the rel lookups (one 22 KB row per chunk: L1)
// and the 16-byte stores, which the L2 merges into full sectors because neighbouring ranks of a bin are written by
// neighbouring chunks (the kernel runs in g order).
#pragma once

#include "tmd_common.cuh"

namespace tmd {

struct ScatterArgs {
  const uint2* inter;       // [n_attached] {T, P | bin << 16}
  const uint16_t* rank16;   // [n_attached]
  const uint32_t* rel;      // [n_chunks][n_bins]
  const uint16_t* a_qtot; const uint16_t* a_qmax; const uint8_t* a_flags; const uint8_t* a_sigpad; const uint8_t* a_sigtime;
  uint4* clusters;
  uint32_t n_attached, n_clusters_total;
};

constexpr int SCATTER_THREADS = 256;
constexpr int SCATTER_VEC = 4;

__device__ __forceinline__ uint4 pack_cluster(uint32_t T, uint32_t P, uint32_t qtot, uint32_t qmax, uint32_t sigpad, uint32_t sigtime,
                                              uint32_t flags, uint32_t row, uint32_t sec) {
  uint4 v;
  v.x = T;
  v.y = P | (qtot << 16);
  v.z = qmax | (sigpad << 16) | (sigtime << 24);
  v.w = flags | (row << 8) | (sec << 16);
  return v;
}

// position of a record in `clusters`, or UINT32_MAX if it has no output bin (reading 20)
__device__ __forceinline__ uint32_t scatter_pos(const uint32_t* __restrict__ rel_row, uint2 rec, uint32_t rank) {
  const uint32_t bin = rec.y >> 16;
  return bin == BIN_INVALID ? 0xFFFFFFFFu : __ldg(rel_row + bin) + rank;
}

__device__ __forceinline__ void scatter_store(const DevGeo& G, uint4* __restrict__ clusters, uint32_t n_total, uint32_t pos, uint2 rec,
                                              uint32_t qtot, uint32_t qmax, uint32_t sigpad, uint32_t sigtime, uint32_t flags) {
  const uint32_t bin = rec.y >> 16;
  const uint32_t sec = (bin * G.rows_magic) >> 24, row = bin - sec * G.n_rows;
  if (pos < n_total) clusters[pos] = pack_cluster(rec.x, rec.y & 0xFFFFu, qtot, qmax, sigpad, sigtime, flags, row, sec);
}

__global__ void __launch_bounds__(SCATTER_THREADS) k_scatter(DevGeo G, ScatterArgs A) {
  const uint32_t g0 = (blockIdx.x * SCATTER_THREADS + threadIdx.x) * SCATTER_VEC;
  if (g0 >= A.n_attached) return;
  // CHUNK_WINDOW is a multiple of SCATTER_VEC: the four clusters share a chunk
  const uint32_t* __restrict__ rel_row = A.rel + (size_t)(g0 >> CHUNK_SHIFT) * G.n_bins;
  uint4* __restrict__ clusters = A.clusters;
  if (g0 + SCATTER_VEC <= A.n_attached) {
    const uint4 r01 = __ldg(reinterpret_cast<const uint4*>(A.inter) + (g0 >> 1));
    const uint4 r23 = __ldg(reinterpret_cast<const uint4*>(A.inter) + (g0 >> 1) + 1);
    const uint2 rk = __ldg(reinterpret_cast<const uint2*>(A.rank16) + (g0 >> 2));
    const uint2 qt = __ldg(reinterpret_cast<const uint2*>(A.a_qtot) + (g0 >> 2));
    const uint2 qm = __ldg(reinterpret_cast<const uint2*>(A.a_qmax) + (g0 >> 2));
    const uint32_t sp = __ldg(reinterpret_cast<const uint32_t*>(A.a_sigpad) + (g0 >> 2));
    const uint32_t st = __ldg(reinterpret_cast<const uint32_t*>(A.a_sigtime) + (g0 >> 2));
    const uint32_t fl = __ldg(reinterpret_cast<const uint32_t*>(A.a_flags) + (g0 >> 2));
    const uint2 c0 = make_uint2(r01.x, r01.y), c1 = make_uint2(r01.z, r01.w), c2 = make_uint2(r23.x, r23.y), c3 = make_uint2(r23.z, r23.w);
    // the four dependent lookups first, so that they are in flight together
    const uint32_t p0 = scatter_pos(rel_row, c0, rk.x & 0xFFFFu), p1 = scatter_pos(rel_row, c1, rk.x >> 16);
    const uint32_t p2 = scatter_pos(rel_row, c2, rk.y & 0xFFFFu), p3 = scatter_pos(rel_row, c3, rk.y >> 16);
    scatter_store(G, clusters, A.n_clusters_total, p0, c0, qt.x & 0xFFFFu, qm.x & 0xFFFFu, sp & 0xFFu, st & 0xFFu, fl & 0xFFu);
    scatter_store(G, clusters, A.n_clusters_total, p1, c1, qt.x >> 16, qm.x >> 16, (sp >> 8) & 0xFFu, (st >> 8) & 0xFFu, (fl >> 8) & 0xFFu);
    scatter_store(G, clusters, A.n_clusters_total, p2, c2, qt.y & 0xFFFFu, qm.y & 0xFFFFu, (sp >> 16) & 0xFFu, (st >> 16) & 0xFFu,
                  (fl >> 16) & 0xFFu);
    scatter_store(G, clusters, A.n_clusters_total, p3, c3, qt.y >> 16, qm.y >> 16, sp >> 24, st >> 24, fl >> 24);
  } else {
    for (uint32_t g = g0; g < A.n_attached; ++g) {
      const uint2 c = A.inter[g];
      scatter_store(G, clusters, A.n_clusters_total, scatter_pos(rel_row, c, A.rank16[g]), c, A.a_qtot[g], A.a_qmax[g], A.a_sigpad[g],
                    A.a_sigtime[g], A.a_flags[g]);
    }
  }
}

}  // namespace tmd
