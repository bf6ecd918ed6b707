// tmd_scatter.cuh -- A6: copy-through of the charge / width / flag fields and the deterministic scatter of the attached
// clusters into canonical order (DESIGN.md §3 reading 11):
//   position(g) = rel[g >> CHUNK_SHIFT][bin(g)] + rank16[g]
// with bin(g), T, P from the track-decode kernel's intermediate record, rank16 from the rank kernel (tmd_rank.cuh) and
// rel from the column scan (tmd_scan.cuh).  One thread per attached cluster g: every read is coalesced in g, the only
// irregular access is the 16-byte store.  Integer / byte moves only.
#pragma once

#include "tmd_common.cuh"
#include "tmd_decode.cuh"

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

__global__ void __launch_bounds__(SCATTER_THREADS) k_scatter(DevGeo G, ScatterArgs A) {
  const uint32_t g = blockIdx.x * SCATTER_THREADS + threadIdx.x;
  if (g >= A.n_attached) return;
  const uint2 rec = A.inter[g];
  const uint32_t bin = rec.y >> 16;
  if (bin == BIN_INVALID) return;   // decoded sector has no output bin (reading 20)
  const uint32_t pos = A.rel[(size_t)(g >> CHUNK_SHIFT) * G.n_bins + bin] + A.rank16[g];
  const uint32_t sec = bin / G.n_rows, row = bin - sec * G.n_rows;
  if (pos < A.n_clusters_total)
    A.clusters[pos] = pack_cluster(rec.x, rec.y & 0xFFFFu, A.a_qtot[g], A.a_qmax[g], A.a_sigpad[g], A.a_sigtime[g], A.a_flags[g], row, sec);
}

}  // namespace tmd
