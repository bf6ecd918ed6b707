// tmd_unattached.cuh -- A7: unattached clusters.
//
// "computes each coordinate summing the difference taken from the input array with the coordinates of the
// last decoded cluster; each thread decodes clusters from a specific region of the TPC."  Region = one (sector,row) bin,
// running values reset to (0,0) at the bin start (DESIGN.md §3 reading 9).  Sums are mod 2^16 / 2^32, hence associative:
// the per-thread serial loop of the paper becomes a segmented parallel prefix sum, exact under any order.
#pragma once

#include "tmd_common.cuh"
#include "tmd_scan.cuh"

namespace tmd {

struct UnattachedArgs {
  tmd_compressed in;
  const uint32_t* u_start;     // [n_bins+1] exclusive scan of u_bin_count
  const uint32_t* bin_offset;  // [n_bins+1]
  const uint32_t* att_cnt;     // [n_bins]
  uint4* clusters;
  uint32_t n_clusters_total;
};

constexpr int UNATT_THREADS = 256;
constexpr int UNATT_ITEMS = 4;

// v1: one block per bin, tiles of UNATT_THREADS * UNATT_ITEMS consecutive clusters, block scan with a running carry.
__global__ void __launch_bounds__(UNATT_THREADS) k_unattached(DevGeo G, UnattachedArgs A) {
  __shared__ uint32_t ws[33];
  const uint32_t b = blockIdx.x;
  const uint32_t i0 = A.u_start[b], cnt = A.u_start[b + 1] - i0;
  if (cnt == 0) return;
  const uint32_t dst0 = A.bin_offset[b] + A.att_cnt[b];
  const uint32_t sec = b / G.n_rows, row = b - sec * G.n_rows;
  uint32_t carry_p = 0, carry_t = 0;
  for (uint32_t base = 0; base < cnt; base += UNATT_THREADS * UNATT_ITEMS) {
    const uint32_t k0 = base + threadIdx.x * UNATT_ITEMS;
    uint32_t p[UNATT_ITEMS], t[UNATT_ITEMS];
    uint32_t sp = 0, st = 0;
#pragma unroll
    for (int k = 0; k < UNATT_ITEMS; ++k) {
      const bool in = k0 + k < cnt;
      sp += in ? A.in.u_paddiff[i0 + k0 + k] : 0u;
      st += in ? A.in.u_timediff[i0 + k0 + k] : 0u;
      p[k] = sp;
      t[k] = st;
    }
    uint32_t tot_p, tot_t;
    const uint32_t ex_p = carry_p + block_excl_scan(sp, ws, &tot_p);
    const uint32_t ex_t = carry_t + block_excl_scan(st, ws, &tot_t);
#pragma unroll
    for (int k = 0; k < UNATT_ITEMS; ++k) {
      const uint32_t i = k0 + k;
      if (i < cnt && dst0 + i < A.n_clusters_total) {
        const size_t s = (size_t)i0 + i;
        uint4 v;
        v.x = ex_t + t[k];
        v.y = ((ex_p + p[k]) & 0xFFFFu) | ((uint32_t)A.in.u_qtot[s] << 16);
        v.z = (uint32_t)A.in.u_qmax[s] | ((uint32_t)A.in.u_sigpad[s] << 16) | ((uint32_t)A.in.u_sigtime[s] << 24);
        v.w = (uint32_t)A.in.u_flags[s] | (row << 8) | (sec << 16);
        A.clusters[dst0 + i] = v;
      }
    }
    carry_p += tot_p;
    carry_t += tot_t;
  }
}

}  // namespace tmd
