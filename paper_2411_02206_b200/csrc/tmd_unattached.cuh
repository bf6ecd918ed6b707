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
constexpr int UNATT_WARPS = UNATT_THREADS / 32;
constexpr int UNATT_ITEMS = 4;
constexpr uint32_t UNATT_SMALL = 1024;     // bins up to this many clusters are decoded by one warp, larger ones by the block

__device__ __forceinline__ UnattachedArgs unattached_args(const FrameArgs& F) {
  UnattachedArgs A;
  A.in = F.in; A.u_start = F.at<uint32_t>(F.W.o_u_start); A.bin_offset = F.bin_offset; A.att_cnt = F.at<uint32_t>(F.W.o_att_cnt);
  A.clusters = F.clusters; A.n_clusters_total = (uint32_t)(F.in.n_attached + F.in.n_unattached);
  return A;
}

// Decode bin b with NT cooperating threads (thread index `tid` in 0..NT-1): NT = 32 is one warp (shuffle scan, no block
// barrier), NT = UNATT_THREADS the whole block (NT is uniform over the calling warp, and over the block when it is the block).  Tiles of NT * 4 consecutive clusters, aligned to 4 in the global cluster
// index so that every stream is read with one vector load per thread (8 B of pad differences, 16 B of time differences,
// 8 + 8 B of charges, 3 x 4 B of widths / flags); scan of the per-thread sums with a running carry; 4 x 16-byte stores per thread.
__device__ __forceinline__ void unattached_bin(const DevGeo& G, const UnattachedArgs& A, uint32_t b, uint32_t tid, const uint32_t NT, uint32_t* ws) {
  const uint32_t i0 = A.u_start[b], i1 = A.u_start[b + 1];
  if (i1 == i0) return;
  const uint32_t n_un = (uint32_t)A.in.n_unattached;
  const uint32_t dst0 = A.bin_offset[b] + A.att_cnt[b];
  const uint32_t sec = b / G.n_rows, row = b - sec * G.n_rows;
  const uint32_t tail = (row << 8) | (sec << 16);
  uint32_t carry_p = 0, carry_t = 0;
  // raw words of the four clusters a thread takes from a tile; the NEXT tile's are requested before the current tile is scanned
  struct Raw { uint2 p2; uint4 t4; uint2 q2, m2; uint32_t a, c, f; };
  auto load_raw = [&](uint32_t k0) -> Raw {
    Raw r;
    r.p2 = make_uint2(0, 0); r.t4 = make_uint4(0, 0, 0, 0); r.q2 = make_uint2(0, 0); r.m2 = make_uint2(0, 0); r.a = r.c = r.f = 0;
    if (k0 < i1 && k0 + 4 > i0) {
      if (k0 + 4 <= n_un) {
        r.p2 = __ldg(reinterpret_cast<const uint2*>(A.in.u_paddiff + k0));
        r.t4 = __ldg(reinterpret_cast<const uint4*>(A.in.u_timediff + k0));
        r.q2 = __ldg(reinterpret_cast<const uint2*>(A.in.u_qtot + k0));
        r.m2 = __ldg(reinterpret_cast<const uint2*>(A.in.u_qmax + k0));
        r.a = __ldg(reinterpret_cast<const uint32_t*>(A.in.u_sigpad + k0));
        r.c = __ldg(reinterpret_cast<const uint32_t*>(A.in.u_sigtime + k0));
        r.f = __ldg(reinterpret_cast<const uint32_t*>(A.in.u_flags + k0));
      } else {                                                   // the last clusters of the arrays
        uint32_t pd[4], td[4], qt[4], qm[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          const uint32_t i = min(k0 + k, n_un - 1);
          pd[k] = A.in.u_paddiff[i]; td[k] = A.in.u_timediff[i]; qt[k] = A.in.u_qtot[i]; qm[k] = A.in.u_qmax[i];
          r.a |= (uint32_t)A.in.u_sigpad[i] << (8 * k); r.c |= (uint32_t)A.in.u_sigtime[i] << (8 * k); r.f |= (uint32_t)A.in.u_flags[i] << (8 * k);
        }
        r.p2 = make_uint2(pd[0] | (pd[1] << 16), pd[2] | (pd[3] << 16)); r.t4 = make_uint4(td[0], td[1], td[2], td[3]);
        r.q2 = make_uint2(qt[0] | (qt[1] << 16), qt[2] | (qt[3] << 16)); r.m2 = make_uint2(qm[0] | (qm[1] << 16), qm[2] | (qm[3] << 16));
      }
    }
    return r;
  };
  Raw nxt = load_raw((i0 & ~3u) + tid * UNATT_ITEMS);
  for (uint32_t base = i0 & ~3u; base < i1; base += NT * UNATT_ITEMS) {
    const uint32_t k0 = base + tid * UNATT_ITEMS;        // multiple of 4
    const Raw cur = nxt;
    if (base + NT * UNATT_ITEMS < i1) nxt = load_raw(k0 + NT * UNATT_ITEMS);
    uint32_t pd[4], td[4], qt[4], qm[4], sp[4], st[4], fl[4];
    pd[0] = cur.p2.x & 0xFFFFu; pd[1] = cur.p2.x >> 16; pd[2] = cur.p2.y & 0xFFFFu; pd[3] = cur.p2.y >> 16;
    td[0] = cur.t4.x; td[1] = cur.t4.y; td[2] = cur.t4.z; td[3] = cur.t4.w;
    qt[0] = cur.q2.x & 0xFFFFu; qt[1] = cur.q2.x >> 16; qt[2] = cur.q2.y & 0xFFFFu; qt[3] = cur.q2.y >> 16;
    qm[0] = cur.m2.x & 0xFFFFu; qm[1] = cur.m2.x >> 16; qm[2] = cur.m2.y & 0xFFFFu; qm[3] = cur.m2.y >> 16;
#pragma unroll
    for (int k = 0; k < 4; ++k) { sp[k] = (cur.a >> (8 * k)) & 0xFFu; st[k] = (cur.c >> (8 * k)) & 0xFFu; fl[k] = (cur.f >> (8 * k)) & 0xFFu; }
    uint32_t sum_p = 0, sum_t = 0;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const bool in = k0 + k >= i0 && k0 + k < i1;               // clusters of neighbouring bins in the vector do not count
      sum_p += in ? pd[k] : 0u;
      sum_t += in ? td[k] : 0u;
      pd[k] = sum_p;
      td[k] = sum_t;
    }
    uint32_t tot_p, tot_t, ex_p, ex_t;
    if (NT == 32) {
      const uint32_t inc_p = warp_incl_scan(sum_p), inc_t = warp_incl_scan(sum_t);
      tot_p = __shfl_sync(0xffffffffu, inc_p, 31); tot_t = __shfl_sync(0xffffffffu, inc_t, 31);
      ex_p = carry_p + inc_p - sum_p; ex_t = carry_t + inc_t - sum_t;
    } else {
      block_excl_scan2(sum_p, sum_t, ws, &ex_p, &ex_t, &tot_p, &tot_t);
      ex_p += carry_p; ex_t += carry_t;
    }
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const uint32_t i = k0 + k;
      if (i >= i0 && i < i1 && dst0 + (i - i0) < A.n_clusters_total) {
        uint4 v;
        v.x = ex_t + td[k];
        v.y = ((ex_p + pd[k]) & 0xFFFFu) | (qt[k] << 16);
        v.z = qm[k] | (sp[k] << 16) | (st[k] << 24);
        v.w = fl[k] | tail;
        A.clusters[dst0 + (i - i0)] = v;
      }
    }
    carry_p += tot_p;
    carry_t += tot_t;
  }
}

// A block owns `bins_per_block` consecutive bins (1 for full time frames, UNATT_WARPS for frames with few clusters per
// bin: single events, batches of small frames).  Bins with more than UNATT_SMALL clusters are decoded by the whole block,
// one after the other (the decision is uniform over the block); the others by one warp each.
template <bool BATCH>
__global__ void __launch_bounds__(UNATT_THREADS) k_unattached(const __grid_constant__ DevGeo G, const __grid_constant__ FrameArgs F0,
                                                              const FrameArgs* __restrict__ table, uint32_t bins_per_block) {
  __shared__ uint32_t ws[66];
  const UnattachedArgs A = unattached_args(frame_of<BATCH>(F0, table, blockIdx.y));
  if (A.in.n_unattached == 0) return;
  const uint32_t b0 = blockIdx.x * bins_per_block, b1 = min(b0 + bins_per_block, G.n_bins);
  const uint32_t wid = threadIdx.x >> 5, lane = lane_id();
  for (uint32_t b = b0; b < b1; ++b) {
    const uint32_t n = A.u_start[b + 1] - A.u_start[b];
    const bool whole_block = n > UNATT_SMALL;
    if (whole_block || (b - b0) % UNATT_WARPS == wid)
      unattached_bin(G, A, b, whole_block ? threadIdx.x : lane, whole_block ? (uint32_t)UNATT_THREADS : 32u, ws);
  }
}

}  // namespace tmd
