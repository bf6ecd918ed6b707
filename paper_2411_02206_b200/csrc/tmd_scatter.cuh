// tmd_scatter.cuh -- A6: copy-through of the charge / width / flag fields and the deterministic scatter of the attached
// clusters into canonical order (DESIGN.md §3 reading 11):
//   position(g) = rel[g >> chunk_shift][bin(g)] + rank16[g]
// with bin(g), T, P from the track-decode kernel's intermediate record, rank16 from the rank kernel (tmd_rank.cuh) and
// rel from the column scan (tmd_scan.cuh).  Integer / byte moves only.
//
// Every input stream is read coalesced in g.  What bounded the first version (one thread per cluster, a 16-byte store
// each: 3.51 ms at c3) was measured to be the half-sector stores spread over the whole output: with sequential store
// addresses the same kernel ran at 6.2 TB/s, with whole-sector stores a third faster.  Hence the sort
// through distributed shared memory below.
#pragma once

#include <cooperative_groups.h>

#include "tmd_common.cuh"
#include "tmd_rank.cuh"
#include "tmd_scan.cuh"

namespace tmd {

namespace cg = cooperative_groups;

// Streamed loads of the scatter: read-only path, kept in the L1 (evict_last).  Measured on c3: L1::no_allocate
// or ld.global.cg 3.09 ms, evict_first 2.86, default 2.82, evict_last 2.79.
#define LDPOL "L1::evict_last"
__device__ __forceinline__ uint4 ldx(const uint4* p) { uint4 v; asm volatile("ld.global.nc." LDPOL ".v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p)); return v; }
__device__ __forceinline__ uint2 ldx(const uint2* p) { uint2 v; asm volatile("ld.global.nc." LDPOL ".v2.u32 {%0,%1}, [%2];" : "=r"(v.x), "=r"(v.y) : "l"(p)); return v; }
__device__ __forceinline__ uint32_t ldx(const uint32_t* p) { uint32_t v; asm volatile("ld.global.nc." LDPOL ".u32 %0, [%1];" : "=r"(v) : "l"(p)); return v; }
#undef LDPOL
struct ScatterArgs {
  const uint2* inter;       // [n_attached] {T, P | bin << 16}
  const uint16_t* rank16;   // [n_attached]
  const uint32_t* rel;      // [n_chunks][n_bins]
  const uint16_t* start16;  // [n_chunks][start_stride] first slot of every bin in the chunk's (bin, rank) order; [n_bins] = total
  const uint16_t* a_qtot; const uint16_t* a_qmax; const uint8_t* a_flags; const uint8_t* a_sigpad; const uint8_t* a_sigtime;
  uint4* clusters;
  uint32_t n_attached, n_clusters_total, chunk_shift, start_stride;
};


__device__ __forceinline__ uint4 pack_cluster(uint32_t T, uint32_t P, uint32_t qtot, uint32_t qmax, uint32_t sigpad, uint32_t sigtime,
                                              uint32_t flags, uint32_t row, uint32_t sec) {
  uint4 v;
  v.x = T;
  v.y = P | (qtot << 16);
  v.z = qmax | (sigpad << 16) | (sigtime << 24);
  v.w = flags | (row << 8) | (sec << 16);
  return v;
}

// ---- scatter through distributed shared memory -----------------------------------------------------------------------
// A thread-block cluster of SC_CLUSTER = 8 CTAs owns one chunk.  The chunk's records are first sorted by (bin, rank) INSIDE
// the cluster: record g goes to slot start[bin] + rank16[g] of a 2^chunk_shift-record array that is spread over the shared
// memories of the 8 CTAs (start = exclusive scan of the chunk's histogram row, from the rank kernel; the store is a DSMEM store,
// st.shared::cluster).  After a cluster barrier every CTA writes its part of the sorted array: records of one bin are now
// neighbours, so the ~6 records a chunk adds to a bin leave as one contiguous piece and most 32-byte sectors are written
// whole.  Measured: 16-byte stores that fill half a sector are what bounded the one-thread-per-cluster
// scatter (a partial-sector write is a read-modify-write in the ECC-protected L2).
constexpr int SC_CLUSTER = 8;                       // CTAs per cluster.  Measured at c3: 16 CTAs x 2048 records, 5 CTAs per SM 2.64 ms (a cluster of 16 needs
constexpr int SC_CLUSTER_SHIFT = 3;                 // 16 free CTA slots in ONE GPC: 38 resident clusters = 608 of 740 slots); 8 x 4096, 3 per SM 2.54; 4 x 8192 4.10
constexpr int SC_THREADS = 256;
constexpr int SC_UNROLL = 4;                       // records per thread and batch (the vector loads below are written for 4)
constexpr uint32_t SC_MAX_PER_CTA = (1u << CHUNK_SHIFT_MAX) / SC_CLUSTER;   // 4096 records = 64 KB

__host__ __device__ inline size_t sc_smem_bytes(uint32_t n_bins) { return (size_t)SC_MAX_PER_CTA * 16 + (size_t)sc_start_stride(n_bins) * 2; }

__device__ __forceinline__ ScatterArgs scatter_args(const FrameArgs& F, uint32_t n_bins) {
  ScatterArgs A;
  A.inter = F.at<uint2>(F.W.o_inter); A.rank16 = F.at<uint16_t>(F.W.o_rank16); A.rel = F.at<uint32_t>(F.W.o_rel);
  A.start16 = F.at<uint16_t>(F.W.o_start16);
  A.a_qtot = F.in.a_qtot; A.a_qmax = F.in.a_qmax; A.a_flags = F.in.a_flags; A.a_sigpad = F.in.a_sigpad; A.a_sigtime = F.in.a_sigtime;
  A.clusters = F.clusters;
  A.n_attached = (uint32_t)F.in.n_attached; A.n_clusters_total = (uint32_t)(F.in.n_attached + F.in.n_unattached);
  A.chunk_shift = F.W.chunk_shift; A.start_stride = sc_start_stride(n_bins);
  return A;
}

template <bool BATCH>
__global__ void __launch_bounds__(SC_THREADS, 3) k_scatter(const __grid_constant__ DevGeo G, const __grid_constant__ FrameArgs F0,
                                                           const FrameArgs* __restrict__ table) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const FrameArgs& F = frame_of<BATCH>(F0, table, blockIdx.y);
  if ((blockIdx.x >> SC_CLUSTER_SHIFT) >= F.W.n_chunks) return;     // uniform over the cluster: nobody is left waiting
  const ScatterArgs A = scatter_args(F, G.n_bins);
  uint4* recs = reinterpret_cast<uint4*>(smem_raw);                                   // this CTA's part of the sorted chunk
  const uint32_t recs_addr = (uint32_t)__cvta_generic_to_shared(smem_raw);
  uint16_t* start = reinterpret_cast<uint16_t*>(smem_raw + (size_t)SC_MAX_PER_CTA * 16);  // [n_bins + 1] first slot of every bin
  cg::cluster_group cluster = cg::this_cluster();
  const uint32_t rank_in_cluster = cluster.block_rank();
  const uint32_t c = blockIdx.x >> SC_CLUSTER_SHIFT, tid = threadIdx.x, n_bins = G.n_bins;
  const uint32_t per_shift = A.chunk_shift - SC_CLUSTER_SHIFT, per_cta = 1u << per_shift;
  // ---- arrival of the sorted records is tracked by a transaction barrier in every CTA: a remote store (st.async) completes
  // 16 bytes on the DESTINATION's barrier, and a CTA waits only until the bytes of ITS part have landed -- no cluster-wide
  // barrier with release semantics (MEMBAR.ALL.GPU + ERRBAR + the wait for the slowest CTA: 26 % of the stall samples).
  __shared__ __align__(8) unsigned long long mbar;
  const uint32_t mbar_addr = (uint32_t)__cvta_generic_to_shared(&mbar);
  if (tid == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(mbar_addr) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  // This chunk's row of `rel` is looked up in the write-out phase, a few microseconds from now, in a dependent load in front of
  // every store: each CTA asks for its share of it into the L2 now.
  {
    const uint32_t row_lines = (n_bins * 4u + 127u) >> 7, per = (row_lines + SC_CLUSTER - 1) / SC_CLUSTER, l = rank_in_cluster * per + tid;
    if (tid < per && l < row_lines) asm volatile("prefetch.global.L2 [%0];" ::"l"(reinterpret_cast<const unsigned char*>(A.rel + (size_t)c * n_bins) + l * 128u));
  }
  // "this CTA is running and its barrier exists": waited for just before the first remote store
  asm volatile("barrier.cluster.arrive.relaxed.aligned;" ::: "memory");     // (the mbarrier_init fence above is the release it needs)
  // ---- this CTA's share of g: loads in flight before the cluster barrier
  const uint32_t g_base = (c << A.chunk_shift) + (rank_in_cluster << per_shift);
  bool first = true;
  uint32_t local_bytes = 0;                            // bytes of the records this thread stored into its own CTA's part
  for (uint32_t i0 = 0; i0 < per_cta; i0 += SC_THREADS * SC_UNROLL) {
    uint2 rec[SC_UNROLL];
    uint32_t rk[SC_UNROLL], qt[SC_UNROLL], qm[SC_UNROLL], sp[SC_UNROLL], st[SC_UNROLL], fl[SC_UNROLL];
    // thread tid takes the SC_UNROLL = 4 consecutive records i0 + 4 tid .. + 3: every stream is read with ONE vector load per
    // thread (two for the 8-byte records) instead of one narrow load per record and stream
    const uint32_t ib = i0 + tid * SC_UNROLL, gb = g_base + ib;
#pragma unroll
    for (int k = 0; k < SC_UNROLL; ++k) rec[k] = make_uint2(0u, 0xFFFF0000u);
    if (ib < per_cta && gb + SC_UNROLL <= A.n_attached) {        // (per_cta is a multiple of 4 * 32: whole groups of four)
      const uint4 r01 = ldx(reinterpret_cast<const uint4*>(A.inter + gb)), r23 = ldx(reinterpret_cast<const uint4*>(A.inter + gb) + 1);
      const uint2 rk2 = ldx(reinterpret_cast<const uint2*>(A.rank16 + gb));
      const uint2 qt2 = ldx(reinterpret_cast<const uint2*>(A.a_qtot + gb)), qm2 = ldx(reinterpret_cast<const uint2*>(A.a_qmax + gb));
      const uint32_t sp4 = ldx(reinterpret_cast<const uint32_t*>(A.a_sigpad + gb)), st4 = ldx(reinterpret_cast<const uint32_t*>(A.a_sigtime + gb));
      const uint32_t fl4 = ldx(reinterpret_cast<const uint32_t*>(A.a_flags + gb));
      rec[0] = make_uint2(r01.x, r01.y); rec[1] = make_uint2(r01.z, r01.w); rec[2] = make_uint2(r23.x, r23.y); rec[3] = make_uint2(r23.z, r23.w);
      rk[0] = rk2.x & 0xFFFFu; rk[1] = rk2.x >> 16; rk[2] = rk2.y & 0xFFFFu; rk[3] = rk2.y >> 16;
      qt[0] = qt2.x & 0xFFFFu; qt[1] = qt2.x >> 16; qt[2] = qt2.y & 0xFFFFu; qt[3] = qt2.y >> 16;
      qm[0] = qm2.x & 0xFFFFu; qm[1] = qm2.x >> 16; qm[2] = qm2.y & 0xFFFFu; qm[3] = qm2.y >> 16;
#pragma unroll
      for (int k = 0; k < SC_UNROLL; ++k) {
        sp[k] = (sp4 >> (8 * k)) & 0xFFu; st[k] = (st4 >> (8 * k)) & 0xFFu; fl[k] = (fl4 >> (8 * k)) & 0xFFu;
      }
    } else if (ib < per_cta) {                                    // the last records of the frame
#pragma unroll
      for (int k = 0; k < SC_UNROLL; ++k) {
        const uint32_t g = gb + k;
        if (g < A.n_attached) {
          rec[k] = __ldg(A.inter + g);
          rk[k] = __ldg(A.rank16 + g); qt[k] = __ldg(A.a_qtot + g); qm[k] = __ldg(A.a_qmax + g);
          sp[k] = __ldg(A.a_sigpad + g); st[k] = __ldg(A.a_sigtime + g); fl[k] = __ldg(A.a_flags + g);
        }
      }
    }
    if (first) {
      // start[bin]: the chunk's row of the table the rank kernel wrote (every CTA keeps a copy); requested AFTER the first
      // batch of record loads so that its latency overlaps theirs
      const uint4* src = reinterpret_cast<const uint4*>(A.start16 + (size_t)c * A.start_stride);
      for (uint32_t i = tid; i < A.start_stride / 8; i += SC_THREADS) cp_async16(reinterpret_cast<uint4*>(start) + i, src + i, 16);
      cp_async_commit();
      cp_async_wait<0>();                            // (asynchronous copies: no registers held next to the record loads)
      __syncthreads();                               // start[] visible
      asm volatile("barrier.cluster.wait.aligned;" ::: "memory");   // every CTA of the cluster is running (they arrived before their loads)
      first = false;
    }
#pragma unroll
    for (int k = 0; k < SC_UNROLL; ++k) {
      const uint32_t bin = rec[k].y >> 16;
      if (bin == BIN_INVALID) continue;              // no output bin (reading 20), or past the end
      const uint32_t sec = (bin * G.rows_magic) >> 24, row = bin - sec * G.n_rows;
      const uint32_t slot = (uint32_t)start[bin] + rk[k];
      const uint4 v = pack_cluster(rec[k].x, rec[k].y & 0xFFFFu, qt[k], qm[k], sp[k], st[k], fl[k], row, sec);
      const uint32_t dst_cta = slot >> per_shift;
      if (dst_cta == rank_in_cluster) {                 // stays in this CTA: a plain shared-memory store instead of a request on the
        recs[slot & (per_cta - 1)] = v;                 // SM's crossbar port (what bounds this kernel); its bytes are counted below
        local_bytes += 16u;
        continue;
      }
      uint32_t r_addr, r_mbar;
      asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r_addr) : "r"(recs_addr + ((slot & (per_cta - 1)) << 4)), "r"(dst_cta));
      asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r_mbar) : "r"(mbar_addr), "r"(dst_cta));
      asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v4.b32 [%0], {%1, %2, %3, %4}, [%5];" ::"r"(r_addr),
                   "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w), "r"(r_mbar)
                   : "memory");
    }
  }
  // ---- wait until this CTA's part of the sorted chunk is complete (phase 0 of the transaction barrier).  The expected byte
  // count is posted only now (the remote completions may come first: the barrier's pending count goes negative meanwhile)
  if (local_bytes) asm volatile("mbarrier.complete_tx.relaxed.cta.shared::cta.b64 [%0], %1;" ::"r"(mbar_addr), "r"(local_bytes) : "memory");
  const uint32_t my_first = rank_in_cluster << per_shift;
  const uint32_t n_valid = start[n_bins];                           // records of the chunk that have a bin (last entry of the row)
  const uint32_t n_expected = n_valid > my_first ? min(n_valid - my_first, per_cta) : 0u;   // records that land here
  if (tid == 0) asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mbar_addr), "r"(n_expected * 16u) : "memory");
  if (n_expected) {
    uint32_t done = 0;
    while (!done)
      asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0; selp.u32 %0, 1, 0, p; }" : "=r"(done) : "r"(mbar_addr) : "memory");
  }
  __syncthreads();                                     // the locally stored records are visible to every thread of the CTA
  // ---- this CTA's part of the sorted chunk to its canonical positions
  const uint32_t* __restrict__ rel_row = A.rel + (size_t)c * n_bins;
  uint4* __restrict__ out = A.clusters;
  for (uint32_t i0 = 0; i0 < per_cta; i0 += SC_THREADS * SC_UNROLL) {
    uint4 v[SC_UNROLL];
    uint32_t pos[SC_UNROLL];
#pragma unroll
    for (int k = 0; k < SC_UNROLL; ++k) {                     // the lookups of the batch in flight together
      const uint32_t i = i0 + k * SC_THREADS + tid, p = (rank_in_cluster << per_shift) + i;
      pos[k] = 0xFFFFFFFFu;
      if (i < per_cta && p < n_valid) {
        v[k] = recs[i];
        const uint32_t bin = ((v[k].w >> 16) & 0xFFu) * G.n_rows + ((v[k].w >> 8) & 0xFFu);
        pos[k] = __ldg(rel_row + bin) + (p - (uint32_t)start[bin]);
      }
    }
#pragma unroll
    for (int k = 0; k < SC_UNROLL; ++k)
      if (pos[k] < A.n_clusters_total) out[pos[k]] = v[k];
  }
}

}  // namespace tmd
