// tmd_api.cu -- the C ABI of libtmd.so (include/tmd.h): context, workspace layout, kernel sequencing.
// Every step of the path runs in the kernels of this directory; the host code only checks arguments and enqueues.
#include <algorithm>
#include <new>
#include <stdlib.h>
#include <string.h>

#include "tmd_common.cuh"
#include "tmd_decode.cuh"
#include "tmd_encode.cuh"
#include "tmd_encode_unattached.cuh"
#include "tmd_rank.cuh"
#include "tmd_scan.cuh"
#include "tmd_scatter.cuh"
#include "tmd_sort.cuh"
#include "tmd_unattached.cuh"

using namespace tmd;

struct tmd_ctx {
  DevGeo geo;
  RowGeo* d_rows;
  int device;
  int n_sm;                    // cudaDevAttrMultiProcessorCount
  size_t smem_per_sm;          // cudaDevAttrMaxSharedMemoryPerMultiprocessor
  size_t smem_reserved;        // cudaDevAttrReservedSharedMemoryPerBlock
  size_t decode_smem, decode_smem_max, rank_smem, scatter_smem;
  // Per-call state.  `launches` is the launch count of the last tmd_decode / tmd_decode_batch (the same for every call
  // with the same flags and emptiness, so concurrent calls store the same value).  The TMD_TIMING event pairs and the
  // host-pipeline slots are the only other state a call touches: calls with TMD_TIMING, and the tmd_decode_host* entry
  // points, must not run concurrently on one context; plain tmd_decode calls on different streams may, with distinct
  // workspaces.
  int launches;
  cudaEvent_t ev_t0[TMD_MAX_KERNELS], ev_t1[TMD_MAX_KERNELS];
  const char* kernel_names[TMD_MAX_KERNELS];
  int timed_launches;
  bool events_created, timing_valid;
  // tmd_decode_host / tmd_decode_host_async: TMD_HOST_SLOTS frames in flight, each with its own device arena (inputs,
  // outputs, workspace; grown on demand); host->device copies, decode and device->host copies on three streams so that
  // the upload of one frame overlaps the download of the previous one (Fig. 2: transfers beside kernels)
  struct HostSlot {
    void* arena;
    size_t arena_bytes;
    cudaEvent_t h2d_done, dec_done, d2h_done;
    bool busy;
    uint32_t* h_err;            // pinned: error word of the slot's last container decode (tmd_decode_container_host_async)
    bool container;             // the frame in flight came from a container: tmd_host_wait looks at *h_err
  } slots[TMD_HOST_SLOTS];
  cudaStream_t s_h2d, s_dec, s_d2h;
  bool host_ready;
};

namespace {

constexpr size_t ALIGN = 256;
inline size_t align_up(size_t v) { return (v + ALIGN - 1) & ~(ALIGN - 1); }

// frames per k_store_frames launch: the table travels as a by-value kernel parameter (4 KB parameter space)
constexpr uint32_t STORE_FRAMES = 8;
struct FrameChunk { FrameArgs f[STORE_FRAMES]; };
static_assert(sizeof(FrameChunk) <= 3800, "k_store_frames parameters must fit the 4 KB parameter space");

Workspace layout(uint32_t n_bins, uint32_t n_tracks, uint64_t n_att, int n_sm) {
  Workspace w;
  w.n_tiles = (n_tracks + SCAN_TILE - 1) / SCAN_TILE;
  // Chunk size (a pure function of (n_att, SM count), so tmd_workspace_bytes and tmd_decode agree).  The rank kernel runs one
  // warp per chunk, 20 warps per SM: its time goes with ceil(chunks / warps) * chunk size.  The scatter writes one piece per
  // (chunk, bin): the smaller the chunk the shorter the pieces, measured 14 % per halving (c2, 2^14 -> 2^15: 0.80 -> 0.71 ms).
  // Cost model in units of "one cluster through the scatter at 2^15": a rank slot costs 6 of them.  Ties go to the larger chunk
  // (smaller tables).  c3, c4: 2^15; c2: 2^15 (was 2^14 under the round-1 rule "one chunk per resident warp"); c1: 2^11.
  const uint64_t rank_warps = (uint64_t)n_sm * 20;
  int shift = CHUNK_SHIFT_MAX;
  uint64_t best = ~0ull;
  for (int s = CHUNK_SHIFT_MAX; s >= CHUNK_SHIFT_MIN; --s) {
    const uint64_t chunks = (n_att + (1ull << s) - 1) >> s, rounds = (chunks + rank_warps - 1) / rank_warps;
    const uint64_t cost = rounds * (1ull << s) * 600 + n_att * (100 + 14 * (uint64_t)(CHUNK_SHIFT_MAX - s)) / 100;
    if (cost < best) { best = cost; shift = s; }
  }
  w.chunk_shift = (uint32_t)shift;
  w.n_chunks = (uint32_t)((n_att + (1ull << shift) - 1) >> shift);
  w.n_groups = (w.n_chunks + COL_GROUP - 1) / COL_GROUP;
  size_t o = 0;
  auto take = [&](size_t bytes) { size_t at = o; o += align_up(bytes); return at; };
  w.o_err = take(ERR_WORDS * 4);
  w.o_tile_sum = take(((size_t)w.n_tiles + 1) * 4);
  w.o_off = take(((size_t)n_tracks + 1) * 4);
  w.o_hdr = take((size_t)n_tracks * 16);      // per-track header records in load-balance order (A2), see tmd_sort.cuh
  w.o_hdr2 = take((size_t)n_tracks * 4);
  w.o_att_cnt = take((size_t)n_bins * 4);
  w.o_u_start = take(((size_t)n_bins + 1) * 4);
  w.o_gsum = take((size_t)w.n_groups * n_bins * 4);
  w.o_hist = take((size_t)w.n_chunks * n_bins * 2);
  w.o_start16 = take((size_t)w.n_chunks * sc_start_stride(n_bins) * 2);
  w.o_rel = take((size_t)w.n_chunks * n_bins * 4);
  w.o_rank16 = take((size_t)n_att * 2);
  w.o_inter = take((size_t)n_att * 8);
  w.o_table = take((size_t)TMD_MAX_BATCH * sizeof(FrameArgs));   // the frame table of a batch lives in frame 0's workspace
  w.total = o;
  return w;
}

inline bool misaligned(const void* p, size_t a) { return (reinterpret_cast<uintptr_t>(p) & (a - 1)) != 0; }

// the frame table of tmd_decode_batch: STORE_FRAMES entries per launch, passed by value
__global__ void k_store_frames(const __grid_constant__ FrameChunk C, FrameArgs* __restrict__ table, uint32_t first, uint32_t count) {
  const uint32_t words = sizeof(FrameArgs) / 4;
  static_assert(sizeof(FrameArgs) % 4 == 0, "FrameArgs is copied word by word");
  for (uint32_t i = threadIdx.x; i < count * words; i += blockDim.x)
    reinterpret_cast<uint32_t*>(table + first)[i] = reinterpret_cast<const uint32_t*>(C.f)[i];
}

// TMD_VALIDATE, part 1 (before anything indexes with the counts): per-track fields and the two totals.
// The sum of trk_ncl is taken in 64 bits (the 32-bit offsets wrap for malformed counts).
__global__ void k_validate(DevGeo G, tmd_compressed in, uint32_t* __restrict__ err) {
  __shared__ unsigned long long s_sum, s_ncl;
  if (threadIdx.x == 0) { s_sum = 0; s_ncl = 0; }
  __syncthreads();
  uint32_t bad = 0;
  unsigned long long ncl = 0;
  for (uint32_t t = blockIdx.x * blockDim.x + threadIdx.x; t < in.n_tracks; t += gridDim.x * blockDim.x) {
    const uint32_t n = in.trk_ncl[t];
    ncl += n;
    bad |= (n < 1) | (in.trk_row0[t] >= G.n_rows) | (in.trk_sec0[t] >= G.n_az * G.n_sides);
  }
  if (bad) atomicOr(&err[ERR_TRACK_FIELD], 1u);
  atomicAdd(&s_ncl, ncl);
  if (blockIdx.x == 0) {
    unsigned long long s = 0;
    for (uint32_t b = threadIdx.x; b < G.n_bins; b += blockDim.x) s += in.u_bin_count[b];
    atomicAdd(&s_sum, s);
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    atomicAdd(reinterpret_cast<unsigned long long*>(err + ERR_NCL_SUM_LO), s_ncl);
    if (blockIdx.x == 0 && s_sum != in.n_unattached) atomicOr(&err[ERR_TRACK_FIELD], 2u);
  }
}

int check_args(const tmd_ctx* ctx, const tmd_compressed* in, const tmd_output* out, bool device_side) {
  if (!ctx || !in || !out) return TMD_ERR_ARG;
  if (in->n_attached + in->n_unattached > TMD_MAX_CLUSTERS) return TMD_ERR_ARG;
  if (in->n_attached < in->n_tracks) return TMD_ERR_ARG;
  if ((in->n_tracks == 0) != (in->n_attached == 0)) return TMD_ERR_ARG;
  const bool has_trk = in->n_tracks > 0, has_res = in->n_attached > in->n_tracks, has_un = in->n_unattached > 0;
  const void* trk[] = {in->trk_ncl, in->trk_qpt, in->trk_row0, in->trk_sec0, in->trk_pad0, in->trk_time0,
                       in->a_qtot, in->a_qmax, in->a_flags, in->a_sigpad, in->a_sigtime};
  const void* res[] = {in->a_rowdiff, in->a_secleg, in->a_padres, in->a_timeres};
  const void* un[] = {in->u_qtot, in->u_qmax, in->u_flags, in->u_sigpad, in->u_sigtime, in->u_paddiff, in->u_timediff};
  for (const void* p : trk) if (has_trk && !p) return TMD_ERR_ARG;
  for (const void* p : res) if (has_res && !p) return TMD_ERR_ARG;
  for (const void* p : un) if (has_un && !p) return TMD_ERR_ARG;
  if (!in->u_bin_count || !out->bin_offset) return TMD_ERR_ARG;
  if ((in->n_attached + in->n_unattached) > 0 && !out->clusters) return TMD_ERR_ARG;
  if (device_side) {
    for (const void* p : trk) if (has_trk && misaligned(p, 16)) return TMD_ERR_ALIGN;
    for (const void* p : res) if (has_res && misaligned(p, 16)) return TMD_ERR_ALIGN;
    for (const void* p : un) if (has_un && misaligned(p, 16)) return TMD_ERR_ALIGN;
    if (misaligned(in->u_bin_count, 16) || misaligned(out->clusters, 16) || misaligned(out->bin_offset, 4) ||
        misaligned(out->probe_state, 4))
      return TMD_ERR_ALIGN;
  }
  return TMD_OK;
}

// argument / alignment / workspace checks of one frame and its FrameArgs
int make_frame(const tmd_ctx* ctx, const tmd_compressed* in, const tmd_output* out, uint32_t flags, FrameArgs* F) {
  int rc = check_args(ctx, in, out, true);
  if (rc != TMD_OK) return rc;
  const Workspace W = layout(ctx->geo.n_bins, in->n_tracks, in->n_attached, ctx->n_sm);
  if (!out->workspace || out->workspace_bytes < W.total) return TMD_ERR_WORKSPACE;
  if (misaligned(out->workspace, ALIGN)) return TMD_ERR_ALIGN;
  F->in = *in;
  F->clusters = (uint4*)out->clusters;
  F->bin_offset = out->bin_offset;
  F->probe_state = out->probe_state;
  F->probe_step = out->probe_step;
  F->validate = (flags & TMD_VALIDATE) ? 1u : 0u;
  F->ws = (unsigned char*)out->workspace;
  F->W = W;
  return TMD_OK;
}

#define TMD_CUDA(call)                                   \
  do {                                                   \
    if ((call) != cudaSuccess) return TMD_ERR_CUDA;      \
  } while (0)

// Launch bookkeeping: an event pair around the kernel with TMD_TIMING
struct Launcher {
  tmd_ctx* ctx;
  cudaStream_t st;
  bool timing;
  int n = 0;
  bool before() {
    return !(timing && n < TMD_MAX_KERNELS && cudaEventRecord(ctx->ev_t0[n], st) != cudaSuccess);
  }
  bool after(const char* name) {
    if (cudaGetLastError() != cudaSuccess) return false;
    if (timing && n < TMD_MAX_KERNELS) {
      ctx->kernel_names[n] = name;
      if (cudaEventRecord(ctx->ev_t1[n], st) != cudaSuccess) return false;
    }
    ++n;
    return true;
  }
};
#define TMD_LAUNCH(name, ...)                      \
  do {                                             \
    if (!L.before()) return TMD_ERR_CUDA;          \
    __VA_ARGS__;                                   \
    if (!L.after(name)) return TMD_ERR_CUDA;       \
  } while (0)

// The launch sequence of rows A1-A7 over `n_frames` frames.  BATCH = false: one frame, its FrameArgs
// passed by value.  BATCH = true: the frames' FrameArgs are in device memory (`table`) and every grid has a frame
// coordinate; `mx` holds the per-kernel maxima of the frames' grid extents.
struct Extents { uint32_t n_tiles, n_tracks, n_chunks, n_groups; uint64_t n_unattached; bool any_probe; uint32_t mean_len; };   // mean_len: attached clusters per track (all frames)

template <bool BATCH>
int enqueue(tmd_ctx* ctx, const FrameArgs& F0, const FrameArgs* table, uint32_t n_frames, const Extents& mx, Launcher& L) {
  const DevGeo& G = ctx->geo;
  const uint32_t n_bins = G.n_bins, nf = n_frames;
  cudaStream_t st = L.st;
  const uint32_t bin_blocks = (n_bins + 255) / 256;
  if (mx.n_tracks > 0) {
    // A1: track offsets
    TMD_LAUNCH("track_tile_sums", k_track_tile_sums<BATCH><<<dim3(mx.n_tiles, nf), SCAN_THREADS, 0, st>>>(F0, table));
    TMD_LAUNCH("scan_tile_sums", k_scan_tile_sums<BATCH><<<dim3(1, nf), 1024, 0, st>>>(F0, table));
    TMD_LAUNCH("track_offsets", k_track_offsets<BATCH><<<dim3(mx.n_tiles, nf), SCAN_THREADS, 0, st>>>(F0, table));
    // A2: load-balance order (counting sort by cluster count, longest first, inside windows of consecutive tracks)
    TMD_LAUNCH("len_sort_window",
               k_len_sort_window<BATCH><<<dim3((mx.n_tracks + SORT_WINDOW - 1) / SORT_WINDOW, nf), SORT_THREADS, 0, st>>>(F0, table));
    // A3 (walk) + A5: track-model decode -> intermediate records {T, P, bin} in g order
    // Blocks per SM: registers allow DECODE_BLOCKS_PER_SM = 6; for long tracks 5 are faster (c3 2.39 -> 2.28 ms, 4: 2.30, 7: 2.52,
    // 8: 2.62: every track in flight keeps five 128-byte lines alive in the L2 -- four streams and its output -- and 113 k tracks
    // x 5 lines overflow it: sectors are evicted between the two cells that share them), for short tracks 6 (c4 1.24 vs 1.28 ms:
    // more tracks start per unit of time).  The cap is set through the size of the dynamic shared memory.
    const dim3 dg((mx.n_tracks + DECODE_THREADS - 1) / DECODE_THREADS, nf);
    size_t dsm = ctx->decode_smem;
    if (mx.mean_len >= DECODE_LONG_TRACKS) {
      const size_t cap = ctx->smem_per_sm / DECODE_BLOCKS_PER_SM - ctx->smem_reserved + 128;   // DECODE_BLOCKS_PER_SM blocks of this size do not fit
      if (cap > dsm && cap <= ctx->decode_smem_max) dsm = cap;
    }
    if (mx.any_probe) TMD_LAUNCH("track_decode", k_track_decode<true, BATCH><<<dg, DECODE_THREADS, dsm, st>>>(G, F0, table));
    else TMD_LAUNCH("track_decode", k_track_decode<false, BATCH><<<dg, DECODE_THREADS, dsm, st>>>(G, F0, table));
    // A3 (count): per-chunk histogram + ranks; one warp per chunk, as many warps resident as shared memory allows
    uint32_t per_sm = (uint32_t)(ctx->smem_per_sm / (ctx->rank_smem + 1024));
    if (per_sm < 1) per_sm = 1;
    if (per_sm > 16) per_sm = 16;
    uint32_t rank_blocks = (mx.n_chunks + WR_WARPS - 1) / WR_WARPS;
    const uint32_t rank_cap = (per_sm * (uint32_t)ctx->n_sm + nf - 1) / nf;
    if (rank_blocks > rank_cap) rank_blocks = rank_cap;
    if (rank_blocks < 1) rank_blocks = 1;
    TMD_LAUNCH("rank", k_rank<BATCH><<<dim3(rank_blocks, nf), WR_THREADS, ctx->rank_smem, st>>>(G, F0, table));
    // A4: column scan over chunks
    TMD_LAUNCH("col_group_sums", k_col_group_sums<BATCH><<<dim3(bin_blocks, mx.n_groups, nf), 256, 0, st>>>(n_bins, F0, table));
  }
  // att_cnt (zero for a frame without tracks), then bin offsets
  TMD_LAUNCH("col_group_scan", k_col_group_scan<BATCH><<<dim3(bin_blocks, nf), 256, 0, st>>>(n_bins, F0, table));
  TMD_LAUNCH("bin_offsets", k_bin_offsets<BATCH><<<dim3(1, nf), 1024, 0, st>>>(n_bins, F0, table));
  if (mx.n_tracks > 0)
    TMD_LAUNCH("col_apply", k_col_apply<BATCH><<<dim3(bin_blocks, mx.n_groups, nf), 256, 0, st>>>(n_bins, F0, table));
  // A7: unattached clusters
  // A7: unattached clusters; a block per bin for full time frames, a warp per bin where bins hold few clusters
  const uint32_t un_bpb = mx.n_unattached / n_bins >= 512 ? 1u : (uint32_t)UNATT_WARPS;
  TMD_LAUNCH("unattached", k_unattached<BATCH><<<dim3((n_bins + un_bpb - 1) / un_bpb, nf), UNATT_THREADS, 0, st>>>(G, F0, table, un_bpb));
  if (mx.n_tracks > 0) {
    // A6: copy-through + scatter (a thread-block cluster of SC_CLUSTER CTAs per chunk)
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(mx.n_chunks * SC_CLUSTER, nf);
    cfg.blockDim = dim3(SC_THREADS);
    cfg.dynamicSmemBytes = ctx->scatter_smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = SC_CLUSTER; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    TMD_LAUNCH("scatter", if (cudaLaunchKernelEx(&cfg, k_scatter<BATCH>, G, F0, table) != cudaSuccess) return TMD_ERR_CUDA);
  }
  return TMD_OK;
}

int prepare_timing(tmd_ctx* ctx, bool timing) {
  ctx->timing_valid = false;
  if (timing && !ctx->events_created) {
    for (int i = 0; i < TMD_MAX_KERNELS; ++i) {
      TMD_CUDA(cudaEventCreate(&ctx->ev_t0[i]));
      TMD_CUDA(cudaEventCreate(&ctx->ev_t1[i]));
    }
    ctx->events_created = true;
  }
  return TMD_OK;
}

// tmd_selftest_ieee: the unchecked IEEE sequences of the decode kernel against the intrinsics they replace.
// counts[0]: sqrt_rn_safe vs __fsqrt_rn on EVERY binary32 pattern in [2^-100, 2^100];
// counts[1]: div_rn_safe vs __fdiv_rn on 2^log2_pairs hashed (dividend, divisor) pairs, |dividend| in [2^-40, 2^84],
//            |divisor| in [2^-10, 2^80], plus every combination of 16 edge mantissas and all exponents of those ranges;
// counts[2]: floor_clamp vs (int)clamp(floorf(w), 0, hi) on every binary32 pattern, both limits.
__device__ __forceinline__ uint32_t mix32(uint32_t x) {
  x ^= x >> 16; x *= 0x7feb352du; x ^= x >> 15; x *= 0x846ca68bu; x ^= x >> 16;
  return x;
}
__device__ __forceinline__ bool same_float(float a, float b) {
  return __float_as_uint(a) == __float_as_uint(b) || (a != a && b != b);
}
__device__ __forceinline__ bool div_agrees(float a, float b) { return same_float(div_rn_safe(a, b, recip_refined(b)), __fdiv_rn(a, b)); }

__global__ void k_selftest_ieee(uint32_t log2_pairs, unsigned long long* __restrict__ counts) {
  const uint64_t tid = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x, nthr = (uint64_t)gridDim.x * blockDim.x;
  unsigned long long bad_sqrt = 0, bad_div = 0, bad_floor = 0;
  for (uint64_t v = tid; v < (1ull << 32); v += nthr) {
    const float x = __uint_as_float((uint32_t)v);
    if (x >= 7.888609052210118e-31f && x <= 1.2676506002282294e30f) bad_sqrt += !same_float(sqrt_rn_safe(x), __fsqrt_rn(x));
    const uint32_t wantP = (uint32_t)(int)clampf(floorf(x), 0.0f, 65535.0f), wantT = (uint32_t)(int)clampf(floorf(x), 0.0f, 16777215.0f);
    bad_floor += (floor_clamp(x, 65535) != wantP) + (floor_clamp(x, 16777215) != wantT);
  }
  const uint64_t n_pairs = 1ull << log2_pairs;
  for (uint64_t v = tid; v < n_pairs; v += nthr) {
    const uint32_t h1 = mix32((uint32_t)v * 2u + 1u), h2 = mix32(h1 ^ (uint32_t)(v >> 31) ^ 0x9e3779b9u), h3 = mix32(h2 + 0x85ebca6bu);
    const uint32_t ea = 127u - 40u + h3 % 125u;            // dividend exponent 2^-40 .. 2^84
    const uint32_t eb = 127u - 10u + (h3 >> 8) % 91u;      // divisor exponent 2^-10 .. 2^80
    const float a = __uint_as_float((h1 & 0x807FFFFFu) | (ea << 23)), b = __uint_as_float((h2 & 0x807FFFFFu) | (eb << 23));
    bad_div += !div_agrees(a, b);
  }
  const uint32_t edge[16] = {0u, 1u, 2u, 0x7FFFFFu, 0x7FFFFEu, 0x400000u, 0x400001u, 0x3FFFFFu, 0x555555u, 0x2AAAAAu, 0x000FFFu, 0x7FF000u,
                             0x100000u, 0x600000u, 0x123456u, 0x654321u};
  for (uint64_t v = tid; v < 125ull * 91ull * 256ull * 4ull; v += nthr) {
    const uint32_t ia = (uint32_t)(v % 125), ib = (uint32_t)(v / 125 % 91), m = (uint32_t)(v / (125 * 91) % 256), sg = (uint32_t)(v / (125 * 91 * 256));
    const float a = __uint_as_float(edge[m & 15] | ((127u - 40u + ia) << 23) | ((sg & 1u) << 31));
    const float b = __uint_as_float(edge[m >> 4] | ((127u - 10u + ib) << 23) | ((sg >> 1) << 31));
    bad_div += !div_agrees(a, b);
  }
  if (bad_sqrt) atomicAdd(&counts[0], bad_sqrt);
  if (bad_div) atomicAdd(&counts[1], bad_div);
  if (bad_floor) atomicAdd(&counts[2], bad_floor);
}

template <typename K>
cudaError_t allow_smem(K kernel, size_t bytes) {
  return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}

}  // namespace

extern "C" {

int tmd_create(const tmd_geometry* g, const tmd_field* f, tmd_ctx** out_ctx) {
  if (!g || !f || !out_ctx) return TMD_ERR_ARG;
  if (!g->row_x || !g->row_padw || !g->row_inv_padw || !g->row_npads) return TMD_ERR_ARG;
  if (g->n_az < 1 || g->n_az > 63 || g->n_sides < 1 || g->n_sides > 2 || g->n_rows < 1 || g->n_rows > 255) return TMD_ERR_ARG;
  if (g->n_sectors_out < 1 || g->n_sectors_out > g->n_az * g->n_sides) return TMD_ERR_ARG;
  if ((uint64_t)g->n_sectors_out * g->n_rows > MAX_BINS) return TMD_ERR_ARG;
  // finite, bounded tables (bounds: tmd_decode.cuh TMD_GEO_*): they keep every magnitude of the model far from overflow
  if (!(fabsf(f->bz_tesla) <= TMD_MAX_BZ) || !(fabsf(g->cos_a) <= 1.0f) || !(fabsf(g->sin_a) <= 1.0f)) return TMD_ERR_ARG;
  for (uint32_t r = 0; r < g->n_rows; ++r) {
    if (!(fabsf(g->row_x[r]) <= TMD_GEO_MAX_X) || !(g->row_padw[r] >= TMD_GEO_MIN_PADW && g->row_padw[r] <= TMD_GEO_MAX_PADW) ||
        !(g->row_inv_padw[r] >= 1.0f / TMD_GEO_MAX_PADW && g->row_inv_padw[r] <= 1.0f / TMD_GEO_MIN_PADW))
      return TMD_ERR_ARG;
  }
  tmd_ctx* ctx = new (std::nothrow) tmd_ctx();
  if (!ctx) return TMD_ERR_CUDA;
  memset(ctx, 0, sizeof(*ctx));
  if (cudaGetDevice(&ctx->device) != cudaSuccess) { delete ctx; return TMD_ERR_CUDA; }
  RowGeo* h = (RowGeo*)malloc(sizeof(RowGeo) * g->n_rows);
  if (!h) { delete ctx; return TMD_ERR_CUDA; }
  for (uint32_t r = 0; r < g->n_rows; ++r) {
    h[r].x = g->row_x[r];
    h[r].padw = g->row_padw[r];
    h[r].inv_padw = g->row_inv_padw[r];
    h[r].half = (float)(g->row_npads[r] / 2);   // exact in binary32
  }
  cudaError_t e = cudaMalloc(&ctx->d_rows, sizeof(RowGeo) * g->n_rows);
  if (e == cudaSuccess) e = cudaMemcpy(ctx->d_rows, h, sizeof(RowGeo) * g->n_rows, cudaMemcpyHostToDevice);
  free(h);
  int smem_sm = 0;
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&ctx->n_sm, cudaDevAttrMultiProcessorCount, ctx->device);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&smem_sm, cudaDevAttrMaxSharedMemoryPerMultiprocessor, ctx->device);
  ctx->smem_per_sm = (size_t)smem_sm;
  int smem_res = 0;
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&smem_res, cudaDevAttrReservedSharedMemoryPerBlock, ctx->device);
  ctx->smem_reserved = (size_t)smem_res;
  const uint32_t n_bins_c = g->n_sectors_out * g->n_rows;
  ctx->rank_smem = (size_t)WR_WARPS * wr_warp_smem(n_bins_c);
  ctx->scatter_smem = sc_smem_bytes(n_bins_c);
  ctx->decode_smem = decode_smem_bytes(g->n_rows);
  // The dynamic shared-memory limit is a per-function, process-wide attribute: always set it to the maximum any geometry
  // can need (MAX_BINS bins, 255 rows), so that contexts of different geometries never lower it for one another.
  const size_t rank_max = (size_t)WR_WARPS * wr_warp_smem(MAX_BINS), scatter_max = sc_smem_bytes(MAX_BINS);
  // (the decode kernel may be launched with more than it needs: that is how its blocks per SM are capped, see enqueue)
  const size_t decode_max = std::max(decode_smem_bytes(255), ctx->smem_per_sm / (DECODE_BLOCKS_PER_SM - 1) - ctx->smem_reserved);
  ctx->decode_smem_max = decode_max;
  if (e == cudaSuccess) e = allow_smem(k_rank<false>, rank_max);
  if (e == cudaSuccess) e = allow_smem(k_rank<true>, rank_max);
  if (e == cudaSuccess) e = allow_smem(k_scatter<false>, scatter_max);
  if (e == cudaSuccess) e = allow_smem(k_scatter<true>, scatter_max);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_scatter<false>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_scatter<true>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
  if (e == cudaSuccess) e = allow_smem(k_track_decode<false, false>, decode_max);
  if (e == cudaSuccess) e = allow_smem(k_track_decode<true, false>, decode_max);
  if (e == cudaSuccess) e = allow_smem(k_track_decode<false, true>, decode_max);
  if (e == cudaSuccess) e = allow_smem(k_track_decode<true, true>, decode_max);
  if (e != cudaSuccess) {
    cudaGetLastError();
    tmd_destroy(ctx);
    return TMD_ERR_CUDA;
  }
  {  // the scatter kernel needs a thread-block cluster of SC_CLUSTER CTAs: say so here, not at the first decode
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(SC_CLUSTER);
    cfg.blockDim = dim3(SC_THREADS);
    cfg.dynamicSmemBytes = ctx->scatter_smem;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = SC_CLUSTER; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    int n_clusters = 0;
    if (cudaOccupancyMaxActiveClusters(&n_clusters, k_scatter<false>, &cfg) != cudaSuccess || n_clusters < 1) {
      cudaGetLastError();
      tmd_destroy(ctx);
      return TMD_ERR_DEVICE;
    }
  }
  DevGeo& G = ctx->geo;
  G.n_az = g->n_az; G.n_sides = g->n_sides; G.n_sectors_out = g->n_sectors_out; G.n_rows = g->n_rows;
  G.n_bins = g->n_sectors_out * g->n_rows;
  G.cos_a = g->cos_a; G.sin_a = g->sin_a;
  // KB = bz * 0.00299792458f; QK = 0.0625f * KB: two single binary32 multiplications (volatile: no folding into one)
  volatile float kb = f->bz_tesla * 0.00299792458f;
  volatile float qk = 0.0625f * kb;
  G.qk = qk;
  G.rows = ctx->d_rows;
  G.rows_magic = (1u << 24) / g->n_rows + 1u;
  G.az_magic = (1u << 24) / g->n_az + 1u;
  *out_ctx = ctx;
  return TMD_OK;
}

int tmd_workspace_bytes(const tmd_ctx* ctx, uint32_t n_tracks, uint64_t n_att, uint64_t n_unatt, size_t* out_bytes) {
  if (!ctx || !out_bytes) return TMD_ERR_ARG;
  if (n_att + n_unatt > TMD_MAX_CLUSTERS || n_att < n_tracks) return TMD_ERR_ARG;
  *out_bytes = layout(ctx->geo.n_bins, n_tracks, n_att, ctx->n_sm).total;
  return TMD_OK;
}

int tmd_decode(tmd_ctx* ctx, const tmd_compressed* in, tmd_output* out, uint32_t flags, void* cuda_stream) {
  FrameArgs F;
  int rc = make_frame(ctx, in, out, flags, &F);
  if (rc != TMD_OK) return rc;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const bool validate = (flags & TMD_VALIDATE) != 0, timing = (flags & TMD_TIMING) != 0;
  rc = prepare_timing(ctx, timing);
  if (rc != TMD_OK) return rc;
  uint32_t* d_err = F.at<uint32_t>(F.W.o_err);
  if (validate) {
    // part 1, before anything indexes with the counts: per-track fields, sum(trk_ncl) in 64 bits, sum(u_bin_count)
    uint32_t h_err[ERR_WORDS];
    TMD_CUDA(cudaMemsetAsync(d_err, 0, ERR_WORDS * 4, st));
    k_validate<<<ctx->n_sm, 256, 0, st>>>(ctx->geo, *in, d_err);
    TMD_CUDA(cudaGetLastError());
    TMD_CUDA(cudaMemcpyAsync(h_err, d_err, sizeof(h_err), cudaMemcpyDeviceToHost, st));
    TMD_CUDA(cudaStreamSynchronize(st));
    const uint64_t ncl_sum = (uint64_t)h_err[ERR_NCL_SUM_LO] | ((uint64_t)h_err[ERR_NCL_SUM_HI] << 32);
    if (h_err[ERR_TRACK_FIELD] || ncl_sum != in->n_attached) return TMD_ERR_CORRUPT;
    TMD_CUDA(cudaMemsetAsync(d_err, 0, ERR_WORDS * 4, st));
  }
  Launcher L{ctx, st, timing};
  const Extents mx = {F.W.n_tiles, in->n_tracks, F.W.n_chunks, F.W.n_groups, in->n_unattached, out->probe_state != nullptr,
                      in->n_tracks ? (uint32_t)(in->n_attached / in->n_tracks) : 0u};
  rc = enqueue<false>(ctx, F, nullptr, 1, mx, L);
  ctx->launches = L.n + (validate ? 1 : 0);
  if (rc != TMD_OK) return rc;
  ctx->timed_launches = L.n;
  ctx->timing_valid = timing;
  if (validate) {   // part 2: a decoded sector without output bins (reading 20)
    uint32_t h_err[ERR_WORDS];
    TMD_CUDA(cudaMemcpyAsync(h_err, d_err, sizeof(h_err), cudaMemcpyDeviceToHost, st));
    TMD_CUDA(cudaStreamSynchronize(st));
    if (h_err[ERR_TRACK_FIELD] || h_err[ERR_SECTOR_OUT]) return TMD_ERR_CORRUPT;
  }
  return TMD_OK;
}

int tmd_decode_batch(tmd_ctx* ctx, uint32_t n_frames, const tmd_compressed* in, tmd_output* out, uint32_t flags, void* cuda_stream) {
  if (!ctx || !in || !out || n_frames < 1 || n_frames > TMD_MAX_BATCH) return TMD_ERR_ARG;
  if (flags & TMD_VALIDATE) return TMD_ERR_ARG;          // it synchronises: validate frames one by one with tmd_decode
  if (n_frames == 1) return tmd_decode(ctx, in, out, flags, cuda_stream);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const bool timing = (flags & TMD_TIMING) != 0;
  int rc = prepare_timing(ctx, timing);
  if (rc != TMD_OK) return rc;
  Extents mx = {0, 0, 0, 0, 0, false, 0};
  FrameArgs* table = nullptr;
  FrameChunk chunk;
  // Chunk size of the batch: the one a single frame holding ALL the attached clusters would get (larger than any
  // frame's own, so its tables fit the frame's workspace): a batch has chunks enough with every frame cut coarsely.
  uint64_t att_total = 0;
  uint64_t trk_total = 0;
  for (uint32_t i = 0; i < n_frames; ++i) { att_total += in[i].n_attached; trk_total += in[i].n_tracks; }
  mx.mean_len = trk_total ? (uint32_t)(att_total / trk_total) : 0u;
  const uint32_t batch_shift = layout(ctx->geo.n_bins, 0, att_total, ctx->n_sm).chunk_shift;
  auto make_batch_frame = [&](uint32_t i, FrameArgs* F) -> int {
    const int r = make_frame(ctx, &in[i], &out[i], flags, F);
    if (r != TMD_OK) return r;
    if (batch_shift > F->W.chunk_shift) {
      F->W.chunk_shift = batch_shift;
      F->W.n_chunks = (uint32_t)((in[i].n_attached + (1ull << batch_shift) - 1) >> batch_shift);
      F->W.n_groups = (F->W.n_chunks + COL_GROUP - 1) / COL_GROUP;
    }
    return TMD_OK;
  };
  // every frame is checked before anything is enqueued
  for (uint32_t i = 0; i < n_frames; ++i) {
    FrameArgs F;
    rc = make_batch_frame(i, &F);
    if (rc != TMD_OK) return rc;
    if (i == 0) table = F.at<FrameArgs>(F.W.o_table);
    mx.n_tiles = mx.n_tiles > F.W.n_tiles ? mx.n_tiles : F.W.n_tiles;
    mx.n_tracks = mx.n_tracks > in[i].n_tracks ? mx.n_tracks : in[i].n_tracks;
    mx.n_chunks = mx.n_chunks > F.W.n_chunks ? mx.n_chunks : F.W.n_chunks;
    mx.n_groups = mx.n_groups > F.W.n_groups ? mx.n_groups : F.W.n_groups;
    mx.n_unattached = mx.n_unattached > in[i].n_unattached ? mx.n_unattached : in[i].n_unattached;
    mx.any_probe = mx.any_probe || out[i].probe_state != nullptr;
  }
  Launcher L{ctx, st, timing};
  // The frame table goes up STORE_FRAMES entries per launch.  With TMD_TIMING the whole upload is ONE timed row
  // ("store_frames"): a pair per launch would use up the TMD_MAX_KERNELS pairs at ~100 frames and push the decode
  // kernels off the end of tmd_kernel_times.
  int store_launches = 0;
  if (!L.before()) return TMD_ERR_CUDA;
  for (uint32_t first = 0; first < n_frames; first += STORE_FRAMES) {
    const uint32_t count = n_frames - first < STORE_FRAMES ? n_frames - first : STORE_FRAMES;
    for (uint32_t k = 0; k < count; ++k) make_batch_frame(first + k, &chunk.f[k]);
    k_store_frames<<<1, 256, 0, st>>>(chunk, table, first, count);
    ++store_launches;
  }
  if (!L.after("store_frames")) return TMD_ERR_CUDA;
  rc = enqueue<true>(ctx, chunk.f[0], table, n_frames, mx, L);
  ctx->launches = L.n + store_launches - 1;      // L counted the upload as one
  if (rc != TMD_OK) return rc;
  ctx->timed_launches = L.n;
  ctx->timing_valid = timing;
  return TMD_OK;
}

int tmd_kernel_times(tmd_ctx* ctx, int max_kernels, const char** names, float* ms) {
  if (!ctx || !names || !ms || max_kernels < 0) return TMD_ERR_ARG;
  if (!ctx->timing_valid) return 0;
  const int n = ctx->timed_launches < TMD_MAX_KERNELS ? ctx->timed_launches : TMD_MAX_KERNELS;
  int k = 0;
  for (; k < n && k < max_kernels; ++k) {
    names[k] = ctx->kernel_names[k];
    if (cudaEventSynchronize(ctx->ev_t1[k]) != cudaSuccess) return TMD_ERR_CUDA;
    if (cudaEventElapsedTime(&ms[k], ctx->ev_t0[k], ctx->ev_t1[k]) != cudaSuccess) return TMD_ERR_CUDA;
  }
  return k;
}

int tmd_encode_attached(tmd_ctx* ctx, const tmd_attached_truth* in, tmd_compressed* out, void* workspace, size_t workspace_bytes,
                        void* cuda_stream) {
  if (!ctx || !in || !out) return TMD_ERR_ARG;
  if (in->n_attached > TMD_MAX_CLUSTERS || in->n_attached < in->n_tracks) return TMD_ERR_ARG;
  if (in->n_tracks == 0) return in->n_attached == 0 ? TMD_OK : TMD_ERR_ARG;
  if (!in->trk_ncl || !in->trk_qptf || !in->att || !in->leg) return TMD_ERR_ARG;
  void* outs[] = {(void*)out->trk_qpt, (void*)out->trk_row0, (void*)out->trk_sec0, (void*)out->trk_pad0, (void*)out->trk_time0,
                  (void*)out->a_qtot, (void*)out->a_qmax, (void*)out->a_flags, (void*)out->a_sigpad, (void*)out->a_sigtime};
  for (void* p : outs) if (!p) return TMD_ERR_ARG;
  if (in->n_attached > in->n_tracks && (!out->a_rowdiff || !out->a_secleg || !out->a_padres || !out->a_timeres)) return TMD_ERR_ARG;
  if (misaligned(in->trk_ncl, 16) || misaligned(in->att, 16)) return TMD_ERR_ALIGN;
  const Workspace W = layout(ctx->geo.n_bins, in->n_tracks, in->n_attached, ctx->n_sm);
  if (!workspace || workspace_bytes < W.total) return TMD_ERR_WORKSPACE;
  if (misaligned(workspace, ALIGN)) return TMD_ERR_ALIGN;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  FrameArgs F;
  memset(&F, 0, sizeof(F));
  F.in.n_tracks = in->n_tracks; F.in.n_attached = in->n_attached; F.in.trk_ncl = in->trk_ncl;
  F.ws = (unsigned char*)workspace;
  F.W = W;
  uint32_t* d_err = F.at<uint32_t>(W.o_err);
  uint32_t* d_off = F.at<uint32_t>(W.o_off);
  if (cudaMemsetAsync(d_err, 0, ERR_WORDS * 4, st) != cudaSuccess) return TMD_ERR_CUDA;
  k_track_tile_sums<false><<<W.n_tiles, SCAN_THREADS, 0, st>>>(F, nullptr);
  k_scan_tile_sums<false><<<1, 1024, 0, st>>>(F, nullptr);
  k_track_offsets<false><<<W.n_tiles, SCAN_THREADS, 0, st>>>(F, nullptr);
  EncodeArgs E;
  E.n_tracks = in->n_tracks; E.off = d_off; E.trk_qptf = in->trk_qptf; E.att = (const uint4*)in->att; E.leg = in->leg;
  E.trk_qpt = (int8_t*)out->trk_qpt; E.trk_row0 = (uint8_t*)out->trk_row0; E.trk_sec0 = (uint8_t*)out->trk_sec0;
  E.trk_pad0 = (uint16_t*)out->trk_pad0; E.trk_time0 = (uint32_t*)out->trk_time0;
  E.a_qtot = (uint16_t*)out->a_qtot; E.a_qmax = (uint16_t*)out->a_qmax; E.a_flags = (uint8_t*)out->a_flags;
  E.a_sigpad = (uint8_t*)out->a_sigpad; E.a_sigtime = (uint8_t*)out->a_sigtime;
  E.a_rowdiff = (uint8_t*)out->a_rowdiff; E.a_secleg = (uint8_t*)out->a_secleg;
  E.a_padres = (uint16_t*)out->a_padres; E.a_timeres = (uint32_t*)out->a_timeres;
  E.err = d_err;
  k_encode_attached<<<(in->n_tracks + 127) / 128, 128, sizeof(RowGeo) * ctx->geo.n_rows, st>>>(ctx->geo, E);
  if (cudaGetLastError() != cudaSuccess) return TMD_ERR_CUDA;
  uint32_t h_err[ERR_WORDS + 1];
  if (cudaMemcpyAsync(h_err, d_err, ERR_WORDS * 4, cudaMemcpyDeviceToHost, st) != cudaSuccess) return TMD_ERR_CUDA;
  if (cudaMemcpyAsync(&h_err[ERR_WORDS], d_off + in->n_tracks, 4, cudaMemcpyDeviceToHost, st) != cudaSuccess) return TMD_ERR_CUDA;
  if (cudaStreamSynchronize(st) != cudaSuccess) return TMD_ERR_CUDA;
  if (h_err[ERR_TRACK_FIELD] || h_err[ERR_WORDS] != (uint32_t)in->n_attached) return TMD_ERR_CORRUPT;
  return TMD_OK;
}

namespace {
struct UnWorkspace { size_t o_err, o_bin_start, o_tile_start, o_cursor, o_max_tiles, o_buf_a, o_buf_b, total; };
UnWorkspace un_layout(uint32_t n_bins, uint64_t n_un) {
  UnWorkspace w;
  size_t o = 0;
  auto take = [&](size_t bytes) { size_t at = o; o += align_up(bytes); return at; };
  w.o_err = take(ERR_WORDS * 4);
  w.o_bin_start = take(((size_t)n_bins + 1) * 4);
  w.o_tile_start = take(((size_t)n_bins + 1) * 4);
  w.o_cursor = take((size_t)n_bins * 4);
  w.o_max_tiles = take(4);
  w.o_buf_a = take((size_t)n_un * 16);
  w.o_buf_b = take((size_t)n_un * 16);
  w.total = o;
  return w;
}
}  // namespace

int tmd_encode_unattached_workspace_bytes(const tmd_ctx* ctx, uint64_t n_unattached, size_t* out_bytes) {
  if (!ctx || !out_bytes || n_unattached > TMD_MAX_CLUSTERS) return TMD_ERR_ARG;
  *out_bytes = un_layout(ctx->geo.n_bins, n_unattached).total;
  return TMD_OK;
}

int tmd_encode_unattached(tmd_ctx* ctx, uint64_t n_unattached, const tmd_cluster* un, tmd_compressed* out, void* workspace,
                          size_t workspace_bytes, void* cuda_stream) {
  if (!ctx || !out || n_unattached > TMD_MAX_CLUSTERS || !out->u_bin_count) return TMD_ERR_ARG;
  if (n_unattached > 0 && (!un || !out->u_qtot || !out->u_qmax || !out->u_flags || !out->u_sigpad || !out->u_sigtime || !out->u_paddiff ||
                           !out->u_timediff))
    return TMD_ERR_ARG;
  if (misaligned(un, 16)) return TMD_ERR_ALIGN;
  const uint32_t n_bins = ctx->geo.n_bins, n_un = (uint32_t)n_unattached;
  const UnWorkspace W = un_layout(n_bins, n_unattached);
  if (!workspace || workspace_bytes < W.total) return TMD_ERR_WORKSPACE;
  if (misaligned(workspace, ALIGN)) return TMD_ERR_ALIGN;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  unsigned char* ws = (unsigned char*)workspace;
  UnEncodeArgs A;
  A.n_un = n_un; A.n_bins = n_bins; A.n_rows = ctx->geo.n_rows;
  A.un = (const uint4*)un;
  A.bin_count = (uint32_t*)out->u_bin_count;
  A.bin_start = (uint32_t*)(ws + W.o_bin_start); A.tile_start = (uint32_t*)(ws + W.o_tile_start);
  A.cursor = (uint32_t*)(ws + W.o_cursor); A.max_tiles = (uint32_t*)(ws + W.o_max_tiles);
  A.buf_a = (uint4*)(ws + W.o_buf_a); A.buf_b = (uint4*)(ws + W.o_buf_b);
  uint32_t* d_err = (uint32_t*)(ws + W.o_err);
  TMD_CUDA(cudaMemsetAsync(d_err, 0, ERR_WORDS * 4, st));
  TMD_CUDA(cudaMemsetAsync(A.bin_count, 0, (size_t)n_bins * 4, st));
  const uint32_t stream_blocks = (uint32_t)ctx->n_sm * 8;
  if (n_un > 0) k_un_count<<<stream_blocks, 256, 0, st>>>(A, d_err);
  k_un_offsets<<<1, 1024, 0, st>>>(A);
  TMD_CUDA(cudaGetLastError());
  uint32_t h_err[ERR_WORDS], h_max_tiles = 0;
  TMD_CUDA(cudaMemcpyAsync(h_err, d_err, sizeof(h_err), cudaMemcpyDeviceToHost, st));
  TMD_CUDA(cudaMemcpyAsync(&h_max_tiles, A.max_tiles, 4, cudaMemcpyDeviceToHost, st));
  TMD_CUDA(cudaStreamSynchronize(st));
  if (h_err[ERR_TRACK_FIELD]) return TMD_ERR_CORRUPT;       // a row / sector without an output bin
  if (n_un == 0) return TMD_OK;
  static_assert((size_t)UN_TILE * 16 <= 48 * 1024, "below the default dynamic shared-memory limit: no per-function attribute needed");
  const uint32_t tile_bound = n_un / UN_TILE + n_bins;      // >= number of tiles; surplus blocks return at once
  k_un_bucket<<<stream_blocks, 256, 0, st>>>(A);
  k_un_sort_tiles<<<tile_bound, UN_THREADS, (size_t)UN_TILE * 16, st>>>(A);
  const uint4* src = A.buf_a;
  uint4* dst = A.buf_b;
  for (uint32_t p = 0; (1u << p) < h_max_tiles; ++p) {      // runs of 2^p tiles -> runs of 2^(p+1) tiles
    k_un_merge<<<tile_bound, UN_THREADS, (size_t)UN_TILE * 16, st>>>(A, src, dst, p);
    const uint4* t = src; src = dst; dst = (uint4*)t;
  }
  UnDiffOut O;
  O.u_qtot = (uint16_t*)out->u_qtot; O.u_qmax = (uint16_t*)out->u_qmax; O.u_flags = (uint8_t*)out->u_flags;
  O.u_sigpad = (uint8_t*)out->u_sigpad; O.u_sigtime = (uint8_t*)out->u_sigtime;
  O.u_paddiff = (uint16_t*)out->u_paddiff; O.u_timediff = (uint32_t*)out->u_timediff;
  k_un_diff<<<stream_blocks, 256, 0, st>>>(A, src, O);
  TMD_CUDA(cudaGetLastError());
  TMD_CUDA(cudaStreamSynchronize(st));
  return TMD_OK;
}

// the three streams of the host pipeline (uploads, decode, downloads), created on first use
static int host_streams(tmd_ctx* ctx) {
  if (!ctx->host_ready) {
    TMD_CUDA(cudaStreamCreateWithFlags(&ctx->s_h2d, cudaStreamNonBlocking));
    TMD_CUDA(cudaStreamCreateWithFlags(&ctx->s_dec, cudaStreamNonBlocking));
    TMD_CUDA(cudaStreamCreateWithFlags(&ctx->s_d2h, cudaStreamNonBlocking));
    ctx->host_ready = true;
  }
  return TMD_OK;
}

// Enqueue one host-to-host decode in slot `slot`: copies in on `s_in`, decode on `s_run`, copies out on `s_out` (the three
// may be the same stream), ordered by the slot's events.  Does not wait for the result.
// With `blob` (a TMDZ container in HOST memory) the inputs are not the arrays of `in` but the container: it alone is copied
// to the device, the entropy stage decodes it into the slot's arrays on `s_run`, and tmd_decode follows on the same stream.
static int host_enqueue(tmd_ctx* ctx, const tmd_compressed* in, const void* blob, size_t blob_bytes, tmd_output* out, uint32_t flags,
                        int slot, cudaStream_t s_in, cudaStream_t s_run, cudaStream_t s_out) {
  int rc;
  tmd_compressed counts;                         // container path: the counts of its header, no pointers
  if (blob) {
    if (!ctx || !out || !out->bin_offset) return TMD_ERR_ARG;
    memset(&counts, 0, sizeof(counts));
    uint32_t z_bins = 0;
    size_t z_total = 0;
    rc = tmd_entropy_sizes(blob, blob_bytes, &counts.n_tracks, &counts.n_attached, &counts.n_unattached, &z_bins, &z_total);
    if (rc != TMD_OK) return rc;
    if (z_total > blob_bytes || z_total < TMD_ENTROPY_HEAD_BYTES) return TMD_ERR_CORRUPT;
    if (z_bins != ctx->geo.n_bins) return TMD_ERR_ARG;                      // written for another geometry
    if (counts.n_attached + counts.n_unattached > TMD_MAX_CLUSTERS) return TMD_ERR_ARG;
    if ((counts.n_tracks == 0) != (counts.n_attached == 0)) return TMD_ERR_CORRUPT;
    if (counts.n_attached + counts.n_unattached > 0 && !out->clusters) return TMD_ERR_ARG;
    blob_bytes = z_total;
    in = &counts;
  } else {
    rc = check_args(ctx, in, out, false);
    if (rc != TMD_OK) return rc;
  }
  tmd_ctx::HostSlot& S = ctx->slots[slot];
  if (!S.h2d_done) {
    TMD_CUDA(cudaEventCreateWithFlags(&S.h2d_done, cudaEventDisableTiming));
    TMD_CUDA(cudaEventCreateWithFlags(&S.dec_done, cudaEventDisableTiming));
    TMD_CUDA(cudaEventCreateWithFlags(&S.d2h_done, cudaEventDisableTiming));
  }
  if (blob && !S.h_err) TMD_CUDA(cudaHostAlloc((void**)&S.h_err, 4, cudaHostAllocDefault));
  const uint32_t n_bins = ctx->geo.n_bins;
  const size_t n_trk = in->n_tracks, n_att = in->n_attached, n_res = n_att - n_trk, n_un = in->n_unattached;
  const Workspace W = layout(n_bins, in->n_tracks, n_att, ctx->n_sm);
  // arena: inputs, outputs, workspace
  struct Seg { const void* src; size_t bytes; size_t at; };
  Seg segs[] = {
      {in->trk_ncl, n_trk * 2, 0},   {in->trk_qpt, n_trk, 0},      {in->trk_row0, n_trk, 0},    {in->trk_sec0, n_trk, 0},
      {in->trk_pad0, n_trk * 2, 0},  {in->trk_time0, n_trk * 4, 0},
      {in->a_rowdiff, n_res, 0},     {in->a_secleg, n_res, 0},     {in->a_padres, n_res * 2, 0}, {in->a_timeres, n_res * 4, 0},
      {in->a_qtot, n_att * 2, 0},    {in->a_qmax, n_att * 2, 0},   {in->a_flags, n_att, 0},     {in->a_sigpad, n_att, 0},
      {in->a_sigtime, n_att, 0},
      {in->u_qtot, n_un * 2, 0},     {in->u_qmax, n_un * 2, 0},    {in->u_flags, n_un, 0},      {in->u_sigpad, n_un, 0},
      {in->u_sigtime, n_un, 0},      {in->u_paddiff, n_un * 2, 0}, {in->u_timediff, n_un * 4, 0},
      {in->u_bin_count, (size_t)n_bins * 4, 0}};
  size_t o = 0;
  for (Seg& s : segs) { s.at = o; o += align_up(s.bytes); }
  const size_t o_clusters = o; o += align_up((n_att + n_un) * 16);
  const size_t o_binoff = o;   o += align_up(((size_t)n_bins + 1) * 4);
  const size_t o_probe = o;    o += align_up(out->probe_state ? n_trk * 24 : 0);
  const size_t o_ws = o;       o += W.total;
  const size_t o_blob = o;     o += align_up(blob ? blob_bytes : 0);
  const size_t o_err = o;      o += align_up(blob ? 4 : 0);
  if (S.busy) {                                   // the slot's previous frame must have left the arena
    TMD_CUDA(cudaEventSynchronize(S.d2h_done));
    S.busy = false;
  }
  if (o > S.arena_bytes) {
    if (S.arena) cudaFree(S.arena);
    S.arena = nullptr; S.arena_bytes = 0;
    if (cudaMalloc(&S.arena, o) != cudaSuccess) { cudaGetLastError(); return TMD_ERR_CUDA; }
    S.arena_bytes = o;
  }
  unsigned char* a = (unsigned char*)S.arena;
  if (blob) {
    TMD_CUDA(cudaMemcpyAsync(a + o_blob, blob, blob_bytes, cudaMemcpyHostToDevice, s_in));
  } else {
    for (const Seg& s : segs)
      if (s.bytes) TMD_CUDA(cudaMemcpyAsync(a + s.at, s.src, s.bytes, cudaMemcpyHostToDevice, s_in));
  }
  tmd_compressed d = *in;
  const void** dst[] = {(const void**)&d.trk_ncl, (const void**)&d.trk_qpt, (const void**)&d.trk_row0, (const void**)&d.trk_sec0,
                        (const void**)&d.trk_pad0, (const void**)&d.trk_time0, (const void**)&d.a_rowdiff, (const void**)&d.a_secleg,
                        (const void**)&d.a_padres, (const void**)&d.a_timeres, (const void**)&d.a_qtot, (const void**)&d.a_qmax,
                        (const void**)&d.a_flags, (const void**)&d.a_sigpad, (const void**)&d.a_sigtime, (const void**)&d.u_qtot,
                        (const void**)&d.u_qmax, (const void**)&d.u_flags, (const void**)&d.u_sigpad, (const void**)&d.u_sigtime,
                        (const void**)&d.u_paddiff, (const void**)&d.u_timediff, (const void**)&d.u_bin_count};
  for (size_t i = 0; i < sizeof(segs) / sizeof(segs[0]); ++i) *dst[i] = a + segs[i].at;
  tmd_output dout = *out;
  dout.clusters = (tmd_cluster*)(a + o_clusters);
  dout.bin_offset = (uint32_t*)(a + o_binoff);
  dout.probe_state = out->probe_state ? (uint32_t*)(a + o_probe) : nullptr;
  dout.workspace = a + o_ws;
  dout.workspace_bytes = W.total;
  if (s_run != s_in) {
    TMD_CUDA(cudaEventRecord(S.h2d_done, s_in));
    TMD_CUDA(cudaStreamWaitEvent(s_run, S.h2d_done, 0));
  }
  if (blob) {   // entropy stage on the decode stream: container -> the slot's arrays (the header is read from the HOST copy)
    rc = tmd_entropy_decode(blob, TMD_ENTROPY_HEAD_BYTES, a + o_blob, blob_bytes, &d, a + o_err, (void*)s_run);
    if (rc != TMD_OK) return rc;
  }
  rc = tmd_decode(ctx, &d, &dout, flags, (void*)s_run);
  if (rc != TMD_OK) return rc;
  if (s_out != s_run) {
    TMD_CUDA(cudaEventRecord(S.dec_done, s_run));
    TMD_CUDA(cudaStreamWaitEvent(s_out, S.dec_done, 0));
  }
  if (n_att + n_un) TMD_CUDA(cudaMemcpyAsync(out->clusters, dout.clusters, (n_att + n_un) * 16, cudaMemcpyDeviceToHost, s_out));
  TMD_CUDA(cudaMemcpyAsync(out->bin_offset, dout.bin_offset, ((size_t)n_bins + 1) * 4, cudaMemcpyDeviceToHost, s_out));
  if (out->probe_state && n_trk)
    TMD_CUDA(cudaMemcpyAsync(out->probe_state, dout.probe_state, n_trk * 24, cudaMemcpyDeviceToHost, s_out));
  if (blob) TMD_CUDA(cudaMemcpyAsync(S.h_err, a + o_err, 4, cudaMemcpyDeviceToHost, s_out));
  S.container = blob != nullptr;
  TMD_CUDA(cudaEventRecord(S.d2h_done, s_out));
  S.busy = true;
  return TMD_OK;
}

int tmd_decode_host(tmd_ctx* ctx, const tmd_compressed* in, tmd_output* out, uint32_t flags, void* cuda_stream) {
  if (!ctx) return TMD_ERR_ARG;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int rc = host_enqueue(ctx, in, nullptr, 0, out, flags, 0, st, st, st);
  if (rc != TMD_OK) return rc;
  return tmd_host_wait(ctx, 0);
}

int tmd_decode_host_async(tmd_ctx* ctx, const tmd_compressed* in, tmd_output* out, uint32_t flags, int slot) {
  if (!ctx || slot < 0 || slot >= TMD_HOST_SLOTS || (flags & TMD_VALIDATE)) return TMD_ERR_ARG;
  const int rc_s = host_streams(ctx);
  if (rc_s != TMD_OK) return rc_s;
  return host_enqueue(ctx, in, nullptr, 0, out, flags, slot, ctx->s_h2d, ctx->s_dec, ctx->s_d2h);
}

int tmd_decode_container_host_async(tmd_ctx* ctx, const void* blob, size_t blob_bytes, tmd_output* out, uint32_t flags, int slot) {
  if (!ctx || !blob || slot < 0 || slot >= TMD_HOST_SLOTS || (flags & TMD_VALIDATE)) return TMD_ERR_ARG;
  if (blob_bytes < TMD_ENTROPY_HEAD_BYTES) return TMD_ERR_ARG;
  const int rc = host_streams(ctx);
  if (rc != TMD_OK) return rc;
  return host_enqueue(ctx, nullptr, blob, blob_bytes, out, flags, slot, ctx->s_h2d, ctx->s_dec, ctx->s_d2h);
}

int tmd_host_wait(tmd_ctx* ctx, int slot) {
  if (!ctx || slot < 0 || slot >= TMD_HOST_SLOTS) return TMD_ERR_ARG;
  tmd_ctx::HostSlot& S = ctx->slots[slot];
  if (!S.busy) return TMD_OK;
  TMD_CUDA(cudaEventSynchronize(S.d2h_done));
  S.busy = false;
  if (S.container && *S.h_err) return TMD_ERR_CORRUPT;      // the entropy stage found the container damaged
  return TMD_OK;
}

int tmd_selftest_ieee(uint32_t log2_pairs, uint64_t mismatches[3]) {
  if (!mismatches || log2_pairs > 40) return TMD_ERR_ARG;
  unsigned long long* d = nullptr;
  int n_sm = 0, dev = 0;
  TMD_CUDA(cudaGetDevice(&dev));
  TMD_CUDA(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
  TMD_CUDA(cudaMalloc(&d, 3 * sizeof(unsigned long long)));
  cudaError_t e = cudaMemset(d, 0, 3 * sizeof(unsigned long long));
  if (e == cudaSuccess) {
    k_selftest_ieee<<<n_sm * 8, 256>>>(log2_pairs, d);
    e = cudaGetLastError();
  }
  unsigned long long h[3] = {0, 0, 0};
  if (e == cudaSuccess) e = cudaMemcpy(h, d, sizeof(h), cudaMemcpyDeviceToHost);
  cudaFree(d);
  if (e != cudaSuccess) return TMD_ERR_CUDA;
  for (int i = 0; i < 3; ++i) mismatches[i] = h[i];
  return TMD_OK;
}

int tmd_destroy(tmd_ctx* ctx) {
  if (!ctx) return TMD_OK;
  for (tmd_ctx::HostSlot& S : ctx->slots) {
    if (S.busy) cudaEventSynchronize(S.d2h_done);
    if (S.arena) cudaFree(S.arena);
    if (S.h2d_done) { cudaEventDestroy(S.h2d_done); cudaEventDestroy(S.dec_done); cudaEventDestroy(S.d2h_done); }
    if (S.h_err) cudaFreeHost(S.h_err);
  }
  if (ctx->host_ready) { cudaStreamDestroy(ctx->s_h2d); cudaStreamDestroy(ctx->s_dec); cudaStreamDestroy(ctx->s_d2h); }
  if (ctx->d_rows) cudaFree(ctx->d_rows);
  if (ctx->events_created)
    for (int i = 0; i < TMD_MAX_KERNELS; ++i) { cudaEventDestroy(ctx->ev_t0[i]); cudaEventDestroy(ctx->ev_t1[i]); }
  delete ctx;
  return TMD_OK;
}

const char* tmd_status_string(int status) {
  switch (status) {
    case TMD_OK: return "ok";
    case TMD_ERR_ARG: return "bad argument";
    case TMD_ERR_ALIGN: return "misaligned pointer";
    case TMD_ERR_WORKSPACE: return "workspace missing or too small";
    case TMD_ERR_CUDA: return "CUDA runtime error";
    case TMD_ERR_CORRUPT: return "inconsistent compressed input";
    case TMD_ERR_DEVICE: return "device cannot run the kernels (thread-block clusters of 8 CTAs)";
    case TMD_ERR_LIMIT: return "sizes exceed the built-in scratch of the no-allocation entry point";
    default: return "unknown status";
  }
}

int tmd_last_launch_count(const tmd_ctx* ctx) { return ctx ? ctx->launches : 0; }

}  // extern "C"
