// tmd_api.cu -- the C ABI of libtmd.so (include/tmd.h): context, workspace layout, kernel sequencing.
// Every step of the path runs in the kernels of this directory; the host code only checks arguments and enqueues.
#include <new>
#include <stdlib.h>
#include <string.h>

#include "tmd_common.cuh"
#include "tmd_decode.cuh"
#include "tmd_encode.cuh"
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
  int launches;
  // Second stream of tmd_decode: the unattached clusters (A7) are decoded there while the attached ones are scattered
  // (A6) on the caller's stream.
  cudaStream_t side;
  cudaEvent_t ev_fork, ev_join;
  // TMD_TIMING: one event pair around every kernel of the last tmd_decode, recorded on the stream it ran on
  cudaEvent_t ev_t0[TMD_MAX_KERNELS], ev_t1[TMD_MAX_KERNELS];
  const char* kernel_names[TMD_MAX_KERNELS];
  bool events_created, timing_valid;
  // tmd_decode_host / tmd_decode_host_async: TMD_HOST_SLOTS frames in flight, each with its own device arena (inputs,
  // outputs, workspace; grown on demand); host->device copies, decode and device->host copies on three streams so that
  // the upload of one frame overlaps the download of the previous one (Fig. 2: transfers beside kernels)
  struct HostSlot {
    void* arena;
    size_t arena_bytes;
    cudaEvent_t h2d_done, dec_done, d2h_done;
    bool busy;
  } slots[TMD_HOST_SLOTS];
  cudaStream_t s_h2d, s_dec, s_d2h;
  bool host_ready;
  size_t decode_smem, rank_smem, scatter_smem;
  int n_sm;
};

namespace {

constexpr size_t ALIGN = 256;
inline size_t align_up(size_t v) { return (v + ALIGN - 1) & ~(ALIGN - 1); }

struct Workspace {
  uint32_t n_tiles, n_chunks, n_groups, chunk_shift;
  size_t o_err, o_tile_sum, o_off, o_perm, o_att_cnt, o_u_start, o_gsum, o_hist, o_start16, o_rel, o_rank16, o_inter, total;
};

Workspace layout(uint32_t n_bins, uint32_t n_tracks, uint64_t n_att) {
  Workspace w;
  w.n_tiles = (n_tracks + SCAN_TILE - 1) / SCAN_TILE;
  // chunk size: the largest power of two that still leaves about one chunk per resident warp of the rank kernel
  // (B200: 148 SMs x 20 warps); a pure function of n_att, so tmd_workspace_bytes and tmd_decode agree
  int shift = CHUNK_SHIFT_MIN;
  while (shift < CHUNK_SHIFT_MAX && (n_att >> (shift + 1)) >= 2960) ++shift;
  w.chunk_shift = (uint32_t)shift;
  w.n_chunks = (uint32_t)((n_att + (1ull << shift) - 1) >> shift);
  w.n_groups = (w.n_chunks + COL_GROUP - 1) / COL_GROUP;
  size_t o = 0;
  auto take = [&](size_t bytes) { size_t at = o; o += align_up(bytes); return at; };
  w.o_err = take(ERR_WORDS * 4);
  w.o_tile_sum = take(((size_t)w.n_tiles + 1) * 4);
  w.o_off = take(((size_t)n_tracks + 1) * 4);
  w.o_perm = take((size_t)n_tracks * 4);
  w.o_att_cnt = take((size_t)n_bins * 4);
  w.o_u_start = take(((size_t)n_bins + 1) * 4);
  w.o_gsum = take((size_t)w.n_groups * n_bins * 4);
  w.o_hist = take((size_t)w.n_chunks * n_bins * 2);
  w.o_start16 = take((size_t)w.n_chunks * sc_start_stride(n_bins) * 2);
  w.o_rel = take((size_t)w.n_chunks * n_bins * 4);
  w.o_rank16 = take((size_t)n_att * 2);
  w.o_inter = take((size_t)n_att * 8);
  w.total = o;
  return w;
}

inline bool misaligned(const void* p, size_t a) { return (reinterpret_cast<uintptr_t>(p) & (a - 1)) != 0; }

// TMD_VALIDATE, part 1 (before anything indexes with the counts): per-track fields and the two totals.
__global__ void k_validate(DevGeo G, tmd_compressed in, const uint32_t* __restrict__ off, uint32_t* __restrict__ err) {
  __shared__ unsigned long long s_sum;
  if (threadIdx.x == 0) s_sum = 0;
  __syncthreads();
  uint32_t bad = 0;
  for (uint32_t t = blockIdx.x * blockDim.x + threadIdx.x; t < in.n_tracks; t += gridDim.x * blockDim.x)
    bad |= (in.trk_ncl[t] < 1) | (in.trk_row0[t] >= G.n_rows) | (in.trk_sec0[t] >= G.n_az * G.n_sides);
  if (bad) atomicOr(&err[ERR_TRACK_FIELD], 1u);
  if (blockIdx.x == 0) {
    unsigned long long s = 0;
    for (uint32_t b = threadIdx.x; b < G.n_bins; b += blockDim.x) s += in.u_bin_count[b];
    atomicAdd(&s_sum, s);
    __syncthreads();
    if (threadIdx.x == 0) {
      if (s_sum != in.n_unattached) atomicOr(&err[ERR_TRACK_FIELD], 2u);
      if (in.n_tracks > 0 && off[in.n_tracks] != (uint32_t)in.n_attached) atomicOr(&err[ERR_TRACK_FIELD], 4u);
    }
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

// Launch bookkeeping: TMD_BEFORE(stream) ... kernel<<<>>> ... TMD_AFTER(name, stream)
#define TMD_BEFORE(stream)                                                                                  \
  do {                                                                                                      \
    if (timing && ctx->launches < TMD_MAX_KERNELS &&                                                        \
        cudaEventRecord(ctx->ev_t0[ctx->launches], stream) != cudaSuccess) return TMD_ERR_CUDA;             \
  } while (0)
#define TMD_AFTER(name, stream)                                                                             \
  do {                                                                                                      \
    if (cudaGetLastError() != cudaSuccess) return TMD_ERR_CUDA;                                             \
    if (timing && ctx->launches < TMD_MAX_KERNELS) {                                                        \
      ctx->kernel_names[ctx->launches] = name;                                                              \
      if (cudaEventRecord(ctx->ev_t1[ctx->launches], stream) != cudaSuccess) return TMD_ERR_CUDA;           \
    }                                                                                                       \
    ctx->launches++;                                                                                        \
  } while (0)
#define TMD_CUDA(call)                                   \
  do {                                                   \
    if ((call) != cudaSuccess) return TMD_ERR_CUDA;      \
  } while (0)

}  // namespace

extern "C" {

int tmd_create(const tmd_geometry* g, const tmd_field* f, tmd_ctx** out_ctx) {
  if (!g || !f || !out_ctx) return TMD_ERR_ARG;
  if (!g->row_x || !g->row_padw || !g->row_inv_padw || !g->row_npads) return TMD_ERR_ARG;
  if (g->n_az < 1 || g->n_az > 63 || g->n_sides < 1 || g->n_sides > 2 || g->n_rows < 1 || g->n_rows > 255) return TMD_ERR_ARG;
  if (g->n_sectors_out < 1 || g->n_sectors_out > g->n_az * g->n_sides) return TMD_ERR_ARG;
  if ((uint64_t)g->n_sectors_out * g->n_rows > MAX_BINS) return TMD_ERR_ARG;
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
  const uint32_t n_bins_c = g->n_sectors_out * g->n_rows;
  ctx->rank_smem = (size_t)WR_WARPS * wr_warp_smem(n_bins_c);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_rank, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ctx->rank_smem);
  ctx->scatter_smem = sc_smem_bytes(n_bins_c);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_scatter, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ctx->scatter_smem);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_scatter, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
  ctx->decode_smem = DECODE_STAGE_BYTES + sizeof(RowGeo) * g->n_rows;
  if (e == cudaSuccess)
    e = cudaFuncSetAttribute(k_track_decode<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ctx->decode_smem);
  if (e == cudaSuccess)
    e = cudaFuncSetAttribute(k_track_decode<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ctx->decode_smem);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&ctx->n_sm, cudaDevAttrMultiProcessorCount, ctx->device);
  if (e == cudaSuccess) {
    int lo = 0, hi = 0;   // numerically lowest = highest priority: the short integer kernels should not queue behind the decode
    e = cudaDeviceGetStreamPriorityRange(&lo, &hi);
    if (e == cudaSuccess) e = cudaStreamCreateWithPriority(&ctx->side, cudaStreamNonBlocking, hi);
  }
  if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->ev_fork, cudaEventDisableTiming);
  if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->ev_join, cudaEventDisableTiming);
  if (e != cudaSuccess) {
    cudaGetLastError();
    tmd_destroy(ctx);
    return TMD_ERR_CUDA;
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
  *out_bytes = layout(ctx->geo.n_bins, n_tracks, n_att).total;
  return TMD_OK;
}

int tmd_decode(tmd_ctx* ctx, const tmd_compressed* in, tmd_output* out, uint32_t flags, void* cuda_stream) {
  int rc = check_args(ctx, in, out, true);
  if (rc != TMD_OK) return rc;
  const DevGeo& G = ctx->geo;
  const uint32_t n_trk = in->n_tracks, n_bins = G.n_bins;
  const uint32_t n_att = (uint32_t)in->n_attached, n_un = (uint32_t)in->n_unattached;
  const Workspace W = layout(n_bins, n_trk, n_att);
  if (!out->workspace || out->workspace_bytes < W.total) return TMD_ERR_WORKSPACE;
  if (misaligned(out->workspace, ALIGN)) return TMD_ERR_ALIGN;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  unsigned char* ws = (unsigned char*)out->workspace;
  uint32_t* d_err = (uint32_t*)(ws + W.o_err);
  uint32_t* d_tile = (uint32_t*)(ws + W.o_tile_sum);
  uint32_t* d_off = (uint32_t*)(ws + W.o_off);
  uint32_t* d_perm = (uint32_t*)(ws + W.o_perm);
  uint32_t* d_attcnt = (uint32_t*)(ws + W.o_att_cnt);
  uint32_t* d_ustart = (uint32_t*)(ws + W.o_u_start);
  uint32_t* d_gsum = (uint32_t*)(ws + W.o_gsum);
  uint16_t* d_hist = (uint16_t*)(ws + W.o_hist);
  uint16_t* d_start16 = (uint16_t*)(ws + W.o_start16);
  uint32_t* d_rel = (uint32_t*)(ws + W.o_rel);
  uint16_t* d_rank = (uint16_t*)(ws + W.o_rank16);
  uint2* d_inter = (uint2*)(ws + W.o_inter);
  const bool validate = (flags & TMD_VALIDATE) != 0, timing = (flags & TMD_TIMING) != 0;
  cudaStream_t s2 = (flags & TMD_SERIAL) ? st : ctx->side;   // TMD_SERIAL: one stream, kernels back to back
  ctx->launches = 0;
  ctx->timing_valid = false;
  if (timing && !ctx->events_created) {
    for (int i = 0; i < TMD_MAX_KERNELS; ++i) {
      TMD_CUDA(cudaEventCreate(&ctx->ev_t0[i]));
      TMD_CUDA(cudaEventCreate(&ctx->ev_t1[i]));
    }
    ctx->events_created = true;
  }
  TMD_CUDA(cudaMemsetAsync(d_err, 0, ERR_WORDS * 4, st));

  if (n_trk > 0) {  // A1: track offsets
    TMD_BEFORE(st);
    k_track_tile_sums<<<W.n_tiles, SCAN_THREADS, 0, st>>>(in->trk_ncl, n_trk, d_tile);
    TMD_AFTER("track_tile_sums", st);
    TMD_BEFORE(st);
    k_scan_tile_sums<<<1, 1024, 0, st>>>(d_tile, W.n_tiles);
    TMD_AFTER("scan_tile_sums", st);
    TMD_BEFORE(st);
    k_track_offsets<<<W.n_tiles, SCAN_THREADS, 0, st>>>(in->trk_ncl, n_trk, d_tile, W.n_tiles, d_off);
    TMD_AFTER("track_offsets", st);
  }
  if (validate) {
    TMD_BEFORE(st);
    k_validate<<<ctx->n_sm, 256, 0, st>>>(G, *in, d_off, d_err);
    TMD_AFTER("validate", st);
    uint32_t h_err[ERR_WORDS];
    TMD_CUDA(cudaMemcpyAsync(h_err, d_err, sizeof(h_err), cudaMemcpyDeviceToHost, st));
    TMD_CUDA(cudaStreamSynchronize(st));
    if (h_err[ERR_TRACK_FIELD]) return TMD_ERR_CORRUPT;
  }
  if (n_trk > 0) {
    // A2: load-balance order (counting sort by cluster count, longest first, inside windows of consecutive tracks)
    TMD_BEFORE(st);
    k_len_sort_window<<<(n_trk + SORT_WINDOW - 1) / SORT_WINDOW, SORT_THREADS, 0, st>>>(in->trk_ncl, n_trk, d_perm);
    TMD_AFTER("len_sort_window", st);
    // A3 (walk) + A5: track-model decode -> intermediate records {T, P, bin} in g order
    DecodeArgs D;
    D.off = d_off; D.perm = d_perm; D.in = *in; D.inter = d_inter;
    D.probe_state = out->probe_state; D.probe_step = out->probe_step; D.err = d_err;
    TMD_BEFORE(st);
    const uint32_t decode_blocks = (n_trk + DECODE_THREADS - 1) / DECODE_THREADS;
    if (out->probe_state) k_track_decode<true><<<decode_blocks, DECODE_THREADS, ctx->decode_smem, st>>>(G, D);
    else k_track_decode<false><<<decode_blocks, DECODE_THREADS, ctx->decode_smem, st>>>(G, D);
    TMD_AFTER("track_decode", st);
    // A3 (count): per-chunk histogram + ranks; one warp per chunk, as many warps resident as shared memory allows
    RankArgs R;
    R.inter = d_inter; R.hist = d_hist; R.rank16 = d_rank; R.n_attached = n_att; R.n_chunks = W.n_chunks; R.chunk_shift = W.chunk_shift; R.start16 = d_start16; R.start_stride = sc_start_stride(n_bins);
    uint32_t per_sm = (uint32_t)((size_t)(227 * 1024) / (ctx->rank_smem + 1024));
    if (per_sm < 1) per_sm = 1;
    if (per_sm > 16) per_sm = 16;
    uint32_t rank_blocks = (W.n_chunks + WR_WARPS - 1) / WR_WARPS;
    if (rank_blocks > per_sm * (uint32_t)ctx->n_sm) rank_blocks = per_sm * (uint32_t)ctx->n_sm;
    TMD_BEFORE(st);
    k_rank<<<rank_blocks, WR_THREADS, ctx->rank_smem, st>>>(G, R);
    TMD_AFTER("rank", st);
    // A4: column scan over chunks
    dim3 cg((n_bins + 255) / 256, W.n_groups);
    TMD_BEFORE(st);
    k_col_group_sums<<<cg, 256, 0, st>>>(d_hist, W.n_chunks, n_bins, d_gsum);
    TMD_AFTER("col_group_sums", st);
    TMD_BEFORE(st);
    k_col_group_scan<<<(n_bins + 255) / 256, 256, 0, st>>>(d_gsum, W.n_groups, n_bins, d_attcnt);
    TMD_AFTER("col_group_scan", st);
  } else {
    TMD_CUDA(cudaMemsetAsync(d_attcnt, 0, (size_t)n_bins * 4, st));
  }
  TMD_BEFORE(st);
  k_bin_offsets<<<1, 1024, 0, st>>>(d_attcnt, in->u_bin_count, n_bins, out->bin_offset, d_ustart);
  TMD_AFTER("bin_offsets", st);
  if (n_trk > 0) {
    dim3 cg((n_bins + 255) / 256, W.n_groups);
    TMD_BEFORE(st);
    k_col_apply<<<cg, 256, 0, st>>>(d_hist, d_gsum, out->bin_offset, W.n_chunks, n_bins, d_rel);
    TMD_AFTER("col_apply", st);
  }
  // ---- fork: A7 (unattached clusters) on the context's second stream, next to A6 on the caller's
  const bool fork = n_un > 0 && n_trk > 0 && s2 != st;
  if (n_un > 0) {
    cudaStream_t su = fork ? s2 : st;
    if (fork) {
      TMD_CUDA(cudaEventRecord(ctx->ev_fork, st));
      TMD_CUDA(cudaStreamWaitEvent(s2, ctx->ev_fork, 0));
    }
    UnattachedArgs U;
    U.in = *in; U.u_start = d_ustart; U.bin_offset = out->bin_offset; U.att_cnt = d_attcnt;
    U.clusters = (uint4*)out->clusters; U.n_clusters_total = n_att + n_un;
    TMD_BEFORE(su);
    k_unattached<<<n_bins, UNATT_THREADS, 0, su>>>(G, U);
    TMD_AFTER("unattached", su);
    if (fork) TMD_CUDA(cudaEventRecord(ctx->ev_join, s2));
  }
  if (n_trk > 0) {
    // A6: copy-through + scatter
    ScatterArgs S;
    S.inter = d_inter; S.rank16 = d_rank; S.rel = d_rel;
    S.a_qtot = in->a_qtot; S.a_qmax = in->a_qmax; S.a_flags = in->a_flags; S.a_sigpad = in->a_sigpad; S.a_sigtime = in->a_sigtime;
    S.clusters = (uint4*)out->clusters; S.n_attached = n_att; S.n_clusters_total = n_att + n_un; S.chunk_shift = W.chunk_shift;
    S.start16 = d_start16; S.start_stride = sc_start_stride(n_bins);
    TMD_BEFORE(st);
    {
      cudaLaunchConfig_t cfg = {};
      cfg.gridDim = dim3(W.n_chunks * SC_CLUSTER);
      cfg.blockDim = dim3(SC_THREADS);
      cfg.dynamicSmemBytes = ctx->scatter_smem;
      cfg.stream = st;
      cudaLaunchAttribute attr[1];
      attr[0].id = cudaLaunchAttributeClusterDimension;
      attr[0].val.clusterDim.x = SC_CLUSTER; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
      cfg.attrs = attr;
      cfg.numAttrs = 1;
      if (cudaLaunchKernelEx(&cfg, k_scatter, G, S) != cudaSuccess) return TMD_ERR_CUDA;
    }
    TMD_AFTER("scatter", st);
  }
  if (fork) TMD_CUDA(cudaStreamWaitEvent(st, ctx->ev_join, 0));   // join: everything is ordered before later work on `st`
  ctx->timing_valid = timing;
  if (validate) {
    uint32_t h_err[ERR_WORDS];
    TMD_CUDA(cudaMemcpyAsync(h_err, d_err, sizeof(h_err), cudaMemcpyDeviceToHost, st));
    TMD_CUDA(cudaStreamSynchronize(st));
    if (h_err[ERR_TRACK_FIELD] || h_err[ERR_SECTOR_OUT]) return TMD_ERR_CORRUPT;
  }
  return TMD_OK;
}

int tmd_kernel_times(tmd_ctx* ctx, int max_kernels, const char** names, float* ms) {
  if (!ctx || !names || !ms || max_kernels < 0) return TMD_ERR_ARG;
  if (!ctx->timing_valid) return 0;
  const int n = ctx->launches < TMD_MAX_KERNELS ? ctx->launches : TMD_MAX_KERNELS;
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
  const Workspace W = layout(ctx->geo.n_bins, in->n_tracks, in->n_attached);
  if (!workspace || workspace_bytes < W.total) return TMD_ERR_WORKSPACE;
  if (misaligned(workspace, ALIGN)) return TMD_ERR_ALIGN;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  unsigned char* ws = (unsigned char*)workspace;
  uint32_t* d_err = (uint32_t*)(ws + W.o_err);
  uint32_t* d_tile = (uint32_t*)(ws + W.o_tile_sum);
  uint32_t* d_off = (uint32_t*)(ws + W.o_off);
  if (cudaMemsetAsync(d_err, 0, ERR_WORDS * 4, st) != cudaSuccess) return TMD_ERR_CUDA;
  k_track_tile_sums<<<W.n_tiles, SCAN_THREADS, 0, st>>>(in->trk_ncl, in->n_tracks, d_tile);
  k_scan_tile_sums<<<1, 1024, 0, st>>>(d_tile, W.n_tiles);
  k_track_offsets<<<W.n_tiles, SCAN_THREADS, 0, st>>>(in->trk_ncl, in->n_tracks, d_tile, W.n_tiles, d_off);
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

// Enqueue one host-to-host decode in slot `slot`: copies in on `s_in`, decode on `s_run`, copies out on `s_out` (the three
// may be the same stream), ordered by the slot's events.  Does not wait for the result.
static int host_enqueue(tmd_ctx* ctx, const tmd_compressed* in, tmd_output* out, uint32_t flags, int slot, cudaStream_t s_in,
                        cudaStream_t s_run, cudaStream_t s_out) {
  int rc = check_args(ctx, in, out, false);
  if (rc != TMD_OK) return rc;
  tmd_ctx::HostSlot& S = ctx->slots[slot];
  if (!S.h2d_done) {
    TMD_CUDA(cudaEventCreateWithFlags(&S.h2d_done, cudaEventDisableTiming));
    TMD_CUDA(cudaEventCreateWithFlags(&S.dec_done, cudaEventDisableTiming));
    TMD_CUDA(cudaEventCreateWithFlags(&S.d2h_done, cudaEventDisableTiming));
  }
  const uint32_t n_bins = ctx->geo.n_bins;
  const size_t n_trk = in->n_tracks, n_att = in->n_attached, n_res = n_att - n_trk, n_un = in->n_unattached;
  const Workspace W = layout(n_bins, in->n_tracks, n_att);
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
  for (const Seg& s : segs)
    if (s.bytes) TMD_CUDA(cudaMemcpyAsync(a + s.at, s.src, s.bytes, cudaMemcpyHostToDevice, s_in));
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
  TMD_CUDA(cudaEventRecord(S.d2h_done, s_out));
  S.busy = true;
  return TMD_OK;
}

int tmd_decode_host(tmd_ctx* ctx, const tmd_compressed* in, tmd_output* out, uint32_t flags, void* cuda_stream) {
  if (!ctx) return TMD_ERR_ARG;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int rc = host_enqueue(ctx, in, out, flags, 0, st, st, st);
  if (rc != TMD_OK) return rc;
  return tmd_host_wait(ctx, 0);
}

int tmd_decode_host_async(tmd_ctx* ctx, const tmd_compressed* in, tmd_output* out, uint32_t flags, int slot) {
  if (!ctx || slot < 0 || slot >= TMD_HOST_SLOTS || (flags & TMD_VALIDATE)) return TMD_ERR_ARG;
  if (!ctx->host_ready) {
    TMD_CUDA(cudaStreamCreateWithFlags(&ctx->s_h2d, cudaStreamNonBlocking));
    TMD_CUDA(cudaStreamCreateWithFlags(&ctx->s_dec, cudaStreamNonBlocking));
    TMD_CUDA(cudaStreamCreateWithFlags(&ctx->s_d2h, cudaStreamNonBlocking));
    ctx->host_ready = true;
  }
  return host_enqueue(ctx, in, out, flags, slot, ctx->s_h2d, ctx->s_dec, ctx->s_d2h);
}

int tmd_host_wait(tmd_ctx* ctx, int slot) {
  if (!ctx || slot < 0 || slot >= TMD_HOST_SLOTS) return TMD_ERR_ARG;
  tmd_ctx::HostSlot& S = ctx->slots[slot];
  if (!S.busy) return TMD_OK;
  TMD_CUDA(cudaEventSynchronize(S.d2h_done));
  S.busy = false;
  return TMD_OK;
}

int tmd_destroy(tmd_ctx* ctx) {
  if (!ctx) return TMD_OK;
  if (ctx->side) { cudaStreamSynchronize(ctx->side); cudaStreamDestroy(ctx->side); }
  if (ctx->ev_fork) cudaEventDestroy(ctx->ev_fork);
  if (ctx->ev_join) cudaEventDestroy(ctx->ev_join);
  for (tmd_ctx::HostSlot& S : ctx->slots) {
    if (S.busy) cudaEventSynchronize(S.d2h_done);
    if (S.arena) cudaFree(S.arena);
    if (S.h2d_done) { cudaEventDestroy(S.h2d_done); cudaEventDestroy(S.dec_done); cudaEventDestroy(S.d2h_done); }
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
    default: return "unknown status";
  }
}

int tmd_last_launch_count(const tmd_ctx* ctx) { return ctx ? ctx->launches : 0; }

}  // extern "C"
