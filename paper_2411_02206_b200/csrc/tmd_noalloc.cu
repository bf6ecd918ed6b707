// tmd_noalloc.cu -- tmd_decode_unattached_noalloc (include/tmd.h): row A7 for a caller that may not allocate.
//
// Who this is for.  Every other decode entry point wants a context from tmd_create (which calls cudaMalloc for its geometry
// table) and a caller-allocated workspace.  Some hosts of this library can do neither: a reconstruction framework that takes
// the device's memory as one block when it starts and forbids driver allocations afterwards (every later cudaMalloc would
// either fail or eat into memory the framework believes it owns); a plug-in that is handed device pointers by such a host and
// has no pool of its own; a loop with a latency budget, where cudaMalloc / cudaFree are unwelcome because they serialise with
// all work on the device.  For them the scratch of the unattached decode -- the per-bin start table the decode kernel reads --
// lives in the file-scope array below, which is part of the library image: the driver places it in device memory when the
// library's code is loaded on a GPU and it stays there until the process ends.  Cost: NA_SCRATCH_BYTES (64.25 KiB) on every GPU
// that loads libtmd.so, whether or not this entry point is ever called.
//
// The kernels below are variants of k_bin_offsets (tmd_scan.cuh) and k_unattached (tmd_unattached.cuh): same arithmetic (the
// per-bin decode is the shared device function unattached_bin), workspace pointers replaced by offsets into the static array.
// No existing kernel or entry point is touched.
#include <mutex>

#include "tmd_common.cuh"
#include "tmd_scan.cuh"
#include "tmd_unattached.cuh"

using namespace tmd;

namespace {

constexpr uint32_t NA_MAX_BINS = TMD_NOALLOC_MAX_BINS;
constexpr size_t na_align(size_t v) { return (v + 255) & ~(size_t)255; }
// Layout of the scratch: u_start[NA_MAX_BINS + 1] (exclusive scan of u_bin_count: where a bin's differences begin in the u_*
// arrays), then att_cnt[NA_MAX_BINS] (attached clusters in front of a bin's unattached ones: none here, so all zero).
constexpr size_t NA_O_U_START = 0;
constexpr size_t NA_O_ATT_CNT = na_align((size_t)(NA_MAX_BINS + 1) * 4);
constexpr size_t NA_SCRATCH_BYTES = NA_O_ATT_CNT + na_align((size_t)NA_MAX_BINS * 4);
static_assert(NA_SCRATCH_BYTES == 65792, "the size stated in include/tmd.h and README.md");

// The scratch.  In HOST code this name is only a handle for the runtime's symbol calls, not a device address: it must never be
// handed to a kernel as it is (the kernel would fault, or on a system where the GPU can reach host memory quietly use the
// wrong bytes).  Host code gets the address with cudaGetSymbolAddress, see scratch_of_current_device().
static __device__ __align__(256) unsigned char g_na_scratch[NA_SCRATCH_BYTES];

// One device address per GPU (each device that loads the library has its own copy of the array).
constexpr int NA_MAX_DEVICES = 64;
std::mutex g_na_lock;
unsigned char* g_na_addr[NA_MAX_DEVICES];   // zero-initialised: "not looked up yet"

// Address of g_na_scratch on the CURRENT device; looked up once per device, with that device current.
int scratch_of_current_device(unsigned char** out) {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return TMD_ERR_CUDA; }
  if (dev < 0 || dev >= NA_MAX_DEVICES) return TMD_ERR_DEVICE;
  std::lock_guard<std::mutex> hold(g_na_lock);
  if (!g_na_addr[dev]) {
    void* p = nullptr;
    if (cudaGetSymbolAddress(&p, g_na_scratch) != cudaSuccess || !p) { cudaGetLastError(); return TMD_ERR_CUDA; }
    g_na_addr[dev] = (unsigned char*)p;
  }
  *out = g_na_addr[dev];
  return TMD_OK;
}

// Single block.  bin_offset[b] = u_start[b] = exclusive scan of u_bin_count (no attached clusters: a bin holds only its
// unattached ones); att_cnt[b] = 0.  Everything the decode kernel reads from the scratch is written here on every call: the
// array still holds the previous call's tables, possibly of a geometry with more bins.
__global__ void __launch_bounds__(1024) k_na_bin_starts(uint32_t n_bins, const uint32_t* __restrict__ u_cnt, uint32_t* __restrict__ bin_offset,
                                                        unsigned char* __restrict__ scratch) {
  __shared__ uint32_t ws[33];
  uint32_t* __restrict__ u_start = reinterpret_cast<uint32_t*>(scratch + NA_O_U_START);
  uint32_t* __restrict__ att_cnt = reinterpret_cast<uint32_t*>(scratch + NA_O_ATT_CNT);
  const uint32_t per = (n_bins + blockDim.x - 1) / blockDim.x;
  const uint32_t b0 = min(threadIdx.x * per, n_bins), b1 = min(b0 + per, n_bins);
  uint32_t s = 0;
  for (uint32_t b = b0; b < b1; ++b) s += u_cnt[b];
  uint32_t total;
  uint32_t run = block_excl_scan(s, ws, &total);
  for (uint32_t b = b0; b < b1; ++b) {
    bin_offset[b] = run;
    u_start[b] = run;
    att_cnt[b] = 0;
    run += u_cnt[b];
  }
  if (threadIdx.x == 0) {
    bin_offset[n_bins] = total;
    u_start[n_bins] = total;
  }
}

// k_unattached with its two workspace tables taken from the static scratch
__global__ void __launch_bounds__(UNATT_THREADS) k_na_unattached(const __grid_constant__ DevGeo G, const __grid_constant__ tmd_compressed in,
                                                                 uint4* __restrict__ clusters, const uint32_t* __restrict__ bin_offset,
                                                                 const unsigned char* __restrict__ scratch, uint32_t bins_per_block) {
  __shared__ uint32_t ws[66];
  UnattachedArgs A;
  A.in = in;
  A.u_start = reinterpret_cast<const uint32_t*>(scratch + NA_O_U_START);
  A.bin_offset = bin_offset;
  A.att_cnt = reinterpret_cast<const uint32_t*>(scratch + NA_O_ATT_CNT);
  A.clusters = clusters;
  A.n_clusters_total = (uint32_t)in.n_unattached;
  const uint32_t b0 = blockIdx.x * bins_per_block, b1 = min(b0 + bins_per_block, G.n_bins);
  const uint32_t wid = threadIdx.x >> 5, lane = lane_id();
  for (uint32_t b = b0; b < b1; ++b) {
    const uint32_t n = A.u_start[b + 1] - A.u_start[b];
    const bool whole_block = n > UNATT_SMALL;
    if (whole_block || (b - b0) % UNATT_WARPS == wid)
      unattached_bin(G, A, b, whole_block ? threadIdx.x : lane, whole_block ? (uint32_t)UNATT_THREADS : 32u, ws);
  }
}

inline bool na_misaligned(const void* p, size_t a) { return (reinterpret_cast<uintptr_t>(p) & (a - 1)) != 0; }

}  // namespace

extern "C" int tmd_decode_unattached_noalloc(uint32_t n_sectors_out, uint32_t n_rows, const tmd_compressed* in, tmd_cluster* clusters,
                                             uint32_t* bin_offset, void* cuda_stream) {
  // Argument checks first, before any CUDA call: a refused call leaves the device and the scratch untouched.
  if (!in || !bin_offset || n_sectors_out < 1 || n_rows < 1 || n_rows > 255) return TMD_ERR_ARG;
  const uint64_t n_bins64 = (uint64_t)n_sectors_out * n_rows;
  if (n_bins64 > NA_MAX_BINS) return TMD_ERR_LIMIT;                         // the tables would not fit the static scratch
  if (in->n_unattached > TMD_MAX_CLUSTERS) return TMD_ERR_LIMIT;
  if (in->n_tracks != 0 || in->n_attached != 0) return TMD_ERR_ARG;         // attached clusters need tmd_decode and its workspace
  if (!in->u_bin_count) return TMD_ERR_ARG;
  const void* un[] = {in->u_qtot, in->u_qmax, in->u_flags, in->u_sigpad, in->u_sigtime, in->u_paddiff, in->u_timediff};
  if (in->n_unattached > 0) {
    if (!clusters) return TMD_ERR_ARG;
    for (const void* p : un) if (!p) return TMD_ERR_ARG;
    for (const void* p : un) if (na_misaligned(p, 16)) return TMD_ERR_ALIGN;
  }
  if (na_misaligned(in->u_bin_count, 16) || na_misaligned(clusters, 16) || na_misaligned(bin_offset, 4)) return TMD_ERR_ALIGN;

  unsigned char* scratch = nullptr;                // the DEVICE address of g_na_scratch, never the host-side name
  const int rc = scratch_of_current_device(&scratch);
  if (rc != TMD_OK) return rc;

  const uint32_t n_bins = (uint32_t)n_bins64;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  k_na_bin_starts<<<1, 1024, 0, st>>>(n_bins, in->u_bin_count, bin_offset, scratch);
  if (cudaGetLastError() != cudaSuccess) return TMD_ERR_CUDA;
  if (in->n_unattached == 0) return TMD_OK;
  DevGeo G = {};
  G.n_sectors_out = n_sectors_out; G.n_rows = n_rows; G.n_bins = n_bins;    // all that the unattached decode reads of the geometry
  // a block per bin for full time frames, a warp per bin where bins hold few clusters (the rule of tmd_decode)
  const uint32_t bpb = in->n_unattached / n_bins >= 512 ? 1u : (uint32_t)UNATT_WARPS;
  k_na_unattached<<<(n_bins + bpb - 1) / bpb, UNATT_THREADS, 0, st>>>(G, *in, (uint4*)clusters, bin_offset, scratch, bpb);
  if (cudaGetLastError() != cudaSuccess) return TMD_ERR_CUDA;
  return TMD_OK;
}
