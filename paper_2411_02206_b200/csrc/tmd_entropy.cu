// tmd_entropy.cu -- the entropy stage in front of the track-model decoder: rANS decoding of a TMDZ
// container on the GPU, straight into the compressed-cluster SoA that tmd_decode reads, plus the host-side encoder that
// writes such containers.
//
// the compressed time frames are entropy-coded with "lossless ANS"; L49 (Table 2): "TPC Entropy Decoding" is
// 4.65 % of the asynchronous CPU time, the step right before this library's path (L68: "after the entropy decoding, the
// clusters' coordinates must be decoded").  The paper gives no format: TMDZ is this build's own.  The
// coder is range-ANS (Duda, arXiv:1311.2540) with 12-bit tables, a 32-bit state in [2^16, 2^32) and 16-bit
// renormalisation; a plane of byte symbols is cut into blocks of 8192, coded by 32 interleaved coders (symbol k belongs to
// coder k mod 32), the words stored in the order the decoder reads them.  No code is shared with oracle/.
#include <stdlib.h>
#include <string.h>

#include <algorithm>
#include <new>
#include <vector>

#include "tmd_common.cuh"
#include "tmd_scan.cuh"

namespace tmd {

constexpr uint32_t Z_MAGIC = 0x5A444D54u, Z_VERSION = 1, Z_BLOCK = 8192, Z_LANES = 32, Z_PROB_BITS = 12, Z_M = 1u << Z_PROB_BITS;
constexpr uint32_t Z_L = 1u << 16;
constexpr uint32_t Z_HEADER = 64, Z_PLANE = 32, Z_ARRAYS = 23, Z_PLANES = 43;
constexpr int Z_THREADS = 256, Z_WARPS = 8;
constexpr uint32_t Z_CHUNK_BYTES = Z_WARPS * Z_BLOCK;        // bytes of output one CTA assembles (65536)

// widths (bytes per element) of the 23 arrays of tmd_compressed, in struct order
__host__ __device__ inline uint32_t z_width(uint32_t a) {
  const uint8_t w[Z_ARRAYS] = {2, 1, 1, 1, 2, 4, 2, 2, 1, 1, 1, 1, 1, 2, 4, 2, 2, 1, 1, 1, 2, 4, 4};
  return w[a];
}

struct ZArray {
  unsigned char* out;       // DEVICE destination array
  uint64_t n_elem;
  uint32_t width, first_plane, first_chunk, n_chunks;
};
struct ZPlane { uint64_t table_offset, blocks_offset; };
struct ZArgs {
  const unsigned char* blob;   // DEVICE
  uint64_t blob_bytes;
  ZArray arr[Z_ARRAYS];
  ZPlane pl[Z_PLANES];
};
static_assert(sizeof(ZArgs) < 3800, "kernel parameter space");

// One CTA assembles Z_CHUNK_BYTES of one output array: warp wi decodes block (chunk * (8 / w) + wi / w) of byte plane
// (wi mod w) into shared memory, then the CTA interleaves the planes into elements and writes them with coalesced stores.
__global__ void __launch_bounds__(Z_THREADS) k_entropy_decode(const __grid_constant__ ZArgs Z, uint32_t* __restrict__ err) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  unsigned char* stage = smem_raw;                                            // [Z_WARPS][Z_BLOCK] decoded symbols
  unsigned char* lut = smem_raw + Z_CHUNK_BYTES;                              // [w][4096] slot -> symbol
  uint32_t* tab = reinterpret_cast<uint32_t*>(lut + 4 * Z_M);                  // [w][256] freq | cum << 16
  __shared__ uint32_t ws[33];
  // ---- which array, which chunk
  uint32_t a = 0;
  while (a + 1 < Z_ARRAYS && blockIdx.x >= Z.arr[a + 1].first_chunk) ++a;      // first_chunk is non-decreasing
  const ZArray& A = Z.arr[a];
  const uint32_t chunk = blockIdx.x - A.first_chunk, w = A.width;
  if (chunk >= A.n_chunks) return;
  const uint32_t tid = threadIdx.x, lane = tid & 31u, wi = tid >> 5;
  // ---- tables of the w planes: cum by a block scan over the 256 symbols, slot -> symbol by binary search
  for (uint32_t j = 0; j < w; ++j) {
    const uint16_t* freq = reinterpret_cast<const uint16_t*>(Z.blob + Z.pl[A.first_plane + j].table_offset);
    const uint32_t f = freq[tid];
    uint32_t total;
    const uint32_t c = block_excl_scan(f, ws, &total);
    tab[j * 256 + tid] = f | (c << 16);                                        // c <= 4096 fits the upper half
    if (tid == 0 && total != Z_M) atomicOr(&err[0], 1u);
    __syncthreads();
    for (uint32_t slot = tid; slot < Z_M; slot += Z_THREADS) {
      // the largest symbol whose cumulative frequency is <= slot: symbols of frequency 0 share the cumulative value of their
      // successor, so the largest index is the one that covers the slot
      uint32_t lo = 0, hi = 255;
      while (lo < hi) {
        const uint32_t mid = (lo + hi + 1) >> 1;
        if ((tab[j * 256 + mid] >> 16) <= slot) lo = mid; else hi = mid - 1;
      }
      lut[j * Z_M + slot] = (unsigned char)lo;
    }
    __syncthreads();
  }
  // ---- decode: one block per warp
  const uint32_t j = wi % w, q = wi / w, per_plane = Z_WARPS / w;
  const uint64_t n_sym = A.n_elem;
  const uint64_t b = (uint64_t)chunk * per_plane + q;                           // block index inside the plane
  const uint64_t first = b * Z_BLOCK;
  if (first < n_sym) {
    const uint32_t n = (uint32_t)min((uint64_t)Z_BLOCK, n_sym - first);
    const uint32_t* starts = reinterpret_cast<const uint32_t*>(Z.blob + Z.pl[A.first_plane + j].blocks_offset);
    uint32_t s0 = starts[b], s1 = starts[b + 1];
    if (s1 < s0 || s1 > Z.blob_bytes || s1 - s0 < 4 * Z_LANES) {               // corrupt block table: decode nothing from it
      if (lane == 0) atomicOr(&err[0], 4u);
      s0 = 0; s1 = 4 * Z_LANES;
    }
    const unsigned char* blk = Z.blob + s0;
    uint32_t x = reinterpret_cast<const uint32_t*>(blk)[lane];
    const uint16_t* words = reinterpret_cast<const uint16_t*>(blk + 4 * Z_LANES);
    const uint32_t max_words = s1 > s0 + 4 * Z_LANES ? (s1 - s0 - 4 * Z_LANES) / 2 : 0;
    uint32_t used = 0;
    const unsigned char* my_lut = lut + j * Z_M;
    const uint32_t* my_tab = tab + j * 256;
    unsigned char* dst = stage + wi * Z_BLOCK;
    for (uint32_t k0 = 0; k0 < n; k0 += 32) {
      const bool active = k0 + lane < n;
      const uint32_t slot = x & (Z_M - 1), s = my_lut[slot], fc = my_tab[s];
      uint32_t xn = (fc & 0xFFFFu) * (x >> Z_PROB_BITS) + slot - (fc >> 16);
      const bool need = active && xn < Z_L;
      const uint32_t mask = __ballot_sync(0xffffffffu, need);
      if (need) {
        const uint32_t at = used + __popc(mask & ((1u << lane) - 1u));
        xn = (xn << 16) | (at < max_words ? (uint32_t)words[at] : 0u);
      }
      used += __popc(mask);
      if (active) { x = xn; dst[k0 + lane] = (unsigned char)s; }
    }
    if (lane == 0 && used > max_words) atomicOr(&err[0], 2u);                  // a block shorter than its symbols need
  }
  __syncthreads();
  // ---- interleave the planes into elements: output byte o of the chunk = byte (o mod w) of element (o / w)
  const uint64_t out0 = (uint64_t)chunk * Z_CHUNK_BYTES, total_bytes = n_sym * w;
  const uint32_t n_out = (uint32_t)min((uint64_t)Z_CHUNK_BYTES, total_bytes - out0);
  const uint32_t wshift = w == 4 ? 2 : (w == 2 ? 1 : 0);
  auto byte_at = [&](uint32_t o) -> uint32_t {
    const uint32_t e = o >> wshift, jj = o & (w - 1);                          // element (inside the chunk), plane
    return stage[((e / Z_BLOCK) * w + jj) * Z_BLOCK + (e % Z_BLOCK)];
  };
  uint32_t* out32 = reinterpret_cast<uint32_t*>(A.out + out0);                 // 16-byte aligned array, out0 multiple of 65536
  for (uint32_t o = tid * 4; o + 4 <= n_out; o += Z_THREADS * 4)
    out32[o >> 2] = byte_at(o) | (byte_at(o + 1) << 8) | (byte_at(o + 2) << 16) | (byte_at(o + 3) << 24);
  if (tid < (n_out & 3u)) A.out[out0 + (n_out & ~3u) + tid] = (unsigned char)byte_at((n_out & ~3u) + tid);
}

// ---------------------------------------------------------------------------------------------------------------- host side
namespace {

struct Head {
  uint32_t n_tracks, n_bins, n_planes;
  uint64_t n_attached, n_unattached, total;
};

inline uint32_t rd32(const unsigned char* p) { uint32_t v; memcpy(&v, p, 4); return v; }
inline uint64_t rd64(const unsigned char* p) { uint64_t v; memcpy(&v, p, 8); return v; }
inline void wr32(unsigned char* p, uint32_t v) { memcpy(p, &v, 4); }
inline void wr64(unsigned char* p, uint64_t v) { memcpy(p, &v, 8); }

int parse_head(const void* head, size_t head_bytes, Head* h) {
  if (!head || head_bytes < Z_HEADER) return TMD_ERR_ARG;
  const unsigned char* p = (const unsigned char*)head;
  if (rd32(p) != Z_MAGIC || rd32(p + 4) != Z_VERSION || rd32(p + 36) != Z_BLOCK) return TMD_ERR_CORRUPT;
  h->n_tracks = rd32(p + 8); h->n_bins = rd32(p + 12);
  h->n_attached = rd64(p + 16); h->n_unattached = rd64(p + 24);
  h->n_planes = rd32(p + 32); h->total = rd64(p + 40);
  if (h->n_planes != Z_PLANES || h->n_attached < h->n_tracks || h->total < Z_HEADER + (uint64_t)Z_PLANE * Z_PLANES) return TMD_ERR_CORRUPT;
  return TMD_OK;
}

// number of elements of array `a` of the compressed SoA
uint64_t elems_of(uint32_t a, const Head& h) {
  if (a < 6) return h.n_tracks;
  if (a < 11) return h.n_attached;
  if (a < 15) return h.n_attached - h.n_tracks;
  if (a < 22) return h.n_unattached;
  return h.n_bins;
}

// frequencies that sum to 4096, every present symbol >= 1: largest-remainder apportionment
void normalise(const uint64_t cnt[256], uint64_t n, uint16_t freq[256]) {
  memset(freq, 0, 512);
  if (n == 0) return;
  struct Rem { uint64_t rem; int s; };
  std::vector<Rem> order;
  int64_t left = Z_M;
  uint32_t f[256] = {0};
  for (int s = 0; s < 256; ++s) {
    if (!cnt[s]) continue;
    const uint64_t scaled = cnt[s] * Z_M;
    f[s] = (uint32_t)std::max<uint64_t>(1, scaled / n);
    left -= f[s];
    order.push_back({scaled % n, s});
  }
  std::sort(order.begin(), order.end(), [](const Rem& x, const Rem& y) { return x.rem != y.rem ? x.rem > y.rem : x.s < y.s; });
  for (size_t i = 0; left > 0; i = (i + 1) % order.size(), --left) f[order[i].s]++;      // hand out what floor() left over
  while (left < 0) {                                                                      // the >= 1 floor took too much
    int best = -1;
    for (int s = 0; s < 256; ++s) if (f[s] > 1 && (best < 0 || f[s] > f[best])) best = s;
    f[best]--; ++left;
  }
  for (int s = 0; s < 256; ++s) freq[s] = (uint16_t)f[s];
}

}  // namespace
}  // namespace tmd

using namespace tmd;

extern "C" {

int tmd_entropy_bound(uint32_t n_tracks, uint64_t n_attached, uint64_t n_unattached, uint32_t n_bins, size_t* out_bytes) {
  if (!out_bytes || n_attached < n_tracks) return TMD_ERR_ARG;
  Head h = {n_tracks, n_bins, Z_PLANES, n_attached, n_unattached, 0};
  uint64_t total = Z_HEADER + (uint64_t)Z_PLANE * Z_PLANES;
  for (uint32_t a = 0; a < Z_ARRAYS; ++a) {
    const uint64_t n = elems_of(a, h), blocks = (n + Z_BLOCK - 1) / Z_BLOCK;
    // per plane: table, block starts, and per block the 32 states + at most one word per symbol (incompressible data), padding
    total += (uint64_t)z_width(a) * (512 + 16 + 4 * (blocks + 1) + 16 + blocks * (4 * Z_LANES + 4) + 2 * n);
  }
  *out_bytes = (size_t)total;
  return TMD_OK;
}

int tmd_entropy_encode_host(const tmd_compressed* in, uint32_t n_bins, void* blob, size_t capacity, size_t* out_bytes) {
  if (!in || !blob || !out_bytes || in->n_attached < in->n_tracks) return TMD_ERR_ARG;
  size_t bound = 0;
  if (tmd_entropy_bound(in->n_tracks, in->n_attached, in->n_unattached, n_bins, &bound) != TMD_OK) return TMD_ERR_ARG;
  if (capacity < bound) return TMD_ERR_WORKSPACE;
  const Head h = {in->n_tracks, n_bins, Z_PLANES, in->n_attached, in->n_unattached, 0};
  const void* arrays[Z_ARRAYS] = {in->trk_ncl, in->trk_qpt, in->trk_row0, in->trk_sec0, in->trk_pad0, in->trk_time0, in->a_qtot, in->a_qmax,
                                  in->a_flags, in->a_sigpad, in->a_sigtime, in->a_rowdiff, in->a_secleg, in->a_padres, in->a_timeres,
                                  in->u_qtot, in->u_qmax, in->u_flags, in->u_sigpad, in->u_sigtime, in->u_paddiff, in->u_timediff,
                                  in->u_bin_count};
  unsigned char* out = (unsigned char*)blob;
  uint64_t pos = Z_HEADER + (uint64_t)Z_PLANE * Z_PLANES;
  auto align_to = [&](uint64_t a) { while (pos % a) out[pos++] = 0; };
  std::vector<unsigned char> plane;
  std::vector<uint16_t> rev;
  uint32_t p_index = 0;
  for (uint32_t a = 0; a < Z_ARRAYS; ++a) {
    const uint64_t n = elems_of(a, h);
    const uint32_t w = z_width(a);
    if (n && !arrays[a]) return TMD_ERR_ARG;
    const unsigned char* src = (const unsigned char*)arrays[a];
    for (uint32_t j = 0; j < w; ++j, ++p_index) {
      plane.resize(n);
      uint64_t cnt[256] = {0};
      for (uint64_t e = 0; e < n; ++e) { plane[e] = src[e * w + j]; cnt[plane[e]]++; }
      uint16_t freq[256];
      normalise(cnt, n, freq);
      uint32_t cum[257];
      cum[0] = 0;
      for (int s = 0; s < 256; ++s) cum[s + 1] = cum[s] + freq[s];
      align_to(16);
      const uint64_t table_off = pos;
      memcpy(out + pos, freq, 512); pos += 512;
      const uint64_t blocks = (n + Z_BLOCK - 1) / Z_BLOCK;
      align_to(16);
      const uint64_t starts_off = pos;
      pos += 4 * (blocks + 1);
      for (uint64_t b = 0; b < blocks; ++b) {
        align_to(4);
        if (pos > 0xFFFFFFFFull) return TMD_ERR_ARG;                     // block starts are 32-bit: containers stay below 4 GiB
        wr32(out + starts_off + 4 * b, (uint32_t)pos);
        const uint64_t first = b * Z_BLOCK;
        const uint32_t m = (uint32_t)std::min<uint64_t>(Z_BLOCK, n - first);
        uint32_t x[Z_LANES];
        for (uint32_t l = 0; l < Z_LANES; ++l) x[l] = Z_L;
        rev.clear();
        for (uint32_t k = m; k-- > 0;) {                                 // backwards: the decoder pops what was pushed last
          const uint32_t s = plane[first + k], f = freq[s], l = k % Z_LANES;
          if ((uint64_t)x[l] >= ((uint64_t)f << 20)) { rev.push_back((uint16_t)x[l]); x[l] >>= 16; }
          x[l] = ((x[l] / f) << Z_PROB_BITS) + (x[l] % f) + cum[s];
        }
        memcpy(out + pos, x, sizeof(x)); pos += sizeof(x);
        for (size_t i = rev.size(); i-- > 0;) { memcpy(out + pos, &rev[i], 2); pos += 2; }
      }
      align_to(4);
      if (pos > 0xFFFFFFFFull) return TMD_ERR_ARG;
      wr32(out + starts_off + 4 * blocks, (uint32_t)pos);
      unsigned char* d = out + Z_HEADER + (uint64_t)Z_PLANE * p_index;
      wr32(d, a); wr32(d + 4, j); wr64(d + 8, n); wr64(d + 16, table_off); wr64(d + 24, starts_off);
    }
  }
  memset(out, 0, Z_HEADER);
  wr32(out, Z_MAGIC); wr32(out + 4, Z_VERSION); wr32(out + 8, h.n_tracks); wr32(out + 12, h.n_bins);
  wr64(out + 16, h.n_attached); wr64(out + 24, h.n_unattached); wr32(out + 32, Z_PLANES); wr32(out + 36, Z_BLOCK); wr64(out + 40, pos);
  *out_bytes = (size_t)pos;
  return TMD_OK;
}

int tmd_entropy_sizes(const void* head, size_t head_bytes, uint32_t* n_tracks, uint64_t* n_attached, uint64_t* n_unattached,
                      uint32_t* n_bins, size_t* blob_bytes) {
  Head h;
  const int rc = parse_head(head, head_bytes, &h);
  if (rc != TMD_OK) return rc;
  if (n_tracks) *n_tracks = h.n_tracks;
  if (n_attached) *n_attached = h.n_attached;
  if (n_unattached) *n_unattached = h.n_unattached;
  if (n_bins) *n_bins = h.n_bins;
  if (blob_bytes) *blob_bytes = (size_t)h.total;
  return TMD_OK;
}

int tmd_entropy_decode(const void* head, size_t head_bytes, const void* d_blob, size_t blob_bytes, tmd_compressed* out, void* d_err4,
                       void* cuda_stream) {
  Head h;
  int rc = parse_head(head, head_bytes, &h);
  if (rc != TMD_OK) return rc;
  if (!d_blob || !out || !d_err4 || head_bytes < Z_HEADER + (size_t)Z_PLANE * Z_PLANES || blob_bytes < h.total) return TMD_ERR_ARG;
  if ((reinterpret_cast<uintptr_t>(d_blob) & 15u) || (reinterpret_cast<uintptr_t>(d_err4) & 3u)) return TMD_ERR_ALIGN;
  if (out->n_tracks != h.n_tracks || out->n_attached != h.n_attached || out->n_unattached != h.n_unattached) return TMD_ERR_ARG;
  void* arrays[Z_ARRAYS] = {(void*)out->trk_ncl, (void*)out->trk_qpt, (void*)out->trk_row0, (void*)out->trk_sec0, (void*)out->trk_pad0,
                            (void*)out->trk_time0, (void*)out->a_qtot, (void*)out->a_qmax, (void*)out->a_flags, (void*)out->a_sigpad,
                            (void*)out->a_sigtime, (void*)out->a_rowdiff, (void*)out->a_secleg, (void*)out->a_padres, (void*)out->a_timeres,
                            (void*)out->u_qtot, (void*)out->u_qmax, (void*)out->u_flags, (void*)out->u_sigpad, (void*)out->u_sigtime,
                            (void*)out->u_paddiff, (void*)out->u_timediff, (void*)out->u_bin_count};
  ZArgs Z;
  memset(&Z, 0, sizeof(Z));
  Z.blob = (const unsigned char*)d_blob;
  Z.blob_bytes = h.total;
  const unsigned char* dir = (const unsigned char*)head + Z_HEADER;
  uint32_t p_index = 0, chunk = 0;
  for (uint32_t a = 0; a < Z_ARRAYS; ++a) {
    const uint64_t n = elems_of(a, h);
    const uint32_t w = z_width(a);
    if (n && (!arrays[a] || (reinterpret_cast<uintptr_t>(arrays[a]) & 15u))) return arrays[a] ? TMD_ERR_ALIGN : TMD_ERR_ARG;
    Z.arr[a].out = (unsigned char*)arrays[a];
    Z.arr[a].n_elem = n; Z.arr[a].width = w; Z.arr[a].first_plane = p_index; Z.arr[a].first_chunk = chunk;
    const uint64_t chunks = (n * w + Z_CHUNK_BYTES - 1) / Z_CHUNK_BYTES;
    if (chunk + chunks > 0x7FFFFFFFull) return TMD_ERR_ARG;
    Z.arr[a].n_chunks = (uint32_t)chunks;
    chunk += (uint32_t)chunks;
    for (uint32_t j = 0; j < w; ++j, ++p_index) {
      const unsigned char* d = dir + (size_t)Z_PLANE * p_index;
      const uint64_t blocks = (n + Z_BLOCK - 1) / Z_BLOCK;
      if (rd32(d) != a || rd32(d + 4) != j || rd64(d + 8) != n) return TMD_ERR_CORRUPT;
      Z.pl[p_index].table_offset = rd64(d + 16);
      Z.pl[p_index].blocks_offset = rd64(d + 24);
      if (Z.pl[p_index].table_offset + 512 > h.total || Z.pl[p_index].blocks_offset + 4 * (blocks + 1) > h.total ||
          (Z.pl[p_index].table_offset & 1u) || (Z.pl[p_index].blocks_offset & 3u))
        return TMD_ERR_CORRUPT;
    }
  }
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (cudaMemsetAsync(d_err4, 0, 4, st) != cudaSuccess) return TMD_ERR_CUDA;
  if (chunk == 0) return TMD_OK;
  const size_t smem = Z_CHUNK_BYTES + 4 * (size_t)Z_M + 4 * 256 * 4;
  static bool attr_set = false;
  if (!attr_set) {
    if (cudaFuncSetAttribute(k_entropy_decode, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return TMD_ERR_CUDA;
    attr_set = true;
  }
  k_entropy_decode<<<chunk, Z_THREADS, smem, st>>>(Z, (uint32_t*)d_err4);
  return cudaGetLastError() == cudaSuccess ? TMD_OK : TMD_ERR_CUDA;
}

}  // extern "C"
