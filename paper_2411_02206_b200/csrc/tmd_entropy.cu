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
constexpr uint32_t Z_PARTS = 4, Z_PART = Z_BLOCK / Z_PARTS;   // a warp's block is decoded and written out in parts of 2048 symbols

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
static_assert(Z_HEADER + Z_PLANE * Z_PLANES == TMD_ENTROPY_HEAD_BYTES, "include/tmd.h states the size of header + plane directory");

// One CTA assembles Z_CHUNK_BYTES of one output array: warp wi decodes block (chunk * (8 / w) + wi / w) of byte plane
// (wi mod w) into shared memory, then the CTA interleaves the planes into elements and writes them with coalesced stores.
__global__ void __launch_bounds__(Z_THREADS) k_entropy_decode(const __grid_constant__ ZArgs Z, uint32_t* __restrict__ err) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  unsigned char* stage = smem_raw;                                            // [Z_WARPS][Z_PART] decoded symbols of the current part
  unsigned char* lut = smem_raw + Z_WARPS * Z_PART;                           // [w][4096] slot -> symbol
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
    {
      // slot -> symbol: the largest symbol whose cumulative frequency is <= slot (symbols of frequency 0 share the cumulative
      // value of their successor, so the largest index is the one that covers the slot).  A thread fills 16 consecutive
      // slots: one binary search for the first, then it walks up the cumulative table.
      const uint32_t* t = tab + j * 256;
      uint32_t slot = tid * (Z_M / Z_THREADS), lo = 0, hi = 255;
      while (lo < hi) {
        const uint32_t mid = (lo + hi + 1) >> 1;
        if ((t[mid] >> 16) <= slot) lo = mid; else hi = mid - 1;
      }
      uint32_t packed[Z_M / Z_THREADS / 4];
#pragma unroll
      for (uint32_t k = 0; k < Z_M / Z_THREADS; ++k, ++slot) {
        while (lo < 255 && (t[lo + 1] >> 16) <= slot) ++lo;
        if ((k & 3u) == 0) packed[k >> 2] = 0;
        packed[k >> 2] |= lo << (8 * (k & 3u));
      }
      uint4* dst4 = reinterpret_cast<uint4*>(lut + j * Z_M + tid * (Z_M / Z_THREADS));
      static_assert(Z_M / Z_THREADS == 16, "one 16-byte store per thread");
      *dst4 = make_uint4(packed[0], packed[1], packed[2], packed[3]);
    }
    __syncthreads();
  }
  // ---- decode: one block per warp, in Z_PARTS parts of Z_PART symbols; after each part the CTA interleaves the planes into
  // elements and writes them out (a part-sized staging buffer keeps six CTAs resident per SM: the decode loop is a chain
  // of dependent look-ups and shuffles, it needs many warps to hide its latency)
  const uint32_t j = wi % w, q = wi / w, per_plane = Z_WARPS / w;
  const uint64_t n_sym = A.n_elem;
  const uint64_t b = (uint64_t)chunk * per_plane + q;                           // block index inside the plane
  const uint64_t first = b * Z_BLOCK;
  const uint32_t n = first < n_sym ? (uint32_t)min((uint64_t)Z_BLOCK, n_sym - first) : 0u;   // symbols of this warp's block
  uint32_t x = 0, used = 0, base = 0, w0 = 0, w1 = 0, max_words = 0;
  const uint16_t* words = nullptr;
  if (n) {
    const uint32_t* starts = reinterpret_cast<const uint32_t*>(Z.blob + Z.pl[A.first_plane + j].blocks_offset);
    uint32_t s0 = starts[b], s1 = starts[b + 1];
    if (s1 < s0 || s1 > Z.blob_bytes || s1 - s0 < 4 * Z_LANES || (s0 & 3u)) {   // corrupt block table (out of order, out of bounds,
                                                                               // too short, states not 4-byte aligned): decode nothing from it
      if (lane == 0) atomicOr(&err[0], 4u);
      s0 = 0; s1 = 4 * Z_LANES;
    }
    const unsigned char* blk = Z.blob + s0;
    x = reinterpret_cast<const uint32_t*>(blk)[lane];
    words = reinterpret_cast<const uint16_t*>(blk + 4 * Z_LANES);
    max_words = (s1 - s0 - 4 * Z_LANES) / 2;
    // the whole block into the L2 now: lane l asks for line l of every 4 KB (a block is at most 16.1 KB).  2.31 -> 2.19 ms on a
    // full c2 container (profiles/r03_entropy_experiments.md)
    for (uint32_t o = lane * 128u; o < s1 - s0; o += 4096u) asm volatile("prefetch.global.L2 [%0];" ::"l"(blk + o));
  }
  // The words the warp will read next sit in two registers per lane (a 64-word window starting at `base`): a lane takes
  // its word with a shuffle, and the window is refilled 32 words ahead of its use, so no global-memory latency is on the
  // loop-carried path (state -> table look-ups -> ballot -> word).
  auto load_words = [&](uint32_t at) -> uint32_t { return at < max_words ? (uint32_t)__ldg(words + at) : 0u; };
  w0 = load_words(lane); w1 = load_words(32 + lane);
  // shared-memory addresses of this warp's tables and staging row, computed once (the loop below is issue-bound)
  const uint32_t lut_a = (uint32_t)__cvta_generic_to_shared(lut + j * Z_M), tab_a = (uint32_t)__cvta_generic_to_shared(tab + j * 256);
  const uint32_t dst_a = (uint32_t)__cvta_generic_to_shared(stage + wi * Z_PART) + lane;
  const uint32_t wshift = w == 4 ? 2 : (w == 2 ? 1 : 0);
  const uint64_t total_bytes = n_sym * w;
  for (uint32_t part = 0; part < Z_PARTS; ++part) {
    const uint32_t k_lo = part * Z_PART, k_hi = min(n, k_lo + Z_PART);
    for (uint32_t k0 = k_lo; k0 < k_hi; k0 += 32) {
      const bool active = k0 + lane < n;
      const uint32_t slot = x & (Z_M - 1);
      uint32_t s, fc;
      asm volatile("ld.shared.u8 %0, [%1];" : "=r"(s) : "r"(lut_a + slot));
      asm volatile("ld.shared.u32 %0, [%1];" : "=r"(fc) : "r"(tab_a + (s << 2)));
      uint32_t xn = (fc & 0xFFFFu) * (x >> Z_PROB_BITS) + slot - (fc >> 16);
      const bool need = active && xn < Z_L;
      const uint32_t mask = __ballot_sync(0xffffffffu, need);
      const uint32_t idx = used - base + __popc(mask & ((1u << lane) - 1u));          // 0 .. 63 inside the window
      const uint32_t c0 = __shfl_sync(0xffffffffu, w0, idx & 31u), c1 = __shfl_sync(0xffffffffu, w1, idx & 31u);
      if (need) xn = (xn << 16) | (idx < 32u ? c0 : c1);
      used += __popc(mask);
      if (used - base >= 32u) {                                                      // warp-uniform
        base += 32u;
        w0 = w1;
        w1 = load_words(base + 32u + lane);
      }
      if (active) {
        x = xn;
        asm volatile("st.shared.u8 [%0], %1;" ::"r"(dst_a + (k0 - k_lo)), "r"(s) : "memory");
      }
    }
    __syncthreads();
    // interleave the planes into elements.  The part holds, for every block q of the chunk, elements [q * 8192 + part * 2048,
    // + 2048): byte jj of local element i of block q is stage[(q * w + jj) * Z_PART + i].
    // 16 output bytes per thread and step: 16 / w consecutive elements, their bytes fetched with one vector load per plane
    const uint32_t vec_per_q = (Z_PART * w) >> 4;                                     // 16-byte vectors of output per block and part
    for (uint32_t t = tid; t < per_plane * vec_per_q; t += Z_THREADS) {
      const uint32_t qq = t / vec_per_q, o = (t - qq * vec_per_q) << 4;               // byte offset inside the (block, part) piece
      const uint64_t out_byte = (uint64_t)chunk * Z_CHUNK_BYTES + ((uint64_t)qq * Z_BLOCK + (uint64_t)part * Z_PART) * w + o;
      if (out_byte >= total_bytes) continue;
      const unsigned char* src = stage + (qq * w) * Z_PART + (o >> wshift);           // plane 0 of the first element of the vector
      uint4 v;
      if (w == 1) {
        v = *reinterpret_cast<const uint4*>(src);
      } else if (w == 2) {
        const uint2 lo = *reinterpret_cast<const uint2*>(src), hi = *reinterpret_cast<const uint2*>(src + Z_PART);
        v.x = __byte_perm(lo.x, hi.x, 0x5140); v.y = __byte_perm(lo.x, hi.x, 0x7362);
        v.z = __byte_perm(lo.y, hi.y, 0x5140); v.w = __byte_perm(lo.y, hi.y, 0x7362);
      } else {
        const uint32_t p0 = *reinterpret_cast<const uint32_t*>(src), p1 = *reinterpret_cast<const uint32_t*>(src + Z_PART);
        const uint32_t p2 = *reinterpret_cast<const uint32_t*>(src + 2 * Z_PART), p3 = *reinterpret_cast<const uint32_t*>(src + 3 * Z_PART);
        const uint32_t a01 = __byte_perm(p0, p1, 0x5140), b01 = __byte_perm(p0, p1, 0x7362);   // (p0.b0 p1.b0 p0.b1 p1.b1), (.. b2 .. b3)
        const uint32_t a23 = __byte_perm(p2, p3, 0x5140), b23 = __byte_perm(p2, p3, 0x7362);
        v.x = __byte_perm(a01, a23, 0x5410); v.y = __byte_perm(a01, a23, 0x7632);
        v.z = __byte_perm(b01, b23, 0x5410); v.w = __byte_perm(b01, b23, 0x7632);
      }
      if (out_byte + 16 <= total_bytes) *reinterpret_cast<uint4*>(A.out + out_byte) = v;
      else {
        const uint32_t vv[4] = {v.x, v.y, v.z, v.w};
        for (uint32_t kb = 0; out_byte + kb < total_bytes; ++kb) A.out[out_byte + kb] = (unsigned char)(vv[kb >> 2] >> (8 * (kb & 3u)));
      }
    }
    __syncthreads();
  }
  if (n) {
    // The encoder starts every coder at Z_L and the decoder undoes its steps exactly, so an intact block leaves all 32 states at
    // Z_L (coders without a symbol never moved) and has consumed every word but at most the one that pads the block to 4 bytes.
    const bool off_end = __any_sync(0xffffffffu, x != Z_L);
    if (lane == 0) {
      if (used > max_words) atomicOr(&err[0], 2u);                              // a block shorter than its symbols need
      else if (off_end || max_words - used > 1u) atomicOr(&err[0], 8u);         // damaged words or states (bit flips inside the block)
    }
  }
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
        if (pos > 0xFFFFFFFFull) return TMD_ERR_LIMIT;                   // block starts are 32-bit: containers stay below 4 GiB
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
      if (pos > 0xFFFFFFFFull) return TMD_ERR_LIMIT;
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
      // (written without sums that could wrap for offsets near 2^64)
      const uint64_t t_off = Z.pl[p_index].table_offset, b_off = Z.pl[p_index].blocks_offset, starts_bytes = 4 * (blocks + 1);
      if (t_off > h.total || h.total - t_off < 512 || b_off > h.total || h.total - b_off < starts_bytes || (t_off & 1u) || (b_off & 3u))
        return TMD_ERR_CORRUPT;
    }
  }
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (cudaMemsetAsync(d_err4, 0, 4, st) != cudaSuccess) return TMD_ERR_CUDA;
  if (chunk == 0) return TMD_OK;
  constexpr size_t smem = (size_t)Z_WARPS * Z_PART + 4 * (size_t)Z_M + 4 * 256 * 4;
  static_assert(smem <= 48 * 1024, "below the default dynamic shared-memory limit: no per-function attribute (and no per-process flag) needed");
  k_entropy_decode<<<chunk, Z_THREADS, smem, st>>>(Z, (uint32_t*)d_err4);
  return cudaGetLastError() == cudaSuccess ? TMD_OK : TMD_ERR_CUDA;
}

}  // extern "C"
