/*
 * tmd.h -- C ABI of the B200-native TPC track-model decoder (libtmd.so).
 *
 * The operation is the one arXiv:2411.02206 describes in §4:
 *   L68  "after the entropy decoding, the clusters' coordinates must be decoded to the absolute values instead of
 *         residuals or differences" -- input = the entropy-decoded compressed-cluster arrays, output = clusters;
 *   L70  attached clusters: "every GPU-thread receives one track, it propagates it through the TPC and computes the
 *         absolute values of the coordinates using the residuals given in input and the reconstructed track";
 *         unattached clusters: "computes each coordinate summing the difference taken from the input array with the
 *         coordinates of the last decoded cluster; each thread decodes clusters from a specific region of the TPC";
 *         the input is a "Structure Of Arrays (SOA)".
 * The paper fixes no layout, geometry, quantisation or output order; those are the readings in DESIGN.md §3
 * (model = SURVEY.md §8(c) C1-C5).  Step names A1..A7 below are the rows of SURVEY.md §8(a).
 *
 * Conventions for every function:
 *   - returns TMD_OK (0) or a negative tmd_status; never throws, aborts or prints;
 *   - "HOST" / "DEVICE" says in which address space a pointer lives;
 *   - the library owns only tmd_ctx; all data buffers, outputs and the workspace belong to the caller.
 */
#ifndef TMD_H_
#define TMD_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  TMD_OK = 0,
  TMD_ERR_ARG = -1,       /* null pointer, size out of the limits below, bad geometry                         */
  TMD_ERR_ALIGN = -2,     /* a device pointer is not aligned as required                                     */
  TMD_ERR_WORKSPACE = -3, /* workspace missing or smaller than tmd_workspace_bytes()                         */
  TMD_ERR_CUDA = -4,      /* a CUDA runtime call failed (allocation, copy, launch)                           */
  TMD_ERR_CORRUPT = -5,   /* TMD_VALIDATE only: counts / first-cluster fields are inconsistent               */
  TMD_ERR_DEVICE = -6,    /* tmd_create: the device cannot run the kernels (no 8-CTA thread-block clusters)  */
  TMD_ERR_LIMIT = -7      /* a fixed built-in size is exceeded: the scratch of tmd_decode_unattached_noalloc,
                             the 4 GiB of a TMDZ container (tmd_entropy_encode_host)                          */
} tmd_status;

#define TMD_MAX_CLUSTERS 0xFFFF0000ull /* n_attached + n_unattached <= this (32-bit indices with headroom for tile overshoot) */

/* Limits: n_attached + n_unattached <= TMD_MAX_CLUSTERS; trk_ncl in [1, 65535]; n_rows <= 255; n_az <= 63; n_sides in {1,2};
 * n_sectors_out <= n_az * n_sides; n_sectors_out * n_rows <= 8192. */

/* Pad-plane geometry (DESIGN.md §3 reading 1).  HOST pointers; deep-copied by tmd_create. */
typedef struct {
  uint32_t n_az;           /* azimuthal sectors per side (18)                                                  */
  uint32_t n_sides;        /* 2; sector = side * n_az + az                                                     */
  uint32_t n_sectors_out;  /* sectors that own output bins: 36, or 2 for the tiny config (sectors 0,1)         */
  uint32_t n_rows;         /* pad rows per sector (152)                                                        */
  float cos_a, sin_a;      /* cos / sin of the sector angle (20 deg) as binary32                               */
  const float* row_x;        /* [n_rows] cm, x of the pad row in the sector frame                              */
  const float* row_padw;     /* [n_rows] cm, pad width                                                         */
  const float* row_inv_padw; /* [n_rows] 1/cm, binary32 of the double reciprocal                               */
  const uint16_t* row_npads; /* [n_rows] pads in the row (even)                                                */
} tmd_geometry;

typedef struct {
  float bz_tesla;          /* solenoid field; the curvature unit is KB = bz_tesla * 0.00299792458f             */
} tmd_field;

/*
 * Compressed-cluster SoA of one time frame ("input Structure Of Arrays"; layout DESIGN.md §3 / SURVEY C2).
 * All arrays: DEVICE pointers in tmd_decode (HOST pointers in tmd_decode_host), caller-owned, read-only for the
 * library, each aligned to 16 bytes.  Little endian.  Arrays of length 0 may be null.
 *   off[t]  = sum of trk_ncl[0..t)   (computed by the library, A1; the paper precomputes these indices on the CPU, L70)
 *   per track t, cluster j = 0 is stored absolute; cluster j >= 1 uses residual index  off[t] - t + j - 1.
 */
typedef struct {
  uint32_t n_tracks;
  uint64_t n_attached;     /* = sum trk_ncl                                                                    */
  uint64_t n_unattached;   /* = sum u_bin_count                                                                */
  /* per track [n_tracks] */
  const uint16_t* trk_ncl;   /* clusters on the track, >= 1                                                    */
  const int8_t* trk_qpt;     /* q/pT in 1/16 c/GeV                                                             */
  const uint8_t* trk_row0;   /* first cluster: pad row, sector, pad code (pad*64), time code (bin*64)          */
  const uint8_t* trk_sec0;
  const uint16_t* trk_pad0;
  const uint32_t* trk_time0;
  /* per attached cluster incl. the first of each track [n_attached], index g = off[t] + j; copied through        */
  const uint16_t* a_qtot;
  const uint16_t* a_qmax;
  const uint8_t* a_flags;
  const uint8_t* a_sigpad;
  const uint8_t* a_sigtime;
  /* per attached cluster excl. the first of each track [n_attached - n_tracks]                                   */
  const uint8_t* a_rowdiff;   /* (row - row_prev) * dir  mod n_rows  (values are reduced mod n_rows)             */
  const uint8_t* a_secleg;    /* bit 7: leg change; bits 0-5: (az - az_prev) mod n_az (reduced mod n_az); bit 6 ignored */
  const uint16_t* a_padres;   /* (P - P_pred) mod 2^16                                                           */
  const uint32_t* a_timeres;  /* (T - T_pred) mod 2^32                                                           */
  /* per unattached cluster [n_unattached], bin after bin in bin order                                            */
  const uint16_t* u_qtot;
  const uint16_t* u_qmax;
  const uint8_t* u_flags;
  const uint8_t* u_sigpad;
  const uint8_t* u_sigtime;
  const uint16_t* u_paddiff;  /* difference to the preceding cluster of the bin, mod 2^16 (first: to 0)          */
  const uint32_t* u_timediff; /* same for time, mod 2^32                                                         */
  const uint32_t* u_bin_count; /* [n_sectors_out * n_rows] unattached clusters per bin = sector * n_rows + row   */
} tmd_compressed;

/* One decoded cluster: 16 bytes, little endian, naturally aligned. */
typedef struct {
  uint32_t time;   /* time code T = time bin * 64                                                              */
  uint16_t pad;    /* pad code  P = pad * 64                                                                   */
  uint16_t qtot;
  uint16_t qmax;
  uint8_t sigpad;
  uint8_t sigtime;
  uint8_t flags;
  uint8_t row;
  uint8_t sector;
  uint8_t zero;    /* always 0                                                                                 */
} tmd_cluster;

/*
 * Output (DEVICE pointers in tmd_decode, HOST pointers in tmd_decode_host; caller-owned, written by the library).
 * Canonical order (DESIGN.md §3 reading 11): bin b = sector * n_rows + row owns clusters[bin_offset[b] .. bin_offset[b+1]):
 * first the attached clusters of the bin in ascending global attached index g, then its unattached clusters in
 * stored order.
 */
typedef struct {
  tmd_cluster* clusters;   /* [n_attached + n_unattached], 16-byte aligned                                     */
  uint32_t* bin_offset;    /* [n_sectors_out * n_rows + 1]                                                     */
  uint32_t* probe_state;   /* nullable: [n_tracks][6] binary32 bit patterns of the track state (x,y,u,sp,dt,k)
                              after cluster min(probe_step, trk_ncl-1) has been rebuilt and the state updated  */
  uint32_t probe_step;     /* UINT32_MAX = final state                                                         */
  void* workspace;         /* DEVICE scratch, 256-byte aligned; ignored by tmd_decode_host                     */
  size_t workspace_bytes;  /* >= tmd_workspace_bytes(...)                                                      */
} tmd_output;

typedef struct tmd_ctx tmd_ctx;

/* flags of tmd_decode */
#define TMD_VALIDATE 1u /* check on the device that sum(trk_ncl) == n_attached (summed in 64 bits), sum(u_bin_count) ==
                           n_unattached, every trk_ncl >= 1, trk_row0 < n_rows, trk_sec0 < n_az*n_sides -- BEFORE any decode
                           work is enqueued: the call synchronises the stream, and returns TMD_ERR_CORRUPT with nothing
                           decoded if a check fails -- and, after the decode, that every decoded sector is
                           < n_sectors_out (second synchronisation; TMD_ERR_CORRUPT, the offending clusters dropped).
                           Without it such inputs are undefined except that nothing is written out of bounds
                           of `clusters` for a decoded sector >= n_sectors_out (the cluster is dropped). */

#define TMD_TIMING 2u   /* record a CUDA event pair around every kernel (tmd_kernel_times).  The first such call on a
                           context creates the 2 x TMD_MAX_KERNELS events; calls with TMD_TIMING must not run concurrently
                           on one context */
#define TMD_MAX_KERNELS 24
#define TMD_MAX_BATCH 1024 /* frames per tmd_decode_batch call */

/* Uploads the geometry tables to the current CUDA device.  *out_ctx is set only on success. */
int tmd_create(const tmd_geometry* geometry, const tmd_field* field, tmd_ctx** out_ctx);

/* Scratch bytes tmd_decode needs for a time frame of this size (a pure function of the sizes). */
int tmd_workspace_bytes(const tmd_ctx* ctx, uint32_t n_tracks, uint64_t n_attached, uint64_t n_unattached, size_t* out_bytes);

/*
 * Decode one time frame (rows A1-A7).  Only enqueues kernels on `cuda_stream` (a cudaStream_t; null =
 * default stream) and returns: no allocation, no host synchronisation and no device-to-host copy unless TMD_VALIDATE
 * (two synchronisations, see above) or TMD_TIMING (event creation on first use) is set.  All kernels run on that one
 * stream in order: A1 offsets, A2 length sort, A3 + A5 track decode, A3 ranks, A4 column scan and bin offsets, A7
 * unattached clusters, A6 scatter.  Results are valid once the stream has been synchronised.
 * Concurrency: the context is read-only during the call (apart from the launch counter, which every call sets to the
 * same value), so calls on one context from different streams / host threads are allowed as long as they use different
 * workspaces and outputs and none of them sets TMD_TIMING.
 */
int tmd_decode(tmd_ctx* ctx, const tmd_compressed* in, tmd_output* out, uint32_t flags, void* cuda_stream);

/*
 * Decode `n_frames` independent time frames with ONE launch sequence (PAPER.md L70 runs "multiple
 * instances ... concurrently": small frames -- single events, pp-like frames -- do not fill the GPU one at a time).
 * `in` / `out` are HOST arrays of n_frames structs holding DEVICE pointers exactly as for tmd_decode; every frame has its
 * own outputs and its own workspace (>= tmd_workspace_bytes of ITS sizes).  The result of frame i is what
 * tmd_decode(ctx, &in[i], &out[i], ...) produces.  Every kernel's grid gets a frame coordinate; the per-frame arguments
 * live in frame 0's workspace for the duration of the call.  1 <= n_frames <= TMD_MAX_BATCH; TMD_VALIDATE is not
 * accepted (TMD_ERR_ARG): it synchronises.  All frames are checked before anything is enqueued.
 */
int tmd_decode_batch(tmd_ctx* ctx, uint32_t n_frames, const tmd_compressed* in, tmd_output* out, uint32_t flags, void* cuda_stream);

/*
 * End-to-end convenience: every pointer in `in` / `out` is a HOST pointer (pinned memory makes the copies asynchronous;
 * out->workspace is ignored).  Copies the inputs to device buffers owned by the context (grown on demand and reused),
 * runs tmd_decode, copies clusters / bin_offset / probe_state back and synchronises the stream.
 */
int tmd_decode_host(tmd_ctx* ctx, const tmd_compressed* in, tmd_output* out, uint32_t flags, void* cuda_stream);

/*
 * Pipelined form of tmd_decode_host (the deployment shape of PAPER.md L64 / L70: "multiple instances are executed
 * concurrently on different streams, reducing the memory transfer latency").  The context owns TMD_HOST_SLOTS device
 * arenas and three streams (uploads, decode, downloads).  tmd_decode_host_async enqueues the upload, the decode and the
 * download of one time frame in slot `slot` (0 .. TMD_HOST_SLOTS-1) and returns; if the slot still holds an earlier
 * frame it first waits for that frame's download.  With two slots used alternately the upload of frame i+1 runs beside
 * the download of frame i.  HOST pointers as in tmd_decode_host; they must be pinned for the copies to overlap and must
 * stay valid until tmd_host_wait(slot) returns.  TMD_VALIDATE is not accepted (it synchronises): TMD_ERR_ARG.
 * tmd_host_wait blocks until the frame in `slot` is complete in the host buffers (no-op for an idle slot).
 */
#define TMD_HOST_SLOTS 2
int tmd_decode_host_async(tmd_ctx* ctx, const tmd_compressed* in, tmd_output* out, uint32_t flags, int slot);
int tmd_host_wait(tmd_ctx* ctx, int slot);

/*
 * Unattached clusters only (row A7 with the bin offsets of A4, second kernel: "computes each coordinate
 * summing the difference taken from the input array with the coordinates of the last decoded cluster"), for callers that
 * MAY NOT ALLOCATE device memory -- neither here nor at set-up.  Typical cases: the library runs inside a framework that
 * claimed the whole device memory as one block at start-up and rules out any later cudaMalloc; the caller is a plug-in that
 * only ever sees device pointers handed to it; the call sits in a loop that cannot afford the device-wide serialisation of
 * cudaMalloc / cudaFree.  Such a caller cannot use tmd_create (it allocates the geometry table) or provide a workspace, so
 * this call takes neither: no context, no workspace, and it calls no cudaMalloc, cudaFree or other allocating routine.
 *
 * Its scratch (the per-bin start table, 4 bytes x 2 per bin) is a fixed array of 65 792 bytes compiled into libtmd.so;
 * every GPU on which the library's code is loaded holds that array from then until the process exits, used or not.
 * Hence the limit: n_sectors_out * n_rows <= TMD_NOALLOC_MAX_BINS, else TMD_ERR_LIMIT (also for n_unattached >
 * TMD_MAX_CLUSTERS); nothing is enqueued for a refused call.
 *
 *   n_sectors_out, n_rows : the bin grid, bin = sector * n_rows + row (n_rows <= 255), as in tmd_geometry;
 *   in        : HOST struct; n_tracks and n_attached must be 0 (TMD_ERR_ARG otherwise: attached clusters need tmd_decode);
 *               u_bin_count [n_bins] and the seven u_* arrays [n_unattached] are DEVICE pointers, 16-byte aligned,
 *               caller-owned, read-only; the trk_* / a_* members are ignored;
 *   clusters  : DEVICE [n_unattached], 16-byte aligned, written; bin after bin, each bin in stored order;
 *   bin_offset: DEVICE [n_bins + 1], written;
 *   both outputs equal, byte for byte, what tmd_decode writes for the same frame.
 * Enqueues two kernels on `cuda_stream` and returns; results are valid once the stream has been synchronised.
 *
 * Set-up: the FIRST call on each device looks up the array's device address (cudaGetSymbolAddress, with the caller's
 * current device; checked, TMD_ERR_CUDA on failure) and remembers it per device.  Make that first call during
 * initialisation, before any stream capture begins on that device.
 * Sharing: all calls on one device use the same array, and it keeps what the previous call left there.  Each call rewrites
 * every entry it will read (including the part that must be zero) before reading it, so calls that run one after the other
 * -- same stream, or ordered by events -- are independent of each other.  Two calls whose kernels can overlap on the GPU
 * (different streams or host threads, no ordering between them) RACE on the array: the results of both are undefined.
 */
#define TMD_NOALLOC_MAX_BINS 8192u
int tmd_decode_unattached_noalloc(uint32_t n_sectors_out, uint32_t n_rows, const tmd_compressed* in, tmd_cluster* clusters,
                                  uint32_t* bin_offset, void* cuda_stream);

/*
 * Self test of the arithmetic the track-decode kernel relies on (every model operation is ONE IEEE-754
 * binary32 round-to-nearest operation).  The kernel issues the fast sequences of IEEE division and square root without
 * their per-operation range checks (one merged check per cluster instead) and a fused floor-clamp-convert; this call
 * compares them on the current device with __fdiv_rn / __fsqrt_rn / floorf + clamp: mismatches[0] = square root over
 * every binary32 argument in [2^-100, 2^100]; mismatches[1] = division over 2^log2_pairs pseudo-random operand pairs
 * (dividend magnitude in [2^-40, 2^84], divisor magnitude in [2^-10, 2^80]: the ranges the kernel sends down the fast
 * path) plus an exhaustive grid of edge mantissas x exponents; mismatches[2] = the floor-clamp conversion over every
 * binary32 pattern.  All three must be 0.  Synchronous; HOST pointer; log2_pairs <= 40.
 */
int tmd_selftest_ieee(uint32_t log2_pairs, uint64_t mismatches[3]);

/* Frees the context and its device tables / buffers.  Null is accepted. */
int tmd_destroy(tmd_ctx* ctx);

const char* tmd_status_string(int status);

/* Number of kernel launches the last tmd_decode on this context enqueued (for bench.py's gpu_launches). */
int tmd_last_launch_count(const tmd_ctx* ctx);

/*
 * Per-kernel device times of the last tmd_decode / tmd_decode_batch that ran with TMD_TIMING: waits for that call's last
 * event, then fills names[i] (static strings) and ms[i] for its kernels in launch order.  Returns the number filled (0 if
 * the last call did not use TMD_TIMING) or a negative tmd_status.  A batch reports the upload of its frame table (one
 * small launch per 8 frames) as a single row "store_frames", so the rows never exceed TMD_MAX_KERNELS.
 */
int tmd_kernel_times(tmd_ctx* ctx, int max_kernels, const char** names, float* ms);

/*
 * Track-model ENCODING of the attached clusters (the synchronous-side step of PAPER.md L68: each coordinate is stored
 * "as the residual to the correspondent track"; model and formats as above).  DEVICE pointers.
 * `att` holds the attached clusters in g order (track after track); `leg` the leg index of each inside its track;
 * trk_qptf the signed curvature / KB in c/GeV.  Writes the trk_* (except trk_ncl) and a_* arrays `out` points to
 * (as writable device memory; the u_* members are ignored).  `workspace` as for tmd_decode with n_unattached = 0.
 * Synchronises the stream; TMD_ERR_CORRUPT if sum(trk_ncl) != n_attached, a row/sector is out of range or a track
 * changes side.
 */
typedef struct {
  uint32_t n_tracks;
  uint64_t n_attached;
  const uint16_t* trk_ncl;   /* [n_tracks]   */
  const float* trk_qptf;     /* [n_tracks]   */
  const tmd_cluster* att;    /* [n_attached] */
  const uint8_t* leg;        /* [n_attached] */
} tmd_attached_truth;

int tmd_encode_attached(tmd_ctx* ctx, const tmd_attached_truth* in, tmd_compressed* out, void* workspace, size_t workspace_bytes,
                        void* cuda_stream);

/*
 * Track-model ENCODING of the unattached clusters ("unassigned clusters are sorted by coordinate position
 * ... stored as differences relative to the preceding cluster"): per (sector,row) bin, sort ascending
 * by the tuple (time, pad, qtot, qmax, sigpad, sigtime, flags), store pad / time as differences to the predecessor (first
 * of a bin: to (0,0)), copy the other fields through.  `un` = DEVICE array of n_unattached clusters in ANY order (sector
 * and row name the bin).  Writes out->u_bin_count [n_sectors_out * n_rows] and the seven u_* arrays [n_unattached] (as
 * writable DEVICE memory; every other member of `out` is ignored).  `workspace` >= tmd_encode_unattached_workspace_bytes,
 * 256-byte aligned.  Synchronises the stream.  TMD_ERR_CORRUPT if a cluster's row / sector has no output bin.
 * With tmd_encode_attached this is the whole encoder: tmd_decode(encode(x)) reproduces x in canonical order.
 */
int tmd_encode_unattached_workspace_bytes(const tmd_ctx* ctx, uint64_t n_unattached, size_t* out_bytes);
int tmd_encode_unattached(tmd_ctx* ctx, uint64_t n_unattached, const tmd_cluster* un, tmd_compressed* out, void* workspace,
                          size_t workspace_bytes, void* cuda_stream);

/*
 * Entropy stage in front of the decoder.  PAPER.md L20: the compressed time frames are written with
 * "lossless ANS"; L49: "TPC Entropy Decoding" is the step right before track-model decoding; L68: the decoder's input is
 * what "the entropy decoding" produces.  The paper gives no format; "TMDZ" is this build's own: every array
 * of tmd_compressed is split into byte planes, each plane range-ANS coded (12-bit static table per plane, 32-bit state,
 * 16-bit renormalisation) in blocks of 8192 symbols by 32 interleaved coders.
 *
 * tmd_entropy_bound:       upper bound of the container size for these counts.
 * tmd_entropy_encode_host: HOST arrays in (`in`: host pointers), TMDZ container out (`blob`, HOST, capacity >= the bound).
 *                          Runs on the calling host thread (the paper's rANS encoding is a CPU step of the synchronous
 *                          phase, L40).  A container is limited to 4 GiB (block positions are 32-bit byte offsets from
 *                          its start): TMD_ERR_LIMIT when the coded data passes that, `blob` is then unspecified.  The
 *                          bound is not the test (it assumes incompressible data): a full Pb-Pb frame, 4.8 GB of
 *                          arrays, codes to about 2.1 GB.
 * tmd_entropy_sizes:       counts stored in a container's header (`head` = at least its first 64 bytes, HOST).
 * tmd_entropy_decode:      decodes a container resident in DEVICE memory (`d_blob`, 16-byte aligned) into the DEVICE arrays
 *                          `out` points to (caller-allocated with the counts of tmd_entropy_sizes, 16-byte aligned; out's
 *                          n_tracks / n_attached / n_unattached must equal the header's).  `head` = HOST copy of the
 *                          container's first 64 + 32 * 43 bytes (header + plane directory; the caller read the container
 *                          from storage through host memory anyway).  Only enqueues one kernel on `cuda_stream`; one CTA
 *                          decodes eight blocks (one per warp) and assembles 64 KiB of one array.  `d_err4` = 4 bytes of
 *                          DEVICE memory that are non-zero afterwards if the container is corrupt (bit 0: a table does
 *                          not sum to 4096; bit 1: a block is shorter than its symbols need; bit 2: a block position is
 *                          out of order, out of bounds or misaligned; bit 3: a block's coder states do not return to
 *                          their start value or words are left over, i.e. its data was altered); the output is then
 *                          unspecified but nothing is read or written out of bounds.  A plane directory that points
 *                          outside the container is refused on the host (TMD_ERR_CORRUPT).
 *                          The arrays can be handed to tmd_decode on the same stream right away.
 */
#define TMD_ENTROPY_HEAD_BYTES 1440u /* 64-byte header + 43 plane records of 32 bytes */
int tmd_entropy_bound(uint32_t n_tracks, uint64_t n_attached, uint64_t n_unattached, uint32_t n_bins, size_t* out_bytes);
int tmd_entropy_encode_host(const tmd_compressed* in, uint32_t n_bins, void* blob, size_t capacity, size_t* out_bytes);
int tmd_entropy_sizes(const void* head, size_t head_bytes, uint32_t* n_tracks, uint64_t* n_attached, uint64_t* n_unattached,
                      uint32_t* n_bins, size_t* blob_bytes);
int tmd_entropy_decode(const void* head, size_t head_bytes, const void* d_blob, size_t blob_bytes, tmd_compressed* out, void* d_err4,
                       void* cuda_stream);

/*
 * The deployment shape end to end (entropy decoding, then track-model decoding, transfers beside the
 * kernels): a TMDZ container in HOST memory in, decoded clusters in HOST memory out.  Works like tmd_decode_host_async --
 * same slots, same three streams, same tmd_host_wait -- but uploads the CONTAINER (about 2.3x smaller than the arrays it
 * codes), runs tmd_entropy_decode into arrays inside the slot's device arena and tmd_decode right behind it on the same
 * stream; the compressed arrays never exist in host memory.
 *   blob / blob_bytes : HOST, the whole container (at least the size its header states); pinned memory makes the copy
 *                       asynchronous; must stay valid until tmd_host_wait(slot) returns.  Its bin count must be the
 *                       context's (TMD_ERR_ARG otherwise); a header that is not TMDZ: TMD_ERR_CORRUPT.
 *   out               : HOST pointers as in tmd_decode_host (clusters sized from tmd_entropy_sizes; workspace ignored).
 * tmd_host_wait(slot) returns TMD_ERR_CORRUPT if the entropy stage flagged the container (see tmd_entropy_decode); the
 * output is then unspecified.  TMD_VALIDATE is not accepted (TMD_ERR_ARG).  May be mixed with tmd_decode_host_async calls
 * on other slots.  The first call on a slot allocates (device arena, a pinned error word, events).
 */
int tmd_decode_container_host_async(tmd_ctx* ctx, const void* blob, size_t blob_bytes, tmd_output* out, uint32_t flags, int slot);

#ifdef __cplusplus
}
#endif
#endif /* TMD_H_ */
