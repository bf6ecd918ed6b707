// tmd_encode.cuh -- track-model ENCODING of the attached clusters (the synchronous-side step: "stores
// each coordinate as the residual to the correspondent track").  SURVEY.md §8(f)-3 / §8(c)-C6.
//
// Same model as the decoder (tmd_decode.cuh): for cluster j >= 1 the residual to the quantised prediction is stored and
// the state is updated with the TRUE cluster.  Used by bench.py to turn synthetic helix events into the compressed SoA
// on the device, and checked bit for bit against the oracle's encoder in the GPU tests.
#pragma once

#include "tmd_common.cuh"
#include "tmd_decode.cuh"

namespace tmd {

struct EncodeArgs {
  uint32_t n_tracks;
  const uint32_t* off;          // [n_tracks+1]
  const float* trk_qptf;        // [n_tracks] signed curvature / KB in c/GeV (C6)
  const uint4* att;             // [n_attached] g-ordered 16-byte cluster records
  const uint8_t* leg;           // [n_attached] leg index inside the track
  // outputs (device, writable)
  int8_t* trk_qpt; uint8_t* trk_row0; uint8_t* trk_sec0; uint16_t* trk_pad0; uint32_t* trk_time0;
  uint16_t* a_qtot; uint16_t* a_qmax; uint8_t* a_flags; uint8_t* a_sigpad; uint8_t* a_sigtime;
  uint8_t* a_rowdiff; uint8_t* a_secleg; uint16_t* a_padres; uint32_t* a_timeres;
  uint32_t* err;
};

__global__ void __launch_bounds__(128) k_encode_attached(DevGeo G, EncodeArgs A) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  RowGeo* rows = reinterpret_cast<RowGeo*>(smem_raw);
  for (uint32_t r = threadIdx.x; r < G.n_rows; r += blockDim.x) rows[r] = G.rows[r];
  __syncthreads();
  const uint32_t t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= A.n_tracks) return;
  const uint32_t g0 = A.off[t], ncl = A.off[t + 1] - g0;
  const float q = clampf(floorf(fadd(fmul(A.trk_qptf[t], 16.0f), 0.5f)), -127.0f, 127.0f);
  const int qpt = (int)q;
  uint4 c = A.att[g0];
  uint32_t T = c.x, P = c.y & 0xFFFFu, row = (c.w >> 8) & 0xFFu, sec = (c.w >> 16) & 0xFFu;
  if (row >= G.n_rows || sec >= G.n_az * G.n_sides) {
    atomicOr(&A.err[ERR_TRACK_FIELD], 1u);
    return;
  }
  A.trk_qpt[t] = (int8_t)qpt; A.trk_row0[t] = (uint8_t)row; A.trk_sec0[t] = (uint8_t)sec;
  A.trk_pad0[t] = (uint16_t)P; A.trk_time0[t] = T;
  TrackState s;
  track_init(s, G, rows[row], qpt, P, T);
  int dir = +1;
  uint32_t az = sec % G.n_az, leg_prev = A.leg[g0];
  for (uint32_t j = 0; j < ncl; ++j) {
    const uint32_t g = g0 + j;
    if (j > 0) c = A.att[g];
    A.a_qtot[g] = (uint16_t)(c.y >> 16); A.a_qmax[g] = (uint16_t)(c.z & 0xFFFFu);
    A.a_sigpad[g] = (uint8_t)(c.z >> 16); A.a_sigtime[g] = (uint8_t)(c.z >> 24); A.a_flags[g] = (uint8_t)(c.w & 0xFFu);
    if (j == 0) continue;
    const uint32_t row_n = (c.w >> 8) & 0xFFu, sec_n = (c.w >> 16) & 0xFFu, leg_n = A.leg[g];
    if (row_n >= G.n_rows || sec_n / G.n_az != sec / G.n_az) {  // tracks never change side
      atomicOr(&A.err[ERR_TRACK_FIELD], 2u);
      return;
    }
    const bool legflag = leg_n != leg_prev;
    if (legflag) dir = -dir;
    const int dr = ((int)row_n - (int)row) * dir;
    const uint32_t rd = (uint32_t)(((dr % (int)G.n_rows) + (int)G.n_rows) % (int)G.n_rows);
    const uint32_t az_n = sec_n % G.n_az;
    const uint32_t d = (az_n + G.n_az - az) % G.n_az;
    const size_t i = (size_t)g - t - 1;
    A.a_rowdiff[i] = (uint8_t)rd;
    A.a_secleg[i] = (uint8_t)((legflag ? 0x80u : 0u) | d);
    track_leg_and_sector(s, G, legflag, d);
    const Prediction p = track_predict(s, rows[row_n], P, T);
    const uint32_t Pn = c.y & 0xFFFFu, Tn = c.x;
    A.a_padres[i] = (uint16_t)((Pn - p.P) & 0xFFFFu);
    A.a_timeres[i] = Tn - p.T;
    track_update(s, rows[row_n], j, p, Pn, Tn);
    P = Pn; T = Tn; row = row_n; sec = sec_n; az = az_n; leg_prev = leg_n;
  }
}

}  // namespace tmd
