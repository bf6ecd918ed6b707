/*
 * tmd_oracle.c -- plain, slow, single-threaded CPU oracle for TPC track-model coding.
 *
 * TEST INFRASTRUCTURE ONLY.  Nothing in the product path (paper_2411_02206_b200/) may include, link or call this
 * file; only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs use it.
 * It shares no code with the CUDA library (own structs, own constants, own helpers).
 *
 * What it follows.  The paper (PAPER.md = arXiv:2411.02206) describes the method in two paragraphs:
 *   L68 (§4 ¶1): each coordinate of a cluster attached to a track is stored "as the residual to the correspondent
 *                track"; unassigned clusters are "sorted by coordinate position" and stored "as differences relative
 *                to the preceding cluster"; decoding restores "the absolute values".
 *   L70 (§4 ¶2): attached: a track is propagated "through the TPC" and the absolute coordinates are computed
 *                "using the residuals given in input and the reconstructed track"; unattached: "summing the
 *                difference taken from the input array with the coordinates of the last decoded cluster", per
 *                "specific region of the TPC".
 * The paper gives no formula, geometry, quantisation or ordering; those are the readings listed in DESIGN.md §3
 * (taken from SURVEY.md §8(c) C1-C7).  Step numbers "C3-n" below are that op list.  Every `f*` helper is ONE IEEE-754
 * binary32 round-to-nearest-even operation; build with -ffp-contract=off -fno-fast-math (oracle/build.py does).
 *
 * Parity pins (tests/test_oracle_*.py, all `-m "not gpu"`): worked trace tests/golden/c9_trace.txt; closed forms
 * (straight radial track, mirror twice); noiseless exact helices give residuals of a few codes (physical fidelity:
 * a dropped term / wrong sign / wrong index blows this up); numpy.cumsum / stable argsort for offsets, unattached
 * sums and the canonical order; decode(encode(x)) == x; brute-force checks on tiny inputs; and, for every branch of
 * orc_init / orc_step (the `!ok` path, multi-step rotations, the saturation constants, reading 19's reductions), an
 * independent numpy-float32 evaluation of the op list (tests/c3_numpy.py, tests/test_oracle_independent.py) compared
 * per step on all 20 trace columns; the encoder's own lines (trk_qpt rounding / clamp, the unattached sort key) by
 * hand-worked values and numpy.lexsort, the short-step branch with dx != 0 by constructed tracks, the whole file under
 * ASan + UBSan (tests/test_oracle_encoder_pins.py).  DESIGN.md §4 lists mutation -> failing test.  No function here is
 * "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORC_OK 0
#define ORC_ERR_ARG (-1)
#define ORC_ERR_CORRUPT (-5)
#define ORC_ERR_NOMEM (-6)

typedef struct {
  uint32_t n_az, n_sides, n_sectors_out, n_rows;
  float cos_a, sin_a, bz_tesla;
  const float *row_x, *row_padw, *row_inv_padw;
  const uint16_t *row_npads;
} orc_geometry;

typedef struct { /* compressed SoA, host pointers (DESIGN.md §4 / SURVEY C2) */
  uint32_t n_tracks;
  uint64_t n_attached, n_unattached;
  const uint16_t *trk_ncl; const int8_t *trk_qpt; const uint8_t *trk_row0, *trk_sec0;
  const uint16_t *trk_pad0; const uint32_t *trk_time0;
  const uint16_t *a_qtot, *a_qmax; const uint8_t *a_flags, *a_sigpad, *a_sigtime;
  const uint8_t *a_rowdiff, *a_secleg; const uint16_t *a_padres; const uint32_t *a_timeres;
  const uint16_t *u_qtot, *u_qmax; const uint8_t *u_flags, *u_sigpad, *u_sigtime;
  const uint16_t *u_paddiff; const uint32_t *u_timediff;
  const uint32_t *u_bin_count;
} orc_compressed;

typedef struct { /* 16-byte output record */
  uint32_t time; uint16_t pad, qtot, qmax; uint8_t sigpad, sigtime, flags, row, sector, zero;
} orc_cluster;

typedef struct { /* per-step trace row, bit patterns as in SURVEY C9's table */
  uint32_t sec, row; int32_t dir, ok;
  uint32_t x, y, sp;           /* after steps 3-5 */
  uint32_t sp2, y2, u2, s;     /* step 6 (only meaningful if ok) */
  uint32_t P_pred, T_pred, P, T;
  uint32_t yn, un, spn, dtn, kn; /* after step 9 */
} orc_trace_row;

/* ---- single IEEE binary32 operations ------------------------------------------------------------------ */
static inline float fadd(float a, float b) { return a + b; }
static inline float fsub(float a, float b) { return a - b; }
static inline float fmul(float a, float b) { return a * b; }
static inline float fdiv(float a, float b) { return a / b; }
static inline float fsqrt(float a) { return sqrtf(a); }
static inline float clampf(float v, float lo, float hi) { /* == fminf(fmaxf(v,lo),hi); NaN -> lo */
  if (!(v >= lo)) v = lo;
  if (v > hi) v = hi;
  return v;
}
static inline uint32_t fbits(float f) { uint32_t u; memcpy(&u, &f, 4); return u; }

/* ---- constants ----------------------------------------------------------------------------- */
static const float SP_MAX = 0.95f, S_MIN = 0.001f, DT_MAX = 8.0f, ALPHA = 0.5f, BETA = 0.25f, INV64 = 0.015625f;
static const float C24 = 0.041666668f; /* fp32(1/24) = 0x3d2aaaab */

typedef struct {
  float x, y, u, sp, dt, k;
  int dir;
  uint32_t sec, row, P, T; /* last rebuilt cluster */
} orc_state;

static inline float half_of(const orc_geometry *g, uint32_t r) { return (float)(g->row_npads[r] / 2); }

/* pad2y / time2u / quantP / quantT: SURVEY C3 "Helpers" */
static inline float pad2y(const orc_geometry *g, uint32_t r, uint32_t P) {
  return fmul(fsub(fmul((float)P, INV64), half_of(g, r)), g->row_padw[r]);
}
static inline float time2u(uint32_t T) { return fmul((float)T, INV64); }
static inline uint32_t quantP(const orc_geometry *g, float y, uint32_t r) {
  float pf = fadd(fmul(y, g->row_inv_padw[r]), half_of(g, r));
  float v = floorf(fadd(fmul(pf, 64.0f), 0.5f));
  v = clampf(v, 0.0f, 65535.0f);
  return (uint32_t)(int32_t)v;
}
static inline uint32_t quantT(float u) {
  float v = floorf(fadd(fmul(u, 64.0f), 0.5f));
  v = clampf(v, 0.0f, 16777215.0f);
  return (uint32_t)(int32_t)v;
}

/* C3-1, C3-2: state at a track's first cluster (stored absolute: PAPER.md L68 + north_star) */
static void orc_init(const orc_geometry *g, orc_state *st, int8_t qpt, uint32_t sec0, uint32_t row0, uint32_t P0,
                     uint32_t T0) {
  const float KB = fmul(g->bz_tesla, 0.00299792458f);
  const float QK = fmul(0.0625f, KB);
  st->k = fmul((float)qpt, QK);
  st->x = g->row_x[row0];
  st->y = pad2y(g, row0, P0);
  st->u = time2u(T0);
  st->dt = 0.0f;
  st->dir = +1;
  float L = fsqrt(fadd(fmul(st->x, st->x), fmul(st->y, st->y)));
  float sd = clampf(fmul(fmul(0.5f, st->k), L), -SP_MAX, SP_MAX);
  float cd = fsqrt(fsub(1.0f, fmul(sd, sd)));
  st->sp = clampf(fdiv(fadd(fmul(st->y, cd), fmul(st->x, sd)), L), -SP_MAX, SP_MAX);
  st->sec = sec0; st->row = row0; st->P = P0; st->T = T0;
}

/*
 * C3-3 .. C3-9 for cluster j >= 1 of a track.  PAPER.md L70: "propagates it through the TPC and computes the absolute
 * values of the coordinates using the residuals given in input and the reconstructed track".
 * encode == 0: *P_io,*T_io carry the stored residuals in and the rebuilt (P,T) out  (C3-8).
 * encode != 0: *P_io,*T_io carry the true (P,T) in and the residuals out            (C6).
 */
static void orc_step(const orc_geometry *g, orc_state *st, uint32_t j, uint8_t rowdiff, uint8_t secleg, int encode,
                     uint32_t *P_io, uint32_t *T_io, orc_trace_row *tr) {
  const uint32_t n_rows = g->n_rows, n_az = g->n_az;
  /* C3-3 leg */
  if (secleg & 0x80) { st->dir = -st->dir; st->sp = -st->sp; st->dt = -st->dt; st->k = -st->k; }
  /* C3-4 row (reading 19: stored values are reduced mod n_rows / mod n_az, so any byte is defined) */
  uint32_t rd = (uint32_t)rowdiff % n_rows;
  st->row = (st->row + (st->dir > 0 ? rd : n_rows - rd)) % n_rows;
  /* C3-5 sector */
  uint32_t d = (uint32_t)(secleg & 0x3F) % n_az;
  if (d != 0) {
    uint32_t az = st->sec % n_az, side = st->sec / n_az;
    az = (az + d) % n_az;
    st->sec = side * n_az + az;
    int steps = (d <= n_az / 2) ? (int)d : (int)d - (int)n_az;
    float sn = steps > 0 ? g->sin_a : -g->sin_a;
    int n = steps > 0 ? steps : -steps;
    for (int q = 0; q < n; ++q) {
      float cp = fsqrt(fsub(1.0f, fmul(st->sp, st->sp)));
      float xn = fadd(fmul(st->x, g->cos_a), fmul(st->y, sn));
      float yn = fsub(fmul(st->y, g->cos_a), fmul(st->x, sn));
      float spn = clampf(fsub(fmul(st->sp, g->cos_a), fmul(cp, sn)), -SP_MAX, SP_MAX);
      st->x = xn; st->y = yn; st->sp = spn;
    }
  }
  if (tr) { tr->sec = st->sec; tr->row = st->row; tr->dir = st->dir; tr->x = fbits(st->x); tr->y = fbits(st->y); tr->sp = fbits(st->sp); }
  /* C3-6 propagate to the new row's x */
  const uint32_t row = st->row;
  const float xt = g->row_x[row];
  float dx = fsub(xt, st->x);
  float sp2 = fadd(st->sp, fmul(st->k, dx));
  int ok = !(fabsf(sp2) > SP_MAX);
  float y2 = 0.0f, u2 = 0.0f, s = 0.0f;
  if (ok) {
    float cp1 = fsqrt(fsub(1.0f, fmul(st->sp, st->sp)));
    float cp2 = fsqrt(fsub(1.0f, fmul(sp2, sp2)));
    float dy = fdiv(fmul(dx, fadd(st->sp, sp2)), fadd(cp1, cp2));
    float ch = fsqrt(fadd(fmul(dx, dx), fmul(dy, dy)));
    if (dx < 0.0f) ch = -ch;
    float kc = fmul(st->k, ch);
    s = fmul(ch, fadd(1.0f, fmul(fmul(kc, kc), C24)));
    y2 = fadd(st->y, dy);
    u2 = fadd(st->u, fmul(st->dt, s));
  }
  /* C3-7 predict */
  uint32_t P_pred, T_pred;
  if (ok) { P_pred = quantP(g, y2, row); T_pred = quantT(u2); }
  else { P_pred = st->P; T_pred = st->T; }
  /* C3-8 rebuild (decode) or residual (encode, C6) */
  uint32_t P, T;
  if (encode) {
    P = *P_io & 0xFFFFu; T = *T_io;
    *P_io = (P - P_pred) & 0xFFFFu;
    *T_io = T - T_pred;
  } else {
    P = (P_pred + *P_io) & 0xFFFFu;
    T = T_pred + *T_io;
    *P_io = P; *T_io = T;
  }
  /* C3-9 update with the rebuilt cluster */
  float ym = pad2y(g, row, P), um = time2u(T);
  st->x = xt;
  if (!ok) {
    st->y = ym; st->u = um; st->sp = clampf(sp2, -SP_MAX, SP_MAX);
  } else {
    float ry = fsub(ym, y2), ru = fsub(um, u2);
    st->y = fadd(y2, fmul(ALPHA, ry));
    st->u = fadd(u2, fmul(ALPHA, ru));
    if (fabsf(s) >= S_MIN) {
      st->sp = clampf(fadd(sp2, fdiv(fmul(BETA, ry), s)), -SP_MAX, SP_MAX);
      float bu = (j == 1) ? 1.0f : BETA;
      st->dt = clampf(fadd(st->dt, fdiv(fmul(bu, ru), s)), -DT_MAX, DT_MAX);
    } else {
      st->sp = clampf(sp2, -SP_MAX, SP_MAX);
    }
  }
  st->P = P; st->T = T;
  if (tr) {
    tr->ok = ok; tr->sp2 = fbits(sp2); tr->y2 = fbits(y2); tr->u2 = fbits(u2); tr->s = fbits(s);
    tr->P_pred = P_pred; tr->T_pred = T_pred; tr->P = P; tr->T = T;
    tr->yn = fbits(st->y); tr->un = fbits(st->u); tr->spn = fbits(st->sp); tr->dtn = fbits(st->dt); tr->kn = fbits(st->k);
  }
}

static void store_probe(uint32_t *dst, const orc_state *st) {
  dst[0] = fbits(st->x); dst[1] = fbits(st->y); dst[2] = fbits(st->u);
  dst[3] = fbits(st->sp); dst[4] = fbits(st->dt); dst[5] = fbits(st->k);
}

/*
 * Decode ONE track given its own slices of the streams (rowdiff/secleg/padres/timeres have ncl-1 entries).
 * Outputs sec/row/P/T[ncl]; optional trace[ncl-1] (row j-1 describes cluster j); optional init/probe state.
 */
int orc_decode_track(const orc_geometry *g, int8_t qpt, uint32_t sec0, uint32_t row0, uint32_t P0, uint32_t T0,
                     uint32_t ncl, const uint8_t *rowdiff, const uint8_t *secleg, const uint16_t *padres,
                     const uint32_t *timeres, uint8_t *sec, uint8_t *row, uint16_t *P, uint32_t *T,
                     orc_trace_row *trace, uint32_t probe_step, uint32_t *probe6) {
  if (!g || ncl < 1 || row0 >= g->n_rows || sec0 >= g->n_az * g->n_sides) return ORC_ERR_ARG;
  orc_state st;
  orc_init(g, &st, qpt, sec0, row0, P0, T0);
  sec[0] = (uint8_t)sec0; row[0] = (uint8_t)row0; P[0] = (uint16_t)P0; T[0] = T0;
  uint32_t pstep = probe_step < ncl - 1 ? probe_step : ncl - 1;
  if (probe6 && pstep == 0) store_probe(probe6, &st);
  for (uint32_t j = 1; j < ncl; ++j) {
    uint32_t p = padres[j - 1], t = timeres[j - 1];
    orc_step(g, &st, j, rowdiff[j - 1], secleg[j - 1], 0, &p, &t, trace ? &trace[j - 1] : NULL);
    sec[j] = (uint8_t)st.sec; row[j] = (uint8_t)st.row; P[j] = (uint16_t)p; T[j] = t;
    if (probe6 && pstep == j) store_probe(probe6, &st);
  }
  return ORC_OK;
}

/*
 * Full decode (output order C5).
 *   clusters[n_attached+n_unattached], bin_offset[n_bins+1], probe_state nullable [n_tracks][6].
 */
int orc_decode(const orc_geometry *g, const orc_compressed *c, orc_cluster *clusters, uint32_t *bin_offset,
               uint32_t *probe_state, uint32_t probe_step) {
  if (!g || !c || !clusters || !bin_offset) return ORC_ERR_ARG;
  const uint32_t n_bins = g->n_sectors_out * g->n_rows;
  const uint64_t n_att = c->n_attached, n_un = c->n_unattached;
  if (n_att + n_un >= 4294967296ull) return ORC_ERR_ARG;
  /* A1: exclusive prefix sum of trk_ncl (the "indices to access the input SOA") */
  uint64_t *off = (uint64_t *)malloc(sizeof(uint64_t) * ((size_t)c->n_tracks + 1));
  uint8_t *sec = (uint8_t *)malloc(n_att ? n_att : 1), *row = (uint8_t *)malloc(n_att ? n_att : 1);
  uint16_t *P = (uint16_t *)malloc(2 * (n_att ? n_att : 1));
  uint32_t *T = (uint32_t *)malloc(4 * (n_att ? n_att : 1));
  uint32_t *att_cnt = (uint32_t *)calloc(n_bins ? n_bins : 1, 4), *cursor = (uint32_t *)malloc(4 * (n_bins ? n_bins : 1));
  int rc = ORC_OK;
  if (!off || !sec || !row || !P || !T || !att_cnt || !cursor) { rc = ORC_ERR_NOMEM; goto done; }
  off[0] = 0;
  for (uint32_t t = 0; t < c->n_tracks; ++t) {
    if (c->trk_ncl[t] < 1) { rc = ORC_ERR_CORRUPT; goto done; }
    off[t + 1] = off[t] + c->trk_ncl[t];
  }
  if (off[c->n_tracks] != n_att) { rc = ORC_ERR_CORRUPT; goto done; }
  { uint64_t su = 0; for (uint32_t b = 0; b < n_bins; ++b) su += c->u_bin_count[b]; if (su != n_un) { rc = ORC_ERR_CORRUPT; goto done; } }
  /* A5 (+A3): every track, serially, in input order -> g-ordered stream */
  for (uint32_t t = 0; t < c->n_tracks; ++t) {
    uint64_t g0 = off[t], r0 = off[t] - t; /* roff[t] = off[t] - t */
    if (c->trk_row0[t] >= g->n_rows || c->trk_sec0[t] >= g->n_az * g->n_sides) { rc = ORC_ERR_CORRUPT; goto done; }
    rc = orc_decode_track(g, c->trk_qpt[t], c->trk_sec0[t], c->trk_row0[t], c->trk_pad0[t], c->trk_time0[t],
                          c->trk_ncl[t], c->a_rowdiff + r0, c->a_secleg + r0, c->a_padres + r0, c->a_timeres + r0,
                          sec + g0, row + g0, P + g0, T + g0, NULL, probe_step,
                          probe_state ? probe_state + 6 * (size_t)t : NULL);
    if (rc) goto done;
  }
  /* A3 count, A4 bin offsets */
  for (uint64_t i = 0; i < n_att; ++i) {
    if (sec[i] >= g->n_sectors_out) { rc = ORC_ERR_CORRUPT; goto done; }
    att_cnt[(uint32_t)sec[i] * g->n_rows + row[i]]++;
  }
  bin_offset[0] = 0;
  for (uint32_t b = 0; b < n_bins; ++b) bin_offset[b + 1] = bin_offset[b] + att_cnt[b] + c->u_bin_count[b];
  /* A6: copy-through + stable placement in ascending g (C5) */
  for (uint32_t b = 0; b < n_bins; ++b) cursor[b] = bin_offset[b];
  for (uint64_t i = 0; i < n_att; ++i) {
    orc_cluster *o = &clusters[cursor[(uint32_t)sec[i] * g->n_rows + row[i]]++];
    o->time = T[i]; o->pad = P[i]; o->qtot = c->a_qtot[i]; o->qmax = c->a_qmax[i];
    o->sigpad = c->a_sigpad[i]; o->sigtime = c->a_sigtime[i]; o->flags = c->a_flags[i];
    o->row = row[i]; o->sector = sec[i]; o->zero = 0;
  }
  /* A7 / C4: unattached, running sums reset at every (sector,row) bin */
  {
    uint64_t i0 = 0;
    for (uint32_t b = 0; b < n_bins; ++b) {
      uint32_t pad = 0, time = 0, cnt = c->u_bin_count[b];
      for (uint32_t i = 0; i < cnt; ++i) {
        pad = (pad + c->u_paddiff[i0 + i]) & 0xFFFFu;
        time = time + c->u_timediff[i0 + i];
        orc_cluster *o = &clusters[cursor[b] + i];
        o->time = time; o->pad = (uint16_t)pad; o->qtot = c->u_qtot[i0 + i]; o->qmax = c->u_qmax[i0 + i];
        o->sigpad = c->u_sigpad[i0 + i]; o->sigtime = c->u_sigtime[i0 + i]; o->flags = c->u_flags[i0 + i];
        o->row = (uint8_t)(b % g->n_rows); o->sector = (uint8_t)(b / g->n_rows); o->zero = 0;
      }
      i0 += cnt;
    }
  }
done:
  free(off); free(sec); free(row); free(P); free(T); free(att_cnt); free(cursor);
  return rc;
}

/* ---- encoder (C6) -------------------------------------------------------------------------- */

static int cmp_unattached(const void *a, const void *b) {
  const orc_cluster *x = (const orc_cluster *)a, *y = (const orc_cluster *)b;
#define ORC_CMP(f) if (x->f != y->f) return x->f < y->f ? -1 : 1;
  ORC_CMP(time) ORC_CMP(pad) ORC_CMP(qtot) ORC_CMP(qmax) ORC_CMP(sigpad) ORC_CMP(sigtime) ORC_CMP(flags)
#undef ORC_CMP
  return 0;
}

/*
 * Encode.  Inputs:
 *   att[n_attached]   attached clusters in g order (track after track, in track order), fields sector,row,pad,time +
 *                     copy-through; leg[n_attached] leg index of each cluster within its track (0,1,2..);
 *   trk_ncl[n_tracks], trk_qptf[n_tracks] (q/pT in c/GeV as defined in C6);
 *   un[n_unattached]  unattached clusters in any order (sector,row give the bin).
 * Outputs: every array of the compressed SoA (caller-allocated, sizes as in C2).
 */
int orc_encode(const orc_geometry *g, uint32_t n_tracks, const uint16_t *trk_ncl, const float *trk_qptf,
               uint64_t n_attached, const orc_cluster *att, const uint8_t *leg,
               uint64_t n_unattached, const orc_cluster *un,
               int8_t *o_qpt, uint8_t *o_row0, uint8_t *o_sec0, uint16_t *o_pad0, uint32_t *o_time0,
               uint16_t *o_aqtot, uint16_t *o_aqmax, uint8_t *o_aflags, uint8_t *o_asigpad, uint8_t *o_asigtime,
               uint8_t *o_rowdiff, uint8_t *o_secleg, uint16_t *o_padres, uint32_t *o_timeres,
               uint16_t *o_uqtot, uint16_t *o_uqmax, uint8_t *o_uflags, uint8_t *o_usigpad, uint8_t *o_usigtime,
               uint16_t *o_paddiff, uint32_t *o_timediff, uint32_t *o_bin_count) {
  if (!g) return ORC_ERR_ARG;
  const uint32_t n_rows = g->n_rows, n_az = g->n_az, n_bins = g->n_sectors_out * n_rows;
  uint64_t gi = 0;
  for (uint32_t t = 0; t < n_tracks; ++t) {
    uint32_t ncl = trk_ncl[t];
    if (ncl < 1 || gi + ncl > n_attached) return ORC_ERR_ARG;
    float q = clampf(floorf(fadd(fmul(trk_qptf[t], 16.0f), 0.5f)), -127.0f, 127.0f);
    int8_t qpt = (int8_t)(int32_t)q;
    const orc_cluster *c0 = &att[gi];
    if (c0->row >= n_rows || c0->sector >= n_az * g->n_sides) return ORC_ERR_ARG;
    o_qpt[t] = qpt; o_row0[t] = c0->row; o_sec0[t] = c0->sector; o_pad0[t] = c0->pad; o_time0[t] = c0->time;
    orc_state st;
    orc_init(g, &st, qpt, c0->sector, c0->row, c0->pad, c0->time);
    int dir = +1;
    for (uint32_t j = 0; j < ncl; ++j) {
      const orc_cluster *c = &att[gi + j];
      o_aqtot[gi + j] = c->qtot; o_aqmax[gi + j] = c->qmax; o_aflags[gi + j] = c->flags;
      o_asigpad[gi + j] = c->sigpad; o_asigtime[gi + j] = c->sigtime;
      if (j == 0) continue;
      const orc_cluster *p = &att[gi + j - 1];
      if (c->row >= n_rows || c->sector / n_az != p->sector / n_az) return ORC_ERR_ARG; /* tracks never change side */
      uint8_t legflag = (leg[gi + j] != leg[gi + j - 1]) ? 0x80 : 0x00;
      if (legflag) dir = -dir;
      int32_t dr = ((int32_t)c->row - (int32_t)p->row) * dir;
      uint32_t rd = (uint32_t)(((dr % (int32_t)n_rows) + (int32_t)n_rows) % (int32_t)n_rows);
      uint32_t d = ((c->sector % n_az) + n_az - (p->sector % n_az)) % n_az;
      uint64_t i = gi + j - t - 1; /* roff[t] + j - 1 */
      o_rowdiff[i] = (uint8_t)rd; o_secleg[i] = (uint8_t)(legflag | d);
      uint32_t P = c->pad, T = c->time;
      orc_step(g, &st, j, (uint8_t)rd, (uint8_t)(legflag | d), 1, &P, &T, NULL);
      if (st.row != c->row || st.sec != c->sector) return ORC_ERR_CORRUPT;
      o_padres[i] = (uint16_t)P; o_timeres[i] = T;
    }
    gi += ncl;
  }
  if (gi != n_attached) return ORC_ERR_ARG;
  /* unattached: per bin, sort by (time,pad,qtot,qmax,sigpad,sigtime,flags), store differences (L68) */
  memset(o_bin_count, 0, 4 * (size_t)n_bins);
  for (uint64_t i = 0; i < n_unattached; ++i) {
    if (un[i].sector >= g->n_sectors_out || un[i].row >= n_rows) return ORC_ERR_ARG;
    o_bin_count[(uint32_t)un[i].sector * n_rows + un[i].row]++;
  }
  uint64_t *start = (uint64_t *)malloc(8 * ((size_t)n_bins + 1));
  orc_cluster *tmp = (orc_cluster *)malloc(sizeof(orc_cluster) * (n_unattached ? n_unattached : 1));
  if (!start || !tmp) { free(start); free(tmp); return ORC_ERR_NOMEM; }
  start[0] = 0;
  for (uint32_t b = 0; b < n_bins; ++b) start[b + 1] = start[b] + o_bin_count[b];
  {
    uint64_t *cur = (uint64_t *)malloc(8 * ((size_t)n_bins + 1));
    if (!cur) { free(start); free(tmp); return ORC_ERR_NOMEM; }
    memcpy(cur, start, 8 * ((size_t)n_bins + 1));
    for (uint64_t i = 0; i < n_unattached; ++i) tmp[cur[(uint32_t)un[i].sector * n_rows + un[i].row]++] = un[i];
    free(cur);
  }
  for (uint32_t b = 0; b < n_bins; ++b) {
    uint64_t s0 = start[b], n = start[b + 1] - s0;
    qsort(tmp + s0, n, sizeof(orc_cluster), cmp_unattached);
    uint32_t pp = 0, pt = 0;
    for (uint64_t i = 0; i < n; ++i) {
      const orc_cluster *c = &tmp[s0 + i];
      o_paddiff[s0 + i] = (uint16_t)((c->pad - pp) & 0xFFFFu);
      o_timediff[s0 + i] = c->time - pt;
      o_uqtot[s0 + i] = c->qtot; o_uqmax[s0 + i] = c->qmax; o_uflags[s0 + i] = c->flags;
      o_usigpad[s0 + i] = c->sigpad; o_usigtime[s0 + i] = c->sigtime;
      pp = c->pad; pt = c->time;
    }
  }
  free(start); free(tmp);
  return ORC_OK;
}
