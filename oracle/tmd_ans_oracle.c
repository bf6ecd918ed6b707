/*
 * tmd_ans_oracle.c -- plain, slow, single-threaded CPU oracle of the entropy stage in front of the track-model decoder.
 *
 * TEST INFRASTRUCTURE ONLY (same rules as tmd_oracle.c): nothing in the product path may include, link or call this file;
 * it shares no code with the CUDA library or with the library's host-side encoder.
 *
 * What it follows.  PAPER.md L20 (§1): the compressed time frames are written with "lossless ANS" entropy coding; L49
 * (Table 2): "TPC Entropy Decoding" is the step just before track-model decoding (4.65 % of the asynchronous CPU time);
 * L68: the track-model decoder's input is what "the entropy decoding" produces.  The paper gives no stream format, no
 * alphabet, no table precision and no interleaving, and the real CTF dictionaries are not available: the format is this
 * build's own ("TMDZ"), the coder is range-ANS (rANS) as published by J. Duda (arXiv:1311.2540), restated
 * here step by step:
 *     encode symbol s (frequency f, cumulative c, M = 2^12):   x' = floor(x / f) * M + c + (x mod f)
 *     decode:   slot = x mod M;  s = the symbol with c <= slot < c + f;   x' = f * floor(x / M) + slot - c
 * with a 32-bit state kept in [2^16, 2^32) by moving 16-bit words (encoder: emit the low word while x >= 2^20 * f; decoder:
 * read one word while x < 2^16).  A plane of bytes is cut into blocks of 8192 symbols; inside a block 32 coders work
 * interleaved (symbol k belongs to coder k mod 32) so that 32 symbols can be decoded per step.  The words of a block are
 * stored in the order the decoder reads them: step by step, and inside a step by ascending coder index.
 *
 * Pins (tests/test_ans_oracle.py, `-m "not gpu"`): hand-derived streams (one-symbol alphabet: no word is ever emitted and
 * the states stay 2^16; a three-symbol stream whose states are derived in the test's comments), the Shannon bound
 * (compressed size within [n H, n H + overhead] of the quantised distribution), an independent big-integer model of the
 * coder in the test (Python integers, one coder, no renormalisation) compared state by state, decode(encode(x)) == x on
 * skewed / uniform / degenerate planes.  No function here is "parity unpinned".
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ANS_OK 0
#define ANS_ERR_ARG (-1)
#define ANS_ERR_SPACE (-3)
#define ANS_ERR_CORRUPT (-5)

#define ANS_PROB_BITS 12
#define ANS_M (1u << ANS_PROB_BITS)
#define ANS_L (1u << 16)
#define ANS_LANES 32
#define ANS_BLOCK 8192

/* Quantise symbol counts to frequencies that sum to M, every present symbol >= 1 (any such table decodes; this is only
 * the oracle encoder's choice: floor-scale, then hand the remainder to / take the excess from the most frequent symbols). */
int orc_ans_build_table(const uint8_t *sym, uint64_t n, uint16_t freq[256]) {
  uint64_t cnt[256];
  memset(cnt, 0, sizeof(cnt));
  memset(freq, 0, 512);
  if (n == 0) return ANS_OK;
  for (uint64_t i = 0; i < n; ++i) cnt[sym[i]]++;
  uint32_t f[256], total = 0;
  for (int s = 0; s < 256; ++s) {
    f[s] = 0;
    if (cnt[s]) {
      uint64_t v = cnt[s] * ANS_M / n;
      f[s] = v ? (uint32_t)v : 1u;
      total += f[s];
    }
  }
  while (total != ANS_M) { /* adjust the currently largest frequency by one, until the sum is M */
    int best = -1;
    for (int s = 0; s < 256; ++s)
      if (f[s] && (best < 0 || f[s] > f[best])) best = s;
    if (total < ANS_M) { f[best]++; total++; }
    else {
      if (f[best] <= 1) return ANS_ERR_ARG; /* cannot happen: at most 256 symbols of frequency 1 */
      f[best]--; total--;
    }
  }
  for (int s = 0; s < 256; ++s) freq[s] = (uint16_t)f[s];
  return ANS_OK;
}

/* Encode one block of n <= ANS_BLOCK symbols.  out: 32 u32 final states (= the decoder's initial states) followed by the
 * 16-bit words in decoder order.  Returns the number of bytes written (a multiple of 4) or a negative error. */
int64_t orc_ans_encode_block(const uint8_t *sym, uint32_t n, const uint16_t freq[256], uint8_t *out, uint64_t cap) {
  if (n > ANS_BLOCK) return ANS_ERR_ARG;
  uint32_t cum[257];
  cum[0] = 0;
  for (int s = 0; s < 256; ++s) cum[s + 1] = cum[s] + freq[s];
  if (n && cum[256] != ANS_M) return ANS_ERR_ARG;
  uint32_t x[ANS_LANES];
  for (int l = 0; l < ANS_LANES; ++l) x[l] = ANS_L;
  uint16_t *words = (uint16_t *)malloc(2 * ((size_t)n + 1));
  if (!words) return ANS_ERR_SPACE;
  uint64_t nw = 0;
  /* the encoder runs backwards: last step first, and inside a step the highest coder first */
  for (int64_t k = (int64_t)n - 1; k >= 0; --k) {
    const uint32_t l = (uint32_t)(k % ANS_LANES), s = sym[k], f = freq[s], c = cum[s];
    if (f == 0) { free(words); return ANS_ERR_ARG; }
    const uint64_t x_max = ((uint64_t)(ANS_L >> ANS_PROB_BITS) << 16) * f; /* 2^20 f */
    if ((uint64_t)x[l] >= x_max) { words[nw++] = (uint16_t)(x[l] & 0xFFFFu); x[l] >>= 16; }
    x[l] = (x[l] / f) * ANS_M + c + (x[l] % f);
  }
  const uint64_t bytes = 4 * ANS_LANES + ((2 * nw + 3) & ~(uint64_t)3);
  if (bytes > cap) { free(words); return ANS_ERR_SPACE; }
  memset(out, 0, bytes);
  memcpy(out, x, 4 * ANS_LANES);
  uint16_t *w = (uint16_t *)(out + 4 * ANS_LANES);
  for (uint64_t i = 0; i < nw; ++i) w[i] = words[nw - 1 - i]; /* emitted last = read first */
  free(words);
  return (int64_t)bytes;
}

/* Decode one block of n symbols from `in` (block_bytes long).  Optional trace[n]: the state of the symbol's coder right
 * after the symbol has been decoded and the state renormalised. */
int orc_ans_decode_block(const uint8_t *in, uint64_t block_bytes, uint32_t n, const uint16_t freq[256], uint8_t *sym,
                         uint32_t *trace) {
  if (n > ANS_BLOCK || block_bytes < 4 * ANS_LANES) return ANS_ERR_ARG;
  uint32_t cum[257];
  uint8_t lut[ANS_M];
  cum[0] = 0;
  for (int s = 0; s < 256; ++s) cum[s + 1] = cum[s] + freq[s];
  if (n && cum[256] != ANS_M) return ANS_ERR_CORRUPT;
  for (int s = 0; s < 256; ++s)
    for (uint32_t v = cum[s]; v < cum[s + 1]; ++v) lut[v] = (uint8_t)s;
  uint32_t x[ANS_LANES];
  memcpy(x, in, 4 * ANS_LANES);
  const uint16_t *w = (const uint16_t *)(in + 4 * ANS_LANES);
  const uint64_t max_words = (block_bytes - 4 * ANS_LANES) / 2;
  uint64_t iw = 0;
  for (uint32_t k = 0; k < n; ++k) {
    const uint32_t l = k % ANS_LANES;
    const uint32_t slot = x[l] & (ANS_M - 1), s = lut[slot];
    x[l] = freq[s] * (x[l] >> ANS_PROB_BITS) + slot - cum[s];
    if (x[l] < ANS_L) {
      if (iw >= max_words) return ANS_ERR_CORRUPT;
      x[l] = (x[l] << 16) | w[iw++];
    }
    sym[k] = (uint8_t)s;
    if (trace) trace[k] = x[l];
  }
  return ANS_OK;
}
