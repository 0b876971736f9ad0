/* ORACLE -- test infrastructure, NOT part of the product.
 *
 * Entropy coding of the octree occupancy bytes ("GS-NFS then runs a GPU-based entropy encoder, ANS";
 * L283 "compresses position using the ANS entropy coder from NVIDIA's nvCOMP library"; L801 "ANS entropy coding of the
 * octree occupancy bytes adds only ~0.3 ms but roughly halves the compressed size").  The paper uses a closed library;
 * what is restated here is the published range-ANS construction (rANS, static order-0 model), reading [R17] of
 * DESIGN.md.  PARITY UNPINNED by the paper; pinned by a hand-computed stream, an independent big-integer restatement in
 * the tests, decode(encode(x)) = x, block independence and the entropy bound.
 *
 *   model: one table per frame.  hist[s] = occurrences of byte s in the whole stream, total = S.  Quantised to sum
 *     M = 4096: f[s] = 0 if hist[s] = 0, else max(1, floor(hist[s] * 4096 / S)); d = 4096 - sum f; d > 0: added to the
 *     most frequent symbol (largest hist, lowest index); d < 0: one at a time taken from the symbol with the largest
 *     f (lowest index among equals), which always has f > 1.  cum[s] = sum_{t < s} f[t].
 *   blocks of RANS_BLOCK = 1024 bytes are independent streams (one GPU thread each).  32-bit state x, lower bound
 *     L = 2^16, 16-bit renormalisation.  Encoding walks the block BACKWARDS from x = L: for symbol s with f = f[s]:
 *     if x >= (f << 20): emit the low 16 bits of x, x >>= 16; then x = (x / f) * 4096 + (x % f) + cum[s].
 *     Decoding walks forwards from the final state: slot = x & 4095, s = symbol with cum[s] <= slot < cum[s] + f[s],
 *     x = f[s] * (x >> 12) + slot - cum[s]; if x < L: x = (x << 16) | next word.  The words are stored in the order the
 *     decoder reads them (the reverse of emission).
 *   block stream = final state (uint32, little endian) followed by its 16-bit words (little endian); the header holds
 *     f[256] (uint16) and the word count of every block (uint16).
 */
#include <stdint.h>
#include <string.h>

#define RANS_BLOCK 1024u
#define RANS_M 4096u
#define RANS_L 65536u

void rans_oracle_model(const uint8_t* data, uint64_t n, uint16_t f[256]) {
  uint64_t hist[256];
  memset(hist, 0, sizeof(hist));
  for (uint64_t i = 0; i < n; ++i) hist[data[i]]++;
  int64_t sum = 0;
  for (int s = 0; s < 256; ++s) {
    uint64_t v = 0;
    if (hist[s]) { v = hist[s] * RANS_M / n; if (v == 0) v = 1; }
    f[s] = (uint16_t)v;
    sum += (int64_t)v;
  }
  if (n == 0) return;
  int64_t d = (int64_t)RANS_M - sum;
  if (d > 0) {
    int best = 0;
    for (int s = 1; s < 256; ++s) if (hist[s] > hist[best]) best = s;
    f[best] = (uint16_t)(f[best] + d);
  }
  while (d < 0) {
    int best = 0;
    for (int s = 1; s < 256; ++s) if (f[s] > f[best]) best = s;
    f[best]--;
    d++;
  }
}

/* one block: returns the number of 16-bit words; words (capacity >= n) in decoder order; *state = final state */
uint32_t rans_oracle_encode_block(const uint8_t* data, uint32_t n, const uint16_t f[256], uint16_t* words, uint32_t* state) {
  uint32_t cum[256], c = 0;
  for (int s = 0; s < 256; ++s) { cum[s] = c; c += f[s]; }
  uint16_t tmp[RANS_BLOCK + 8];
  uint32_t nw = 0;
  uint32_t x = RANS_L;
  for (uint32_t i = n; i-- > 0;) {
    const uint32_t s = data[i], fs = f[s];
    if ((uint64_t)x >= ((uint64_t)fs << 20)) { tmp[nw++] = (uint16_t)(x & 0xffffu); x >>= 16; }
    x = (x / fs) * RANS_M + (x % fs) + cum[s];
  }
  for (uint32_t i = 0; i < nw; ++i) words[i] = tmp[nw - 1 - i];
  *state = x;
  return nw;
}

/* returns 0 if consistent, 1 if the block ran out of words or did not return to the initial state */
int rans_oracle_decode_block(uint32_t state, const uint16_t* words, uint32_t nw, const uint16_t f[256], uint8_t* out, uint32_t n) {
  uint32_t cum[257], c = 0;
  uint8_t sym[RANS_M];
  for (int s = 0; s < 256; ++s) { cum[s] = c; for (uint32_t k = 0; k < f[s]; ++k) sym[c + k] = (uint8_t)s; c += f[s]; }
  cum[256] = c;
  if (c != RANS_M) return 1;
  uint32_t x = state, w = 0;
  int bad = 0;
  for (uint32_t i = 0; i < n; ++i) {
    const uint32_t slot = x & (RANS_M - 1u);
    const uint32_t s = sym[slot];
    out[i] = (uint8_t)s;
    x = f[s] * (x >> 12) + slot - cum[s];
    if (x < RANS_L) {
      if (w >= nw) { bad = 1; x = (x << 16); } else x = (x << 16) | words[w++];
    }
  }
  if (w != nw || x != RANS_L) bad = 1;
  return bad;
}

/* whole stream: f[256], nwords[nblk] (uint16), payload = per block: state (4 bytes LE) + words (2 bytes LE each).
 * Returns the payload bytes.  payload may be NULL (sizes only). */
uint64_t rans_oracle_encode(const uint8_t* data, uint64_t n, uint16_t f[256], uint16_t* nwords, uint8_t* payload) {
  rans_oracle_model(data, n, f);
  const uint64_t nblk = (n + RANS_BLOCK - 1) / RANS_BLOCK;
  uint64_t off = 0;
  for (uint64_t b = 0; b < nblk; ++b) {
    const uint32_t cnt = (uint32_t)((b + 1) * RANS_BLOCK <= n ? RANS_BLOCK : n - b * RANS_BLOCK);
    uint16_t words[RANS_BLOCK + 8];
    uint32_t state;
    const uint32_t nw = rans_oracle_encode_block(data + b * RANS_BLOCK, cnt, f, words, &state);
    nwords[b] = (uint16_t)nw;
    if (payload) {
      payload[off] = (uint8_t)state; payload[off + 1] = (uint8_t)(state >> 8);
      payload[off + 2] = (uint8_t)(state >> 16); payload[off + 3] = (uint8_t)(state >> 24);
      for (uint32_t i = 0; i < nw; ++i) { payload[off + 4 + 2 * i] = (uint8_t)words[i]; payload[off + 5 + 2 * i] = (uint8_t)(words[i] >> 8); }
    }
    off += 4 + 2ull * nw;
  }
  return off;
}

int rans_oracle_decode(const uint8_t* payload, uint64_t payload_bytes, const uint16_t f[256], const uint16_t* nwords,
                       uint8_t* out, uint64_t n) {
  const uint64_t nblk = (n + RANS_BLOCK - 1) / RANS_BLOCK;
  uint64_t off = 0;
  int bad = 0;
  for (uint64_t b = 0; b < nblk; ++b) {
    const uint32_t cnt = (uint32_t)((b + 1) * RANS_BLOCK <= n ? RANS_BLOCK : n - b * RANS_BLOCK);
    const uint32_t nw = nwords[b];
    if (off + 4 + 2ull * nw > payload_bytes) { memset(out + b * RANS_BLOCK, 0, cnt); bad = 1; continue; }
    const uint32_t state = (uint32_t)payload[off] | ((uint32_t)payload[off + 1] << 8) | ((uint32_t)payload[off + 2] << 16) |
                           ((uint32_t)payload[off + 3] << 24);
    uint16_t words[RANS_BLOCK + 8];
    for (uint32_t i = 0; i < nw && i < RANS_BLOCK + 8; ++i)
      words[i] = (uint16_t)(payload[off + 4 + 2 * i] | (payload[off + 5 + 2 * i] << 8));
    bad |= rans_oracle_decode_block(state, words, nw, f, out + b * RANS_BLOCK, cnt);
    off += 4 + 2ull * nw;
  }
  return bad;
}
