// Entropy coding of the octree occupancy bytes: static order-0 range-ANS (rANS), in place of the closed nvCOMP ANS the
// paper calls ("runs a GPU-based entropy encoder, ANS"; L283; L801 "adds only ~0.3 ms but roughly halves
// the compressed size").  Rules = reading [R17] of DESIGN.md: one 12-bit
// frequency table per frame, independent blocks of 1024 bytes, 32-bit state with lower bound 2^16 and 16-bit
// renormalisation words, a block = final state + words in decoder order.
//
// Five small launches: histogram -> model (one warp quantises the 256 counts to sum 4096) -> one thread per block
// encodes backwards from a padded shared-memory copy of its 1024 bytes into a strided scratch -> scan of the word counts
// -> compaction into the caller's payload.  Decoding is one launch (+ the offset scan): a 4096-entry packed slot table and
// the CTA's payload span in shared memory, one thread per block (see rans_decode_kernel).
#include <mutex>

#include "common.cuh"

namespace gsnfs {

namespace {

constexpr uint32_t kRansBlock = GSNFS_RANS_BLOCK;
constexpr uint32_t kRansM = 4096u;
constexpr uint32_t kRansL = 65536u;
constexpr int kRansCta = 32;                           // blocks (= threads) per CTA
constexpr uint32_t kRansPitch = kRansBlock + 4u;       // bytes per staged block: + 4 keeps the 32 threads on 32 banks
constexpr uint32_t kRansScratchWords = kRansBlock;     // a block never needs more than 12 bits per byte = 768 words

__global__ void __launch_bounds__(256) rans_hist_kernel(const uint8_t* __restrict__ data, uint64_t n_host,
                                                        const uint32_t* __restrict__ n_dev, uint32_t* __restrict__ hist) {
  __shared__ uint32_t s_h[256];
  const uint64_t n = n_dev ? min((uint64_t)*n_dev, n_host) : n_host;
  s_h[threadIdx.x] = 0;
  __syncthreads();
  const uint64_t stride = (uint64_t)gridDim.x * 256u * 4u;
  for (uint64_t i = ((uint64_t)blockIdx.x * 256u + threadIdx.x) * 4u; i < n; i += stride) {
    if (i + 4 <= n) {
      const uint32_t w = *reinterpret_cast<const uint32_t*>(data + i);
      atomicAdd(&s_h[w & 0xffu], 1u); atomicAdd(&s_h[(w >> 8) & 0xffu], 1u);
      atomicAdd(&s_h[(w >> 16) & 0xffu], 1u); atomicAdd(&s_h[w >> 24], 1u);
    } else {
      for (uint64_t k = i; k < n; ++k) atomicAdd(&s_h[data[k]], 1u);
    }
  }
  __syncthreads();
  if (s_h[threadIdx.x]) atomicAdd(&hist[threadIdx.x], s_h[threadIdx.x]);
}

// one warp: lane l owns symbols 8l .. 8l+7
__global__ void __launch_bounds__(32) rans_model_kernel(const uint32_t* __restrict__ hist, uint64_t n_host,
                                                        const uint32_t* __restrict__ n_dev, uint16_t* __restrict__ freq) {
  const int lane = threadIdx.x;
  const uint64_t n = n_dev ? min((uint64_t)*n_dev, n_host) : n_host;
  uint32_t h[8], f[8];
  int sum = 0;
#pragma unroll
  for (int j = 0; j < 8; ++j) {
    h[j] = hist[8 * lane + j];
    uint32_t v = 0;
    if (h[j]) { v = (uint32_t)((uint64_t)h[j] * kRansM / n); if (v == 0) v = 1; }
    f[j] = v;
    sum += (int)v;
  }
  sum = __reduce_add_sync(0xffffffffu, sum);
  int d = (int)kRansM - sum;
  if (n == 0) d = 0;
  if (d > 0) {      // to the most frequent symbol (largest count, lowest index)
    uint32_t best = 0; int bj = 0;
#pragma unroll
    for (int j = 0; j < 8; ++j) if (h[j] > best) { best = h[j]; bj = j; }
    const uint32_t gmax = __reduce_max_sync(0xffffffffu, best);
    const unsigned who = __ballot_sync(0xffffffffu, best == gmax);
    if (lane == __ffs(who) - 1) f[bj] += (uint32_t)d;
  }
  while (d < 0) {   // one at a time from the largest quantised frequency (lowest index among equals)
    uint32_t best = 0; int bj = 0;
#pragma unroll
    for (int j = 0; j < 8; ++j) if (f[j] > best) { best = f[j]; bj = j; }
    const uint32_t gmax = __reduce_max_sync(0xffffffffu, best);
    const unsigned who = __ballot_sync(0xffffffffu, best == gmax);
    if (lane == __ffs(who) - 1) f[bj] -= 1u;
    ++d;
  }
#pragma unroll
  for (int j = 0; j < 8; ++j) freq[8 * lane + j] = (uint16_t)f[j];
}

__global__ void __launch_bounds__(kRansCta) rans_encode_kernel(const uint8_t* __restrict__ data, uint64_t n_host,
                                                               const uint32_t* __restrict__ n_dev,
                                                               const uint16_t* __restrict__ freq,
                                                               uint16_t* __restrict__ scratch /* nblk x kRansScratchWords */,
                                                               uint32_t* __restrict__ states, uint16_t* __restrict__ nwords,
                                                               uint64_t nblk_host) {
  extern __shared__ __align__(16) uint8_t s_data[];                 // kRansCta x kRansPitch
  __shared__ uint2 s_e[256];                                        // symbol -> { floor(2^32 / f), f | cum << 16 }
  const uint64_t n = n_dev ? min((uint64_t)*n_dev, n_host) : n_host;
  const int t = threadIdx.x;
  const uint64_t b0 = (uint64_t)blockIdx.x * kRansCta;
  const uint64_t base = b0 * kRansBlock;
  if (base >= n) { if (b0 + t < nblk_host) nwords[b0 + t] = 0; return; }
  // the CTA's 32 blocks into shared memory: asynchronous 4-byte copies (the pitch of 1028 keeps rows 4-byte aligned only),
  // all in flight while the symbol table is built
  const uint64_t span = min((uint64_t)kRansCta * kRansBlock, n - base);
  {
    const uint32_t sbase = (uint32_t)__cvta_generic_to_shared(s_data);
    for (uint64_t i = (uint64_t)t * 4u; i < span; i += kRansCta * 4u) {      // coalesced, 4 bytes per lane
      const uint32_t blk = (uint32_t)(i / kRansBlock), o = (uint32_t)(i % kRansBlock);
      if (i + 4 <= span) {
        asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(sbase + blk * kRansPitch + o), "l"(data + base + i) : "memory");
      } else {
        uint32_t w = 0;
        for (uint64_t k = i; k < span; ++k) w |= (uint32_t)data[base + k] << (8 * (k - i));
        *reinterpret_cast<uint32_t*>(s_data + blk * kRansPitch + o) = w;
      }
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
  }
  {   // lane t owns symbols 8t .. 8t+7: cumulative frequencies by a warp scan; x / f becomes a multiply by floor(2^32 / f)
    uint32_t f8[8], lsum = 0;
#pragma unroll
    for (int j = 0; j < 8; ++j) { f8[j] = freq[8 * t + j]; lsum += f8[j]; }
    uint32_t inc = lsum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const uint32_t v = __shfl_up_sync(0xffffffffu, inc, o); if (t >= o) inc += v; }
    uint32_t c = inc - lsum;
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      const uint32_t f = f8[j];
      s_e[8 * t + j] = make_uint2(f > 1u ? (uint32_t)((1ull << 32) / f) : 0xffffffffu, f | (c << 16));
      c += f;
    }
  }
  asm volatile("cp.async.wait_group 0;" ::: "memory");
  __syncwarp();
  const uint64_t myb = b0 + t;
  const uint64_t mybase = myb * kRansBlock;
  if (mybase >= n) { if (myb < nblk_host) nwords[myb] = 0; return; }
  const uint32_t cnt = (uint32_t)min((uint64_t)kRansBlock, n - mybase);
  const uint8_t* my = s_data + t * kRansPitch;
  uint16_t* out = scratch + myb * kRansScratchWords + kRansScratchWords;      // filled backwards: decoder order
  uint32_t nw = 0, x = kRansL;
  // one symbol: renormalise if x >= f << 20, then x = (x / f) * 4096 + x % f + cum.  q = x / f: umulhi(x, floor(2^32 / f))
  // is q or q - 1 (the reciprocal is short by < 1 ulp and x < 2^32), one fix-up makes it exact.
  auto put = [&](uint2 e) {
    const uint32_t fs = e.y & 0xffffu;
    if ((x >> 20) >= fs) { *--out = (uint16_t)(x & 0xffffu); x >>= 16; ++nw; }
    uint32_t q = __umulhi(x, e.x);
    uint32_t r = x - q * fs;
    if (r >= fs) { ++q; r -= fs; }
    x = q * kRansM + r + (e.y >> 16);
  };
  uint32_t i = cnt;
  while (i & 3u) { --i; put(s_e[my[i]]); }                          // ragged end of the frame's last block
  while (i) {                                                       // 4 symbols per step: their table entries are loaded
    i -= 4u;                                                        // before the first of the 4 dependent state updates
    const uint32_t w4 = *reinterpret_cast<const uint32_t*>(my + i);
    const uint2 e3 = s_e[w4 >> 24], e2 = s_e[(w4 >> 16) & 0xffu], e1 = s_e[(w4 >> 8) & 0xffu], e0 = s_e[w4 & 0xffu];
    put(e3); put(e2); put(e1); put(e0);
  }
  states[myb] = x;
  nwords[myb] = (uint16_t)nw;
}

// one CTA: offsets of the block streams (4 + 2 nwords bytes each); totals and overflow status
__global__ void __launch_bounds__(1024) rans_scan_kernel(const uint16_t* __restrict__ nwords, uint64_t n_host,
                                                         const uint32_t* __restrict__ n_dev, uint64_t nblk_host,
                                                         uint64_t* __restrict__ off, uint64_t capacity,
                                                         gsnfs_rlgr_info* __restrict__ info) {
  __shared__ uint64_t s_warp[33];
  const uint64_t n = n_dev ? min((uint64_t)*n_dev, n_host) : n_host;
  const uint64_t nblk = min(nblk_host, (n + kRansBlock - 1) / kRansBlock);
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  uint64_t carry = 0;
  for (uint64_t base = 0; base < nblk_host; base += 1024) {
    const uint64_t i = base + tid;
    const uint64_t v = i < nblk ? 4ull + 2ull * nwords[i] : 0ull;
    uint64_t inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint64_t tt = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += tt;
    }
    if (lane == 31) s_warp[warp] = inc;
    __syncthreads();
    if (warp == 0) {
      const uint64_t w = s_warp[lane];
      uint64_t winc = w;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const uint64_t tt = __shfl_up_sync(0xffffffffu, winc, o);
        if (lane >= o) winc += tt;
      }
      s_warp[lane] = winc - w;
      if (lane == 31) s_warp[32] = winc;
    }
    __syncthreads();
    if (i < nblk_host) off[i] = carry + s_warp[warp] + inc - v;
    carry += s_warp[32];
    __syncthreads();
  }
  if (tid == 0) {
    off[nblk_host] = carry;
    info->stream_bytes = carry;
    info->n_blocks = (uint32_t)nblk;
    info->status = carry > capacity ? 2u : 0u;
  }
}

__global__ void __launch_bounds__(128) rans_pack_kernel(const uint16_t* __restrict__ scratch, const uint32_t* __restrict__ states,
                                                        const uint16_t* __restrict__ nwords, const uint64_t* __restrict__ off,
                                                        uint8_t* __restrict__ payload, const gsnfs_rlgr_info* __restrict__ info) {
  const uint64_t b = blockIdx.x;
  if (info->status || b >= info->n_blocks) return;
  const uint32_t nw = nwords[b];
  uint8_t* dst = payload + off[b];
  if (threadIdx.x < 4) dst[threadIdx.x] = (uint8_t)(states[b] >> (8 * threadIdx.x));
  const uint16_t* src = scratch + b * kRansScratchWords + (kRansScratchWords - nw);
  for (uint32_t i = threadIdx.x; i < nw; i += 128) {
    const uint16_t w = src[i];
    dst[4 + 2 * i] = (uint8_t)w;
    dst[5 + 2 * i] = (uint8_t)(w >> 8);
  }
}

// Decoder: one thread per block, one warp per CTA.  A block is a serial chain of 1024 dependent symbol steps, so the
// launch is latency bound (6.6 k threads at config 3) and everything on the chain is kept short: ONE shared-memory load
// per symbol from a 4096-entry slot table that packs {symbol, f - 1, slot - cum} in a word, the CTA's whole payload span
// (its 32 block streams lie back to back) staged in shared memory by asynchronous 16-byte copies before the first symbol, the
// next renormalisation word fetched ahead of its use and selected without a branch, 16 decoded bytes stored at a time.
constexpr uint32_t kRansStageBytes = kRansCta * (4u + 2u * kRansScratchWords);   // the encoder cannot emit more per CTA
constexpr uint32_t kRansDecodeSmem = kRansM * 4u + kRansStageBytes + 32u;

__global__ void __launch_bounds__(kRansCta) rans_decode_kernel(const uint8_t* __restrict__ payload, uint64_t payload_bytes,
                                                               const uint16_t* __restrict__ freq,
                                                               const uint16_t* __restrict__ nwords,
                                                               const uint64_t* __restrict__ off, uint64_t n,
                                                               uint8_t* __restrict__ out, gsnfs_rlgr_info* __restrict__ info) {
  extern __shared__ __align__(16) uint8_t s_dyn[];
  uint32_t* s_tab = reinterpret_cast<uint32_t*>(s_dyn);             // slot -> symbol | (f - 1) << 8 | (slot - cum) << 20
  uint8_t* s_pay = s_dyn + kRansM * 4u;                             // payload span of this CTA's blocks (+ slack)
  __shared__ uint16_t s_cum[257];
  const int t = threadIdx.x;
  const uint64_t b0 = (uint64_t)blockIdx.x * kRansCta;
  const uint64_t base = b0 * kRansBlock;
  if (base >= n) return;
  // model: lane t owns symbols 8t .. 8t+7
  uint32_t f8[8], lsum = 0;
#pragma unroll
  for (int j = 0; j < 8; ++j) { f8[j] = freq[8 * t + j]; lsum += f8[j]; }
  uint32_t inc = lsum;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const uint32_t v = __shfl_up_sync(0xffffffffu, inc, o); if (t >= o) inc += v; }
  const uint32_t total = __shfl_sync(0xffffffffu, inc, 31);
  const bool model_ok = total == kRansM;
  if (model_ok) {
    uint32_t c = inc - lsum;
#pragma unroll
    for (int j = 0; j < 8; ++j) { s_cum[8 * t + j] = (uint16_t)c; c += f8[j]; }
    if (t == 31) s_cum[256] = (uint16_t)kRansM;
  }
  __syncwarp();
  // stage the payload span [o0, o1) of the CTA's blocks from the 16-byte boundary at or below its start: asynchronous
  // 16-byte copies, all in flight while the slot table is built
  const uint64_t nblk = (n + kRansBlock - 1) / kRansBlock;
  const uint64_t o0 = off[b0], o1 = min(off[min(b0 + kRansCta, nblk)], payload_bytes);
  uint32_t sh = 0;
  if (o0 < o1) {
    const uint8_t* g = payload + o0;
    const uint32_t len = (uint32_t)min(o1 - o0, (uint64_t)kRansStageBytes);
    if (((uintptr_t)payload & 15u) == 0) {
      sh = (uint32_t)(o0 & 15u);
      g -= sh;                                                      // 16-byte aligned, still inside the payload
      const uint32_t tot = len + sh;                                // bytes [0, tot) of g lie inside the payload
      const uint32_t full = tot & ~15u;
      const uint32_t sbase = (uint32_t)__cvta_generic_to_shared(s_pay);
      for (uint32_t i = 16u * t; i < full; i += 16u * kRansCta)
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(sbase + i), "l"(g + i) : "memory");
      if (t < (int)(tot - full)) s_pay[full + t] = g[full + t];
    } else {
      for (uint32_t i = t; i < len; i += kRansCta) s_pay[i] = g[i];
    }
  }
  asm volatile("cp.async.commit_group;" ::: "memory");
  if (model_ok) {                                                   // lane t fills slots 128t .. 128t+127
    uint32_t slot = 128u * t;
    int lo = 0, hi = 256;                                           // s_cum[lo] <= slot < s_cum[hi]
    while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (s_cum[mid] <= slot) lo = mid; else hi = mid; }
    uint32_t c0 = s_cum[lo], c1 = s_cum[lo + 1];
    for (int k = 0; k < 128; ++k, ++slot) {
      while (slot >= c1) { ++lo; c0 = c1; c1 = s_cum[lo + 1]; }
      s_tab[slot] = (uint32_t)lo | ((c1 - c0 - 1u) << 8) | ((slot - c0) << 20);
    }
  }
  asm volatile("cp.async.wait_group 0;" ::: "memory");
  __syncwarp();
  const uint64_t myb = b0 + t, mybase = myb * kRansBlock;
  if (mybase >= n) return;
  const uint32_t cnt = (uint32_t)min((uint64_t)kRansBlock, n - mybase);
  uint8_t* dst = out + mybase;
  const uint32_t nw = nwords[myb];
  const uint64_t o = off[myb];
  const uint64_t rel = o - o0 + sh;                                 // this block's stream inside s_pay
  bool bad = !model_ok || o + 4ull + 2ull * nw > payload_bytes || rel + 4ull + 2ull * nw > (uint64_t)kRansStageBytes + sh;
  if (bad) {
    for (uint32_t i = 0; i < cnt; ++i) dst[i] = 0;
    atomicOr(&info->status, 1u);
    return;
  }
  const uint16_t* my = reinterpret_cast<const uint16_t*>(s_pay + rel);      // 2-byte aligned: offsets and sh are even
  uint32_t x = (uint32_t)my[0] | ((uint32_t)my[1] << 16);
  const uint16_t* words = my + 2;
  const uint32_t last = nw ? nw - 1u : 0u;
  uint32_t w = 0, nxt = words[0];                                   // (nw == 0: reads the slack, never used)
  const bool vec = (((uintptr_t)out) & 15u) == 0;
  uint32_t i = 0;
  for (; i + 16u <= cnt; i += 16u) {
    uint32_t acc[4] = {0u, 0u, 0u, 0u};
#pragma unroll
    for (int j = 0; j < 16; ++j) {
      const uint32_t slot = x & (kRansM - 1u);
      const uint32_t e = s_tab[slot];
      acc[j >> 2] |= (e & 0xffu) << (8 * (j & 3));
      x = (((e >> 8) & 0xfffu) + 1u) * (x >> 12) + (e >> 20);
      const bool rn = x < kRansL;                                  // renormalise: no branch (lanes diverge on every symbol)
      x = rn ? (x << 16) | nxt : x;
      w += rn ? 1u : 0u;
      nxt = words[min(w, last)];
    }
    if (vec) {
      *reinterpret_cast<uint4*>(dst + i) = make_uint4(acc[0], acc[1], acc[2], acc[3]);
    } else {
#pragma unroll
      for (int j = 0; j < 16; ++j) dst[i + j] = (uint8_t)(acc[j >> 2] >> (8 * (j & 3)));
    }
  }
  for (; i < cnt; ++i) {                                            // ragged end of the last block
    const uint32_t slot = x & (kRansM - 1u);
    const uint32_t e = s_tab[slot];
    dst[i] = (uint8_t)e;
    x = (((e >> 8) & 0xfffu) + 1u) * (x >> 12) + (e >> 20);
    const bool rn = x < kRansL;
    x = rn ? (x << 16) | nxt : x;
    w += rn ? 1u : 0u;
    nxt = words[min(w, last)];
  }
  if (w != nw || x != kRansL) bad = true;       // (more renormalisations than words: w > nw)
  if (bad) atomicOr(&info->status, 1u);
}

}  // namespace

int run_rans_encode(gsnfs_ctx* ctx, cudaStream_t st, const uint8_t* d_data, uint64_t n, const uint32_t* n_dev, uint16_t* d_freq,
                    uint16_t* d_nwords, uint8_t* d_payload, uint64_t capacity, gsnfs_rlgr_info* d_info) {
  const uint64_t nblk = (n + kRansBlock - 1) / kRansBlock;
  if (nblk + kRansCta + 1 > ctx->rans_blocks_cap) return GSNFS_E_CAPACITY;
  GSNFS_CUDA_OK(ctx, cudaMemsetAsync(ctx->rans_hist, 0, 256 * sizeof(uint32_t), st));
  const int hgrid = (int)min((uint64_t)ctx->num_sms * 4u, n / 1024 + 1);
  GSNFS_KERNEL(ctx, st, "rans_hist");
  rans_hist_kernel<<<hgrid, 256, 0, st>>>(d_data, n, n_dev, ctx->rans_hist);
  GSNFS_LAUNCH_CHECK(ctx, st);
  GSNFS_KERNEL(ctx, st, "rans_model");
  rans_model_kernel<<<1, 32, 0, st>>>(ctx->rans_hist, n, n_dev, d_freq);
  GSNFS_LAUNCH_CHECK(ctx, st);
  const int egrid = (int)((nblk + kRansCta - 1) / kRansCta);
  if (egrid > 0) {
    GSNFS_KERNEL(ctx, st, "rans_encode");
    rans_encode_kernel<<<egrid, kRansCta, kRansCta * kRansPitch, st>>>(d_data, n, n_dev, d_freq, ctx->rans_scratch,
                                                                      ctx->rans_states, d_nwords, nblk);
    GSNFS_LAUNCH_CHECK(ctx, st);
  }
  GSNFS_KERNEL(ctx, st, "rans_scan");
  rans_scan_kernel<<<1, 1024, 0, st>>>(d_nwords, n, n_dev, nblk, ctx->rans_off, capacity, d_info);
  GSNFS_LAUNCH_CHECK(ctx, st);
  if (nblk) {
    GSNFS_KERNEL(ctx, st, "rans_pack");
    rans_pack_kernel<<<(unsigned)nblk, 128, 0, st>>>(ctx->rans_scratch, ctx->rans_states, d_nwords, ctx->rans_off, d_payload, d_info);
    GSNFS_LAUNCH_CHECK(ctx, st);
  }
  return GSNFS_OK;
}

int run_rans_decode(gsnfs_ctx* ctx, cudaStream_t st, const uint8_t* d_payload, uint64_t payload_bytes, const uint16_t* d_freq,
                    const uint16_t* d_nwords, uint64_t n, uint8_t* d_out, gsnfs_rlgr_info* d_info) {
  const uint64_t nblk = (n + kRansBlock - 1) / kRansBlock;
  if (nblk + kRansCta + 1 > ctx->rans_blocks_cap) return GSNFS_E_CAPACITY;
  GSNFS_KERNEL(ctx, st, "rans_scan");
  rans_scan_kernel<<<1, 1024, 0, st>>>(d_nwords, n, nullptr, nblk, ctx->rans_off, ~0ull, d_info);
  GSNFS_LAUNCH_CHECK(ctx, st);
  const int grid = (int)((nblk + kRansCta - 1) / kRansCta);
  if (grid > 0) {
    GSNFS_KERNEL(ctx, st, "rans_decode");
    rans_decode_kernel<<<grid, kRansCta, kRansDecodeSmem, st>>>(d_payload, payload_bytes, d_freq, d_nwords,
                                                                              ctx->rans_off, n, d_out, d_info);
    GSNFS_LAUNCH_CHECK(ctx, st);
  }
  return GSNFS_OK;
}

int rans_setup(gsnfs_ctx* ctx) {
  GSNFS_CUDA_OK(ctx, cudaFuncSetAttribute(rans_decode_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                          (int)kRansDecodeSmem));
  GSNFS_CUDA_OK(ctx, cudaFuncSetAttribute(rans_encode_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                          (int)(kRansCta * kRansPitch)));
  return GSNFS_OK;
}

}  // namespace gsnfs

// ---- gsnfs_rans_decode_static: the decoder without a context and without any allocation ---------------------------
// For callers that must not allocate device memory (see gsnfs.h: the GPU belongs to the application's own pool, the
// memory budget is frozen, or a cudaMalloc's device-wide synchronisation has no place in their frame loop).  The one
// piece of working memory the decoder needs -- the byte offset of every block stream, which run_rans_decode() keeps in
// the context scratch -- lives here in a file-scope device array that ships inside the library image.  The kernels are
// the ones above; only where `off` points differs.

namespace gsnfs {
namespace {

constexpr uint64_t kStaticMaxBlocks = GSNFS_RANS_STATIC_MAX_BYTES / kRansBlock;      // 32768 blocks
static_assert(GSNFS_RANS_STATIC_MAX_BYTES % kRansBlock == 0, "limit is a whole number of blocks");

// 256 KB + 8 on every GPU that loads the library, until the process exits.  In HOST code this name is only a handle
// for cudaGetSymbolAddress(): it is not a device address and must never be handed to a kernel as one.
static __device__ __align__(256) uint64_t g_static_off[kStaticMaxBlocks + 1];

constexpr int kStaticMaxDevices = 64;
std::mutex g_static_mu;
uint64_t* g_static_off_dev[kStaticMaxDevices];     // device address of g_static_off on device i; nullptr = not set up

// Once per device, with that device current: resolve the array's device address (every device has its own copy of
// the array at its own address) and raise the decoder's dynamic shared memory limit as rans_setup() does per context.
int static_off_for_current_device(uint64_t** out) {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kStaticMaxDevices) return GSNFS_E_CUDA;
  std::lock_guard<std::mutex> lock(g_static_mu);
  if (!g_static_off_dev[dev]) {
    uint64_t* p = nullptr;
    if (cudaGetSymbolAddress((void**)&p, g_static_off) != cudaSuccess || !p) return GSNFS_E_CUDA;
    if (cudaFuncSetAttribute(rans_decode_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)kRansDecodeSmem) != cudaSuccess)
      return GSNFS_E_CUDA;
    g_static_off_dev[dev] = p;
  }
  *out = g_static_off_dev[dev];
  return GSNFS_OK;
}

}  // namespace
}  // namespace gsnfs

int gsnfs_rans_decode_static(gsnfs_stream stream, const uint8_t* d_payload, uint64_t payload_bytes,
                             const uint16_t* d_freq, const uint16_t* d_nwords, uint64_t n, uint8_t* d_out,
                             gsnfs_rans_info* d_info) {
  using namespace gsnfs;
  if (!d_freq || !d_info || (n && (!d_payload || !d_nwords || !d_out))) return GSNFS_E_INVALID_ARGUMENT;
  if (n >= (1ull << 32)) return GSNFS_E_INVALID_ARGUMENT;
  if (n > GSNFS_RANS_STATIC_MAX_BYTES) return GSNFS_E_CAPACITY;      // the built-in table has no room: nothing is enqueued
  uint64_t* off = nullptr;
  const int rc = static_off_for_current_device(&off);
  if (rc != GSNFS_OK) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  const uint64_t nblk = (n + kRansBlock - 1) / kRansBlock;           // <= kStaticMaxBlocks; the scan writes off[0 .. nblk]
  // The scan rewrites every offset this call's decoder reads, and all of d_info, so the previous call's leftovers in
  // the table are never seen and nothing needs a memset.
  rans_scan_kernel<<<1, 1024, 0, st>>>(d_nwords, n, nullptr, nblk, off, ~0ull, d_info);
  if (cudaPeekAtLastError() != cudaSuccess) return GSNFS_E_CUDA;
  const int grid = (int)((nblk + kRansCta - 1) / kRansCta);
  if (grid > 0) {
    rans_decode_kernel<<<grid, kRansCta, kRansDecodeSmem, st>>>(d_payload, payload_bytes, d_freq, d_nwords, off,
                                                                              n, d_out, d_info);
    if (cudaPeekAtLastError() != cudaSuccess) return GSNFS_E_CUDA;
  }
  return GSNFS_OK;
}
