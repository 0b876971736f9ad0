// Colour decorrelation in front of RAHT (section 4; Table A.8): RGB -> YUV on every SH function
// (DC and AC), then one Karhunen-Loeve transform per YUV channel over the K SH AC coefficients of that channel ("three
// different KLTs").  Readings [R15] (BT.601 analogue YUV; channel layout scale 3, rotation 4, opacity 1, SH DC 3,
// SH AC 3 x K colour-major) and [R16] (covariance about the mean, eigenvectors by descending eigenvalue, largest
// component positive; y = (x - mu) E).
//
// The paper does this with PyTorch matmuls.  Here: one streaming pass accumulates the 3 x (K + K(K+1)/2) first and second
// moments in fp64 (one thread per moment, rows staged through shared memory with cp.async, two tiles in flight, per-CTA
// partials reduced in a fixed order so the fit is deterministic); one warp per YUV channel then diagonalises its K x K
// covariance with cyclic Jacobi rotations in fp64; the transform itself is one streaming pass (row tiles double buffered
// in shared memory; one thread per (row, YUV channel) keeps the K inputs in registers and reads the basis as broadcast
// 16-byte vectors: K + K*K/4 shared-memory loads for K*K multiply-adds, where one thread per output element needed 3 K*K).
#include "common.cuh"

namespace gsnfs {

namespace {

constexpr int kKMax = 15;
constexpr int kColRows = 64;                 // rows per shared-memory tile
constexpr int kMomMax = kKMax + kKMax * (kKMax + 1) / 2;      // 135 moments per YUV channel

__constant__ float c_yuv[9] = {0.299f, 0.587f, 0.114f, -0.14713f, -0.28886f, 0.436f, 0.615f, -0.51499f, -0.10001f};

struct KltLayout {     // offsets (floats) inside the caller's d_klt block of YUV channel c: c * stride + ...
  int K, stride;       // stride = K + K + K*K: mean[K], lambda[K], basis[K][K] (basis[i][j] = component i of eigenvector j)
};
__host__ __device__ inline KltLayout klt_layout(int channels) {
  KltLayout l;
  l.K = (channels - 11) / 3;
  l.stride = 2 * l.K + l.K * l.K;
  return l;
}

// (R, G, B) -> (Y, U, V) of one SH function, in place in a staged row; inv = the fp64-inverted matrix, passed in
__device__ __forceinline__ void mat3(float* r, int i0, int i1, int i2, const float* m) {
  const float a = r[i0], b = r[i1], c = r[i2];
  r[i0] = fmaf(m[0], a, fmaf(m[1], b, m[2] * c));
  r[i1] = fmaf(m[3], a, fmaf(m[4], b, m[5] * c));
  r[i2] = fmaf(m[6], a, fmaf(m[7], b, m[8] * c));
}

__device__ __forceinline__ void cp_async4(void* smem_dst, const void* gmem_src) {
  const unsigned a = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(a), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src) {
  const unsigned a = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(a), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// Stage `cnt` rows (C floats each, contiguous in global memory) into shared memory with row pitch `pitch` floats,
// asynchronously.  pitch == C and a 16-byte aligned source: 16-byte copies; otherwise element-wise.
__device__ __forceinline__ void stage_rows_async(float* s, int pitch, const float* g, uint32_t cnt, int C) {
  const uint32_t tot = cnt * (uint32_t)C;
  if (pitch == C && ((tot | (uint32_t)C) & 3u) == 0u && (reinterpret_cast<uintptr_t>(g) & 15u) == 0u) {
    for (uint32_t i = threadIdx.x; i < tot / 4; i += blockDim.x) cp_async16(s + 4 * i, g + 4 * i);
  } else if ((C & 7) == 0 && (blockDim.x & 7u) == 0u) {
    // 8 lanes per row (one 32-byte sector each), C / 8 independent copies per thread and row pass, no index division
    const uint32_t c0 = threadIdx.x & 7u, rstep = blockDim.x >> 3;
    for (uint32_t r = threadIdx.x >> 3; r < cnt; r += rstep) {
      float* sr = s + (size_t)r * pitch + c0;
      const float* gr = g + (size_t)r * C + c0;
      for (int q = 0; q < C; q += 8) cp_async4(sr + q, gr + q);
    }
  } else {
    for (uint32_t i = threadIdx.x; i < tot; i += blockDim.x) {
      const uint32_t r = i / (uint32_t)C, c = i - r * (uint32_t)C;
      cp_async4(s + (size_t)r * pitch + c, g + i);
    }
  }
}

// ---- 1. moments of the YUV-converted SH AC coefficients -------------------------------------------------------------
// Second moments as 4 x 4 outer-product blocks: the K <= 15 components of a YUV channel are padded to 16 = four blocks of
// four; a thread owns one of the ten block pairs (bi <= bj) of one channel and one of eight row groups, and keeps the 16
// products (+ the 4 sums, on diagonal blocks) in registers: 8 shared-memory loads feed 32 fp64 FMAs per pair of rows,
// where one thread per moment needed 32 loads for them (that version kept the shared-memory pipe 92 % busy).  The row
// groups' accumulators are combined in a fixed order at the end, so the fit stays deterministic.
constexpr int kStatThreads = 256;            // 240 used: 3 channels x 10 block pairs x 8 row groups
constexpr int kStatW = 49;                   // double2 per row pair (3 x 16 columns + 1: odd pitch, conflict-free row groups)
constexpr int kStatAcc = 20;                 // 16 products + 4 sums

__global__ void __launch_bounds__(kStatThreads) color_stats_kernel(const float* __restrict__ attr, uint32_t n_host,
                                                                   const uint32_t* __restrict__ n_dev, int C,
                                                                   double* __restrict__ partial /* gridDim.x x 3 x kMomMax */) {
  extern __shared__ __align__(16) float s_rows[];        // 2 x kColRows x C floats, then (kColRows / 2) x kStatW double2
  const uint32_t n = n_dev ? min(*n_dev, n_host) : n_host;
  const int K = (C - 11) / 3;
  double2* s_d = reinterpret_cast<double2*>(s_rows + 2 * kColRows * C);       // [row pair][column] = {row 2rp, row 2rp + 1}
  const int t = threadIdx.x;
  const int g = t & 7, task = t >> 3;          // row group, (channel, block pair)
  const int c = task / 10, pidx = task - c * 10;
  // block pairs in the order (0,0) (0,1) (0,2) (0,3) (1,1) (1,2) (1,3) (2,2) (2,3) (3,3)
  const int bi = pidx < 4 ? 0 : pidx < 7 ? 1 : pidx < 9 ? 2 : 3;
  const int bj = pidx < 4 ? pidx : pidx < 7 ? pidx - 3 : pidx < 9 ? pidx - 5 : 3;
  const bool active = task < 30, diag = bi == bj;
  double acc[kStatAcc];
#pragma unroll
  for (int i = 0; i < kStatAcc; ++i) acc[i] = 0.0;
  for (int i = t; i < (kColRows / 2) * kStatW; i += kStatThreads) s_d[i] = make_double2(0.0, 0.0);   // padding columns stay zero
  const uint32_t stride = gridDim.x * kColRows;
  uint32_t r0 = blockIdx.x * kColRows;
  int cur = 0;
  if (r0 < n) stage_rows_async(s_rows, C, attr + (size_t)r0 * C, min((uint32_t)kColRows, n - r0), C);
  cp_async_commit();
  for (; r0 < n; r0 += stride) {
    const uint32_t cnt = min((uint32_t)kColRows, n - r0);
    const float* rows = s_rows + (size_t)cur * kColRows * C;
    const uint32_t rn = r0 + stride;
    if (rn < n) stage_rows_async(s_rows + (size_t)(cur ^ 1) * kColRows * C, C, attr + (size_t)rn * C, min((uint32_t)kColRows, n - rn), C);
    cp_async_commit();
    cp_async_wait<1>();
    __syncthreads();                                      // rows(cur) landed; the previous tile's moments are done with s_d
    // AC triples of two rows -> YUV, widened to fp64 once (rows beyond the tile's count are zeros)
    for (uint32_t i = t; i < (uint32_t)(kColRows / 2) * (uint32_t)K; i += kStatThreads) {
      const uint32_t rp = (K == 15) ? (i / 15u) : i / (uint32_t)K, j = i - rp * (uint32_t)K;
      double2 y = make_double2(0.0, 0.0), u = y, v = y;
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        const uint32_t r = 2 * rp + h;
        if (r < cnt) {
          const float* row = rows + (size_t)r * C + 11 + j;
          const float a = row[0], b = row[K], gg = row[2 * K];
          const double yy = (double)fmaf(c_yuv[0], a, fmaf(c_yuv[1], b, c_yuv[2] * gg));
          const double uu = (double)fmaf(c_yuv[3], a, fmaf(c_yuv[4], b, c_yuv[5] * gg));
          const double vv = (double)fmaf(c_yuv[6], a, fmaf(c_yuv[7], b, c_yuv[8] * gg));
          if (h == 0) { y.x = yy; u.x = uu; v.x = vv; } else { y.y = yy; u.y = uu; v.y = vv; }
        }
      }
      double2* d = s_d + (size_t)rp * kStatW + j;
      d[0] = y; d[16] = u; d[32] = v;
    }
    __syncthreads();
    if (active) {
      const double2* pa = s_d + 16 * c + 4 * bi;
      const double2* pb = s_d + 16 * c + 4 * bj;
#pragma unroll
      for (int q = 0; q < kColRows / 16; ++q) {             // this group's row pairs: g, g + 8, ...
        const int rp = g + 8 * q;
        double2 a[4], b[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) { a[u] = pa[(size_t)rp * kStatW + u]; b[u] = pb[(size_t)rp * kStatW + u]; }
#pragma unroll
        for (int u = 0; u < 4; ++u)
#pragma unroll
          for (int v = 0; v < 4; ++v) acc[4 * u + v] = fma(a[u].y, b[v].y, fma(a[u].x, b[v].x, acc[4 * u + v]));
        if (diag) {
#pragma unroll
          for (int u = 0; u < 4; ++u) acc[16 + u] += a[u].x + a[u].y;
        }
      }
    }
    cur ^= 1;
  }
  cp_async_wait<0>();
  __syncthreads();
  // combine the eight row groups in a fixed order: one thread per moment
  double* s_red = reinterpret_cast<double*>(s_rows);        // [task][group][kStatAcc]
  if (active) {
#pragma unroll
    for (int i = 0; i < kStatAcc; ++i) s_red[((size_t)task * 8 + g) * kStatAcc + i] = acc[i];
  }
  __syncthreads();
  const int nmom = K + K * (K + 1) / 2;
  for (int m3 = t; m3 < 3 * nmom; m3 += kStatThreads) {
    const int cc = m3 / nmom, m = m3 - cc * nmom;
    int pi = m, pj = -1;
    if (m >= K) {                                           // the pair (pi, pj), pi <= pj, in row-major upper-triangle order
      int r = m - K;
      pi = 0;
      while (r >= K - pi) { r -= K - pi; ++pi; }
      pj = pi + r;
    }
    const int ti = pi >> 2, tj = (pj < 0 ? pi : pj) >> 2;
    const int pidx2 = ti == 0 ? tj : ti == 1 ? 3 + tj : ti == 2 ? 5 + tj : 9;      // inverse of the block-pair order above
    const int slot = pj < 0 ? 16 + (pi & 3) : 4 * (pi & 3) + (pj & 3);
    const double* src = s_red + (size_t)(cc * 10 + pidx2) * 8 * kStatAcc + slot;
    double a = 0.0;
#pragma unroll
    for (int gg = 0; gg < 8; ++gg) a += src[gg * kStatAcc];
    partial[((size_t)blockIdx.x * 3 + cc) * kMomMax + m] = a;
  }
}

// ---- 2. three K x K eigen-decompositions (cyclic Jacobi, fp64), one warp each ----------------------------------------
// The partials are reduced by one thread per moment in a fixed order.  A sweep applies its K(K-1)/2 rotations in K - 1
// (K even) or K (K odd) rounds of disjoint pairs (round-robin pairing: the rotations of a round commute, so they are
// computed together -- one lane per pair -- and applied together, lanes = rows, then lanes = columns): 15 dependent
// steps per sweep at K = 15 instead of 105.
constexpr int kEigThreads = 416;             // >= 3 * kMomMax

__global__ void __launch_bounds__(kEigThreads) klt_eig_kernel(const double* __restrict__ partial, int nparts, uint32_t n_host,
                                                              const uint32_t* __restrict__ n_dev, int C, float* __restrict__ klt) {
  __shared__ double s_S[3][kKMax][kKMax + 2];             // row pitch 17 doubles: a column walk hits 16 different banks
  __shared__ double s_V[3][kKMax][kKMax + 2];
  __shared__ double s_mom[3][kMomMax];
  __shared__ double s_rot[3][(kKMax + 1) / 2][2];         // (cos, sin) of the round's rotations
  __shared__ int s_pq[3][(kKMax + 1) / 2][2];
  __shared__ int s_ord[3][kKMax];
  const uint32_t n = n_dev ? min(*n_dev, n_host) : n_host;
  const KltLayout L = klt_layout(C);
  const int K = L.K, nmom = K + K * (K + 1) / 2;
  if (K == 0) return;
  {
    const int t = threadIdx.x;
    if (t < 3 * nmom) {                                    // fixed-order reduction of the per-CTA partials
      const int cc = t / nmom, m = t - cc * nmom;
      const double* src = partial + (size_t)cc * kMomMax + m;
      double a = 0.0;
#pragma unroll 16
      for (int p = 0; p < nparts; ++p) a += __ldg(src + (size_t)p * 3 * kMomMax);
      s_mom[cc][m] = a;
    }
  }
  __syncthreads();
  const int c = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (c >= 3) return;
  float* out = klt + (size_t)c * L.stride;
  const double inv_n = n ? 1.0 / (double)n : 0.0;
  {
    int m = K;
    for (int i = 0; i < K; ++i)
      for (int j = i; j < K; ++j, ++m)
        if (lane == ((i * K + j) & 31)) {
          const double v = s_mom[c][m] * inv_n - (s_mom[c][i] * inv_n) * (s_mom[c][j] * inv_n);
          s_S[c][i][j] = v; s_S[c][j][i] = v;
        }
    for (int i = lane; i < K * K; i += 32) s_V[c][i / K][i % K] = (i / K == i % K) ? 1.0 : 0.0;
  }
  __syncwarp();
  const int Kp = K + (K & 1), ring = Kp - 1, npair = Kp / 2;          // players 0 .. Kp-1 (player K is a bye when K is odd)
  constexpr int kItems = (kKMax * ((kKMax + 1) / 2) + 31) / 32;       // (pair, row) items per lane and round
  int it_k[kItems], it_i[kItems];                                    // pair and row / column of this lane's items (-1: none)
#pragma unroll
  for (int it = 0; it < kItems; ++it) {
    const int idx = lane + 32 * it;
    it_k[it] = idx < K * npair ? idx / K : -1;
    it_i[it] = idx < K * npair ? idx % K : 0;
  }
  for (int sweep = 0; sweep < 30; ++sweep) {
    double off = 0.0, dia = 0.0;
    for (int i = lane; i < K * K; i += 32) {
      const double v = s_S[c][i / K][i % K];
      if (i / K == i % K) dia += v * v; else off += v * v;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { off += __shfl_xor_sync(0xffffffffu, off, o); dia += __shfl_xor_sync(0xffffffffu, dia, o); }
    if (off <= 1e-30 * dia || off == 0.0) break;
    for (int round = 0; round < ring; ++round) {
      if (lane < npair) {                     // its pair of this round and the rotation that zeroes S[p][q]
        const int a = lane == 0 ? Kp - 1 : (round + lane) % ring;
        const int b = lane == 0 ? round : (round - lane + ring) % ring;
        const int p = min(a, b), q = max(a, b);
        double cs = 1.0, sn = 0.0;
        if (q < K) {
          const double apq = s_S[c][p][q];
          if (apq != 0.0) {
            // tan of the rotation angle: the smaller root of t^2 + 2 theta t - 1 = 0.  Reciprocal and reciprocal square
            // root instead of division and square root (this lane's chain is the critical path of the round)
            const double theta = (s_S[c][q][q] - s_S[c][p][p]) * __drcp_rn(2.0 * apq);
            const double at = fabs(theta);
            double tt;
            if (at < 1e100) {
              const double w = theta * theta + 1.0;
              tt = __drcp_rn(at + w * rsqrt(w));
            } else {
              tt = 0.5 * __drcp_rn(at);                   // theta^2 would overflow
            }
            if (theta < 0.0) tt = -tt;
            cs = rsqrt(tt * tt + 1.0);
            sn = tt * cs;
          }
        }
        s_pq[c][lane][0] = p; s_pq[c][lane][1] = q < K ? q : p;     // the bye pair (q == K, odd K) is the identity: its operand loads stay inside the K x K matrix
        s_rot[c][lane][0] = cs; s_rot[c][lane][1] = sn;
      }
      __syncwarp();
      // columns p, q of S and V:  [x_p, x_q] <- [c x_p - s x_q, s x_p + c x_q].  The (pair, row) items of a lane are
      // independent: all operands are loaded before the first store (one warp per matrix: nothing else hides the latency)
      {
        double ck[kItems], sk[kItems], sp[kItems], sq[kItems], vp[kItems], vq[kItems];
        int pk[kItems], qk[kItems];
#pragma unroll
        for (int it = 0; it < kItems; ++it) {
          sk[it] = 0.0;
          if (it_k[it] >= 0) {
            ck[it] = s_rot[c][it_k[it]][0]; sk[it] = s_rot[c][it_k[it]][1];
            pk[it] = s_pq[c][it_k[it]][0]; qk[it] = s_pq[c][it_k[it]][1];
            sp[it] = s_S[c][it_i[it]][pk[it]]; sq[it] = s_S[c][it_i[it]][qk[it]];
            vp[it] = s_V[c][it_i[it]][pk[it]]; vq[it] = s_V[c][it_i[it]][qk[it]];
          }
        }
#pragma unroll
        for (int it = 0; it < kItems; ++it) {
          if (sk[it] != 0.0) {
            s_S[c][it_i[it]][pk[it]] = ck[it] * sp[it] - sk[it] * sq[it];
            s_S[c][it_i[it]][qk[it]] = sk[it] * sp[it] + ck[it] * sq[it];
            s_V[c][it_i[it]][pk[it]] = ck[it] * vp[it] - sk[it] * vq[it];
            s_V[c][it_i[it]][qk[it]] = sk[it] * vp[it] + ck[it] * vq[it];
          }
        }
      }
      __syncwarp();
      {   // rows p, q of S
        double ck[kItems], sk[kItems], sp[kItems], sq[kItems];
        int pk[kItems], qk[kItems];
#pragma unroll
        for (int it = 0; it < kItems; ++it) {
          sk[it] = 0.0;
          if (it_k[it] >= 0) {
            ck[it] = s_rot[c][it_k[it]][0]; sk[it] = s_rot[c][it_k[it]][1];
            pk[it] = s_pq[c][it_k[it]][0]; qk[it] = s_pq[c][it_k[it]][1];
            sp[it] = s_S[c][pk[it]][it_i[it]]; sq[it] = s_S[c][qk[it]][it_i[it]];
          }
        }
#pragma unroll
        for (int it = 0; it < kItems; ++it) {
          if (sk[it] != 0.0) {
            s_S[c][pk[it]][it_i[it]] = ck[it] * sp[it] - sk[it] * sq[it];
            s_S[c][qk[it]][it_i[it]] = sk[it] * sp[it] + ck[it] * sq[it];
          }
        }
      }
      __syncwarp();
      if (lane < npair && s_rot[c][lane][1] != 0.0) {
        const int p = s_pq[c][lane][0], q = s_pq[c][lane][1];
        s_S[c][p][q] = 0.0; s_S[c][q][p] = 0.0;
      }
      __syncwarp();
    }
  }
  if (lane == 0) {                             // eigenvalues in descending order (stable selection)
    bool used[kKMax];
    for (int i = 0; i < K; ++i) used[i] = false;
    for (int r = 0; r < K; ++r) {
      int best = -1;
      for (int i = 0; i < K; ++i)
        if (!used[i] && (best < 0 || s_S[c][i][i] > s_S[c][best][best])) best = i;
      used[best] = true;
      s_ord[c][r] = best;
    }
  }
  __syncwarp();
  for (int j = lane; j < K; j += 32) {
    const int src = s_ord[c][j];
    int imax = 0;
    for (int i = 1; i < K; ++i) if (fabs(s_V[c][i][src]) > fabs(s_V[c][imax][src])) imax = i;
    const double sg = s_V[c][imax][src] < 0.0 ? -1.0 : 1.0;                  // largest component positive [R16]
    out[j] = (float)(s_mom[c][j] * inv_n);                                   // mean
    out[K + j] = (float)s_S[c][src][src];                                    // eigenvalue
    for (int i = 0; i < K; ++i) out[2 * K + i * K + j] = (float)(sg * s_V[c][i][src]);
  }
}

// ---- 3. the transform: RGB -> YUV on every SH function, (x - mu) E on the AC coefficients (or the inverse) -------------
// Shared memory: two row tiles (filled by cp.async, transformed in place, copied out coalesced), odd row pitch, the
// basis as [c][q][16] floats (row q of E_c, or of E_c^T for the inverse, padded to four 16-byte vectors) and the means.
constexpr int kEP = 16;                      // padded basis row

template <bool INV>
__global__ void __launch_bounds__(256) color_apply_kernel(const float* __restrict__ in, uint32_t n_host,
                                                          const uint32_t* __restrict__ n_dev, int C,
                                                          const float* __restrict__ klt /* NULL: YUV only */,
                                                          float* __restrict__ out) {
  extern __shared__ __align__(16) float s_dyn[];
  const int P = C | 1;                                     // odd row pitch: a warp's 32 rows fall into 32 different banks
  float* s_in = s_dyn;                                     // 2 x kColRows x P; a tile is transformed in place
  float* s_E = s_in + 2 * kColRows * P;                    // 3 x kKMax x kEP (16-byte aligned: kColRows % 4 == 0)
  float* s_mu = s_E + 3 * kKMax * kEP;                     // 3 x kEP
  __shared__ float s_m[9];
  const uint32_t n = n_dev ? min(*n_dev, n_host) : n_host;
  const KltLayout L = klt_layout(C);
  const int K = L.K;
  const int t = threadIdx.x;
  if (t < 9) {
    if (!INV) {
      s_m[t] = c_yuv[t];
    } else {                                               // the inverse matrix, from fp64 cofactors
      const double m[9] = {0.299, 0.587, 0.114, -0.14713, -0.28886, 0.436, 0.615, -0.51499, -0.10001};
      const double det = m[0] * (m[4] * m[8] - m[5] * m[7]) - m[1] * (m[3] * m[8] - m[5] * m[6]) + m[2] * (m[3] * m[7] - m[4] * m[6]);
      const int r = t / 3, cc = t % 3;                     // inverse[r][cc] = cofactor[cc][r] / det
      const int r1 = (cc + 1) % 3, r2 = (cc + 2) % 3, c1 = (r + 1) % 3, c2 = (r + 2) % 3;
      s_m[t] = (float)((m[r1 * 3 + c1] * m[r2 * 3 + c2] - m[r1 * 3 + c2] * m[r2 * 3 + c1]) / det);
    }
  }
  for (int i = t; i < 3 * kKMax * kEP + 3 * kEP; i += blockDim.x) s_E[i] = 0.f;      // s_E and s_mu are contiguous
  __syncthreads();
  if (klt) {
    // forward: y_j = sum_q (x_q - mu_q) E[q][j]  -> row q holds E[q][.];  inverse: x_j = sum_q y_q E[j][q] + mu_j -> E^T
    for (int i = t; i < 3 * K * K; i += blockDim.x) {
      const int c = i / (K * K), rem = i - c * K * K, q = rem / K, j = rem - q * K;
      const float* kc = klt + (size_t)c * L.stride + 2 * K;
      s_E[(c * kKMax + q) * kEP + j] = INV ? kc[j * K + q] : kc[q * K + j];
    }
    for (int i = t; i < 3 * K; i += blockDim.x) s_mu[(i / K) * kEP + (i % K)] = klt[(size_t)(i / K) * L.stride + (i % K)];
  }
  const uint32_t stride = gridDim.x * kColRows;
  uint32_t r0 = blockIdx.x * kColRows;
  int cur = 0;
  if (r0 < n) stage_rows_async(s_in, P, in + (size_t)r0 * C, min((uint32_t)kColRows, n - r0), C);
  cp_async_commit();
  for (; r0 < n; r0 += stride) {
    const uint32_t cnt = min((uint32_t)kColRows, n - r0);
    float* rows = s_in + (size_t)cur * kColRows * P;
    const uint32_t rn = r0 + stride;
    if (rn < n) stage_rows_async(s_in + (size_t)(cur ^ 1) * kColRows * P, P, in + (size_t)rn * C, min((uint32_t)kColRows, n - rn), C);
    cp_async_commit();
    cp_async_wait<1>();
    __syncthreads();                                       // rows(cur) landed; the previous tile's copy-out is complete
    if (!INV) {
      for (uint32_t i = t; i < cnt * (uint32_t)(K + 1); i += blockDim.x) {       // every SH function -> YUV
        const uint32_t r = (K == 15) ? (i >> 4) : i / (K + 1), j = i - r * (K + 1);
        float* row = rows + (size_t)r * P;
        if (j == 0) mat3(row, 8, 9, 10, s_m); else mat3(row, 11 + (j - 1), 11 + K + (j - 1), 11 + 2 * K + (j - 1), s_m);
      }
      __syncthreads();
    }
    // one thread per (row, YUV channel); the threads of a warp share the channel, so the basis loads are broadcasts
    if (klt) {
      for (uint32_t i = t; i < 3u * kColRows; i += blockDim.x) {
        const uint32_t c = i / kColRows, r = i - c * kColRows;
        if (r >= cnt) continue;
        const float* x = rows + (size_t)r * P + 11 + c * K;
        float* y = rows + (size_t)r * P + 11 + c * K;         // in place: this thread has read all of x by then
        const float* E = s_E + c * kKMax * kEP;
        const float* mu = s_mu + c * kEP;
        float acc[kEP];
#pragma unroll
        for (int j = 0; j < kEP; ++j) acc[j] = 0.f;
#pragma unroll
        for (int q = 0; q < kKMax; ++q) {
          if (q < K) {
            const float xv = INV ? x[q] : x[q] - mu[q];
            const float4* e4 = reinterpret_cast<const float4*>(E + q * kEP);
#pragma unroll
            for (int v = 0; v < kEP / 4; ++v) {
              const float4 e = e4[v];
              acc[4 * v + 0] = fmaf(xv, e.x, acc[4 * v + 0]); acc[4 * v + 1] = fmaf(xv, e.y, acc[4 * v + 1]);
              acc[4 * v + 2] = fmaf(xv, e.z, acc[4 * v + 2]); acc[4 * v + 3] = fmaf(xv, e.w, acc[4 * v + 3]);
            }
          }
        }
#pragma unroll
        for (int j = 0; j < kKMax; ++j) if (j < K) y[j] = INV ? acc[j] + mu[j] : acc[j];
      }
    }
    __syncthreads();
    if (INV) {
      for (uint32_t i = t; i < cnt * (uint32_t)(K + 1); i += blockDim.x) {       // every SH function back to RGB
        const uint32_t r = (K == 15) ? (i >> 4) : i / (K + 1), j = i - r * (K + 1);
        float* row = rows + (size_t)r * P;
        if (j == 0) mat3(row, 8, 9, 10, s_m); else mat3(row, 11 + (j - 1), 11 + K + (j - 1), 11 + 2 * K + (j - 1), s_m);
      }
      __syncthreads();
    }
    float* g = out + (size_t)r0 * C;
    if ((C & 7) == 0) {                                    // 8 lanes per row: full 32-byte sectors, no index division
      for (uint32_t r = t >> 3; r < cnt; r += blockDim.x >> 3) {
        const float* sr = rows + (size_t)r * P + (t & 7);
        float* gr = g + (size_t)r * C + (t & 7);
        for (int q = 0; q < C; q += 8) gr[q] = sr[q];
      }
    } else {
      for (uint32_t r = t >> 5; r < cnt; r += blockDim.x >> 5)                    // a warp per row: coalesced
        for (int ch = t & 31; ch < C; ch += 32) g[(size_t)r * C + ch] = rows[(size_t)r * P + ch];
    }
    __syncthreads();                                       // the next iteration's prefetch refills this buffer
    cur ^= 1;
  }
  cp_async_wait<0>();
}

}  // namespace

int run_klt_fit(gsnfs_ctx* ctx, cudaStream_t st, const float* d_attr, uint32_t n, const gsnfs_counts* d_counts, int channels,
                float* d_klt) {
  const uint32_t* n_dev = d_counts ? &d_counts->n_voxels : nullptr;
  const int K = (channels - 11) / 3;
  if (K == 0) return GSNFS_OK;
  // row tiles + the fp64 copy; the final combine reuses the buffer as [30 tasks][8 groups][kStatAcc] doubles
  const size_t smem = max(sizeof(float) * 2 * kColRows * channels + sizeof(double2) * (kColRows / 2) * kStatW,
                          sizeof(double) * 30 * 8 * kStatAcc);
  int per_sm = ctx->occ_cache[8];
  if (per_sm == 0 || ctx->occ_cache_smem[8] != smem) {
    GSNFS_CUDA_OK(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, color_stats_kernel, kStatThreads, smem));
    ctx->occ_cache[8] = per_sm;
    ctx->occ_cache_smem[8] = smem;
  }
  const uint32_t want = (n + kColRows - 1) / kColRows;
  const int grid = (int)min(min((uint32_t)ctx->color_parts_cap, (uint32_t)max(per_sm, 1) * (uint32_t)ctx->num_sms), want);
  if (grid < 1) return GSNFS_OK;
  GSNFS_KERNEL(ctx, st, "color_stats");
  color_stats_kernel<<<grid, kStatThreads, smem, st>>>(d_attr, n, n_dev, channels, ctx->color_partial);
  GSNFS_LAUNCH_CHECK(ctx, st);
  GSNFS_KERNEL(ctx, st, "klt_eig");
  klt_eig_kernel<<<1, kEigThreads, 0, st>>>(ctx->color_partial, grid, n, n_dev, channels, d_klt);
  GSNFS_LAUNCH_CHECK(ctx, st);
  return GSNFS_OK;
}

int run_color_apply(gsnfs_ctx* ctx, cudaStream_t st, bool inverse, const float* d_in, uint32_t n, const gsnfs_counts* d_counts,
                    int channels, const float* d_klt, float* d_out) {
  if (n == 0) return GSNFS_OK;
  const uint32_t* n_dev = d_counts ? &d_counts->n_voxels : nullptr;
  const KltLayout L = klt_layout(channels);
  (void)L;
  const size_t smem = sizeof(float) * (2 * kColRows * (channels | 1) + 3 * kKMax * kEP + 3 * kEP);
  const int grid = (int)min((uint32_t)ctx->num_sms * 6u, (n + kColRows - 1) / kColRows);
  GSNFS_KERNEL(ctx, st, inverse ? "color_inverse" : "color_forward");
  if (inverse) color_apply_kernel<true><<<grid, 256, smem, st>>>(d_in, n, n_dev, channels, d_klt, d_out);
  else color_apply_kernel<false><<<grid, 256, smem, st>>>(d_in, n, n_dev, channels, d_klt, d_out);
  GSNFS_LAUNCH_CHECK(ctx, st);
  return GSNFS_OK;
}

int color_setup(gsnfs_ctx* ctx) {
  const int smem = (int)(sizeof(float) * (2 * kColRows * 57 + 3 * kKMax * kEP + 3 * kEP));
  GSNFS_CUDA_OK(ctx, cudaFuncSetAttribute(color_stats_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                          (int)(sizeof(float) * 2 * kColRows * 56 + sizeof(double2) * (kColRows / 2) * kStatW)));
  GSNFS_CUDA_OK(ctx, cudaFuncSetAttribute(color_apply_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
  GSNFS_CUDA_OK(ctx, cudaFuncSetAttribute(color_apply_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
  return GSNFS_OK;
}

}  // namespace gsnfs
