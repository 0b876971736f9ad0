// Colour decorrelation in front of RAHT (section 4; Table A.8): RGB -> YUV on every SH function
// (DC and AC), then one Karhunen-Loeve transform per YUV channel over the K SH AC coefficients of that channel ("three
// different KLTs").  Readings [R15] (BT.601 analogue YUV; channel layout scale 3, rotation 4, opacity 1, SH DC 3,
// SH AC 3 x K colour-major) and [R16] (covariance about the mean, eigenvectors by descending eigenvalue, largest
// component positive; y = (x - mu) E).
//
// The paper does this with PyTorch matmuls.  Here: one streaming pass accumulates the 3 x (K + K(K+1)/2) first and second
// moments in fp64 (one thread per moment, rows staged through shared memory, per-CTA partials reduced in a fixed order so
// the fit is deterministic); one warp per YUV channel then diagonalises its K x K covariance with cyclic Jacobi
// rotations in fp64; the transform itself is one streaming pass (a row tile in shared memory, one thread per output
// element, K multiply-adds each).
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

// Stage `cnt` rows (C floats each) of a row-major tensor into shared memory, coalesced.
__device__ __forceinline__ void stage_rows(float* s, const float* g, uint32_t cnt, int C) {
  const uint32_t tot = cnt * (uint32_t)C;
  for (uint32_t i = threadIdx.x; i < tot; i += blockDim.x) s[i] = g[i];
}

// ---- 1. moments of the YUV-converted SH AC coefficients -------------------------------------------------------------
__global__ void __launch_bounds__(448) color_stats_kernel(const float* __restrict__ attr, uint32_t n_host,
                                                          const uint32_t* __restrict__ n_dev, int C,
                                                          double* __restrict__ partial /* gridDim.x x 3 x kMomMax */) {
  extern __shared__ float s_rows[];                      // kColRows x C
  const uint32_t n = n_dev ? min(*n_dev, n_host) : n_host;
  const int K = (C - 11) / 3;
  const int nmom = K + K * (K + 1) / 2;
  // thread -> (YUV channel c, moment m): m < K: sum of component m; else the pair (i, j), i <= j
  const int t = threadIdx.x;
  const int c = t / nmom, m = t - c * nmom;
  int pi = 0, pj = -1;
  if (c < 3 && m >= K) {
    int r = m - K;
    pi = 0;
    while (r >= K - pi) { r -= K - pi; ++pi; }
    pj = pi + r;
  } else if (c < 3) {
    pi = m;
  }
  const int base = 11 + K * c;
  double acc = 0.0;
  for (uint32_t r0 = blockIdx.x * kColRows; r0 < n; r0 += gridDim.x * kColRows) {
    const uint32_t cnt = min((uint32_t)kColRows, n - r0);
    __syncthreads();
    stage_rows(s_rows, attr + (size_t)r0 * C, cnt, C);
    __syncthreads();
    for (uint32_t i = t; i < cnt * (uint32_t)K; i += blockDim.x) {      // AC triples -> YUV
      const uint32_t r = i / K, j = i - r * K;
      mat3(s_rows + (size_t)r * C, 11 + j, 11 + K + j, 11 + 2 * K + j, c_yuv);
    }
    __syncthreads();
    if (c < 3) {
      if (pj < 0) for (uint32_t r = 0; r < cnt; ++r) acc += (double)s_rows[(size_t)r * C + base + pi];
      else for (uint32_t r = 0; r < cnt; ++r) acc += (double)s_rows[(size_t)r * C + base + pi] * (double)s_rows[(size_t)r * C + base + pj];
    }
  }
  if (c < 3) partial[((size_t)blockIdx.x * 3 + c) * kMomMax + m] = acc;
}

// ---- 2. three K x K eigen-decompositions (cyclic Jacobi, fp64), one warp each ----------------------------------------
__global__ void __launch_bounds__(96) klt_eig_kernel(const double* __restrict__ partial, int nparts, uint32_t n_host,
                                                     const uint32_t* __restrict__ n_dev, int C, float* __restrict__ klt) {
  __shared__ double s_S[3][kKMax][kKMax + 1];
  __shared__ double s_V[3][kKMax][kKMax + 1];
  __shared__ double s_mom[3][kMomMax];
  __shared__ double s_cs[3][2];
  __shared__ int s_ord[3][kKMax];
  const uint32_t n = n_dev ? min(*n_dev, n_host) : n_host;
  const KltLayout L = klt_layout(C);
  const int K = L.K, nmom = K + K * (K + 1) / 2;
  const int c = threadIdx.x >> 5, lane = threadIdx.x & 31;
  float* out = klt + (size_t)c * L.stride;
  if (K == 0) return;
  for (int m = lane; m < nmom; m += 32) {                 // fixed-order reduction of the per-CTA partials
    double a = 0.0;
    for (int p = 0; p < nparts; ++p) a += partial[((size_t)p * 3 + c) * kMomMax + m];
    s_mom[c][m] = a;
  }
  __syncwarp();
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
  for (int sweep = 0; sweep < 30; ++sweep) {
    double off = 0.0, dia = 0.0;
    for (int i = lane; i < K * K; i += 32) {
      const double v = s_S[c][i / K][i % K];
      if (i / K == i % K) dia += v * v; else off += v * v;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { off += __shfl_xor_sync(0xffffffffu, off, o); dia += __shfl_xor_sync(0xffffffffu, dia, o); }
    if (off <= 1e-30 * dia || off == 0.0) break;
    for (int p = 0; p < K - 1; ++p) {
      for (int q = p + 1; q < K; ++q) {
        if (lane == 0) {
          const double apq = s_S[c][p][q];
          double cs = 1.0, sn = 0.0;
          if (apq != 0.0) {
            const double theta = (s_S[c][q][q] - s_S[c][p][p]) / (2.0 * apq);
            const double tt = (theta >= 0.0 ? 1.0 : -1.0) / (fabs(theta) + sqrt(theta * theta + 1.0));
            cs = 1.0 / sqrt(tt * tt + 1.0);
            sn = tt * cs;
          }
          s_cs[c][0] = cs; s_cs[c][1] = sn;
        }
        __syncwarp();
        const double cs = s_cs[c][0], sn = s_cs[c][1];
        if (sn != 0.0) {
          if (lane < K) {                      // columns p, q of S and V:  [x_p, x_q] <- [c x_p - s x_q, s x_p + c x_q]
            const double sp = s_S[c][lane][p], sq = s_S[c][lane][q];
            s_S[c][lane][p] = cs * sp - sn * sq;
            s_S[c][lane][q] = sn * sp + cs * sq;
            const double vp = s_V[c][lane][p], vq = s_V[c][lane][q];
            s_V[c][lane][p] = cs * vp - sn * vq;
            s_V[c][lane][q] = sn * vp + cs * vq;
          }
          __syncwarp();
          if (lane < K) {                      // rows p, q of S
            const double sp = s_S[c][p][lane], sq = s_S[c][q][lane];
            s_S[c][p][lane] = cs * sp - sn * sq;
            s_S[c][q][lane] = sn * sp + cs * sq;
          }
          __syncwarp();
          if (lane == 0) { s_S[c][p][q] = 0.0; s_S[c][q][p] = 0.0; }
        }
        __syncwarp();
      }
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
template <bool INV>
__global__ void __launch_bounds__(256) color_apply_kernel(const float* __restrict__ in, uint32_t n_host,
                                                          const uint32_t* __restrict__ n_dev, int C,
                                                          const float* __restrict__ klt /* NULL: YUV only */,
                                                          float* __restrict__ out) {
  extern __shared__ float s_dyn[];
  float* s_rows = s_dyn;                                   // kColRows x C
  float* s_tmp = s_rows + kColRows * C;                    // kColRows x C (transformed)
  float* s_klt = s_tmp + kColRows * C;                     // 3 x stride
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
  if (klt) for (int i = t; i < 3 * L.stride; i += blockDim.x) s_klt[i] = klt[i];
  for (uint32_t r0 = blockIdx.x * kColRows; r0 < n; r0 += gridDim.x * kColRows) {
    const uint32_t cnt = min((uint32_t)kColRows, n - r0);
    __syncthreads();
    stage_rows(s_rows, in + (size_t)r0 * C, cnt, C);
    __syncthreads();
    if (!INV) {
      for (uint32_t i = t; i < cnt * (uint32_t)(K + 1); i += blockDim.x) {       // every SH function -> YUV
        const uint32_t r = i / (K + 1), j = i - r * (K + 1);
        float* row = s_rows + (size_t)r * C;
        if (j == 0) mat3(row, 8, 9, 10, s_m); else mat3(row, 11 + (j - 1), 11 + K + (j - 1), 11 + 2 * K + (j - 1), s_m);
      }
      __syncthreads();
    }
    // one thread per output element; AC element (c, j): sum_i (x_i - mu_i) E[i][j]  (inverse: sum_i y_i E[j][i] + mu_j)
    for (uint32_t i = t; i < cnt * (uint32_t)C; i += blockDim.x) {
      const uint32_t r = i / C, ch = i - r * C;
      const float* row = s_rows + (size_t)r * C;
      float v = row[ch];
      if (klt && ch >= 11) {
        const int c = (int)(ch - 11) / K, j = (int)(ch - 11) - c * K;
        const float* kc = s_klt + c * L.stride;
        const float* x = row + 11 + c * K;
        float acc = 0.f;
        if (!INV) for (int q = 0; q < K; ++q) acc = fmaf(x[q] - kc[q], kc[2 * K + q * K + j], acc);
        else { for (int q = 0; q < K; ++q) acc = fmaf(x[q], kc[2 * K + j * K + q], acc); acc += kc[j]; }
        v = acc;
      }
      s_tmp[i] = v;
    }
    __syncthreads();
    if (INV) {
      for (uint32_t i = t; i < cnt * (uint32_t)(K + 1); i += blockDim.x) {       // every SH function back to RGB
        const uint32_t r = i / (K + 1), j = i - r * (K + 1);
        float* row = s_tmp + (size_t)r * C;
        if (j == 0) mat3(row, 8, 9, 10, s_m); else mat3(row, 11 + (j - 1), 11 + K + (j - 1), 11 + 2 * K + (j - 1), s_m);
      }
      __syncthreads();
    }
    float* g = out + (size_t)r0 * C;
    for (uint32_t i = t; i < cnt * (uint32_t)C; i += blockDim.x) g[i] = s_tmp[i];
  }
}

}  // namespace

int run_klt_fit(gsnfs_ctx* ctx, cudaStream_t st, const float* d_attr, uint32_t n, const gsnfs_counts* d_counts, int channels,
                float* d_klt) {
  const uint32_t* n_dev = d_counts ? &d_counts->n_voxels : nullptr;
  const int K = (channels - 11) / 3;
  if (K == 0) return GSNFS_OK;
  const int nmom = K + K * (K + 1) / 2;
  const int threads = (3 * nmom + 31) & ~31;
  const int grid = (int)min((uint32_t)ctx->color_parts_cap, (n + kColRows - 1) / kColRows);
  if (grid < 1) return GSNFS_OK;
  const size_t smem = sizeof(float) * kColRows * channels;
  GSNFS_KERNEL(ctx, st, "color_stats");
  color_stats_kernel<<<grid, threads, smem, st>>>(d_attr, n, n_dev, channels, ctx->color_partial);
  GSNFS_LAUNCH_CHECK(ctx, st);
  GSNFS_KERNEL(ctx, st, "klt_eig");
  klt_eig_kernel<<<1, 96, 0, st>>>(ctx->color_partial, grid, n, n_dev, channels, d_klt);
  GSNFS_LAUNCH_CHECK(ctx, st);
  return GSNFS_OK;
}

int run_color_apply(gsnfs_ctx* ctx, cudaStream_t st, bool inverse, const float* d_in, uint32_t n, const gsnfs_counts* d_counts,
                    int channels, const float* d_klt, float* d_out) {
  if (n == 0) return GSNFS_OK;
  const uint32_t* n_dev = d_counts ? &d_counts->n_voxels : nullptr;
  const KltLayout L = klt_layout(channels);
  const size_t smem = sizeof(float) * (2 * kColRows * channels + 3 * L.stride);
  const int grid = (int)min((uint32_t)ctx->num_sms * 4u, (n + kColRows - 1) / kColRows);
  GSNFS_KERNEL(ctx, st, inverse ? "color_inverse" : "color_forward");
  if (inverse) color_apply_kernel<true><<<grid, 256, smem, st>>>(d_in, n, n_dev, channels, d_klt, d_out);
  else color_apply_kernel<false><<<grid, 256, smem, st>>>(d_in, n, n_dev, channels, d_klt, d_out);
  GSNFS_LAUNCH_CHECK(ctx, st);
  return GSNFS_OK;
}

int color_setup(gsnfs_ctx* ctx) {
  const int smem = (int)(sizeof(float) * (2 * kColRows * 56 + 3 * (30 + 225)));
  GSNFS_CUDA_OK(ctx, cudaFuncSetAttribute(color_apply_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
  GSNFS_CUDA_OK(ctx, cudaFuncSetAttribute(color_apply_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
  return GSNFS_OK;
}

}  // namespace gsnfs
