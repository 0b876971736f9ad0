/* gsnfs.h -- C ABI of the B200-native (sm_100a) octree + RAHT hot path of GS-NFS's per-frame codec.
 *
 * Paper: arxiv/paper_2606_05650, "GS-NFS: Bandwidth-adaptive Streaming of Dynamic Gaussian Splats and
 * Point Clouds"; citations are PAPER.md:L<line> of the extracted text.  Readings of passages where the
 * paper is silent or garbled are tagged [O*]/[R*] and listed in DESIGN.md.
 *
 * Conventions
 *  - Every `d_*` pointer is CALLER-OWNED DEVICE memory (e.g. a torch tensor), 16-byte aligned.  Every
 *    `h_*` pointer and every pointer documented "(host)" is host memory.  The library never allocates
 *    or frees caller memory; its only state is the context's scratch, sized at gsnfs_create().
 *  - All calls enqueue work on the given stream (a cudaStream_t passed as void*) and return without
 *    synchronising, except the *_host frame calls, which return after their last copy completes.
 *  - Data-dependent sizes are written to a device-resident gsnfs_counts; calls that consume them read
 *    them on the device, so an encode can be chained with no host round trip.
 *  - Return value: GSNFS_OK (0) or a negative gsnfs_status.  Stream corruption found on the device is
 *    reported in gsnfs_counts.status (it cannot be known at enqueue time).
 *  - Limits: 1 <= depth <= 21 (3*depth-bit Morton codes in 64 bits, PAPER.md:L152 [O10]);
 *    n < 2^30; 1 <= channels <= GSNFS_MAX_CHANNELS.
 *  - No C++ types, exceptions or torch types cross this boundary.  There is no CPU fallback.
 */
#ifndef GSNFS_H_
#define GSNFS_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define GSNFS_MAX_DEPTH 21
#define GSNFS_MAX_CHANNELS 208   /* a 256-row tile of fp32 channels + its metadata must fit the 227 KB of shared memory per CTA */

typedef enum gsnfs_status {
  GSNFS_OK = 0,
  GSNFS_E_INVALID_ARGUMENT = -1, /* NULL pointer, depth/channels/n out of range, bbox_max <= bbox_min   */
  GSNFS_E_CAPACITY = -2,         /* n, channels or depth exceed what gsnfs_create() sized; occ too small */
  GSNFS_E_CUDA = -3,             /* CUDA runtime error; text via gsnfs_last_error()                      */
  GSNFS_E_CORRUPT_STREAM = -4,   /* value of gsnfs_counts.status bit 0 (set on the device by decode)     */
  GSNFS_E_UNIMPLEMENTED = -5
} gsnfs_status;

typedef struct gsnfs_ctx gsnfs_ctx; /* opaque; owns only internal device scratch */
typedef void* gsnfs_stream;         /* a cudaStream_t, e.g. torch.cuda.current_stream().cuda_stream */

/* Device-resident result counters written by the encoder / decoder. */
typedef struct gsnfs_counts {
  uint32_t n_voxels;  /* N_v: occupied voxels = |L_J|                                     */
  uint32_t occ_bytes; /* S = sum_{d<J} |L_d|: occupancy bytes emitted                     */
  uint32_t status;    /* 0 = ok; bit 0 = corrupt stream (decode) ; bit 1 = scratch overflow */
  uint32_t reserved;
} gsnfs_counts;

/* Dead-zone quantiser parameters (PAPER.md:L255 names the quantiser; rule is reading [R10]):
 *   q = sign(y) * floor(|y| * (1/qstep_c) + dz_round),   y^ = sign(q) * (|q| + recon_bias*[q != 0]) * qstep_c.
 * Arithmetic of the integer decision (normative, the CPU oracle evaluates the same): y is the fp32 coefficient
 * widened to fp64; 1/qstep_c is the fp64 reciprocal of the fp32 step (one rounding); the product and the sum are
 * each rounded once in fp64 (no fused multiply-add); floor; saturation to int32; sign(+-0) = 0, so an exactly zero
 * coefficient gives q = 0 even at dz_round = 1.
 * NULL => { 1/3, 0 }.  Required: 0 <= dz_round <= 1, 0 <= recon_bias < 1, both finite (else INVALID_ARGUMENT). */
typedef struct gsnfs_quant {
  float dz_round;
  float recon_bias;
} gsnfs_quant;

/* ---- context ---------------------------------------------------------------------------------- */
/* Creates a context on `device` with scratch for frames of up to max_points Gaussians, max_channels
 * attribute channels and octree depth max_depth.  Scratch is one cudaMalloc (about
 * max_points * (80 + 8*max_channels) bytes). */
int gsnfs_create(gsnfs_ctx** out, int device, uint64_t max_points, int max_channels, int max_depth);
void gsnfs_destroy(gsnfs_ctx* ctx);
const char* gsnfs_strerror(int status);
const char* gsnfs_last_error(const gsnfs_ctx* ctx);  /* text of the last GSNFS_E_CUDA / overflow on this context */
/* Errors found on the device after a call has returned (today: a RAHT call whose schedule did not fit the context
 * scratch -- possible only for voxel keys that are not sorted and unique, see DESIGN.md "RAHT phases" -- in which
 * case the transform wrote NO output).  The kernel sets gsnfs_counts.status bit 1 (if the call was given d_counts)
 * and a flag that the next entry point on this context, or this call, reports ONCE as GSNFS_E_CAPACITY.  Does not
 * synchronise: for a definitive answer synchronise the stream first.  GSNFS_OK if nothing is pending. */
int gsnfs_poll_status(gsnfs_ctx* ctx);
const char* gsnfs_version(void);
/* Number of CUDA kernels this context has launched so far (bench.py's gpu_launches). */
uint64_t gsnfs_launch_count(const gsnfs_ctx* ctx);

/* Per-kernel device timing.  gsnfs_profile_start(): from now on every kernel this context launches is
 * bracketed by a CUDA event pair on its stream (up to max_records launches).  gsnfs_profile_stop():
 * synchronises the device, stops recording and writes one text line per kernel name into `out` (host):
 * "<name> <launches> <total_ms>\n".  Used by bench.py for the live roofline figures. */
int gsnfs_profile_start(gsnfs_ctx* ctx, int max_records);
int gsnfs_profile_stop(gsnfs_ctx* ctx, char* out /* host */, uint64_t out_cap);

/* Upper bound on occupancy bytes for n points at `depth`: sum_{d<depth} min(8^d, n), rounded up to 16. */
uint64_t gsnfs_occ_capacity(uint64_t n, int depth);

/* ---- position coder, encoder side (section 2.2, Algorithm A.1) ------------------------- */
/* fp32 positions -> breadth-first per-level occupancy bytes + Morton-sorted voxel permutation.
 *   voxelise  [O1][O2]: v_a = clamp(floor((fp64(p_a) - fp64(lo_a)) * (2^depth / (fp64(hi_a) - fp64(lo_a)))), 0, 2^depth-1)
 *                       with the subtraction and the product each rounded once in fp64 (no FMA).
 *   Morton    (L136):   bit 3b = x_b, 3b+1 = y_b, 3b+2 = z_b.
 *   sort      (L152, A.1 l.4): stable LSD radix sort of (code, original index) [O8].
 *   unique    (L154):   voxel v = v-th run of equal codes; d_voxel_start[v] = its first sorted position.
 *   octree    (L156-168, A.1): L_d = unique(L_{d+1} >> 3); one byte per internal node, bit i <-> child
 *                       (node << 3) + i [O4]; level 0 first, each level contiguous, ascending code [O5].
 * Outputs (all device): d_occ[occ_capacity] (only the first counts.occ_bytes are meaningful; the buffer
 * is cleared by the call), d_level_sizes[depth+1] = (|L_0| .. |L_J|) [O6], d_perm[n],
 * d_voxel_keys[n] (first N_v valid), d_voxel_start[n+1] (first N_v+1 valid; [N_v] == n), d_counts.
 * n == 0 is valid (N_v = 0, no bytes, level sizes 0).  Non-finite positions give an unspecified (but
 * in-range) voxel.  Errors: INVALID_ARGUMENT, CAPACITY (n/depth beyond the context, or occ_capacity <
 * gsnfs_occ_capacity(n, depth)), CUDA. */
int gsnfs_octree_encode(gsnfs_ctx* ctx, gsnfs_stream stream,
                        const float* d_xyz /* n x 3 row-major */, uint64_t n,
                        const float bbox_min[3] /* host */, const float bbox_max[3] /* host */, int depth,
                        uint8_t* d_occ, uint64_t occ_capacity, uint32_t* d_level_sizes,
                        uint32_t* d_perm, uint64_t* d_voxel_keys, uint32_t* d_voxel_start,
                        gsnfs_counts* d_counts);

/* Duplicate-voxel merge: merged[v][c] = mean over the Gaussians of voxel v of
 * attr[g][c] (fp64 accumulation in sorted order, [O9]); weights[v] = count.  Rows v >= N_v untouched.
 * N_v is read on the device from d_counts (written by gsnfs_octree_encode on the same stream). */
int gsnfs_voxel_merge(gsnfs_ctx* ctx, gsnfs_stream stream,
                      const float* d_attr /* n x channels row-major */, int channels, uint64_t n,
                      const uint32_t* d_perm, const uint32_t* d_voxel_start, const gsnfs_counts* d_counts,
                      float* d_merged /* capacity n x channels, Morton order */,
                      uint32_t* d_weights /* capacity n */);

/* ---- position coder, decoder side (section 2.3, Algorithms A.2 and A.3) ---------------- */
/* occupancy bytes -> leaf Morton codes and integer voxel coordinates, in Morton order.
 * level_sizes (host, depth+1 entries) is the stream header [O6]; N_v = level_sizes[depth] and
 * occ_bytes must equal sum_{d<depth} level_sizes[d].  d_voxel_xyz is N_v x 3 (x, y, z) uint32;
 * d_voxel_keys (N_v) may be NULL.  A zero occupancy byte or a level whose popcount sum differs from
 * the header sets d_counts->status bit 0 [O12]; no out-of-bounds access happens either way.
 * occ_bytes must be < 2^29 (GSNFS_E_CAPACITY otherwise). */
int gsnfs_octree_decode(gsnfs_ctx* ctx, gsnfs_stream stream,
                        const uint8_t* d_occ, uint64_t occ_bytes,
                        const uint32_t* level_sizes /* host, depth+1 */, int depth,
                        uint32_t* d_voxel_xyz, uint64_t* d_voxel_keys, gsnfs_counts* d_counts);

/* ---- attribute coder: RAHT (section 3, Eq. (1), Appendix D, Algorithms A.4-A.6) ------- */
/* Forward transform of the N_v x channels attribute rows of the Morton-sorted voxels, bottom-up over
 * the 3*depth binary levels: siblings at level l are adjacent active entries whose codes agree above
 * bit l-1 (A.4 l.10); a = sqrt(w0/(w0+w1)), b = sqrt(w1/(w0+w1)); low = a*y0 + b*y1 stays at the left
 * index, high = -b*y0 + a*y1 goes to the right index (A.6 l.16-17) [R6].  The signal transformed is
 * x_i = sqrt(w_i) * attr_i [R2]; d_weights == NULL means unit leaf weights (the paper's case).
 * Output order ("canonical order", [R8]): row i of the Morton-sorted voxel list, row 0 = DC.
 *   qstep (host, `channels` entries) != NULL: d_qcoeff[i][c] = sign(y) floor(|y| * (1/qstep_c) + dz_round),
 *   saturated to int32, in the arithmetic gsnfs_quant states (fp64, from the fp32 coefficient).  d_coeff (unquantised fp32) and
 *   d_qcoeff may each be NULL, not both; d_qcoeff requires qstep.
 * n_voxels is the row count; if d_counts != NULL the actual N_v is read on the device from it and
 * n_voxels is only an upper bound (rows beyond N_v are untouched); a d_counts whose status is already non-zero
 * (a stream the decoder flagged) makes the call a no-op; a schedule overflow ORs bit 1 into d_counts->status.
 * d_voxel_keys must be sorted and unique, d_weights >= 1 (the caller's responsibility; violations cannot crash
 * or write out of bounds, and end either in unspecified coefficients or in the overflow report above).
 * Schedule reuse: the prelude (sibling pairs, weights, a/b factors: Alg. A.4/A.5) depends on the codes and leaf weights
 * only.  d_voxel_keys == NULL in gsnfs_raht_forward / gsnfs_raht_inverse means "the same voxel list and weights as the
 * previous gsnfs_raht_* / gsnfs_merge_raht_forward call on this context, with the same n_voxels": the prelude is skipped
 * (one rung more of a bitrate ladder costs the transform only).  d_weights must still be passed if it was then.
 * The reusing call must be issued on the SAME stream as the call that built the schedule (nothing else orders the
 * two).  GSNFS_E_INVALID_ARGUMENT if the context holds no schedule of n_voxels rows built on this stream (a failed
 * RAHT call leaves none); other mismatches are the caller's error.  gsnfs_merge_raht_forward never reuses. */
int gsnfs_raht_forward(gsnfs_ctx* ctx, gsnfs_stream stream,
                       const uint64_t* d_voxel_keys, const uint32_t* d_weights, uint64_t n_voxels,
                       gsnfs_counts* d_counts, int depth,
                       const float* d_attr /* N_v x channels */, int channels,
                       const float* qstep /* host */, const gsnfs_quant* quant /* host, may be NULL */,
                       int32_t* d_qcoeff, float* d_coeff);

/* One more quantisation of an unquantised coefficient tensor (d_coeff of gsnfs_raht_forward, N_v x channels,
 * canonical order): d_qcoeff[i][c] = sign(y) floor(|y| * (1/qstep_c) + dz_round), the same rule and arithmetic as the
 * quantiser fused into gsnfs_raht_forward [R10], so a bitrate ladder (one step per
 * attribute and rung) can share one sort/octree/transform and pay only this pass per rung.  qstep: host,
 * `channels` entries, all > 0 and finite; quant may be NULL (dz_round = 1/3).  n_rows is the row count; if
 * d_counts != NULL the actual N_v is read on the device and n_rows is an upper bound (rows beyond N_v are
 * untouched).  Asynchronous on `stream`; d_coeff and d_qcoeff are caller-owned device memory and may not overlap. */
int gsnfs_quantize(gsnfs_ctx* ctx, gsnfs_stream stream,
                   const float* d_coeff /* N_v x channels */, uint64_t n_rows, const gsnfs_counts* d_counts,
                   int channels, const float* qstep /* host */, const gsnfs_quant* quant /* host, may be NULL */,
                   int32_t* d_qcoeff /* N_v x channels */);

/* Fused gsnfs_voxel_merge + gsnfs_raht_forward(weights = counts): the same coefficients, bit for bit, as
 * the two calls in sequence, but phase-1 rows are gathered through d_perm straight into shared memory and
 * the merged N_v x channels tensor is never written (saves a 2 x 4*channels bytes/voxel round trip).
 * d_attr is the UNSORTED n x channels input; d_weights_out (capacity n) receives the run lengths;
 * d_counts (required) supplies N_v on the device; n is the row capacity as in gsnfs_raht_forward. */
int gsnfs_merge_raht_forward(gsnfs_ctx* ctx, gsnfs_stream stream,
                             const uint64_t* d_voxel_keys, const uint32_t* d_perm, const uint32_t* d_voxel_start,
                             uint64_t n, gsnfs_counts* d_counts, int depth,
                             const float* d_attr /* n x channels, input order */, int channels,
                             const float* qstep /* host */, const gsnfs_quant* quant /* host, may be NULL */,
                             uint32_t* d_weights_out, int32_t* d_qcoeff, float* d_coeff);

/* Inverse transform (A.6 l.24-43): de-quantise (if d_qcoeff != NULL, else take d_coeff), run the same
 * schedule top-down with low' = a*y0 - b*y1, high' = b*y0 + a*y1, then divide row i by sqrt(w_i) [R2]. */
int gsnfs_raht_inverse(gsnfs_ctx* ctx, gsnfs_stream stream,
                       const uint64_t* d_voxel_keys, const uint32_t* d_weights, uint64_t n_voxels,
                       gsnfs_counts* d_counts, int depth,
                       const int32_t* d_qcoeff, const float* d_coeff, int channels,
                       const float* qstep /* host */, const gsnfs_quant* quant /* host, may be NULL */,
                       float* d_attr_out /* N_v x channels */);

/* ---- colour decorrelation in front of RAHT (section 4; Table A.8) ---------------
 * "It first transforms RGB to YUV for each SH function ... to all SH coefficients (both DC and AC)"; "a decorrelating
 * transform, Karhunen-Loeve transform, only to the AC coefficients ... three different KLTs, one to each channel in
 * YUV color space"; "We apply KLT before RAHT".
 * Readings: [R15] BT.601 analogue YUV (Y = 0.299 R + 0.587 G + 0.114 B, U = -0.14713 R - 0.28886 G + 0.436 B,
 * V = 0.615 R - 0.51499 G - 0.10001 B; the inverse is the fp64 matrix inverse); channel layout: 8 geometry channels
 * (scale 3, rotation 4, opacity 1), SH DC (R, G, B) at 8..10, SH AC colour-major: AC(c, j) = 11 + K c + j, K = (channels
 * - 11) / 3 in {0, .., 15}.  [R16] KLT of YUV channel c: covariance about the mean of its K AC coefficients over the n
 * rows (fp64 accumulation), eigenvectors by descending eigenvalue, each signed so that its largest-magnitude
 * component is positive; y = (x - mu) E, x = y E^T + mu.
 * d_klt (device, gsnfs_klt_floats(channels) floats) is the frame's side information: per YUV channel mean[K],
 * eigenvalue[K], basis[K][K] (basis[i][j] = component i of eigenvector j).  d_klt == NULL in the transform calls means
 * YUV only.  d_out may equal d_attr (rows are independent).  n_rows / d_counts as in gsnfs_raht_forward.  The fit is
 * deterministic (fixed reduction order).  Errors: INVALID_ARGUMENT (channels not 11 + 3K, K <= 15; NULL), CAPACITY. */
uint64_t gsnfs_klt_floats(int channels);
int gsnfs_klt_fit(gsnfs_ctx* ctx, gsnfs_stream stream, const float* d_attr /* n_rows x channels, RGB */, uint64_t n_rows,
                  const gsnfs_counts* d_counts, int channels, float* d_klt);
int gsnfs_color_forward(gsnfs_ctx* ctx, gsnfs_stream stream, const float* d_attr /* RGB */, uint64_t n_rows,
                        const gsnfs_counts* d_counts, int channels, const float* d_klt, float* d_out /* YUV + KLT */);
int gsnfs_color_inverse(gsnfs_ctx* ctx, gsnfs_stream stream, const float* d_attr /* YUV + KLT */, uint64_t n_rows,
                        const gsnfs_counts* d_counts, int channels, const float* d_klt, float* d_out /* RGB */);

/* ---- entropy coder for the quantised coefficients: block-parallel adaptive RLGR ---------------------
 * PAPER.md:L257 (section 3.4: Run-Length Golomb-Rice [25], run-length coding of zeros, Golomb-Rice coding of non-zero
 * magnitudes with an adaptive parameter, blocks of successive coefficients coded by one GPU thread each), L803
 * (Appendix H: each attribute channel partitioned into fixed-size blocks, encoded independently), Table A.5 (block
 * sizes 256 .. 8192).  The paper gives the coder by citation only; the bit-exact rules are reading [R14]:
 *   u(x) = 2x (x >= 0), -2x - 1 (x < 0);  GR(u, kR): p = u >> kR, p < 32: p ones, a zero, kR low bits of u; else 32
 *   ones and u in 32 bits;  state kP, kRP (k = kP >> 2, kR = kRP >> 2), every block starts at kP = 0, kRP = 8;
 *   k == 0: GR(u(x), kR), then kP += 3 if x == 0 else kP -= 1;  k > 0: 2^k zeros -> bit 0, kP += 2; r < 2^k zeros then
 *   x != 0 -> bit 1, r in k bits, GR(u(x) - 1, kR), kP -= 3; a block ending inside a run -> bit 0 (a 0 bit means
 *   min(2^k, coefficients left) zeros);  after a GR: p == 0: kRP -= 2, p > 1: kRP += min(p, 32) + 1;
 *   0 <= kP <= 64, 0 <= kRP <= 127;  bits MSB first, every block padded to a multiple of 32 bits.
 * Layout: d_qcoeff is n_rows x channels row-major (canonical order [R8]); block (b, c) = rows [b*B, min((b+1)*B, n))
 * of column c; d_block_bits[b * channels + c] = its padded bit length (the stream header); d_stream holds the block
 * streams back to back in that order.  Nothing is transposed: the threads of a CTA are the channels of one row block.
 * All pointers are caller-owned device memory; d_stream 4-byte aligned.  Asynchronous on `stream`. */
#define GSNFS_RLGR_MIN_BLOCK 64
#define GSNFS_RLGR_MAX_BLOCK 65536
typedef struct gsnfs_rlgr_info {  /* device-resident result of the RLGR calls */
  uint64_t stream_bytes;          /* total bytes of the block streams                                          */
  uint32_t n_blocks;              /* entries of d_block_bits                                                   */
  uint32_t status;                /* 0 = ok; bit 0 = corrupt / inconsistent stream (decode);                   */
} gsnfs_rlgr_info;                /*         bit 1 = stream_capacity too small (encode: nothing was written)   */
/* Entries of d_block_bits: ceil(n_rows / block_size) * channels (0 for an invalid block_size). */
uint64_t gsnfs_rlgr_blocks(uint64_t n_rows, int channels, int block_size);
/* A stream capacity that always suffices in practice: the raw size 4 * n_rows * channels plus the per-block padding
 * (an RLGR stream longer than the raw coefficients is reported through status bit 1, never written). */
uint64_t gsnfs_rlgr_capacity(uint64_t n_rows, int channels, int block_size);
/* n_rows is the row count; if d_counts != NULL the actual N_v is read on the device and n_rows is an upper bound
 * (blocks beyond N_v get bit length 0).  Errors: INVALID_ARGUMENT (NULL, block_size outside [64, 65536], misaligned
 * d_stream), CAPACITY (beyond the context). */
int gsnfs_rlgr_encode(gsnfs_ctx* ctx, gsnfs_stream stream,
                      const int32_t* d_qcoeff /* n_rows x channels */, uint64_t n_rows, const gsnfs_counts* d_counts,
                      int channels, int block_size,
                      uint32_t* d_block_bits /* gsnfs_rlgr_blocks() entries */,
                      uint8_t* d_stream, uint64_t stream_capacity, gsnfs_rlgr_info* d_info);
/* Inverse: block streams -> d_qcoeff (n_rows x channels).  A block that runs out of bits, or a header that does not
 * fit stream_bytes, sets status bit 0 (the block's remaining coefficients are zero); never reads out of bounds. */
int gsnfs_rlgr_decode(gsnfs_ctx* ctx, gsnfs_stream stream,
                      const uint8_t* d_stream, uint64_t stream_bytes, const uint32_t* d_block_bits,
                      uint64_t n_rows, int channels, int block_size,
                      int32_t* d_qcoeff /* n_rows x channels */, gsnfs_rlgr_info* d_info);

/* ---- entropy coder for the occupancy bytes: static order-0 rANS -------------------------------------
 * PAPER.md:L170 ("To improve compression efficiency, GS-NFS then runs a GPU-based entropy encoder, ANS"), L283 (nvCOMP),
 * L801 ("adds only ~0.3 ms but roughly halves the compressed size").  The paper calls a closed library; this is the
 * published rANS construction, reading [R17]:
 *   model: hist over the whole stream, quantised to sum 4096: f[s] = max(1, floor(hist[s] * 4096 / n)) for hist[s] > 0;
 *   the remainder goes to the most frequent symbol, an excess is taken one at a time from the largest f;
 *   blocks of GSNFS_RANS_BLOCK bytes are independent: 32-bit state, lower bound 2^16, 16-bit renormalisation, symbols
 *   walked backwards from x = 2^16: if x >= f << 20: emit low 16 bits, x >>= 16; x = (x / f) * 4096 + x % f + cum[s];
 *   block stream = final state (4 bytes LE) + its words (2 bytes LE each) in the order the decoder reads them.
 * Stream header: d_freq[256] (uint16), d_nwords[gsnfs_rans_blocks(n)] (uint16); d_payload holds the blocks back to back.
 * n is the byte count; if d_counts != NULL the actual count is read on the device from d_counts->occ_bytes (chained
 * after gsnfs_octree_encode) and n is an upper bound.  d_info: stream_bytes = payload bytes, n_blocks, status (bit 0:
 * corrupt stream / model on decode, bit 1: payload_capacity too small on encode -- nothing written).  d_data 4-byte
 * aligned.  All pointers are caller-owned device memory; asynchronous on `stream`. */
#define GSNFS_RANS_BLOCK 1024
typedef gsnfs_rlgr_info gsnfs_rans_info;
uint64_t gsnfs_rans_blocks(uint64_t n);
uint64_t gsnfs_rans_capacity(uint64_t n);    /* payload bytes that always suffice (12 bits per byte + block states) */
int gsnfs_rans_encode(gsnfs_ctx* ctx, gsnfs_stream stream, const uint8_t* d_data, uint64_t n, const gsnfs_counts* d_counts,
                      uint16_t* d_freq, uint16_t* d_nwords, uint8_t* d_payload, uint64_t payload_capacity,
                      gsnfs_rans_info* d_info);
int gsnfs_rans_decode(gsnfs_ctx* ctx, gsnfs_stream stream, const uint8_t* d_payload, uint64_t payload_bytes,
                      const uint16_t* d_freq, const uint16_t* d_nwords, uint64_t n, uint8_t* d_out,
                      gsnfs_rans_info* d_info);

/* gsnfs_rans_decode for callers that may not allocate device memory.
 * Who needs it: a player or renderer that decodes occupancy streams from a thread or a phase of its frame loop where
 * device allocation is off limits -- the application has handed the whole GPU to its own pool (a tensor framework's
 * caching allocator, an engine's arena) so a library cudaMalloc can fail or fragment it; or it runs under a memory
 * budget that is frozen after start-up; or it cannot afford the device-wide synchronisation and the unbounded latency
 * a cudaMalloc/cudaFree brings into a real-time loop.  Every other call of this header needs a gsnfs_ctx, and
 * gsnfs_create() is one cudaMalloc.  This call takes NO context and calls no cudaMalloc, cudaFree or any library
 * routine that allocates: its only working memory (the table of block-stream offsets, 8 bytes per 1024-byte block,
 * which gsnfs_rans_decode keeps in the context scratch) is a fixed 256 KB array that is part of the library image, so
 * every GPU that loads libgsnfs.so holds those 256 KB from load until the process exits, used or not.
 * Same arguments, same result (d_out and d_info, bit for bit) and same device-side corruption report as
 * gsnfs_rans_decode; inputs and outputs are still the caller's device buffers.
 * Limit: n <= GSNFS_RANS_STATIC_MAX_BYTES (32 MiB of occupancy bytes: the 16M-Gaussian frame at depth 16 needs about
 * 19 MB); a larger n returns GSNFS_E_CAPACITY before anything is enqueued -- use gsnfs_rans_decode with a context then.
 * Device: the work goes to the CURRENT device of the calling thread, which must be the device `stream` belongs to.
 * First call on each device: it looks up the device address of the built-in table (and sets one kernel attribute),
 * once, under a lock; that lookup is ordinary host-side set-up work, so make this first call before any stream capture
 * is started on that device.  Later calls only enqueue two kernels on `stream` and return without synchronising.
 * Sharing: all calls on one device use the same table.  Calls on one stream are ordered and safe back to back; two
 * calls that can overlap on the GPU (different streams, no event between them) race on the table and decode
 * garbage -- serialise them.  The table keeps the previous call's offsets between calls; nothing in it has to start at
 * zero, every call rewrites the entries it reads (and d_info in full) before it reads them.
 * Errors: INVALID_ARGUMENT (NULL pointer, n >= 2^32), CAPACITY (n beyond the limit above), CUDA (no current device,
 * more than 64 devices, a failed launch; cudaGetLastError() still holds the runtime's code). */
#define GSNFS_RANS_STATIC_MAX_BYTES (32ull << 20)
int gsnfs_rans_decode_static(gsnfs_stream stream, const uint8_t* d_payload, uint64_t payload_bytes,
                             const uint16_t* d_freq, const uint16_t* d_nwords, uint64_t n, uint8_t* d_out,
                             gsnfs_rans_info* d_info);

/* ---- bitstream container (host only) -----------------------------------------------------------------
 * PAPER.md:L176 ("J ... and the number of occupied nodes n_d at each level ... is encoded in the bitstream as
 * metadata"), L526 ("The header stores the number of levels and the node count of each level"), L255 (per-attribute
 * quantisation steps).  One coded frame = a fixed description + tagged sections (the arrays the device calls produce,
 * copied to the host by the caller), framed into one checksummed byte buffer:
 *   header (magic "GSNF", version, section count, gsnfs_frame_desc, CRC-32 of the whole file, total bytes)
 *   | section table (id, offset, bytes) | payloads, each 8-byte aligned.  Little endian.
 * gsnfs_container_unpack() does not copy: the returned sections point into `buf`.  A bad magic / version / checksum /
 * section bound returns GSNFS_E_CORRUPT_STREAM.  This build's [R1] reading needs the leaf weights at the decoder
 * (section GSNFS_SEC_WEIGHTS; absent = unit weights = the paper's stream). */
#define GSNFS_MAX_SECTIONS 16
enum {
  GSNFS_SEC_LEVEL_SIZES = 1,  /* uint32[depth + 1]                                                */
  GSNFS_SEC_QSTEP = 2,        /* float[channels]                                                  */
  GSNFS_SEC_KLT = 3,          /* float[gsnfs_klt_floats(channels)] (optional)                     */
  GSNFS_SEC_OCC_RAW = 4,      /* the occupancy bytes as they are                                  */
  GSNFS_SEC_OCC_FREQ = 5,     /* rANS model: uint16[256]                                          */
  GSNFS_SEC_OCC_NWORDS = 6,   /* rANS block word counts: uint16[gsnfs_rans_blocks(occ_bytes)]     */
  GSNFS_SEC_OCC_PAYLOAD = 7,  /* rANS block streams                                               */
  GSNFS_SEC_WEIGHTS = 8,      /* uint32[n_voxels] leaf weights (optional)                         */
  GSNFS_SEC_COEF_BITS = 9,    /* RLGR header: uint32[gsnfs_rlgr_blocks(n_voxels, channels, rlgr_block)] */
  GSNFS_SEC_COEF_STREAM = 10  /* RLGR block streams                                               */
};
typedef struct gsnfs_frame_desc {
  uint32_t depth, channels, n_voxels, occ_bytes, rlgr_block, flags;   /* flags: free for the application */
  float bbox_min[3], bbox_max[3];
  float dz_round, recon_bias;
} gsnfs_frame_desc;
typedef struct gsnfs_section {
  uint32_t id;
  uint32_t reserved;
  const uint8_t* data;   /* host */
  uint64_t bytes;
} gsnfs_section;
uint64_t gsnfs_container_size(const gsnfs_section* sections, int n_sections);
int gsnfs_container_pack(const gsnfs_frame_desc* desc, const gsnfs_section* sections, int n_sections,
                         uint8_t* out /* host */, uint64_t capacity, uint64_t* written);
int gsnfs_container_unpack(const uint8_t* buf /* host */, uint64_t bytes, gsnfs_frame_desc* desc,
                           gsnfs_section* sections /* out, max_sections entries */, int max_sections, int* n_sections);

/* ---- whole-frame calls on HOST buffers (copies inside; used for end-to-end timing) --------------- */
/* encode = H2D(xyz, attr) -> octree_encode -> voxel_merge -> raht_forward(weights = counts) -> D2H.
 * Host outputs: h_occ[occ_capacity], h_level_sizes[depth+1], h_weights[n] (first N_v valid),
 * h_qcoeff[n x channels] (first N_v rows valid), h_counts.  Host buffers should be pinned.
 * Returns after the results are in host memory. */
int gsnfs_frame_encode_host(gsnfs_ctx* ctx, gsnfs_stream stream,
                            const float* h_xyz, const float* h_attr, uint64_t n, int channels,
                            const float bbox_min[3], const float bbox_max[3], int depth,
                            const float* qstep, const gsnfs_quant* quant,
                            uint8_t* h_occ, uint64_t occ_capacity, uint32_t* h_level_sizes,
                            uint32_t* h_weights, int32_t* h_qcoeff, gsnfs_counts* h_counts);

/* decode = H2D(occ, weights, qcoeff) -> octree_decode -> raht_inverse -> D2H(voxel_xyz, attr).
 * h_weights may be NULL (unit weights).  h_voxel_xyz is N_v x 3 uint32, h_attr N_v x channels fp32. */
int gsnfs_frame_decode_host(gsnfs_ctx* ctx, gsnfs_stream stream,
                            const uint8_t* h_occ, uint64_t occ_bytes, const uint32_t* level_sizes, int depth,
                            const uint32_t* h_weights, const int32_t* h_qcoeff, int channels,
                            const float* qstep, const gsnfs_quant* quant,
                            uint32_t* h_voxel_xyz, float* h_attr, gsnfs_counts* h_counts);

/* The same two frame calls with the quantised coefficients entropy coded on the device (gsnfs_rlgr_encode /
 * gsnfs_rlgr_decode, block size rlgr_block), so that RLGR bytes instead of raw int32 coefficients cross PCIe
 * (everything stays GPU-resident until the bitstream).  Host outputs of the encoder: h_occ,
 * h_level_sizes, h_weights as above; h_block_bits[gsnfs_rlgr_blocks(n, channels, rlgr_block)], h_stream (first
 * h_info->stream_bytes valid), h_counts, h_info.  The attribute tensor is copied on an internal copy stream while the
 * position coder runs on `stream`.  GSNFS_E_CAPACITY if stream_capacity (or the context's 4*n*channels staging) is
 * too small for the stream. */
int gsnfs_frame_encode_host_packed(gsnfs_ctx* ctx, gsnfs_stream stream,
                                   const float* h_xyz, const float* h_attr, uint64_t n, int channels,
                                   const float bbox_min[3], const float bbox_max[3], int depth,
                                   const float* qstep, const gsnfs_quant* quant, int rlgr_block,
                                   uint8_t* h_occ, uint64_t occ_capacity, uint32_t* h_level_sizes, uint32_t* h_weights,
                                   uint32_t* h_block_bits, uint8_t* h_stream, uint64_t stream_capacity,
                                   gsnfs_counts* h_counts, gsnfs_rlgr_info* h_info);
int gsnfs_frame_decode_host_packed(gsnfs_ctx* ctx, gsnfs_stream stream,
                                   const uint8_t* h_occ, uint64_t occ_bytes, const uint32_t* level_sizes, int depth,
                                   const uint32_t* h_weights, const uint32_t* h_block_bits, const uint8_t* h_stream,
                                   uint64_t stream_bytes, int rlgr_block, int channels,
                                   const float* qstep, const gsnfs_quant* quant,
                                   uint32_t* h_voxel_xyz, float* h_attr, gsnfs_counts* h_counts);

#ifdef __cplusplus
}
#endif
#endif /* GSNFS_H_ */
