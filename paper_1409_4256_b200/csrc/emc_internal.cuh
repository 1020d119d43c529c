// Internal declarations shared by the translation units of libemc (sm_100a only).
// Nothing here is part of the C ABI (include/emc.h) and nothing is shared with oracle/.
#pragma once

#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/emc.h"

namespace emc {

// ---------------------------------------------------------------- host-side plumbing
emc_status cuda_fail(cudaError_t e, const char *what);
void note_launch(int n = 1);

#define EMC_TRY_CUDA(expr)                                        \
    do {                                                          \
        cudaError_t e__ = (expr);                                 \
        if (e__ != cudaSuccess) return ::emc::cuda_fail(e__, #expr); \
    } while (0)

#define EMC_TRY(expr)                         \
    do {                                      \
        emc_status s__ = (expr);              \
        if (s__ != EMC_OK) return s__;        \
    } while (0)

// after a kernel launch
#define EMC_LAUNCHED()                        \
    do {                                      \
        ::emc::note_launch();                 \
        EMC_TRY_CUDA(cudaGetLastError());     \
    } while (0)

static inline size_t round_up(size_t x, size_t a) { return (x + a - 1) / a * a; }
static inline int ceil_div(int a, int b) { return (a + b - 1) / b; }

// First 256 bytes of every workspace: what only the device can see (emc_check()).
struct WsHeader {
    int max_count;   // largest unmasked photon count seen by the pack kernel
    int w_range;     // 1 if a slice value left the fp16 range of the Gaussian model's operand planes (>= 65504)
    int shard_stamp[4];   // written by emc_shard_stats: (R_local, N, P, kShardTag) of the L / packed patterns the workspace carries
    int shard_mismatch;   // set by emc_shard_update when the stamp is not the one its own arguments give
    int pad[57];
};
constexpr int kShardTag = 0x53484152;   // "SHAR"
static_assert(sizeof(WsHeader) == 256, "header is one 256-byte line");

// Bump allocator over the caller's workspace.
struct Arena {
    uint8_t *base;
    size_t size, off;
    bool ok;
    Arena(void *p, size_t bytes) : base((uint8_t *)p), size(bytes), off(0), ok(true) {}
    template <class T>
    T *take(size_t count) {
        size_t bytes = round_up(count * sizeof(T), 1024);
        if (off + bytes > size) { ok = false; off += bytes; return nullptr; }
        T *p = (T *)(base + off);
        off += bytes;
        return p;
    }
};

enum PlaneFormat { FMT_F16 = 0, FMT_BF16 = 1 };   // = the UMMA instruction descriptor encoding

// ---------------------------------------------------------------- stage launchers (device work)
// Sample geometry prepared once per call (emc_expand.cu): q and the mask as one float4 per pixel (x, y, z, use ? 1 : 0),
// the rotation matrices as three float4 per rotation (rows of R_r, .w unused), the detector's row length for the tiling.
struct Geometry {
    const float4 *qm;     // [P]
    const float4 *rotm;   // [R][3]
    int n_pix, n_rot, row_len;
};
size_t geometry_float4(int n_pix, int n_rot);   // float4s of scratch behind a Geometry
emc_status launch_geometry(const float *q, const uint8_t *mask, int n_pix, int row_len, const float *quat, int n_rot,
                           float4 *buf, Geometry *out, cudaStream_t st);

// Expand (emc_expand.cu).  Any of W, idx, planes may be null.  planes = [2][R][ld_p] fp16 (hi, lo)
// of logW with masked / outside samples zeroed; S[r] = sum_{p:mask} W (the plain-gather kernel adds into S: zero it first).  gauss: the planes
// hold W itself and S[r] += sum_{p:mask} W^2 (the operands of the paper's Gaussian model).
// `blocked` = scratch of expand_scratch_floats() floats (corner blocks of the model, band partials of S) with `geo`
// prepared, or both null:
// plain gathers from q / mask / quat.
size_t expand_scratch_floats(int n, int n_pix, int n_rot);
emc_status launch_expand(const float *model, int n, const float *q, const uint8_t *mask, int n_pix,
                         const float *quat, int n_rot, float *W, int32_t *idx, __half *planes,
                         int ld_p, float *S, float *blocked, const Geometry *geo, cudaStream_t st, bool gauss = false,
                         bool logw32 = false, int *w_range = nullptr);
// w_range (gauss): set to 1 if an unmasked slice value is >= 65504 (it would become inf in the fp16 planes of W)
// logw32 (blocked path, W given, no idx / planes): W receives log(max(W, 1e-30)) as float32, 0 for masked / outside samples, and
// S the row sums (operands of the photon-list log-likelihood, emc_sparse.cu)
// logW planes + S from a given W (stage API of emc_loglik).
emc_status launch_logw_split(const float *W, const int32_t *idx, const uint8_t *mask, int n_pix,
                             int n_rot, __half *planes, int ld_p, float *S, cudaStream_t st, bool gauss = false);
// gauss: the planes hold W itself and S[r] += sum_{p:mask} W^2 (stage API of the Gaussian model)
// Q[r,d] = B^2 g_d - C_r / (2 sigma^2) and phi[r,d] = A_d / B[r,d] (inf where B = 0) from B = W K^T (eqs. 2.2, 2.3, 2.6 collapsed)
emc_status launch_gauss_q(const float *B, const float *c_row, const float *g_col, const float *ia_col, float inv2s2, int n_rot,
                          int n_pat, int ld_b, float *Q, float *phi, int ld_out, cudaStream_t st);

// Pack photon counts (emc_pack.cu): Kc [Nc][ld_p] fp16 (row = pattern) and/or KT [P][ld_n] fp16
// (row = pixel), masked pixels zeroed, an unmasked count above EMC_MAX_COUNT recorded in hdr->max_count.
emc_status launch_pack(const void *counts, emc_count_type type, int n_pat, int n_pix,
                       const uint8_t *mask, __half *Kc, int ld_p, __half *KT, int ld_n,
                       WsHeader *hdr, cudaStream_t st);
// fills out[0..n) (floats) with NaN if hdr->max_count != 0: a result computed from clamped counts must not be
// consumed unnoticed (emc.h, conventions)
emc_status launch_poison(const WsHeader *hdr, float *out, size_t n, double *out64, int n64, cudaStream_t st);
// rotation shards: emc_shard_stats stamps the header with the sizes of what it leaves in the workspace; emc_shard_update
// verifies the stamp on the device (no host round trip) and records a mismatch, which poisons its results like a count out
// of range does and is reported by emc_check
emc_status launch_shard_stamp(WsHeader *hdr, int n_rot, int n_pat, int n_pix, bool verify, cudaStream_t st);

// A[d] = sum_p Kc[d][p]^2 (fluence numerators of the Gaussian model, eq. 2.6) as g_col[d] = 1 / (2 sigma^2 A_d) and
// ia_col[d] = 1 / A_d (both 0 where A_d = 0)
emc_status launch_rowsq(const __half *Kc, int n_pat, int n_pix, int ld_p, float inv2s2, float *g_col, float *ia_col,
                        cudaStream_t st);

// Plane GEMM on tcgen05 (emc_gemm.cu):  acc[m,n] = sum_pl sum_k A[pl][m][k] * B[n][k]
struct GemmProblem {
    const void *A;      // [n_planes][M][lda] 16-bit elements, K-major
    const void *B;      // [N][ldb] 16-bit elements, K-major
    int n_planes;       // 2
    int M, N, K;
    int lda, ldb;       // row pitches in elements (multiples of 8)
    size_t plane_stride;  // elements between planes of A
    PlaneFormat a_fmt, b_fmt;
    float *out;         // [M][ld_out]
    int ld_out;
    const float *rowv;  // [M] row vector of the epilogue (S for loglik, s for update) or null
    int epilogue;       // EPI_*
    int k_chunk = 0;    // k-blocks (of 64) per TMEM accumulation chunk, 0 = default (8 = 512 elements)
    const float *chunk_scale = nullptr;   // [ceil(K/512)][M] factor applied when a chunk is drained, or null
    // log-likelihood only: fused first sweep of the normalisation.  When stat_m is set (and the CTA-pair kernel
    // runs, see gemm_fuses_stats()) the epilogue writes per-(32-row block, column) partial statistics of
    // a = out + log w_r (reference pair + sum-exp, emc_normalize.cu ColStat) into stat_m, stat_w, stat_z
    // [ceil(M/32)][ld_stat]; weight = [M] prior weights or null = 1/M.
    float *stat_m = nullptr, *stat_w = nullptr, *stat_z = nullptr;
    int ld_stat = 0;
    const float *weight = nullptr;
    float log_uniform = 0.f;          // log_uniform_of(all rotations) for weight == null
    const float *gauss_g = nullptr;   // EPI_GAUSS: [N] g_d = 1 / (2 sigma^2 A_d)
    float inv2s2 = 0.f;               // EPI_GAUSS: 1 / (2 sigma^2)
    bool one_cta = false;   // EMC_GEMM_1CTA: the one-CTA kernel instead of CTA pairs (cta_group::2)
};
enum { EPI_SUB_ROW = 0,     // out = acc - rowv[m]                      (log-likelihood)
       EPI_STORE = 1,       // out = acc                                (raw update numerator)
       EPI_ADD = 2,         // out += acc                               (numerator over chunks)
       EPI_DIV_ROW = 3,     // out = rowv[m] > 0 ? acc / rowv[m] : 0    (eq. 2.5)
       EPI_GAUSS = 4 };     // out = acc = B; rowv = C, gauss_g = g: statistics of Q = (B^2/A - C) / (2 sigma^2)
emc_status launch_plane_gemm(const GemmProblem &g, bool simt_debug, cudaStream_t st);
// true if launch_plane_gemm(g, simt_debug, .) fills g.stat_m / g.stat_z
bool gemm_fuses_stats(const GemmProblem &g, bool simt_debug);

// Gaussian model (eqs. 2.2, 2.3, 2.6): with phi = A_d / B_rd,  Q_rd = (B_rd^2 / A_d - C_r) / (2 sigma^2)
//   = B^2 g_d + (-C_r / (2 sigma^2)),  g_d = 1 / (2 sigma^2 A_d)  (0 for a frame without photons).
// The GEMM epilogue (statistics) and normalize_kernel (second sweep) must form the two terms BIT-IDENTICALLY, hence
// explicit single-rounding intrinsics that the compiler cannot contract differently in the two kernels.
#ifdef __CUDACC__
__device__ __forceinline__ float gauss_col_factor(float a_col, float inv2s2) {
    return a_col > 0.f ? __fdiv_rn(inv2s2, a_col) : 0.f;
}
__device__ __forceinline__ float gauss_elem_term(float b, float g_col) { return __fmul_rn(__fmul_rn(b, b), g_col); }
__device__ __forceinline__ float gauss_row_term(float log_w, float c_row, float inv2s2) {
    return __fsub_rn(log_w, __fmul_rn(c_row, inv2s2));
}
#endif

// Normalise (emc_normalize.cu).  scratch = normalize_scratch_floats() floats.  `planes` (optional) receives the
// operand planes of P for the update GEMM: two fp16 planes scaled per (row, 512-column chunk) with the inverse
// scales in chunk_inv_scale [ceil(ld_n/512)][R].
// Gaussian model: L holds B = W K^T; c_row [R] = sum_p W^2, A_d = sum_p K^2 enters as two column factors, inv2s2 = 1 / (2 sigma^2)
struct GaussTerms {
    const float *c_row, *g_col, *ia_col;   // g_col = 1 / (2 sigma^2 A_d), ia_col = 1 / A_d
    float inv2s2;
    float log_uniform;                     // log_uniform_of(R): the same float in the GEMM's statistics and the second sweep
};
// log(1/R) for weight == NULL, evaluated ONCE on the host and handed to every kernel that needs it (the row terms of
// the Gaussian model nearly cancel: a 1-ulp difference between two evaluations would show in sum_r P)
float log_uniform_of(int n_rot);
size_t normalize_scratch_floats(int n_rot, int ld_n);
int normalize_stat_rows(int n_rot);   // scratch = part_m, part_w, part_z [rows][ld_n] each, then col_m, col_w, col_iz [ld_n] each
emc_status launch_normalize(const float *L, const float *weight, int n_rot, int n_pat, int ld_n,
                            float *P, __half *planes, size_t plane_stride, float *chunk_inv_scale,
                            float *s, double *loglik, bool accumulate, float *scratch, bool stats_ready,
                            cudaStream_t st, const GaussTerms *gauss = nullptr, int n_store = 0, float log_uniform = 0.f,
                            int chunk_mode = 0, bool carry_in = false, int layout_rot = 0);
// chunk_mode (rotation chunks): 0 = the rows are the whole rotation list; 1 = first sweep of a
// chunk: its column statistics are merged into the carried ones (carry_in = false for the first chunk) and nothing else is
// written (loglik, when given, receives the total of the statistics carried so far: pass it with the last chunk only);
// 2 = second sweep of a chunk: P / planes / s with the final statistics left by the last mode-1 call.
// layout_rot: the rotation count the scratch was laid out for (normalize_scratch_floats); 0 = n_rot.  A ragged last chunk
// passes the full chunk size so that the carried statistics stay where they are.
// log_uniform: log w of every row when weight == null; 0 = log_uniform_of(n_rot) (set it when the rows are a chunk of a
// longer rotation list)
// n_store: columns of a row the call may write (planes padding, column arrays); 0 = ld_n.  Smaller when L, planes and
// scratch are views that start inside a row (emc_api.cu, pipelined first iteration).
// Rotation shards (one process per GPU, DESIGN.md section 11 NEXT-4): (m, w, z) pointers of partial row `row` of the statistics
// scratch (row < 0: the carry row), and the merge of the first n_rows partial rows (one per rank, in rank order) into the
// final column statistics (+ the total log-likelihood); launch_normalize(chunk_mode = 2) then writes P.
void normalize_stat_row(float *scratch, int layout_rot, int ld_n, int row, float **m, float **w, float **z);
emc_status launch_colstats_combine_rows(float *scratch, int layout_rot, int n_rows, int n_pat, int ld_n, double *loglik,
                                        cudaStream_t st);
// operand planes of a given P (stage API of emc_update).
emc_status launch_p_split(const float *P, int n_rot, int n_pat, int ld_n, __half *planes, int ld_pl,
                          size_t plane_stride, float *chunk_inv_scale, cudaStream_t st);
// rows of Wnew divided by s[r] (after the last pattern chunk).
emc_status launch_div_rows(float *Wnew, const float *s, int n_rot, int n_pix, cudaStream_t st);

// Photon lists and the sparse form of stages 2 and 4 (emc_sparse.cu, EMC_SPARSE_PHOTONS)
struct SparseList {
    const int *row_ptr;          // [rows + 1]
    const uint32_t *entries;     // column | count << 20, in row order
    int rows;
};
size_t sparse_list_ints(int rows, size_t max_entries);   // ints of scratch behind a SparseList
// both lists straight from the raw counts [rows = frames][cols = pixels] (masked pixels skipped; an unmasked count above
// EMC_MAX_COUNT recorded in hdr); list_pat / list_pix = sparse_list_ints(rows, rows x cols) / (cols, rows x cols) ints
emc_status launch_lists_raw(const void *counts, emc_count_type type, int rows, int cols, const uint8_t *mask, int *list_pat,
                            int *list_pix, WsHeader *hdr, SparseList *by_frame, SparseList *by_pixel, cudaStream_t st);
// rows of L^T [rows][ld] -> rows of P^T in place (soft-max over the n_rot rotations of a row with log weights logw [n_rot] or
// null = uniform, every log w = log_uniform); s[r] += column sums; loglik += total
emc_status launch_softmax_rows(float *LT, int rows, int n_rot, int ld, const float *logw, float log_uniform, float *s,
                               double *loglik, cudaStream_t st);
emc_status launch_logw(const float *weight, int n_rot, float *out, cudaStream_t st);
// Y [rows][ld] = A X (- sub_row) (+ Y), X [K][ld], the first n_rot columns
emc_status launch_spmm_rot(const SparseList &a, const float *X, float *Y, int ld, int n_rot, const float *sub_row,
                           bool accumulate, cudaStream_t st);
emc_status launch_transpose(const float *in, int rows, int cols, int ld_in, float *out, int ld_out, cudaStream_t st);
// logW^T [P][ld_r] from W [R][P] (0 for masked / outside samples) and S[r] += sum_{p:mask} W
emc_status launch_logw_transposed(const float *W, const int32_t *idx, const uint8_t *mask, int n_rot, int n_pix, float *logWT,
                                  int ld_r, float *S, cudaStream_t st);
// W' [R][P] = (W'^T [P][ld_r])^T / s[r]
emc_status launch_transpose_div(const float *WT, int n_pix, int n_rot, int ld_r, float *Wnew, const float *s, cudaStream_t st);

// Compress (emc_compress.cu).  acc = compress_scratch_float2(n) float2 of scratch (one 64-byte (num, den) corner
// block per base corner), zeroed inside.
size_t compress_scratch_float2(int n);
// cache (optional, eq. 2.10 with slice_w only): den survives in `acc` from one call to the next and is reused while the
// set {r: slice_w[r] > 0} stays the one in cache->active; force = accumulate it afresh (first iteration, new list).
struct DenCache {
    uint32_t *active;   // [ceil(R/32)] bit mask of the slices den was accumulated for
    int *changed;       // device flag, scratch
    bool force;
};
enum { COMPRESS_CLEAR = 1, COMPRESS_SCATTER = 2, COMPRESS_DIVIDE = 4, COMPRESS_ALL = 7 };
// numden [2][n^3] = the numerator and denominator grids gathered from the corner blocks (what rotation shards all-reduce)
emc_status launch_compress_export(const float2 *acc, int n, float *numden, cudaStream_t st);
// model' = num / den from such grids (division as the final step)
emc_status launch_numden_divide(const float *numden, int n, float *model_out, cudaStream_t st);
emc_status launch_compress(const float *Wnew, const float *slice_w, bool weighted, const Geometry &geo, int n,
                           float2 *acc, float *model_out, float *den_out, cudaStream_t st,
                           const DenCache *cache = nullptr, int phases = COMPRESS_ALL);
// phases: rotation chunks scatter into the same accumulators (CLEAR with the first, DIVIDE with the last; no cache)

}  // namespace emc
