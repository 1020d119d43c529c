/*
 * emc.h -- C ABI of libemc: one iteration of the Expansion-Maximization-Compression (EMC)
 * algorithm of arXiv 1409.4256 (Ekeberg, Engblom, Liu) on one NVIDIA B200 (sm_100a).
 *
 * Citations are "PAPER.md:<line>" (= /root/reference/PAPER.md of the build container) plus the
 * equation they fall in, and "DESIGN.md §3 Gn" for the readings taken where the paper is silent.
 *
 * Notation (paper -> here): M_rot -> R (index r), M_data -> N (index d), M_pix -> P (index p),
 * M_grid -> G = n^3 (index l); W_ij -> W[r,p]; model grid (blackboard W_l) -> model[l];
 * P_jk -> P[r,d]; w_j -> weight[r].
 *
 * Conventions for EVERY entry point
 *  - Every array pointer is a DEVICE pointer owned by the caller (the Python binding allocates
 *    them with PyTorch) unless the comment says "host".  The library allocates nothing: scratch
 *    comes from the caller's workspace `ws` of at least emc_workspace_bytes(...) bytes, 256-byte
 *    aligned.  Nothing in the workspace survives a call except where stated.
 *  - `stream` is a cudaStream_t.  Calls validate their arguments synchronously, enqueue their
 *    kernels on `stream` and return without synchronising.  The exceptions say so in their own
 *    comment: emc_check, emc_profile_read and emc_refine wait for the device.
 *  - No call creates CUDA objects.  The two features that need some (a copy stream for
 *    host-resident patterns, events for per-stage timing) take them from an emc_context the
 *    caller creates once; one context serves one stream at a time, any number of contexts and
 *    workspaces can be in use on different streams and threads at once.
 *  - Errors are returned as negative emc_status values, never thrown or aborted.  A condition that
 *    only the device can see (a photon count too large for the exact 16-bit operand format) is
 *    recorded in the workspace header: every result of that call is then filled with NaN on the
 *    device, so that it cannot be consumed unnoticed, and emc_check() reports it.
 *  - Matrices are row-major: W is [R][P], L and P are [R][N] with row pitch `ld_n` floats
 *    (ld_n >= N, a multiple of 4; the binding uses N rounded up to 64).  The model is
 *    [n][n][n] with z fastest, voxel (i,j,k) at integer coordinates, origin c = n/2 on every axis
 *    (DESIGN.md §3 G5).
 */
#ifndef EMC_H_
#define EMC_H_

#include <stddef.h>
#include <stdint.h>

#if defined(__GNUC__)
#define EMC_API __attribute__((visibility("default")))
#else
#define EMC_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    EMC_OK = 0,
    EMC_ERR_ARG = -1,          /* null pointer, non-positive size, misaligned pointer or pitch */
    EMC_ERR_UNSUPPORTED = -2,  /* a size outside what the kernels index (see each call) */
    EMC_ERR_WORKSPACE = -3,    /* ws is NULL, misaligned or smaller than emc_workspace_bytes() */
    EMC_ERR_CUDA = -4,         /* a CUDA runtime/driver call failed (emc_last_cuda_error()) */
    EMC_ERR_COUNT_RANGE = -5,  /* an unmasked photon count exceeds EMC_MAX_COUNT (emc_check) */
    EMC_ERR_VALUE_RANGE = -6,  /* emc_iterate_gaussian: an unmasked slice value >= 65504 (fp16 planes of W; emc_check) */
    EMC_ERR_STATIC_SCRATCH = -7 /* emc_normalize_static: these sizes need more than EMC_STATIC_SCRATCH_BYTES */
} emc_status;

typedef enum { EMC_I32 = 0, EMC_U16 = 1, EMC_U8 = 2 } emc_count_type;

/* Largest photon count in an unmasked pixel that the exact 16-bit tensor-core operands hold
 * (fp16 holds every integer up to 2048; DESIGN.md §6 "precision scheme").  Saturated pixels are
 * expected to be masked. */
#define EMC_MAX_COUNT 2048

/* Responsibilities are float32 (the paper works in single precision).  libemc stores them flush-to-zero:
 * a value below the smallest normal float32, 2^-126, is 0, on output (emc_normalize, P_out) and on input (emc_update)
 * (DESIGN.md §3 G20).  The paper is silent on underflow; the plain IEEE cast would keep subnormals down to 2^-149.  Why
 * the library flushes: a subnormal P has lost its 24 significant bits, so a slice whose weights are all subnormal gets a
 * W' (eq. 2.11) that no float32 pipeline can form to 1e-5 -- and the B200's own float32 reduction units (RED.ADD.F32 to
 * global memory, which accumulates s[r]) flush subnormal operands anyway.  A rotation whose whole row is 0 has
 * s[r] = 0: W'[r,:] = 0 and the slice is skipped by Compress (G17).  Which slices that is matters under eq. (2.10)
 * only; the tests gate the difference to the plain cast slice by slice (tests/gates.py). */
#define EMC_P_MIN 1.1754943508222875e-38f

/* flags */
#define EMC_COMPRESS_WEIGHTED 0x1u /* eq. (2.12): slice r enters Compress with
                                      weight s[r] = sum_d P[r,d]; default is eq. (2.10), weight 1 */
#define EMC_ACCUMULATE        0x2u /* emc_normalize: add into s / loglik; emc_update: add into Wnew
                                      (pattern chunks, DESIGN.md §3 G9) */
#define EMC_UPDATE_RAW        0x4u /* emc_update: leave Wnew as the numerator of eq. (2.11),
                                      do not divide by s[r] */
#define EMC_PROFILE_STAGES    0x20u /* emc_iterate records the context's CUDA events on `stream` around every
                                      stage; read (and reset) the sums with emc_profile_read() */
#define EMC_SPARSE_PHOTONS    0x40u /* emc_iterate (Poisson model): stages 2 and 4 from per-frame / per-pixel photon lists on
                                      plain CUDA cores instead of the dense tensor-core contractions; for frames that
                                      are almost empty (DESIGN.md section 11 NEXT-2 has the measured crossover).  Needs
                                      n_pix and the pattern chunk below 2^20 and their product below 2^31 (32-bit list
                                      offsets), else EMC_ERR_UNSUPPORTED; the workspace grows (pass the flag to
                                      emc_workspace_bytes).  Not taken by emc_iterate_rot_chunked (EMC_ERR_UNSUPPORTED). */
#define EMC_GEMM_1CTA         0x200u /* run the two contractions with one CTA per tile (cta_group::1)
                                        instead of CTA pairs (cta_group::2); a comparison / bisecting aid */
#define EMC_DEBUG_SIMT        0x100u /* run the two contractions on plain CUDA cores (slow; a
                                        bisecting aid for the tcgen05 path, never the default) */

/* The 3D intensity model on its Cartesian grid (p_l). */
typedef struct {
    int n;              /* grid is n x n x n, 2 <= n <= 1024 */
    const float *model; /* [n][n][n], z fastest */
} emc_model;

/* Detector geometry: the Ewald-sphere coordinates q_i of every pixel. */
typedef struct {
    int n_pix;           /* P */
    const float *q;      /* [P][3] (x,y,z) in voxel units relative to the origin c */
    const uint8_t *mask; /* [P], 1 = use, 0 = missing/saturated; NULL = use all */
    int row_len;         /* pixels per detector row when the P pixels are a row-major 2-D array (n_pix % row_len == 0),
                            0 = no 2-D structure known.  A locality hint only: Expand and Compress then give each warp a
                            4 x 8 tile of pixels instead of 32 consecutive ones; results do not depend on it. */
} emc_detector;

/* The discretised rotation space (R_j) with prior weights w_j. */
typedef struct {
    int n_rot;           /* R */
    const float *quat;   /* [R][4] unit quaternions (w,x,y,z), active rotation */
    const float *weight; /* [R] prior weights w_j > 0, or NULL = 1/R */
} emc_rotations;

/* The measured frames K_k of photon counts. */
typedef struct {
    int n_pat;           /* N */
    const void *counts;  /* [N][P] row-major; values in masked pixels are ignored */
    emc_count_type type;
} emc_patterns;

/* CUDA objects the library may use on the caller's behalf: one non-blocking copy stream with its events
 * (EMC_PATTERNS_ON_HOST) and a pool of timing events (EMC_PROFILE_STAGES).  Created and destroyed by the
 * caller, outside the hot path; emc_iterate* take it as an argument and need it only with those flags
 * (EMC_ERR_ARG if it is NULL then).  One context serves one stream at a time. */
typedef struct emc_context emc_context;
EMC_API emc_status emc_context_create(emc_context **ctx);
EMC_API emc_status emc_context_destroy(emc_context *ctx);

/* Bytes of workspace sufficient for any call below at these sizes.  n_pat_chunk = patterns
 * resident per chunk (= N when not chunked).  Returns 0 on invalid sizes. */
EMC_API size_t emc_workspace_bytes(int n, int n_pix, int n_rot, int n_pat_chunk, unsigned flags);
/* Bytes sufficient for emc_expand and emc_compress alone (the stage calls that touch no patterns): the corner blocks
 * of the model or of the accumulators plus the packed geometry.  Returns 0 on invalid sizes. */
EMC_API size_t emc_workspace_bytes_geometry(int n, int n_pix, int n_rot);

/* Stage 1, Expand (e-step), eq. (2.9), PAPER.md:113-116:
 *   W[r,p] = sum_l f(p_l - R_r q_p) model[l],  f = trilinear weights of the 8 voxels around
 *   x = R_r q_p + c.  Samples whose 8 neighbours are not all inside the grid give W = 0 (G7).
 * Computed for every pixel, masked or not.
 *   W   [R][P] float, out.
 *   idx [R][P] int32, out, or NULL: linear index (b_x*n + b_y)*n + b_z of the base corner
 *       b = floor(x), or -1 outside the grid.  The coordinate arithmetic is pinned (DESIGN.md §3
 *       G4) so this map is bit-exact against the oracle.
 *   ws  workspace or NULL.  With a workspace the model is first re-laid as one 32-byte block of the 8 corner
 *       values per base corner, so that a sample is one 32-byte load; without, plain gathers. */
EMC_API emc_status emc_expand(const emc_model *model, const emc_detector *det, const emc_rotations *rot,
                      float *W, int32_t *idx, void *ws, size_t ws_bytes, void *stream);

/* Stage 2, Poisson log-likelihood (north_star stage 2; Poisson model of PAPER.md:68; the E-step
 * numerator of PAPER.md:166):
 *   L[r,d] = sum_{p: mask} ( K[d,p] * logW[r,p] - W[r,p] ),
 *   logW = log(max(W, 1e-30)) inside the grid, 0 outside (G7, G8).
 *   W   [R][P] float, in (as written by emc_expand).
 *   idx [R][P] int32, in, or NULL = every sample is inside the grid.
 *   L   [R][ld_n] float, out (columns >= N are not written). */
EMC_API emc_status emc_loglik(const float *W, const int32_t *idx, const emc_detector *det,
                      const emc_patterns *pat, int n_rot, float *L, int ld_n, unsigned flags,
                      void *ws, size_t ws_bytes, void *stream);

/* Stage 3, normalisation over rotations (reconstructed eq. (2.4)):
 *   a = L[r,d] + log w_r;  m_d = max_r a;  P[r,d] = exp(a - m_d) / sum_r exp(a - m_d),
 *   values below EMC_P_MIN stored as 0.
 *   L      [R][ld_n] float, in.
 *   P      [R][ld_n] float, out.
 *   s      [R] float, out: s[r] = sum_d P[r,d]            (added to with EMC_ACCUMULATE)
 *   loglik device double, out: sum_d (m_d + log sum_r exp(a - m_d))   (added to with EMC_ACCUMULATE)
 *   Either of s, loglik may be NULL. */
EMC_API emc_status emc_normalize(const float *L, const emc_rotations *rot, int n_pat, int ld_n, float *P,
                         float *s, double *loglik, unsigned flags, void *ws, size_t ws_bytes,
                         void *stream);

/* Stage 3 again, for callers that have no device memory to hand over as a workspace and no way to get any.
 *
 * Who that is: code that runs where cudaMalloc is off limits or already spent -- a plug-in inside a host
 * application that gave it fixed input / output buffers and nothing else, a real-time acquisition loop at the
 * beamline that must not touch the allocator (cudaMalloc takes a device-wide lock and can stall every stream for
 * milliseconds), a process whose memory pool has been handed out in full to the experiment's frames.  Every other
 * call of this header takes its scratch from the caller's `ws`; this one brings its own.
 *
 * Same arithmetic, same kernels, same results as emc_normalize (P bit for bit; s and loglik up to the order of
 * their atomic additions).  The per-pattern partial statistics of the first sweep live in ONE array of
 * EMC_STATIC_SCRATCH_BYTES that is compiled into the library as a `static __device__` object: every GPU that
 * loads libemc holds these 4 MiB from then until the process exits, whether this call is ever used or not.
 *
 *   Arguments as emc_normalize, without ws / ws_bytes.  L, P, s, loglik are the caller's device buffers.
 *   Limit: emc_normalize_static_bytes(n_rot, n_pat, ld_n) <= EMC_STATIC_SCRATCH_BYTES, else the call returns
 *     EMC_ERR_STATIC_SCRATCH and enqueues nothing.  The need is (3 * row_splits + 3) * ld_n floats with
 *     row_splits <= 64 shrinking as n_pat grows; every n_pat up to 100 000 fits for any n_rot (all of
 *     Table 4.1's pattern counts per chunk).
 *   The call itself never calls cudaMalloc, cudaFree or any library routine that allocates.
 *   First call on a device: looks up the device address of the array (cudaGetSymbolAddress, with the device that
 *     owns `stream` current -- the caller makes it current, as for every other call) and keeps it for later calls on
 *     that device.  Make that first call outside any stream capture.
 *   One array per device, shared by every call in the process: two emc_normalize_static calls whose kernels can
 *     overlap on the GPU (different streams, or different host threads on different streams) race on it and
 *     produce garbage.  Keep them on one stream, or order them with events.  The array keeps whatever the last
 *     call left; nothing in it has to start at zero, because every value a call reads it has written itself
 *     earlier in the same call (s and loglik are cleared by the call unless EMC_ACCUMULATE is set). */
#define EMC_STATIC_SCRATCH_BYTES (4u << 20)
/* bytes of the built-in array a call at these sizes uses; 0 on invalid sizes */
EMC_API size_t emc_normalize_static_bytes(int n_rot, int n_pat, int ld_n);
EMC_API emc_status emc_normalize_static(const float *L, const emc_rotations *rot, int n_pat, int ld_n, float *P,
                                float *s, double *loglik, unsigned flags, void *stream);

/* Stage 4, slice update (M-step), eq. (2.5) with phi == 1 / eq. (2.11), PAPER.md:84-85, 124-125:
 *   Wnew[r,p] = sum_d P[r,d] K[d,p] / s[r]   for unmasked p, 0 for masked p and where s[r] = 0.
 *   P [R][ld_n] float, in;  s [R] float, in (ignored with EMC_UPDATE_RAW);  Wnew [R][P] float, out.
 *   EMC_UPDATE_RAW leaves the numerator; EMC_ACCUMULATE (implies RAW) adds it into Wnew. */
EMC_API emc_status emc_update(const float *P, int ld_n, const float *s, const emc_detector *det,
                      const emc_patterns *pat, int n_rot, float *Wnew, unsigned flags, void *ws,
                      size_t ws_bytes, void *stream);

/* Stage 5, Compress (c-step), eq. (2.10) / (2.12), PAPER.md:118-130, 166, 192:
 *   num[l] = sum_{r,p} f om_r Wnew[r,p],  den[l] = sum_{r,p} f om_r  over unmasked samples inside
 *   the grid, same f as Expand;  model_out[l] = den > 0 ? num/den : 0 (division last).
 *   om_r = 1 if slice_w == NULL; else slices with slice_w[r] == 0 are skipped and
 *   om_r = slice_w[r] with EMC_COMPRESS_WEIGHTED (eq. 2.12), 1 without (eq. 2.10).
 *   model_out [n^3] float, out;  den_out [n^3] float, out or NULL. */
EMC_API emc_status emc_compress(const float *Wnew, const float *slice_w, const emc_detector *det,
                        const emc_rotations *rot, int n, float *model_out, float *den_out,
                        unsigned flags, void *ws, size_t ws_bytes, void *stream);

/* Algorithm 1: `n_iter` iterations of stages 1-5 on one stream with no host
 * synchronisation; model' of one iteration is the model of the next (same rotation list).
 * Patterns are processed in chunks of n_pat_chunk (0 = all at once): stages 2-3 per chunk, s[r]
 * and the update numerators summed over chunks, divided after the last (DESIGN.md §3 G9).
 *   pat->counts may be a PINNED HOST pointer when flags has EMC_PATTERNS_ON_HOST: each chunk is
 *   then copied to the device inside the call, on the context's copy stream into two staging
 *   buffers of the workspace, so that the copy of one chunk overlaps the work on the previous one
 *   (one stream per workspace and per context).  With a single resident chunk of at least 4096
 *   patterns the first iteration runs on four sub-ranges of the chunk while the copies are in flight (the
 *   same arithmetic as pattern chunks).
 *   With eq. (2.10) the denominators of Compress are accumulated in the first iteration and reused by the later
 *   ones for as long as the set of skipped slices (s[r] = 0) stays the same; this is decided on the device.
 *   model_out [n^3] float, out (may not alias model->model).
 *   P_out     [R][ld_n] float of the LAST iteration, out, or NULL (ld_n >= N; needs one chunk).
 *   loglik    [n_iter] device doubles, out: total log-likelihood of each iteration. */
#define EMC_PATTERNS_ON_HOST 0x10u
EMC_API emc_status emc_iterate(const emc_model *model, const emc_detector *det, const emc_rotations *rot,
                       const emc_patterns *pat, int n_iter, int n_pat_chunk, float *model_out,
                       float *P_out, int ld_n, double *loglik, unsigned flags, void *ws,
                       size_t ws_bytes, void *stream, emc_context *ctx);

/* Where emc_iterate / emc_iterate_gaussian left its intermediate results inside the caller's workspace: pointer
 * arithmetic on the host, nothing is enqueued.  For checking the product path itself (tests/): the log-likelihood matrix
 * that the fused Expand (logW operand planes formed in registers) and the contraction produced, which no stage call
 * returns, and the slices W' and their weights s that went into Compress.  Sizes and flags as passed to the emc_iterate
 * call that used `ws`.  Valid after that call's work on its stream has finished and until the next call that uses `ws`;
 * with several pattern chunks the per-chunk buffers hold the LAST chunk of the last iteration.
 *   what = EMC_VIEW_LOGLIK: *ptr = L [R][*ld] float (Gaussian model: B = W K^T); not with EMC_SPARSE_PHOTONS
 *          EMC_VIEW_S:      *ptr = s [R] float, *ld = 0
 *          EMC_VIEW_WNEW:   *ptr = W' [R][*ld] float, *ld = n_pix */
enum { EMC_VIEW_LOGLIK = 0, EMC_VIEW_S = 1, EMC_VIEW_WNEW = 2 };
EMC_API emc_status emc_workspace_view(void *ws, int n, int n_pix, int n_rot, int n_pat_chunk, unsigned flags, int what,
                              void **ptr, int *ld);

/* Algorithm 1 with the ROTATION list streamed in chunks of n_rot_chunk rotations, the paper's own memory scheme
 * ("chunk C_c"; "only maximal rotational probabilities and sums are necessary", PAPER.md:203;
 * DESIGN.md section 11 NEXT-2): nothing of size R x N or R x P is held, the workspace scales with the chunk.  Two
 * sweeps over the chunks per iteration:
 *   sweep 1, per chunk: Expand, log-likelihood, the chunk's per-pattern (max, sum) merged into the running ones
 *   sweep 2, per chunk: Expand, log-likelihood (recomputed), P with the final (max, sum), s[r], update, and the
 *                       chunk's scatter into the numerator / denominator grids of Compress; division after the last.
 * Results are those of emc_iterate up to summation order; the log-likelihood contraction runs twice.
 * Patterns are device-resident, in one pattern chunk.  Arguments as emc_iterate (no P_out);
 * ws >= emc_workspace_bytes_rot_chunked(). */
EMC_API size_t emc_workspace_bytes_rot_chunked(int n, int n_pix, int n_rot, int n_rot_chunk, int n_pat);
EMC_API emc_status emc_iterate_rot_chunked(const emc_model *model, const emc_detector *det, const emc_rotations *rot,
                                   const emc_patterns *pat, int n_iter, int n_rot_chunk, float *model_out,
                                   double *loglik, unsigned flags, void *ws, size_t ws_bytes, void *stream,
                                   emc_context *ctx);

/* One iteration with the ROTATION list sharded over several GPUs, one process per GPU (the paper's decomposition:
 * PAPER.md:170, 188-194 Algorithm 2, 203; DESIGN.md section 11 NEXT-4).  Every rank holds the model, the detector, all
 * patterns and its own share of the rotations.  The library does the device work of a rank in three calls; the two
 * exchanges between them belong to the caller (paper_1409_4256_b200/parallel.py does them with torch.distributed):
 *   emc_shard_stats   Expand, log-likelihood and per-pattern statistics of the rank's rotations
 *                       -> stats_out [3][ld_n] floats (reference L, reference log w, sum; ld_n = N rounded up to 64)
 *   (all-gather of stats_out over the ranks -> stats_all [world][3][ld_n], in rank order)
 *   emc_shard_update  merges the ranks' statistics (the same result on every rank), then P, s[r], the update and the
 *                       Compress scatter of the rank's rotations -> numden_out [2][n^3] (numerator, denominator grids),
 *                       loglik (device double, the total log-likelihood, identical on every rank), s_out [R_local] or NULL
 *   (all-reduce(sum) of numden_out over the ranks)
 *   emc_shard_finish  model_out = num / den (division as the final step).
 * The workspace (emc_workspace_bytes for the rank's rotation count and all N patterns) carries L and the packed
 * patterns from emc_shard_stats to emc_shard_update: same ws, same stream, nothing else in between.  emc_shard_stats
 * stamps the workspace header with its sizes and emc_shard_update checks the stamp on the device: with a workspace that
 * does not come from a matching emc_shard_stats its results are NaN and emc_check returns EMC_ERR_WORKSPACE.
 * n_rot_total = R of the whole list (log(1/R) for weight == NULL).  world <= 64.  Poisson model, device patterns. */
EMC_API emc_status emc_shard_stats(const emc_model *model, const emc_detector *det, const emc_rotations *rot_local,
                           const emc_patterns *pat, int n_rot_total, float *stats_out, unsigned flags, void *ws,
                           size_t ws_bytes, void *stream);
EMC_API emc_status emc_shard_update(const emc_model *model, const emc_detector *det, const emc_rotations *rot_local,
                            const emc_patterns *pat, int n_rot_total, const float *stats_all, int world,
                            float *numden_out, double *loglik, float *s_out, unsigned flags, void *ws, size_t ws_bytes,
                            void *stream);
EMC_API emc_status emc_shard_finish(const float *numden, int n, float *model_out, void *stream);

/* Algorithm 1 with the paper's own likelihood: Gaussian around the slice with a fluence per (rotation, frame),
 * eqs. (2.2), (2.3), (2.5)/(2.11), (2.6), PAPER.md:70-89, 124-130 (NEXT-3, readings GA1-GA7):
 *   phi[r,d]  = sum_p K[d,p]^2 / sum_p W[r,p] K[d,p]                     (2.6), from the slices of this iteration
 *   Q[r,d]    = -sum_p (K[d,p] / phi[r,d] - W[r,p])^2 / (2 sigma^2)      (2.2)-(2.3)
 *   P         = the same normalisation over rotations as emc_normalize, with Q in the place of L
 *   Wnew[r,p] = sum_d P[r,d] K[d,p] / phi[r,d]  /  sum_d P[r,d]          (2.5)
 * over unmasked pixels, then Compress by eq. (2.12) with EMC_COMPRESS_WEIGHTED (what the paper runs) or (2.10).
 * With phi of (2.6), Q collapses to (B^2 / A_d - C_r) / (2 sigma^2), B = sum_p W K (one plane GEMM), A_d = sum_p K^2,
 * C_r = sum_p W^2; float32 evaluation of that form carries an absolute error of about 1e-7 C_r / (2 sigma^2).
 * Pattern chunks as in emc_iterate (the fluence and the E-step are per frame, so chunks are independent; s[r] and the
 * numerators add up), device-resident or host-resident patterns; slices must stay below 65504 (fp16 operand planes).
 * Arguments as emc_iterate; sigma > 0 in the units of the model. */
EMC_API emc_status emc_iterate_gaussian(const emc_model *model, const emc_detector *det, const emc_rotations *rot,
                                const emc_patterns *pat, int n_iter, int n_pat_chunk, float sigma, float *model_out,
                                float *P_out, int ld_n, double *loglik, unsigned flags, void *ws, size_t ws_bytes,
                                void *stream, emc_context *ctx);

/* The E-step of the Gaussian model as a stage of its own (eqs. 2.2, 2.3, 2.6):
 *   phi[r,d] = sum_p K[d,p]^2 / sum_p W[r,p] K[d,p],   Q[r,d] = -sum_p (K[d,p] / phi[r,d] - W[r,p])^2 / (2 sigma^2)
 * over unmasked pixels, evaluated in the collapsed form (B^2 / A_d - C_r) / (2 sigma^2) that emc_iterate_gaussian uses
 * (same kernels), so that the exponent itself can be checked, not only the responsibilities that come out of it.
 *   W [R][P] float in (as written by emc_expand);  Q, phi [R][ld_n] float out, either may be NULL. */
EMC_API emc_status emc_loglik_gaussian(const float *W, const emc_detector *det, const emc_patterns *pat, int n_rot,
                               float sigma, float *Q, float *phi, int ld_n, unsigned flags, void *ws, size_t ws_bytes,
                               void *stream);

/* Adaptive EMC, section 3.4 and eq. (3.1): `n_iter` iterations that start on the coarsest
 * rotation list levels[0] and move on to the next list after an iteration n >= 1 whose total log-likelihood
 * satisfies  |L^n - L^(n-1)| <= threshold |L^n|  (the paper: threshold = 0.01, and the lists are the
 * discretisations d, d+1, ... of eq. (2.7)); the last list is kept.  Each iteration is one emc_iterate().
 *   levels        HOST array of n_levels rotation lists (their quat / weight arrays are device pointers)
 *   model_out     [n^3] float, out: the model after the last iteration
 *   model_tmp     [n^3] float scratch (the iterations alternate between the two; neither may alias model->model)
 *   loglik        [n_iter] device doubles, out
 *   level_of_iter HOST [n_iter] int32, out: index of the list iteration n ran on
 *   ws            sized for the largest list.
 * The criterion is evaluated on the host in float64 from the device's log-likelihood, so this call synchronises
 * `stream` once per iteration (the paper's master node does the same). */
EMC_API emc_status emc_refine(const emc_model *model, const emc_detector *det, const emc_rotations *levels,
                      int n_levels, const emc_patterns *pat, int n_iter, double threshold, int n_pat_chunk,
                      float *model_out, float *model_tmp, double *loglik, int32_t *level_of_iter,
                      unsigned flags, void *ws, size_t ws_bytes, void *stream, emc_context *ctx);

/* Synchronises `stream` and reports what only the device saw during calls that used `ws`:
 * EMC_ERR_COUNT_RANGE if an unmasked count exceeded EMC_MAX_COUNT (the results of that call are NaN),
 * EMC_ERR_VALUE_RANGE if a slice of the Gaussian model left the fp16 range (its results hold inf / NaN),
 * EMC_ERR_WORKSPACE if emc_shard_update found a workspace that no matching emc_shard_stats had prepared (results NaN),
 * EMC_ERR_CUDA if the stream is in error.  Reads and clears the record on `stream` itself. */
EMC_API emc_status emc_check(void *ws, void *stream);

/* Stages timed under EMC_PROFILE_STAGES (at most EMC_MAX_SPANS spans between reads; later ones are dropped). */
#define EMC_MAX_SPANS 4096
enum { EMC_STAGE_EXPAND = 0, EMC_STAGE_PACK = 1, EMC_STAGE_LOGLIK = 2, EMC_STAGE_NORMALIZE = 3,
       EMC_STAGE_UPDATE = 4, EMC_STAGE_COMPRESS = 5, EMC_N_STAGES = 6 };
/* Waits for the recorded events, returns per stage the summed device time in milliseconds (HOST
 * array ms[EMC_N_STAGES]) and the number of spans (HOST array spans[EMC_N_STAGES]), and resets. */
EMC_API emc_status emc_profile_read(emc_context *ctx, double *ms, int *spans);
/* Spans that found the pool of EMC_MAX_SPANS event pairs exhausted since the last call of this function (their time is
 * missing from emc_profile_read's sums: read more often, e.g. once per emc_iterate_rot_chunked iteration); resets the count. */
EMC_API int emc_profile_dropped(emc_context *ctx);

/* Number of kernels this library has launched in this process (for bench.py's gpu_launches). */
EMC_API uint64_t emc_launch_count(void);

EMC_API const char *emc_strerror(emc_status status);
EMC_API const char *emc_last_cuda_error(void); /* text of the last CUDA failure seen by this thread */
EMC_API const char *emc_version(void);

#ifdef __cplusplus
}
#endif
#endif /* EMC_H_ */
