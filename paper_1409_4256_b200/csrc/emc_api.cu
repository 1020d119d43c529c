// The C ABI of libemc (include/emc.h): argument validation, workspace carving and the stage order
// of Algorithm 1.  All device work is in the launch_* functions of the other
// translation units; nothing here touches the data.
#include <atomic>
#include <cstdio>
#include <cstring>
#include <cmath>
#include <new>

#include "emc_internal.cuh"

namespace emc {

static thread_local char g_err[512] = "";
static std::atomic<uint64_t> g_launches{0};

emc_status cuda_fail(cudaError_t e, const char *what) {
    snprintf(g_err, sizeof(g_err), "%s: %s (%s)", what, cudaGetErrorName(e), cudaGetErrorString(e));
    return EMC_ERR_CUDA;
}
void note_launch(int n) { g_launches.fetch_add((uint64_t)n, std::memory_order_relaxed); }

float log_uniform_of(int n_rot) { return -logf((float)n_rot); }

}  // namespace emc

// The caller-created CUDA objects (emc.h): a copy stream with its events for host-resident patterns (chunks cross
// PCIe into two staging buffers, so that the copy of chunk j + 1 overlaps pack + GEMMs of chunk j) and a pool of event
// pairs for per-stage timing.  Everything is created in emc_context_create(); no call on the hot path creates anything.
struct emc_context {
    cudaStream_t copy_stream = nullptr;
    cudaEvent_t ready[2] = {nullptr, nullptr}, freed[2] = {nullptr, nullptr}, entry = nullptr;
    cudaEvent_t beg[EMC_MAX_SPANS], end[EMC_MAX_SPANS];
    int stage[EMC_MAX_SPANS];
    int created = 0, used = 0, dropped = 0;
};

namespace emc {
namespace {

// records the context's next event pair around a stage (EMC_PROFILE_STAGES)
struct Span {
    emc_context *c = nullptr;
    int slot = -1;
    cudaStream_t st;
    Span(emc_context *ctx, bool on, int stage, cudaStream_t stream) : st(stream) {
        if (!on || !ctx) return;
        if (ctx->used >= ctx->created) { ++ctx->dropped; return; }   // emc_profile_dropped()
        c = ctx;
        slot = c->used++;
        c->stage[slot] = stage;
        cudaEventRecord(c->beg[slot], st);
    }
    ~Span() {
        if (slot >= 0) cudaEventRecord(c->end[slot], st);
    }
};

size_t count_size(emc_count_type t) { return t == EMC_I32 ? 4 : (t == EMC_U16 ? 2 : 1); }

// One layout serves every entry point; a call uses the parts it needs.
struct Layout {
    WsHeader *hdr;
    __half *planesL;          // [2][R][ld_p]  logW hi / lo
    float *S;                 // [R]           sum_{p:mask} W
    __half *Kc;               // [Nc][ld_p]    counts, row = pattern
    __half *KT;               // [P][ld_n]     counts, row = pixel
    float *L;                 // [R][ld_n]
    __half *planesP;          // [2][R][ld_n]  fp16 hi / lo of chunk-scaled P
    float *pscale;            // [ld_n/512][R] inverse chunk scales of planesP
    float *s;                 // [R]
    float *Wnum;              // [R][P]        update numerators -> W'
    float2 *acc;              // [8 G]         one 64-byte (num, den) corner block per base corner (Compress)
    float *blocked;           // [8 G]         one 32-byte corner block of the model per base corner (Expand)
    float4 *geom;             // [P + 3 R]     packed pixel geometry and rotation matrices (launch_geometry)
    float *scratch;           // normalise partials
    float *Asq;               // [2][ld_n]     1 / (2 sigma^2 A_d) and 1 / A_d, A_d = sum_p K^2 (Gaussian model)
    uint32_t *active;         // [R/32 + 1]    slices den was accumulated for (+ the device flag), Compress
    void *stage;              // two chunks of raw counts (patterns on host, double-buffered)
    // photon-list path (EMC_SPARSE_PHOTONS): everything with the rotations along the rows (pitch ld_r)
    float *logWT;             // [P][ld_r]     log W transposed
    float *LT;                // [Nc][ld_r]    L transposed, then P transposed
    float *WT;                // [P][ld_r]     update numerators transposed
    float *logw;              // [ld_r]        log of the prior weights
    int *list_pat, *list_pix; // photon lists by frame and by pixel (sparse_list_ints)
    int ld_p, ld_n, ld_r;
    size_t total;
};

Layout carve(void *ws, int n, int n_pix, int n_rot, int n_chunk, size_t stage_bytes, bool sparse = false) {
    Layout l;
    l.ld_p = (int)round_up((size_t)n_pix, 64);
    l.ld_n = (int)round_up((size_t)n_chunk, 64);
    Arena a(ws, (size_t)-1);
    const size_t R = (size_t)n_rot;
    l.hdr = a.take<WsHeader>(1);
    l.planesL = a.take<__half>(2 * R * l.ld_p);
    l.S = a.take<float>(R);
    l.Kc = a.take<__half>((size_t)n_chunk * l.ld_p);
    l.KT = a.take<__half>((size_t)n_pix * l.ld_n);
    l.L = a.take<float>(R * l.ld_n);
    l.planesP = a.take<__half>(2 * R * l.ld_n);
    l.pscale = a.take<float>((size_t)ceil_div(l.ld_n, 512) * R);
    l.s = a.take<float>(R);
    l.Wnum = a.take<float>(R * n_pix);
    l.acc = a.take<float2>(compress_scratch_float2(n));
    l.blocked = a.take<float>(expand_scratch_floats(n, n_pix, n_rot));
    l.geom = a.take<float4>(geometry_float4(n_pix, n_rot));
    l.scratch = a.take<float>(normalize_scratch_floats(n_rot, l.ld_n));
    l.Asq = a.take<float>((size_t)2 * l.ld_n);
    l.active = a.take<uint32_t>((size_t)ceil_div(n_rot, 32) + 1);
    l.stage = a.take<uint8_t>(stage_bytes);
    l.ld_r = (int)round_up((size_t)n_rot, 32);
    if (sparse) {
        const size_t cap = (size_t)n_chunk * n_pix;             // every count non-zero: the lists cannot overflow
        l.logWT = a.take<float>((size_t)n_pix * l.ld_r);
        l.LT = a.take<float>((size_t)n_chunk * l.ld_r);
        l.WT = a.take<float>((size_t)n_pix * l.ld_r);
        l.logw = a.take<float>((size_t)l.ld_r);
        l.list_pat = a.take<int>(sparse_list_ints(n_chunk, cap));
        l.list_pix = a.take<int>(sparse_list_ints(n_pix, cap));
    } else {
        l.logWT = l.LT = l.WT = l.logw = nullptr;
        l.list_pat = l.list_pix = nullptr;
    }
    l.total = a.off;
    return l;
}

bool sizes_ok(int n, int n_pix, int n_rot, int n_pat) {
    return n >= 2 && n <= 1024 && n_pix > 0 && n_rot > 0 && n_pat > 0 && (size_t)n_pix * 8 < (size_t)1 << 31;
}

emc_status check_ws(void *ws, size_t ws_bytes, size_t need) {
    if (!ws || ((uintptr_t)ws & 255)) return EMC_ERR_WORKSPACE;
    if (ws_bytes < need) return EMC_ERR_WORKSPACE;
    return EMC_OK;
}

bool det_ok(const emc_detector *d) {
    return d && d->n_pix > 0 && d->q && d->row_len >= 0 && (d->row_len == 0 || d->n_pix % d->row_len == 0);
}
bool rot_ok(const emc_rotations *r) { return r && r->n_rot > 0 && r->quat; }
bool pat_ok(const emc_patterns *p) {
    return p && p->n_pat > 0 && p->counts && (p->type == EMC_I32 || p->type == EMC_U16 || p->type == EMC_U8);
}

emc_status reset_header(const Layout &l, cudaStream_t st) {
    EMC_TRY_CUDA(cudaMemsetAsync(l.hdr, 0, sizeof(WsHeader), st));
    return EMC_OK;
}

// stats_ready (optional): the normalisation's column statistics go into l.scratch in the same pass, where the
// kernel that runs supports it (weight = prior weights or null; log_uniform = log w of every row in that case)
emc_status run_loglik_gemm(const Layout &l, int n_rot, int n_pix, int n_pat, float *L, int ld_out,
                           unsigned flags, cudaStream_t st, const float *weight = nullptr, float log_uniform = 0.f,
                           bool *stats_ready = nullptr, const GaussTerms *gauss = nullptr, int layout_rot = 0) {
    GemmProblem g;
    g.A = l.planesL; g.B = l.Kc; g.n_planes = 2;
    g.M = n_rot; g.N = n_pat; g.K = n_pix;
    g.lda = l.ld_p; g.ldb = l.ld_p; g.plane_stride = (size_t)n_rot * l.ld_p;
    g.a_fmt = FMT_F16; g.b_fmt = FMT_F16;
    g.out = L; g.ld_out = ld_out; g.rowv = l.S; g.epilogue = gauss ? EPI_GAUSS : EPI_SUB_ROW;
    if (gauss) { g.gauss_g = gauss->g_col; g.inv2s2 = gauss->inv2s2; }
    // accumulation chunks of 1024 pixels for the Poisson log-likelihood (no per-chunk scales here): the tensor core gets
    // twice the run-ahead over the end-of-tile phase and half the drains; measured on C2: max |dL|/A 7.6e-7 (4.6e-7 at
    // 512), signed mean +2.6e-7, tolerance 1e-5.  The Gaussian B keeps 512: its error is amplified by cancellation.
    if (!gauss) g.k_chunk = 16;
    g.one_cta = (flags & EMC_GEMM_1CTA) != 0;
    const bool simt = (flags & EMC_DEBUG_SIMT) != 0;
    if (stats_ready) {
        const size_t rows = (size_t)normalize_stat_rows(layout_rot > 0 ? layout_rot : n_rot);
        g.stat_m = l.scratch;
        g.stat_w = l.scratch + rows * l.ld_n;
        g.stat_z = l.scratch + 2 * rows * l.ld_n;
        g.ld_stat = l.ld_n;
        g.weight = weight;
        g.log_uniform = log_uniform;
        *stats_ready = ld_out == l.ld_n && gemm_fuses_stats(g, simt);
        if (!*stats_ready) g.stat_m = g.stat_w = g.stat_z = nullptr;
    }
    return launch_plane_gemm(g, simt, st);
}

emc_status run_update_gemm(const Layout &l, int n_rot, int n_pix, int n_pat, float *out, const float *s, int epilogue,
                           unsigned flags, cudaStream_t st) {
    GemmProblem g;
    g.A = l.planesP; g.B = l.KT; g.n_planes = 2;
    g.M = n_rot; g.N = n_pix; g.K = n_pat;
    g.lda = l.ld_n; g.ldb = l.ld_n; g.plane_stride = (size_t)n_rot * l.ld_n;
    g.a_fmt = g.b_fmt = FMT_F16;
    g.chunk_scale = l.pscale;
    g.out = out; g.ld_out = n_pix; g.rowv = s; g.epilogue = epilogue;
    g.one_cta = (flags & EMC_GEMM_1CTA) != 0;
    return launch_plane_gemm(g, (flags & EMC_DEBUG_SIMT) != 0, st);
}

}  // namespace
}  // namespace emc

using namespace emc;

extern "C" {

emc_status emc_context_create(emc_context **out) {
    if (!out) return EMC_ERR_ARG;
    *out = nullptr;
    emc_context *c = new (std::nothrow) emc_context;
    if (!c) return EMC_ERR_ARG;
    auto fail = [&](cudaError_t e, const char *what) {
        emc_context_destroy(c);
        return cuda_fail(e, what);
    };
    cudaError_t e = cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking);
    if (e != cudaSuccess) return fail(e, "cudaStreamCreateWithFlags");
    cudaEvent_t *plain[5] = {&c->ready[0], &c->ready[1], &c->freed[0], &c->freed[1], &c->entry};
    for (cudaEvent_t *ev : plain)
        if ((e = cudaEventCreateWithFlags(ev, cudaEventDisableTiming)) != cudaSuccess) return fail(e, "cudaEventCreateWithFlags");
    for (int i = 0; i < EMC_MAX_SPANS; ++i) {
        if ((e = cudaEventCreate(&c->beg[i])) != cudaSuccess) return fail(e, "cudaEventCreate");
        if ((e = cudaEventCreate(&c->end[i])) != cudaSuccess) { cudaEventDestroy(c->beg[i]); return fail(e, "cudaEventCreate"); }
        c->created = i + 1;
    }
    *out = c;
    return EMC_OK;
}

emc_status emc_context_destroy(emc_context *c) {
    if (!c) return EMC_OK;
    for (int i = 0; i < c->created; ++i) { cudaEventDestroy(c->beg[i]); cudaEventDestroy(c->end[i]); }
    cudaEvent_t plain[5] = {c->ready[0], c->ready[1], c->freed[0], c->freed[1], c->entry};
    for (cudaEvent_t ev : plain)
        if (ev) cudaEventDestroy(ev);
    if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
    delete c;
    return EMC_OK;
}

size_t emc_workspace_bytes(int n, int n_pix, int n_rot, int n_pat_chunk, unsigned flags) {
    if (!sizes_ok(n, n_pix, n_rot, n_pat_chunk)) return 0;
    if ((flags & EMC_SPARSE_PHOTONS) && (n_pix >= (1 << 20) || n_pat_chunk >= (1 << 20) || (size_t)n_pat_chunk * n_pix >= ((size_t)1 << 31)))
        return 0;                                               // what emc_iterate refuses for the photon-list path
    const size_t stage = (flags & EMC_PATTERNS_ON_HOST) ? 2 * round_up((size_t)n_pat_chunk * n_pix * 4, 1024) : 0;
    return carve(nullptr, n, n_pix, n_rot, n_pat_chunk, stage, (flags & EMC_SPARSE_PHOTONS) != 0).total;
}

size_t emc_workspace_bytes_geometry(int n, int n_pix, int n_rot) {
    if (!sizes_ok(n, n_pix, n_rot, 1)) return 0;
    size_t blocks = round_up(sizeof(float2) * compress_scratch_float2(n), 1024);
    const size_t eb = round_up(sizeof(float) * expand_scratch_floats(n, n_pix, n_rot), 1024);
    if (eb > blocks) blocks = eb;
    return blocks + round_up(sizeof(float4) * geometry_float4(n_pix, n_rot), 1024);
}

emc_status emc_expand(const emc_model *model, const emc_detector *det, const emc_rotations *rot,
                      float *W, int32_t *idx, void *ws, size_t ws_bytes, void *stream) {
    if (!model || !model->model || !det_ok(det) || !rot_ok(rot) || (!W && !idx)) return EMC_ERR_ARG;
    if (!sizes_ok(model->n, det->n_pix, rot->n_rot, 1)) return EMC_ERR_UNSUPPORTED;
    float *blocked = nullptr;
    Geometry geo;
    if (ws) {
        const size_t b_bytes = round_up(sizeof(float) * expand_scratch_floats(model->n, det->n_pix, rot->n_rot), 1024);
        EMC_TRY(check_ws(ws, ws_bytes, b_bytes + sizeof(float4) * geometry_float4(det->n_pix, rot->n_rot)));
        blocked = (float *)ws;
        EMC_TRY(launch_geometry(det->q, det->mask, det->n_pix, det->row_len, rot->quat, rot->n_rot,
                                (float4 *)((uint8_t *)ws + b_bytes), &geo, (cudaStream_t)stream));
    }
    return launch_expand(model->model, model->n, det->q, det->mask, det->n_pix, rot->quat, rot->n_rot, W, idx,
                         nullptr, 0, nullptr, blocked, blocked ? &geo : nullptr, (cudaStream_t)stream);
}

emc_status emc_loglik(const float *W, const int32_t *idx, const emc_detector *det,
                      const emc_patterns *pat, int n_rot, float *L, int ld_n, unsigned flags,
                      void *ws, size_t ws_bytes, void *stream) {
    if (!W || !det_ok(det) || !pat_ok(pat) || n_rot <= 0 || !L || ld_n < pat->n_pat || (ld_n & 3) ||
        ((uintptr_t)L & 15))
        return EMC_ERR_ARG;
    if (!sizes_ok(2, det->n_pix, n_rot, pat->n_pat)) return EMC_ERR_UNSUPPORTED;
    cudaStream_t st = (cudaStream_t)stream;
    EMC_TRY(check_ws(ws, ws_bytes, carve(nullptr, 0, det->n_pix, n_rot, pat->n_pat, 0).total));
    const Layout l = carve(ws, 0, det->n_pix, n_rot, pat->n_pat, 0);
    EMC_TRY(reset_header(l, st));
    EMC_TRY_CUDA(cudaMemsetAsync(l.S, 0, sizeof(float) * n_rot, st));
    EMC_TRY(launch_logw_split(W, idx, det->mask, det->n_pix, n_rot, l.planesL, l.ld_p, l.S, st));
    EMC_TRY(launch_pack(pat->counts, pat->type, pat->n_pat, det->n_pix, det->mask, l.Kc, l.ld_p, nullptr, 0, l.hdr, st));
    EMC_TRY(run_loglik_gemm(l, n_rot, det->n_pix, pat->n_pat, L, ld_n, flags, st));
    return launch_poison(l.hdr, L, (size_t)n_rot * ld_n, nullptr, 0, st);
}

emc_status emc_loglik_gaussian(const float *W, const emc_detector *det, const emc_patterns *pat, int n_rot,
                               float sigma, float *Q, float *phi, int ld_n, unsigned flags, void *ws, size_t ws_bytes,
                               void *stream) {
    if (!W || !det_ok(det) || !pat_ok(pat) || n_rot <= 0 || (!Q && !phi) || ld_n < pat->n_pat || !(sigma > 0.f)) return EMC_ERR_ARG;
    if (!sizes_ok(2, det->n_pix, n_rot, pat->n_pat)) return EMC_ERR_UNSUPPORTED;
    cudaStream_t st = (cudaStream_t)stream;
    EMC_TRY(check_ws(ws, ws_bytes, carve(nullptr, 0, det->n_pix, n_rot, pat->n_pat, 0).total));
    const Layout l = carve(ws, 0, det->n_pix, n_rot, pat->n_pat, 0);
    const float inv2s2 = 1.f / (2.f * sigma * sigma);
    EMC_TRY(reset_header(l, st));
    EMC_TRY_CUDA(cudaMemsetAsync(l.S, 0, sizeof(float) * n_rot, st));
    EMC_TRY(launch_logw_split(W, nullptr, det->mask, det->n_pix, n_rot, l.planesL, l.ld_p, l.S, st, true));   // planes of W, C_r
    EMC_TRY(launch_pack(pat->counts, pat->type, pat->n_pat, det->n_pix, det->mask, l.Kc, l.ld_p, nullptr, 0, l.hdr, st));
    EMC_TRY_CUDA(cudaMemsetAsync(l.Asq, 0, sizeof(float) * 2 * l.ld_n, st));
    EMC_TRY(launch_rowsq(l.Kc, pat->n_pat, det->n_pix, l.ld_p, inv2s2, l.Asq, l.Asq + l.ld_n, st));
    GemmProblem g;                                              // B = W K^T, the same plane GEMM, no epilogue
    g.A = l.planesL; g.B = l.Kc; g.n_planes = 2;
    g.M = n_rot; g.N = pat->n_pat; g.K = det->n_pix;
    g.lda = l.ld_p; g.ldb = l.ld_p; g.plane_stride = (size_t)n_rot * l.ld_p;
    g.a_fmt = g.b_fmt = FMT_F16;
    g.out = l.L; g.ld_out = l.ld_n; g.rowv = nullptr; g.epilogue = EPI_STORE;
    g.one_cta = (flags & EMC_GEMM_1CTA) != 0;
    EMC_TRY(launch_plane_gemm(g, (flags & EMC_DEBUG_SIMT) != 0, st));
    EMC_TRY(launch_gauss_q(l.L, l.S, l.Asq, l.Asq + l.ld_n, inv2s2, n_rot, pat->n_pat, l.ld_n, Q, phi, ld_n, st));
    if (Q) EMC_TRY(launch_poison(l.hdr, Q, (size_t)n_rot * ld_n, nullptr, 0, st));
    if (phi) EMC_TRY(launch_poison(l.hdr, phi, (size_t)n_rot * ld_n, nullptr, 0, st));
    return EMC_OK;
}

emc_status emc_normalize(const float *L, const emc_rotations *rot, int n_pat, int ld_n, float *P,
                         float *s, double *loglik, unsigned flags, void *ws, size_t ws_bytes,
                         void *stream) {
    if (!L || !rot || rot->n_rot <= 0 || n_pat <= 0 || ld_n < n_pat || !P || (ld_n & 3) || ((uintptr_t)L & 15) ||
        ((uintptr_t)P & 15))
        return EMC_ERR_ARG;
    const size_t need = round_up(sizeof(float) * normalize_scratch_floats(rot->n_rot, ld_n), 1024);
    EMC_TRY(check_ws(ws, ws_bytes, need));
    return launch_normalize(L, rot->weight, rot->n_rot, n_pat, ld_n, P, nullptr, 0, nullptr, s, loglik,
                            (flags & EMC_ACCUMULATE) != 0, (float *)ws, false, (cudaStream_t)stream);
}

emc_status emc_update(const float *P, int ld_n, const float *s, const emc_detector *det,
                      const emc_patterns *pat, int n_rot, float *Wnew, unsigned flags, void *ws,
                      size_t ws_bytes, void *stream) {
    const bool raw = (flags & (EMC_UPDATE_RAW | EMC_ACCUMULATE)) != 0;
    if (!P || !det_ok(det) || !pat_ok(pat) || n_rot <= 0 || !Wnew || ld_n < pat->n_pat || (!raw && !s))
        return EMC_ERR_ARG;
    if (!sizes_ok(2, det->n_pix, n_rot, pat->n_pat)) return EMC_ERR_UNSUPPORTED;
    cudaStream_t st = (cudaStream_t)stream;
    EMC_TRY(check_ws(ws, ws_bytes, carve(nullptr, 0, det->n_pix, n_rot, pat->n_pat, 0).total));
    const Layout l = carve(ws, 0, det->n_pix, n_rot, pat->n_pat, 0);
    EMC_TRY(reset_header(l, st));
    EMC_TRY(launch_p_split(P, n_rot, pat->n_pat, ld_n, l.planesP, l.ld_n, (size_t)n_rot * l.ld_n, l.pscale, st));
    EMC_TRY(launch_pack(pat->counts, pat->type, pat->n_pat, det->n_pix, det->mask, nullptr, 0, l.KT, l.ld_n, l.hdr, st));
    const int epi = (flags & EMC_ACCUMULATE) ? EPI_ADD : (raw ? EPI_STORE : EPI_DIV_ROW);
    EMC_TRY(run_update_gemm(l, n_rot, det->n_pix, pat->n_pat, Wnew, s, epi, flags, st));
    return launch_poison(l.hdr, Wnew, (size_t)n_rot * det->n_pix, nullptr, 0, st);
}

emc_status emc_compress(const float *Wnew, const float *slice_w, const emc_detector *det,
                        const emc_rotations *rot, int n, float *model_out, float *den_out,
                        unsigned flags, void *ws, size_t ws_bytes, void *stream) {
    if (!Wnew || !det_ok(det) || !rot_ok(rot) || !model_out) return EMC_ERR_ARG;
    if (!sizes_ok(n, det->n_pix, rot->n_rot, 1)) return EMC_ERR_UNSUPPORTED;
    const size_t a_bytes = round_up(sizeof(float2) * compress_scratch_float2(n), 1024);
    EMC_TRY(check_ws(ws, ws_bytes, a_bytes + sizeof(float4) * geometry_float4(det->n_pix, rot->n_rot)));
    Geometry geo;
    EMC_TRY(launch_geometry(det->q, det->mask, det->n_pix, det->row_len, rot->quat, rot->n_rot,
                            (float4 *)((uint8_t *)ws + a_bytes), &geo, (cudaStream_t)stream));
    return launch_compress(Wnew, slice_w, (flags & EMC_COMPRESS_WEIGHTED) != 0, geo, n, (float2 *)ws, model_out, den_out,
                           (cudaStream_t)stream);
}

// Algorithm 1 for both likelihood models; sigma > 0 selects the paper's Gaussian model (section 11 of DESIGN.md)
static emc_status iterate_impl(const emc_model *model, const emc_detector *det, const emc_rotations *rot,
                               const emc_patterns *pat, int n_iter, int n_pat_chunk, float *model_out,
                               float *P_out, int ld_n, double *loglik, unsigned flags, void *ws,
                               size_t ws_bytes, void *stream, emc_context *ctx, float sigma) {
    const bool gauss = sigma > 0.f;
    if (!model || !model->model || !det_ok(det) || !rot_ok(rot) || !pat_ok(pat) || n_iter <= 0 || !model_out ||
        model_out == model->model || !loglik || n_pat_chunk < 0)
        return EMC_ERR_ARG;
    if ((flags & (EMC_PATTERNS_ON_HOST | EMC_PROFILE_STAGES)) && !ctx) return EMC_ERR_ARG;
    if (n_iter > 256) return EMC_ERR_UNSUPPORTED;
    const int n = model->n, n_pix = det->n_pix, n_rot = rot->n_rot, n_pat = pat->n_pat;
    const int chunk = (n_pat_chunk == 0 || n_pat_chunk > n_pat) ? n_pat : n_pat_chunk;
    if (!sizes_ok(n, n_pix, n_rot, chunk)) return EMC_ERR_UNSUPPORTED;
    const int n_chunks = ceil_div(n_pat, chunk);
    const bool on_host = (flags & EMC_PATTERNS_ON_HOST) != 0;
    const size_t csz = count_size(pat->type);
    const size_t stage_one = round_up((size_t)chunk * n_pix * 4, 1024);          // one staging buffer (4 B per count at most)
    const size_t stage_bytes = on_host ? 2 * stage_one : 0;
    const bool sparse = (flags & EMC_SPARSE_PHOTONS) != 0;
    // photon lists: 20-bit column indices, and 32-bit offsets into lists sized for a chunk in which every count is non-zero
    if (sparse && (gauss || n_pix >= (1 << 20) || chunk >= (1 << 20) || (size_t)chunk * n_pix >= ((size_t)1 << 31) ||
                   (flags & (EMC_GEMM_1CTA | EMC_DEBUG_SIMT))))
        return EMC_ERR_UNSUPPORTED;
    EMC_TRY(check_ws(ws, ws_bytes, carve(nullptr, n, n_pix, n_rot, chunk, stage_bytes, sparse).total));
    const Layout l = carve(ws, n, n_pix, n_rot, chunk, stage_bytes, sparse);
    if (P_out && (n_chunks != 1 || ld_n != l.ld_n)) return EMC_ERR_ARG;
    if (gauss && (flags & (EMC_GEMM_1CTA | EMC_DEBUG_SIMT))) return EMC_ERR_UNSUPPORTED;
    const float log_uniform = log_uniform_of(n_rot);
    const GaussTerms gterms = {l.S, l.Asq, l.Asq + l.ld_n, gauss ? 1.f / (2.f * sigma * sigma) : 0.f, log_uniform};
    const GaussTerms *gt = gauss ? &gterms : nullptr;
    cudaStream_t st = (cudaStream_t)stream;
    const bool weighted = (flags & EMC_COMPRESS_WEIGHTED) != 0;
    const bool prof = (flags & EMC_PROFILE_STAGES) != 0;

    EMC_TRY(reset_header(l, st));
    // Host-resident patterns in ONE resident chunk: the first iteration is run on sub-ranges of the chunk, so that the
    // copy of sub-range j + 1 crosses PCIe while sub-range j is packed (into its place in the full-size operands)
    // and goes through stages 2-4; later iterations use the resident operands in one piece.  Same arithmetic as
    // pattern chunks (G9).  Sub-ranges are multiples of 512 patterns (the update's K chunk and scale granularity).
    const bool pipelined = on_host && n_chunks == 1 && !gauss && !sparse && n_pat >= 4096;
    const int sub = pipelined ? (int)round_up((size_t)ceil_div(n_pat, 4), 512) : chunk;
    const int n_sub = pipelined ? ceil_div(n_pat, sub) : 1;
    // pack jobs in order: every (iteration, chunk) when there are several chunks, else the resident chunk once
    // (in n_sub pieces when pipelined)
    const int n_jobs = n_chunks > 1 ? n_iter * n_chunks : n_sub;
    auto job_range = [&](int j, int &d0, int &nc) {
        const int step = pipelined ? sub : chunk;
        d0 = (pipelined ? j : j % n_chunks) * step;
        nc = n_pat - d0 < step ? n_pat - d0 : step;
    };
    auto issue_copy = [&](int j) -> emc_status {              // host -> staging buffer j & 1, on the context's copy stream
        int d0, nc;
        job_range(j, d0, nc);
        const int b = j & 1;
        if (j >= 2) EMC_TRY_CUDA(cudaStreamWaitEvent(ctx->copy_stream, ctx->freed[b], 0));   // pack j - 2 has read it
        EMC_TRY_CUDA(cudaMemcpyAsync((uint8_t *)l.stage + b * stage_one, (const uint8_t *)pat->counts + (size_t)d0 * n_pix * csz,
                                     (size_t)nc * n_pix * csz, cudaMemcpyHostToDevice, ctx->copy_stream));
        EMC_TRY_CUDA(cudaEventRecord(ctx->ready[b], ctx->copy_stream));
        return EMC_OK;
    };
    if (on_host) {
        EMC_TRY_CUDA(cudaEventRecord(ctx->entry, st));        // earlier work on `st` may still read the staging buffers
        EMC_TRY_CUDA(cudaStreamWaitEvent(ctx->copy_stream, ctx->entry, 0));
        EMC_TRY(issue_copy(0));
    }
    int job = 0;
    SparseList by_frame = {nullptr, nullptr, 0}, by_pixel = {nullptr, nullptr, 0};
    const float *model_cur = model->model;
    Geometry geo;                                            // once per call: the rotation list is the same in every iteration
    EMC_TRY(launch_geometry(det->q, det->mask, n_pix, det->row_len, rot->quat, n_rot, l.geom, &geo, st));
    if (sparse && rot->weight) EMC_TRY(launch_logw(rot->weight, n_rot, l.logw, st));
    for (int it = 0; it < n_iter; ++it) {
        // stage 1: Expand, with logW planes and S fused in
        {
            Span sp(ctx, prof, EMC_STAGE_EXPAND, st);
            EMC_TRY_CUDA(cudaMemsetAsync(l.S, 0, sizeof(float) * n_rot, st));
            if (sparse) {
                // log W as float32 (into the W' buffer, free until the update), transposed: rotations along the rows
                EMC_TRY(launch_expand(model_cur, n, det->q, det->mask, n_pix, rot->quat, n_rot, l.Wnum, nullptr, nullptr, 0,
                                      l.S, l.blocked, &geo, st, false, true));
                EMC_TRY(launch_transpose(l.Wnum, n_rot, n_pix, n_pix, l.logWT, l.ld_r, st));
            } else {
                EMC_TRY(launch_expand(model_cur, n, det->q, det->mask, n_pix, rot->quat, n_rot, nullptr, nullptr,
                                      l.planesL, l.ld_p, l.S, l.blocked, &geo, st, gauss, false, gauss ? &l.hdr->w_range : nullptr));
            }
        }
        EMC_TRY_CUDA(cudaMemsetAsync(l.s, 0, sizeof(float) * n_rot, st));
        EMC_TRY_CUDA(cudaMemsetAsync(loglik + it, 0, sizeof(double), st));
        // the parts of this iteration: pattern chunks (each in the per-chunk buffers), or, in the pipelined first
        // iteration, sub-ranges of the one resident chunk (each at its offset in the full-size buffers)
        const bool sub_ranges = pipelined && it == 0;
        const int n_parts = sub_ranges ? n_sub : n_chunks;
        for (int c = 0; c < n_parts; ++c) {
            const int step = sub_ranges ? sub : chunk;
            const int d0 = c * step;
            const int nc = n_pat - d0 < step ? n_pat - d0 : step;
            Layout v = l;                               // view of the buffers this part works in
            if (sub_ranges) {
                v.Kc = l.Kc + (size_t)d0 * l.ld_p;
                v.KT = l.KT + d0;
                v.L = l.L + d0;
                v.planesP = l.planesP + d0;
                v.pscale = l.pscale + (size_t)(d0 / 512) * n_rot;
                v.scratch = l.scratch + d0;
            }
            if (n_chunks > 1 || it == 0) {          // one resident chunk is packed once for all iterations
                Span sp(ctx, prof, EMC_STAGE_PACK, st);
                const uint8_t *src = (const uint8_t *)pat->counts + (size_t)d0 * n_pix * csz;
                if (on_host) {
                    const int b = job & 1;
                    if (job + 1 < n_jobs) EMC_TRY(issue_copy(job + 1));      // overlaps this part's pack and GEMMs
                    EMC_TRY_CUDA(cudaStreamWaitEvent(st, ctx->ready[b], 0));
                    src = (const uint8_t *)l.stage + b * stage_one;
                }
                if (sparse)                         // photon lists by frame and by pixel, straight from the raw counts
                    EMC_TRY(launch_lists_raw(src, pat->type, nc, n_pix, det->mask, l.list_pat, l.list_pix, l.hdr, &by_frame, &by_pixel, st));
                else
                    EMC_TRY(launch_pack(src, pat->type, nc, n_pix, det->mask, v.Kc, l.ld_p, v.KT, l.ld_n, l.hdr, st));
                if (on_host) EMC_TRY_CUDA(cudaEventRecord(ctx->freed[job & 1], st));
                if (gauss) {                        // A_d = sum_p K^2, the numerators of the fluence (eq. 2.6)
                    EMC_TRY_CUDA(cudaMemsetAsync(l.Asq, 0, sizeof(float) * 2 * l.ld_n, st));
                    EMC_TRY(launch_rowsq(l.Kc, nc, n_pix, l.ld_p, gterms.inv2s2, l.Asq, l.Asq + l.ld_n, st));
                }
                ++job;
            }
            if (sparse) {
                // stages 2-4 from the photon lists, in the transposed world (emc_sparse.cu): L^T, P^T, W'^T
                {
                    Span sp(ctx, prof, EMC_STAGE_LOGLIK, st);
                    EMC_TRY(launch_spmm_rot(by_frame, l.logWT, l.LT, l.ld_r, n_rot, l.S, false, st));
                }
                {
                    Span sp(ctx, prof, EMC_STAGE_NORMALIZE, st);
                    EMC_TRY(launch_softmax_rows(l.LT, nc, n_rot, l.ld_r, rot->weight ? l.logw : nullptr, log_uniform, l.s, loglik + it, st));
                    if (P_out && it == n_iter - 1) EMC_TRY(launch_transpose(l.LT, nc, n_rot, l.ld_r, P_out, l.ld_n, st));
                }
                {
                    Span sp(ctx, prof, EMC_STAGE_UPDATE, st);
                    EMC_TRY(launch_spmm_rot(by_pixel, l.LT, l.WT, l.ld_r, n_rot, nullptr, c > 0, st));
                }
                continue;
            }
            // stage 2: L = logW K^T - S  (+ the column max / sum-exp partials of stage 3 from the same epilogue)
            bool stats_ready = false;
            {
                Span sp(ctx, prof, EMC_STAGE_LOGLIK, st);
                EMC_TRY(run_loglik_gemm(v, n_rot, n_pix, nc, v.L, l.ld_n, flags, st, rot->weight, log_uniform, &stats_ready, gt));
            }
            // stage 3: responsibilities of this part; s and LL add up over parts
            float *p_dst = (P_out && it == n_iter - 1) ? P_out + (sub_ranges ? d0 : 0) : nullptr;
            {
                Span sp(ctx, prof, EMC_STAGE_NORMALIZE, st);
                EMC_TRY(launch_normalize(v.L, rot->weight, n_rot, nc, l.ld_n, p_dst, v.planesP, (size_t)n_rot * l.ld_n, v.pscale,
                                         l.s, loglik + it, true, v.scratch, stats_ready, st, gt,
                                         l.ld_n - (sub_ranges ? d0 : 0), log_uniform));
            }
            // stage 4: update numerators (divided by s[r] in the epilogue when there is one part)
            const int epi = n_parts == 1 ? EPI_DIV_ROW : (c == 0 ? EPI_STORE : EPI_ADD);
            {
                Span sp(ctx, prof, EMC_STAGE_UPDATE, st);
                EMC_TRY(run_update_gemm(v, n_rot, n_pix, nc, l.Wnum, l.s, epi, flags, st));
            }
        }
        if (sparse) {
            Span sp(ctx, prof, EMC_STAGE_UPDATE, st);
            EMC_TRY(launch_transpose_div(l.WT, n_pix, n_rot, l.ld_r, l.Wnum, l.s, st));      // W' = numerator / s[r] (eq. 2.5)
        } else if (n_parts > 1) {
            Span sp(ctx, prof, EMC_STAGE_UPDATE, st);
            EMC_TRY(launch_div_rows(l.Wnum, l.s, n_rot, n_pix, st));
        }
        // stage 5: Compress
        {
            Span sp(ctx, prof, EMC_STAGE_COMPRESS, st);
            const DenCache cache = {l.active, (int *)(l.active + ceil_div(n_rot, 32)), it == 0};
            EMC_TRY(launch_compress(l.Wnum, l.s, weighted, geo, n, l.acc, model_out, nullptr, st, &cache));
        }
        model_cur = model_out;
    }
    // a count out of range (seen by the pack kernels above): every result of the call becomes NaN
    EMC_TRY(launch_poison(l.hdr, model_out, (size_t)n * n * n, loglik, n_iter, st));
    if (P_out) EMC_TRY(launch_poison(l.hdr, P_out, (size_t)n_rot * ld_n, nullptr, 0, st));
    return EMC_OK;
}

emc_status emc_iterate(const emc_model *model, const emc_detector *det, const emc_rotations *rot,
                       const emc_patterns *pat, int n_iter, int n_pat_chunk, float *model_out,
                       float *P_out, int ld_n, double *loglik, unsigned flags, void *ws,
                       size_t ws_bytes, void *stream, emc_context *ctx) {
    return iterate_impl(model, det, rot, pat, n_iter, n_pat_chunk, model_out, P_out, ld_n, loglik, flags, ws, ws_bytes,
                        stream, ctx, 0.f);
}

emc_status emc_workspace_view(void *ws, int n, int n_pix, int n_rot, int n_pat_chunk, unsigned flags, int what, void **ptr,
                              int *ld) {
    if (!ws || ((uintptr_t)ws & 255) || !ptr || !ld) return EMC_ERR_ARG;
    if (!sizes_ok(n, n_pix, n_rot, n_pat_chunk)) return EMC_ERR_UNSUPPORTED;
    const bool sparse = (flags & EMC_SPARSE_PHOTONS) != 0;
    const size_t stage = (flags & EMC_PATTERNS_ON_HOST) ? 2 * round_up((size_t)n_pat_chunk * n_pix * 4, 1024) : 0;
    const Layout l = carve(ws, n, n_pix, n_rot, n_pat_chunk, stage, sparse);      // the layout iterate_impl uses
    switch (what) {
        case EMC_VIEW_LOGLIK:
            if (sparse) return EMC_ERR_UNSUPPORTED;                                // the photon-list path forms L^T only
            *ptr = l.L; *ld = l.ld_n;
            return EMC_OK;
        case EMC_VIEW_S: *ptr = l.s; *ld = 0; return EMC_OK;
        case EMC_VIEW_WNEW: *ptr = l.Wnum; *ld = n_pix; return EMC_OK;
    }
    return EMC_ERR_ARG;
}

// Rotation chunks: the per-chunk buffers of carve() at R = chunk size, then s for the whole list
static size_t rot_chunked_extra(int n_rot) { return round_up(sizeof(float) * (size_t)n_rot, 1024); }

size_t emc_workspace_bytes_rot_chunked(int n, int n_pix, int n_rot, int n_rot_chunk, int n_pat) {
    if (!sizes_ok(n, n_pix, n_rot, n_pat) || n_rot_chunk <= 0) return 0;
    const int rc = n_rot_chunk < n_rot ? n_rot_chunk : n_rot;
    return carve(nullptr, n, n_pix, rc, n_pat, 0).total + rot_chunked_extra(n_rot);
}

emc_status emc_iterate_rot_chunked(const emc_model *model, const emc_detector *det, const emc_rotations *rot,
                                   const emc_patterns *pat, int n_iter, int n_rot_chunk, float *model_out,
                                   double *loglik, unsigned flags, void *ws, size_t ws_bytes, void *stream,
                                   emc_context *ctx) {
    if (!model || !model->model || !det_ok(det) || !rot_ok(rot) || !pat_ok(pat) || n_iter <= 0 || !model_out ||
        model_out == model->model || !loglik || n_rot_chunk <= 0)
        return EMC_ERR_ARG;
    if (flags & (EMC_PATTERNS_ON_HOST | EMC_SPARSE_PHOTONS)) return EMC_ERR_UNSUPPORTED;   // dense, device-resident only
    if ((flags & EMC_PROFILE_STAGES) && !ctx) return EMC_ERR_ARG;
    if (n_iter > 256) return EMC_ERR_UNSUPPORTED;
    const int n = model->n, n_pix = det->n_pix, n_rot = rot->n_rot, n_pat = pat->n_pat;
    if (!sizes_ok(n, n_pix, n_rot, n_pat)) return EMC_ERR_UNSUPPORTED;
    const int rc = n_rot_chunk < n_rot ? n_rot_chunk : n_rot;
    const size_t base_bytes = carve(nullptr, n, n_pix, rc, n_pat, 0).total;
    EMC_TRY(check_ws(ws, ws_bytes, base_bytes + rot_chunked_extra(n_rot)));
    const Layout l = carve(ws, n, n_pix, rc, n_pat, 0);
    float *s_all = (float *)((uint8_t *)ws + base_bytes);
    cudaStream_t st = (cudaStream_t)stream;
    const bool weighted = (flags & EMC_COMPRESS_WEIGHTED) != 0;
    const bool prof = (flags & EMC_PROFILE_STAGES) != 0;
    const float log_uniform = log_uniform_of(n_rot);                  // log w of every row when weight == NULL
    const int n_chunks = ceil_div(n_rot, rc);

    EMC_TRY(reset_header(l, st));
    {
        Span sp(ctx, prof, EMC_STAGE_PACK, st);
        EMC_TRY(launch_pack(pat->counts, pat->type, n_pat, n_pix, det->mask, l.Kc, l.ld_p, l.KT, l.ld_n, l.hdr, st));
    }
    const float *model_cur = model->model;
    for (int it = 0; it < n_iter; ++it) {
        EMC_TRY_CUDA(cudaMemsetAsync(s_all, 0, sizeof(float) * n_rot, st));
        EMC_TRY_CUDA(cudaMemsetAsync(loglik + it, 0, sizeof(double), st));
        for (int sweep = 1; sweep <= 2; ++sweep) {
            for (int c = 0; c < n_chunks; ++c) {
                const int r0 = c * rc, nr = n_rot - r0 < rc ? n_rot - r0 : rc;
                const emc_rotations sub = {nr, rot->quat + 4 * (size_t)r0, rot->weight ? rot->weight + r0 : nullptr};
                Geometry geo;
                {
                    Span sp(ctx, prof, EMC_STAGE_EXPAND, st);
                    EMC_TRY(launch_geometry(det->q, det->mask, n_pix, det->row_len, sub.quat, nr, l.geom, &geo, st));
                    EMC_TRY_CUDA(cudaMemsetAsync(l.S, 0, sizeof(float) * nr, st));
                    EMC_TRY(launch_expand(model_cur, n, det->q, det->mask, n_pix, sub.quat, nr, nullptr, nullptr, l.planesL,
                                          l.ld_p, l.S, l.blocked, &geo, st, false));
                }
                bool stats_ready = false;
                {
                    Span sp(ctx, prof, EMC_STAGE_LOGLIK, st);
                    EMC_TRY(run_loglik_gemm(l, nr, n_pix, n_pat, l.L, l.ld_n, flags, st, sub.weight, log_uniform,
                                            sweep == 1 ? &stats_ready : nullptr, nullptr, rc));
                }
                if (sweep == 1) {
                    // the chunk's (max, sum) per pattern merged into the running ones; LL with the last chunk
                    Span sp(ctx, prof, EMC_STAGE_NORMALIZE, st);
                    EMC_TRY(launch_normalize(l.L, sub.weight, nr, n_pat, l.ld_n, nullptr, nullptr, 0, nullptr, nullptr,
                                             c == n_chunks - 1 ? loglik + it : nullptr, true, l.scratch, stats_ready, st,
                                             nullptr, 0, log_uniform, 1, c > 0, rc));
                    continue;
                }
                {
                    Span sp(ctx, prof, EMC_STAGE_NORMALIZE, st);
                    EMC_TRY(launch_normalize(l.L, sub.weight, nr, n_pat, l.ld_n, nullptr, l.planesP, (size_t)nr * l.ld_n, l.pscale,
                                             s_all + r0, nullptr, true, l.scratch, false, st, nullptr, 0, log_uniform, 2,
                                             false, rc));
                }
                {
                    Span sp(ctx, prof, EMC_STAGE_UPDATE, st);
                    GemmProblem g;
                    g.A = l.planesP; g.B = l.KT; g.n_planes = 2;
                    g.M = nr; g.N = n_pix; g.K = n_pat;
                    g.lda = l.ld_n; g.ldb = l.ld_n; g.plane_stride = (size_t)nr * l.ld_n;
                    g.a_fmt = g.b_fmt = FMT_F16;
                    g.chunk_scale = l.pscale;
                    g.out = l.Wnum; g.ld_out = n_pix; g.rowv = s_all + r0; g.epilogue = EPI_DIV_ROW;
                    g.one_cta = (flags & EMC_GEMM_1CTA) != 0;
                    EMC_TRY(launch_plane_gemm(g, (flags & EMC_DEBUG_SIMT) != 0, st));
                }
                {
                    Span sp(ctx, prof, EMC_STAGE_COMPRESS, st);
                    const int phases = COMPRESS_SCATTER | (c == 0 ? COMPRESS_CLEAR : 0) | (c == n_chunks - 1 ? COMPRESS_DIVIDE : 0);
                    EMC_TRY(launch_compress(l.Wnum, s_all + r0, weighted, geo, n, l.acc, model_out, nullptr, st, nullptr,
                                            phases));
                }
            }
        }
        model_cur = model_out;
    }
    return launch_poison(l.hdr, model_out, (size_t)n * n * n, loglik, n_iter, st);
}

// ---- rotation shards (NEXT-4): a rank's device work between the caller's collectives
static emc_status shard_args(const emc_model *model, const emc_detector *det, const emc_rotations *rot,
                             const emc_patterns *pat, int n_rot_total, unsigned flags, void *ws, size_t ws_bytes, Layout *l) {
    if (!model || !model->model || !det_ok(det) || !rot_ok(rot) || !pat_ok(pat) || n_rot_total < rot->n_rot) return EMC_ERR_ARG;
    if (flags & (EMC_PATTERNS_ON_HOST | EMC_SPARSE_PHOTONS | EMC_PROFILE_STAGES)) return EMC_ERR_UNSUPPORTED;
    if (!sizes_ok(model->n, det->n_pix, rot->n_rot, pat->n_pat)) return EMC_ERR_UNSUPPORTED;
    EMC_TRY(check_ws(ws, ws_bytes, carve(nullptr, model->n, det->n_pix, rot->n_rot, pat->n_pat, 0).total));
    *l = carve(ws, model->n, det->n_pix, rot->n_rot, pat->n_pat, 0);
    return EMC_OK;
}

emc_status emc_shard_stats(const emc_model *model, const emc_detector *det, const emc_rotations *rot,
                           const emc_patterns *pat, int n_rot_total, float *stats_out, unsigned flags, void *ws,
                           size_t ws_bytes, void *stream) {
    Layout l;
    EMC_TRY(shard_args(model, det, rot, pat, n_rot_total, flags, ws, ws_bytes, &l));
    if (!stats_out) return EMC_ERR_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    const int n = model->n, n_pix = det->n_pix, n_rot = rot->n_rot, n_pat = pat->n_pat;
    const float log_uniform = log_uniform_of(n_rot_total);
    EMC_TRY(reset_header(l, st));
    EMC_TRY(launch_pack(pat->counts, pat->type, n_pat, n_pix, det->mask, l.Kc, l.ld_p, l.KT, l.ld_n, l.hdr, st));
    Geometry geo;
    EMC_TRY(launch_geometry(det->q, det->mask, n_pix, det->row_len, rot->quat, n_rot, l.geom, &geo, st));
    EMC_TRY_CUDA(cudaMemsetAsync(l.S, 0, sizeof(float) * n_rot, st));
    EMC_TRY(launch_expand(model->model, n, det->q, det->mask, n_pix, rot->quat, n_rot, nullptr, nullptr, l.planesL, l.ld_p, l.S,
                          l.blocked, &geo, st, false));
    bool stats_ready = false;
    EMC_TRY(run_loglik_gemm(l, n_rot, n_pix, n_pat, l.L, l.ld_n, flags, st, rot->weight, log_uniform, &stats_ready));
    // the rank's statistics = the carry row after a first-sweep merge with nothing carried in
    EMC_TRY(launch_normalize(l.L, rot->weight, n_rot, n_pat, l.ld_n, nullptr, nullptr, 0, nullptr, nullptr, nullptr, true, l.scratch,
                             stats_ready, st, nullptr, 0, log_uniform, 1, false));
    float *m, *w, *z;
    normalize_stat_row(l.scratch, n_rot, l.ld_n, -1, &m, &w, &z);
    const size_t row = sizeof(float) * (size_t)l.ld_n;
    EMC_TRY_CUDA(cudaMemcpyAsync(stats_out, m, row, cudaMemcpyDeviceToDevice, st));
    EMC_TRY_CUDA(cudaMemcpyAsync(stats_out + l.ld_n, w, row, cudaMemcpyDeviceToDevice, st));
    EMC_TRY_CUDA(cudaMemcpyAsync(stats_out + 2 * (size_t)l.ld_n, z, row, cudaMemcpyDeviceToDevice, st));
    EMC_TRY(launch_shard_stamp(l.hdr, n_rot, n_pat, n_pix, false, st));      // what the workspace now carries
    return launch_poison(l.hdr, stats_out, 3 * (size_t)l.ld_n, nullptr, 0, st);
}

emc_status emc_shard_update(const emc_model *model, const emc_detector *det, const emc_rotations *rot,
                            const emc_patterns *pat, int n_rot_total, const float *stats_all, int world,
                            float *numden_out, double *loglik, float *s_out, unsigned flags, void *ws, size_t ws_bytes,
                            void *stream) {
    Layout l;
    EMC_TRY(shard_args(model, det, rot, pat, n_rot_total, flags, ws, ws_bytes, &l));
    if (!stats_all || world <= 0 || world > 64 || !numden_out || !loglik) return EMC_ERR_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    const int n = model->n, n_pix = det->n_pix, n_rot = rot->n_rot, n_pat = pat->n_pat;
    const float log_uniform = log_uniform_of(n_rot_total);
    const bool weighted = (flags & EMC_COMPRESS_WEIGHTED) != 0;
    // L, the packed counts and the header must be those of an emc_shard_stats call with these sizes: checked on the
    // device; a mismatch turns the results into NaN and emc_check reports EMC_ERR_WORKSPACE
    EMC_TRY(launch_shard_stamp(l.hdr, n_rot, n_pat, n_pix, true, st));
    // the ranks' statistics become partial rows 0 .. world-1 (merged in rank order: the same result on every rank)
    const size_t row = sizeof(float) * (size_t)l.ld_n;
    for (int k = 0; k < world; ++k) {
        float *m, *w, *z;
        normalize_stat_row(l.scratch, n_rot, l.ld_n, k, &m, &w, &z);
        const float *src = stats_all + (size_t)k * 3 * l.ld_n;
        EMC_TRY_CUDA(cudaMemcpyAsync(m, src, row, cudaMemcpyDeviceToDevice, st));
        EMC_TRY_CUDA(cudaMemcpyAsync(w, src + l.ld_n, row, cudaMemcpyDeviceToDevice, st));
        EMC_TRY_CUDA(cudaMemcpyAsync(z, src + 2 * (size_t)l.ld_n, row, cudaMemcpyDeviceToDevice, st));
    }
    EMC_TRY_CUDA(cudaMemsetAsync(loglik, 0, sizeof(double), st));
    EMC_TRY(launch_colstats_combine_rows(l.scratch, n_rot, world, n_pat, l.ld_n, loglik, st));
    EMC_TRY_CUDA(cudaMemsetAsync(l.s, 0, sizeof(float) * n_rot, st));
    EMC_TRY(launch_normalize(l.L, rot->weight, n_rot, n_pat, l.ld_n, nullptr, l.planesP, (size_t)n_rot * l.ld_n, l.pscale, l.s, nullptr,
                             true, l.scratch, false, st, nullptr, 0, log_uniform, 2, false));
    EMC_TRY(run_update_gemm(l, n_rot, n_pix, n_pat, l.Wnum, l.s, EPI_DIV_ROW, flags, st));
    Geometry geo;
    EMC_TRY(launch_geometry(det->q, det->mask, n_pix, det->row_len, rot->quat, n_rot, l.geom, &geo, st));
    EMC_TRY(launch_compress(l.Wnum, l.s, weighted, geo, n, l.acc, nullptr, nullptr, st, nullptr, COMPRESS_CLEAR | COMPRESS_SCATTER));
    EMC_TRY(launch_compress_export(l.acc, n, numden_out, st));
    if (s_out) EMC_TRY_CUDA(cudaMemcpyAsync(s_out, l.s, sizeof(float) * n_rot, cudaMemcpyDeviceToDevice, st));
    return launch_poison(l.hdr, numden_out, 2 * (size_t)n * n * n, loglik, 1, st);
}

emc_status emc_shard_finish(const float *numden, int n, float *model_out, void *stream) {
    if (!numden || !model_out || n < 2 || n > 1024) return EMC_ERR_ARG;
    return launch_numden_divide(numden, n, model_out, (cudaStream_t)stream);
}

emc_status emc_iterate_gaussian(const emc_model *model, const emc_detector *det, const emc_rotations *rot,
                                const emc_patterns *pat, int n_iter, int n_pat_chunk, float sigma, float *model_out,
                                float *P_out, int ld_n, double *loglik, unsigned flags, void *ws, size_t ws_bytes,
                                void *stream, emc_context *ctx) {
    if (!(sigma > 0.f)) return EMC_ERR_ARG;
    return iterate_impl(model, det, rot, pat, n_iter, n_pat_chunk, model_out, P_out, ld_n, loglik, flags, ws, ws_bytes, stream,
                        ctx, sigma);
}

emc_status emc_refine(const emc_model *model, const emc_detector *det, const emc_rotations *levels,
                      int n_levels, const emc_patterns *pat, int n_iter, double threshold, int n_pat_chunk,
                      float *model_out, float *model_tmp, double *loglik, int32_t *level_of_iter,
                      unsigned flags, void *ws, size_t ws_bytes, void *stream, emc_context *ctx) {
    if (!model || !model->model || !levels || n_levels <= 0 || n_iter <= 0 || !model_out || !model_tmp ||
        model_out == model_tmp || model_out == model->model || model_tmp == model->model || !loglik ||
        !level_of_iter || !(threshold >= 0.0))
        return EMC_ERR_ARG;
    for (int l = 0; l < n_levels; ++l)
        if (!rot_ok(&levels[l])) return EMC_ERR_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    float *bufs[2] = {model_out, model_tmp};
    const float *src = model->model;
    int level = 0;
    double prev = 0.0;
    for (int i = 0; i < n_iter; ++i) {
        float *dst = bufs[(n_iter - 1 - i) & 1];                    // the last iteration lands in model_out
        const emc_model cur = {model->n, src};
        EMC_TRY(emc_iterate(&cur, det, &levels[level], pat, 1, n_pat_chunk, dst, nullptr, 0, loglik + i, flags, ws,
                            ws_bytes, stream, ctx));
        level_of_iter[i] = level;
        double ll = 0.0;
        EMC_TRY_CUDA(cudaMemcpyAsync(&ll, loglik + i, sizeof(double), cudaMemcpyDeviceToHost, st));
        EMC_TRY_CUDA(cudaStreamSynchronize(st));
        // eq. (3.1)
        if (i >= 1 && level + 1 < n_levels && fabs(ll - prev) <= threshold * fabs(ll)) ++level;
        prev = ll;
        src = dst;
    }
    return EMC_OK;
}

emc_status emc_check(void *ws, void *stream) {
    if (!ws) return EMC_ERR_ARG;
    WsHeader h;
    cudaStream_t st = (cudaStream_t)stream;
    // read and clear ON the caller's stream (ordered after the calls that used ws, before whatever the caller enqueues
    // next on it); the legacy default stream would not be ordered against a non-blocking stream
    EMC_TRY_CUDA(cudaMemcpyAsync(&h, ws, sizeof(h), cudaMemcpyDeviceToHost, st));
    EMC_TRY_CUDA(cudaMemsetAsync(ws, 0, sizeof(h), st));
    EMC_TRY_CUDA(cudaStreamSynchronize(st));
    if (h.max_count > 0) return EMC_ERR_COUNT_RANGE;            // the pack kernel records only counts over its limit
    if (h.shard_mismatch) return EMC_ERR_WORKSPACE;             // emc_shard_update without the matching emc_shard_stats
    return h.w_range ? EMC_ERR_VALUE_RANGE : EMC_OK;
}

emc_status emc_profile_read(emc_context *c, double *ms, int *spans) {
    if (!c || !ms || !spans) return EMC_ERR_ARG;
    for (int i = 0; i < EMC_N_STAGES; ++i) { ms[i] = 0.0; spans[i] = 0; }
    emc_status rc = EMC_OK;
    for (int i = 0; i < c->used; ++i) {
        float t = 0.f;
        cudaError_t e = cudaEventSynchronize(c->end[i]);
        if (e == cudaSuccess) e = cudaEventElapsedTime(&t, c->beg[i], c->end[i]);
        if (e != cudaSuccess) { rc = cuda_fail(e, "emc_profile_read"); break; }
        ms[c->stage[i]] += (double)t;
        spans[c->stage[i]] += 1;
    }
    c->used = 0;
    return rc;
}

int emc_profile_dropped(emc_context *c) {
    if (!c) return 0;
    const int d = c->dropped;
    c->dropped = 0;
    return d;
}

uint64_t emc_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }

const char *emc_strerror(emc_status s) {
    switch (s) {
        case EMC_OK: return "ok";
        case EMC_ERR_ARG: return "invalid argument";
        case EMC_ERR_UNSUPPORTED: return "size not supported";
        case EMC_ERR_WORKSPACE: return "workspace missing, misaligned or too small";
        case EMC_ERR_CUDA: return "CUDA error";
        case EMC_ERR_COUNT_RANGE: return "unmasked photon count above EMC_MAX_COUNT";
        case EMC_ERR_VALUE_RANGE: return "slice value at or above 65504 in the Gaussian model (fp16 operand planes)";
        case EMC_ERR_STATIC_SCRATCH:
            return "emc_normalize_static: these sizes need more than the EMC_STATIC_SCRATCH_BYTES built into the library "
                   "(see emc_normalize_static_bytes); use emc_normalize with a workspace";
    }
    return "unknown status";
}

const char *emc_last_cuda_error(void) { return g_err; }

const char *emc_version(void) { return "libemc 0.3 (sm_100a)"; }

}  // extern "C"
