// Stage 1, Expand (e-step), eq. (2.9), and the log-slice planes that feed the
// log-likelihood contraction (north_star stage 2).
//
//   W[r,p] = sum over the 8 voxels around x = R_r q_p + c of (trilinear weight) * model[voxel]
//
// Fused into the same pass: logW = log(max(W,1e-30)) split into two fp16 planes
// (hi, lo) with masked / outside samples zeroed, and S[r] = sum_{p:mask} W[r,p].
#include <algorithm>

#include "emc_geometry.cuh"
#include "emc_internal.cuh"

namespace emc {

namespace {

constexpr int kThreads = 256;
constexpr int kPixPerThread = 4;
constexpr int kPixPerBlock = kThreads * kPixPerThread;

__device__ __forceinline__ float block_sum(float v, float *red) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (lane == 0) red[warp] = v;
    __syncthreads();
    float t = 0.f;
    if (warp == 0) {
        t = lane < (kThreads / 32) ? red[lane] : 0.f;
#pragma unroll
        for (int o = 4; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
    }
    return t;   // valid in thread 0
}

// logW -> two fp16 planes: hi = fp16(lw), lo = fp16(lw - hi); 22 significand bits in all.
// gauss (the paper's Gaussian model): the operand is W itself, not log W
// FAST: __logf (one MUFU.LG2 and a multiply; absolute error <= 2^-21.41 on [0.5, 2], else <= 3 ulp, CUDA Math API) in
// the place of logf (about 22 instructions, 1 ulp): |d logW| <= 3.6e-7 max(1, |logW|), against T1's 1e-5 (K |logW| + W)
// summed over the pixels -- the same order as the fp32 accumulation error of the contraction.
template <bool FAST = false>
__device__ __forceinline__ void split_logw(float w, bool live, __half &hi, __half &lo, int gauss = 0) {
    const float lg = FAST ? __logf(fmaxf(w, 1e-30f)) : logf(fmaxf(w, 1e-30f));
    float lw = live ? (gauss ? w : lg) : 0.f;
    hi = __float2half_rn(lw);
    lo = __float2half_rn(lw - __half2float(hi));
}

// grid = (R, ceil(P / kPixPerBlock)); one rotation per block row.
__global__ void __launch_bounds__(kThreads)
expand_kernel(const float *__restrict__ model, int n, const float *__restrict__ q,
              const uint8_t *__restrict__ mask, int n_pix, const float *__restrict__ quat,
              float *__restrict__ W, int32_t *__restrict__ idx, __half *__restrict__ planes, int ld_p,
              size_t plane_stride, float *__restrict__ S, int gauss) {
    __shared__ float rm[9];
    __shared__ float red[kThreads / 32];
    const int r = blockIdx.x;
    if (threadIdx.x == 0) {
        RotMat m = rotation_matrix(quat + 4 * (size_t)r);
#pragma unroll
        for (int i = 0; i < 9; ++i) rm[i] = m.m[i];
    }
    __syncthreads();
    const int nn = n * n;
    float part = 0.f;
#pragma unroll
    for (int j = 0; j < kPixPerThread; ++j) {
        const int p = blockIdx.y * kPixPerBlock + j * kThreads + threadIdx.x;
        if (p >= n_pix) continue;
        const Sample s = locate(rm, q[3 * p], q[3 * p + 1], q[3 * p + 2], n);
        float w = 0.f;
        if (s.base >= 0) {
            const float *b = model + s.base;
            const float z0 = 1.f - s.tz, y0 = 1.f - s.ty, x0 = 1.f - s.tx;
            const float c00 = b[0] * z0 + b[1] * s.tz;
            const float c01 = b[n] * z0 + b[n + 1] * s.tz;
            const float c10 = b[nn] * z0 + b[nn + 1] * s.tz;
            const float c11 = b[nn + n] * z0 + b[nn + n + 1] * s.tz;
            w = (c00 * y0 + c01 * s.ty) * x0 + (c10 * y0 + c11 * s.ty) * s.tx;
        }
        const size_t o = (size_t)r * n_pix + p;
        if (W) W[o] = w;
        if (idx) idx[o] = s.base;
        const bool use = mask ? (mask[p] != 0) : true;
        if (planes) {
            __half hi, lo;
            split_logw(w, use && s.base >= 0, hi, lo, gauss);
            const size_t po = (size_t)r * ld_p + p;
            planes[po] = hi;
            planes[plane_stride + po] = lo;
        }
        if (use) part += gauss ? w * w : w;
    }
    if (S) {
        const float t = block_sum(part, red);
        if (threadIdx.x == 0) atomicAdd(S + r, t);
    }
}

// ---- corner blocks of the model ---------------------------------------------------------------
// A sample reads the 2x2x2 voxels at its base corner b.  In the plain [n][n][n] layout these are 8
// gathers on 4 different cache lines.  Here the model is re-laid as one aligned 32-byte block per BASE
// CORNER: blocked[(b_x n + b_y) n + b_z] = the 8 corner values (order 4 dx + 2 dy + dz), i.e. the block index is
// the index map itself.  One sample = ONE 32-byte gather; a 128-byte line holds the blocks of 4 z-adjacent bases
// (2 x 2 x 5 voxels).  Cost: 32 G bytes written once per iteration (8 MB at 64^3), L2-resident up to n = 128.
__global__ void __launch_bounds__(256)
build_blocked_kernel(const float *__restrict__ model, int n, float4 *__restrict__ blocked) {
    const size_t g = (size_t)n * n * n;
    const size_t t = (size_t)blockIdx.x * 256 + threadIdx.x;
    if (t >= g) return;
    const int bk = (int)(t % n), bj = (int)((t / n) % n), bi = (int)(t / ((size_t)n * n));
    float v[8];
#pragma unroll
    for (int d = 0; d < 8; ++d) {
        const int x = bi + (d >> 2), y = bj + ((d >> 1) & 1), z = bk + (d & 1);
        v[d] = (x < n && y < n && z < n) ? model[((size_t)x * n + y) * n + z] : 0.f;
    }
    blocked[2 * t] = make_float4(v[0], v[1], v[2], v[3]);
    blocked[2 * t + 1] = make_float4(v[4], v[5], v[6], v[7]);
}

// One 32-byte corner block in one request (LDG.256): a divergent gather costs the L1 one tag lookup per distinct
// line and instruction, so two 16-byte loads of the same block cost twice as much as this.
__device__ __forceinline__ void ldg256(const float4 *p, float4 &a, float4 &b) {
    asm volatile("ld.global.nc.v8.f32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                 : "=f"(a.x), "=f"(a.y), "=f"(a.z), "=f"(a.w), "=f"(b.x), "=f"(b.y), "=f"(b.z), "=f"(b.w)
                 : "l"(p));
}

// q and the mask as one float4 per pixel (x, y, z, use ? 1 : 0): one 16-byte load per sample; the rotation matrices
// (float64 arithmetic, G4) once per rotation instead of once per thread block
__global__ void __launch_bounds__(256)
geometry_kernel(const float *__restrict__ q, const uint8_t *__restrict__ mask, int n_pix, const float *__restrict__ quat,
                int n_rot, float4 *__restrict__ qm, float4 *__restrict__ rotm) {
    const int t = blockIdx.x * 256 + threadIdx.x;
    if (t < n_pix) qm[t] = make_float4(q[3 * t], q[3 * t + 1], q[3 * t + 2], (mask && mask[t] == 0) ? 0.f : 1.f);
    if (t < n_rot) {
        const RotMat m = rotation_matrix(quat + 4 * (size_t)t);
        rotm[3 * (size_t)t] = make_float4(m.m[0], m.m[1], m.m[2], 0.f);
        rotm[3 * (size_t)t + 1] = make_float4(m.m[3], m.m[4], m.m[5], 0.f);
        rotm[3 * (size_t)t + 2] = make_float4(m.m[6], m.m[7], m.m[8], 0.f);
    }
}

// One WARP per (rotation, band) work item (a stride loop covers item counts beyond the grid limit).  A warp works on a
// 4 x 8 TILE of detector pixels at a time (its 32 samples cover about 3 x 6 voxels of the slice: 21 distinct corner
// blocks per gather against 25 for 32 pixels of a detector row), four tiles per step in PHASES so that the loads of
// a phase are all in flight together: geometry loads; coordinates; gathers; interpolation and outputs.  The kernel
// is specialised on the outputs it has to write and has no divergent control flow: a lane without a pixel repeats
// pixel 0 and only its stores are predicated.  What bounds it (ncu, profiles/r02_full_ncu.md): the issue
// slots (125 warp instructions per 32 samples, 62 % of the slots used) with the waits for the gather exposed; capping
// registers for more warps per SM (spills) or making the warps persistent over long bands were both slower.
// S_part [R][n_bands]: sum_{p:mask} W (or W^2) of each band, summed per rotation in a fixed order by rowsum_kernel
// (bitwise reproducible S, no atomics).
constexpr int kWarps = kThreads / 32;
// LOGW32 (photon-list path): W receives log W as float32 (0 for masked / outside samples) and S the row sums
// GAUSS: the planes hold W itself (Gaussian model); a compile-time switch so that the Poisson path pays nothing for it
template <bool W_OUT, bool IDX_OUT, bool PLANES, bool LOGW32 = false, bool GAUSS = false>
__global__ void __launch_bounds__(kThreads, 4)
expand_blocked_kernel(const float4 *__restrict__ blocked, int n, const float4 *__restrict__ qm, const TileMap tm,
                      const float4 *__restrict__ rotm, int n_rot, int n_pix, float *__restrict__ W, int32_t *__restrict__ idx,
                      __half *__restrict__ planes, int ld_p, size_t plane_stride, float *__restrict__ S_part, int gauss,
                      int *__restrict__ w_range) {
    const int lane = threadIdx.x & 31;
    const int n_items = n_rot * tm.n_bands;
    for (int item = blockIdx.x * kWarps + (threadIdx.x >> 5); item < n_items; item += gridDim.x * kWarps) {
        const int r = item / tm.n_bands;
        float rm[9];
        load_rotation(rotm, r, rm);
        const Band band(tm, item - r * tm.n_bands, lane);
        float *const w_row = (W_OUT || LOGW32) ? W + (size_t)r * n_pix : nullptr;
        int32_t *const i_row = IDX_OUT ? idx + (size_t)r * n_pix : nullptr;
        __half *const hi_row = PLANES ? planes + (size_t)r * ld_p : nullptr;
        __half *const lo_row = PLANES ? hi_row + plane_stride : nullptr;
        float part = 0.f;
        for (int t0 = 0; t0 < band.n_tiles; t0 += kTilesPerStep) {
            int pix[kTilesPerStep];
            float4 g[kTilesPerStep];
#pragma unroll
            for (int j = 0; j < kTilesPerStep; ++j) {
                pix[j] = band.pixel(t0 + j);
                g[j] = qm[max(pix[j], 0)];
            }
            Sample s[kTilesPerStep];
            float4 lo4[kTilesPerStep], hi4[kTilesPerStep];
#pragma unroll
            for (int j = 0; j < kTilesPerStep; ++j) {
                s[j] = locate(rm, g[j].x, g[j].y, g[j].z, n);
                // outside samples read block 0 (any valid address) and are zeroed afterwards
                ldg256(blocked + 2 * (size_t)(unsigned)max(s[j].base, 0), lo4[j], hi4[j]);
            }
#pragma unroll
            for (int j = 0; j < kTilesPerStep; ++j) {
                const bool in = pix[j] >= 0, inside = s[j].base >= 0;
                const int pc = max(pix[j], 0);
                const float tx = s[j].tx, ty = s[j].ty, tz = s[j].tz;
                const float z0 = 1.f - tz, y0 = 1.f - ty, x0 = 1.f - tx;
                const float c00 = lo4[j].x * z0 + lo4[j].y * tz;
                const float c01 = lo4[j].z * z0 + lo4[j].w * tz;
                const float c10 = hi4[j].x * z0 + hi4[j].y * tz;
                const float c11 = hi4[j].z * z0 + hi4[j].w * tz;
                float w = (c00 * y0 + c01 * ty) * x0 + (c10 * y0 + c11 * ty) * tx;
                w = inside ? w : 0.f;
                const bool use = in && g[j].w != 0.f;
                if (LOGW32) {
                    const float lw = (use && inside) ? __logf(fmaxf(w, 1e-30f)) : 0.f;
                    if (in) w_row[pc] = lw;
                } else if (W_OUT && in) {
                    w_row[pc] = w;
                }
                if (IDX_OUT && in) i_row[pc] = s[j].base;
                if (PLANES) {
                    __half hi, lo;
                    if (GAUSS && use && w >= 65504.f && w_range) *w_range = 1;       // fp16 planes of W itself would hold inf
                    split_logw<true>(w, use && inside, hi, lo, GAUSS ? 1 : 0);
                    if (in) {
                        hi_row[pc] = hi;
                        lo_row[pc] = lo;
                    }
                }
                part += use ? (GAUSS ? w * w : w) : 0.f;
            }
        }
        if (PLANES || LOGW32) {                              // S accompanies the log-likelihood operands
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
            if (lane == 0) S_part[item] = part;
        }
    }
}

// S[r] = sum of the row's band partials, in a fixed order (one warp per rotation)
__global__ void __launch_bounds__(256)
rowsum_kernel(const float *__restrict__ S_part, int n_rot, int n_bands, float *__restrict__ S) {
    const int r = blockIdx.x * 8 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (r >= n_rot) return;
    float t = 0.f;
    for (int b = lane; b < n_bands; b += 32) t += S_part[(size_t)r * n_bands + b];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
    if (lane == 0) S[r] = t;
}

__global__ void __launch_bounds__(kThreads)
logw_split_kernel(const float *__restrict__ W, const int32_t *__restrict__ idx,
                  const uint8_t *__restrict__ mask, int n_pix, __half *__restrict__ planes, int ld_p,
                  size_t plane_stride, float *__restrict__ S, int gauss) {
    __shared__ float red[kThreads / 32];
    const int r = blockIdx.x;
    float part = 0.f;
#pragma unroll
    for (int j = 0; j < kPixPerThread; ++j) {
        const int p = blockIdx.y * kPixPerBlock + j * kThreads + threadIdx.x;
        if (p >= n_pix) continue;
        const size_t o = (size_t)r * n_pix + p;
        const float w = W[o];
        const bool inside = idx ? (idx[o] >= 0) : true;
        const bool use = mask ? (mask[p] != 0) : true;
        __half hi, lo;
        split_logw(w, use && inside, hi, lo, gauss);
        const size_t po = (size_t)r * ld_p + p;
        planes[po] = hi;
        planes[plane_stride + po] = lo;
        if (use) part += gauss ? w * w : w;
    }
    const float t = block_sum(part, red);
    if (threadIdx.x == 0) atomicAdd(S + r, t);
}

}  // namespace

size_t geometry_float4(int n_pix, int n_rot) { return (size_t)n_pix + 3 * (size_t)n_rot; }

emc_status launch_geometry(const float *q, const uint8_t *mask, int n_pix, int row_len, const float *quat, int n_rot,
                           float4 *buf, Geometry *out, cudaStream_t st) {
    float4 *qm = buf, *rotm = buf + n_pix;
    const int n = n_pix > n_rot ? n_pix : n_rot;
    geometry_kernel<<<ceil_div(n, 256), 256, 0, st>>>(q, mask, n_pix, quat, n_rot, qm, rotm);
    EMC_LAUNCHED();
    *out = Geometry{qm, rotm, n_pix, n_rot, row_len};
    return EMC_OK;
}

// corner blocks of the model + the band partials of S (at most one band per 4 pixels... per 32 pixels of a row)
size_t expand_scratch_floats(int n, int n_pix, int n_rot) {
    return (size_t)8 * n * n * n + (size_t)n_rot * (size_t)((n_pix + 31) / 32 + 1);
}

emc_status launch_expand(const float *model, int n, const float *q, const uint8_t *mask, int n_pix,
                         const float *quat, int n_rot, float *W, int32_t *idx, __half *planes,
                         int ld_p, float *S, float *blocked, const Geometry *geo, cudaStream_t st, bool gauss, bool logw32, int *w_range) {
    const int g = gauss ? 1 : 0;
    if (planes && !S) return EMC_ERR_ARG;
    if (blocked && geo) {
        const size_t blocks = (size_t)n * n * n;              // one 32-byte block per base corner
        build_blocked_kernel<<<(unsigned)((blocks + 255) / 256), 256, 0, st>>>(model, n, (float4 *)blocked);
        EMC_LAUNCHED();
        const float4 *b4 = (const float4 *)blocked;
        const size_t ps = (size_t)n_rot * ld_p;
        const TileMap tm = make_tile_map(n_pix, geo->row_len);
        // band partials of S live behind the corner blocks (expand_scratch_floats)
        float *S_part = blocked + (size_t)8 * n * n * n;
        const long long items = (long long)n_rot * tm.n_bands;
        if (items > 0x7fffffffLL) return EMC_ERR_UNSUPPORTED;      // the kernels count work items in 32 bits
        const int grid = (int)std::min<long long>((items + kWarps - 1) / kWarps, (long long)1 << 30);
#define EMC_EXPAND_CASE(w_, i_, p_)                                                                                   \
    expand_blocked_kernel<w_, i_, p_><<<grid, kThreads, 0, st>>>(b4, n, geo->qm, tm, geo->rotm, n_rot, n_pix, W, idx, planes, ld_p, ps, S_part, g, w_range)
        const int sel = (W ? 4 : 0) | (idx ? 2 : 0) | (planes ? 1 : 0);
        switch (sel) {
            case 1:
                if (gauss)
                    expand_blocked_kernel<false, false, true, false, true><<<grid, kThreads, 0, st>>>(b4, n, geo->qm, tm, geo->rotm, n_rot, n_pix, W, idx, planes, ld_p, ps, S_part, g, w_range);
                else
                    EMC_EXPAND_CASE(false, false, true);
                break;
            case 2: EMC_EXPAND_CASE(false, true, false); break;
            case 4:
                if (logw32)                                      // log W and S out instead of W
                    expand_blocked_kernel<false, false, false, true><<<grid, kThreads, 0, st>>>(b4, n, geo->qm, tm, geo->rotm, n_rot, n_pix, W, idx, planes, ld_p, ps, S_part, g, w_range);
                else
                    EMC_EXPAND_CASE(true, false, false);
                break;
            case 6: EMC_EXPAND_CASE(true, true, false); break;
            default: return EMC_ERR_ARG;                         // no caller asks for slices and operand planes at once
        }
#undef EMC_EXPAND_CASE
        EMC_LAUNCHED();
        if (planes || logw32) {
            rowsum_kernel<<<ceil_div(n_rot, 8), 256, 0, st>>>(S_part, n_rot, tm.n_bands, S);
            EMC_LAUNCHED();
        }
        return EMC_OK;
    }
    dim3 grid(n_rot, ceil_div(n_pix, kPixPerBlock));
    expand_kernel<<<grid, kThreads, 0, st>>>(model, n, q, mask, n_pix, quat, W, idx, planes, ld_p,
                                             (size_t)n_rot * ld_p, S, g);
    EMC_LAUNCHED();
    return EMC_OK;
}

emc_status launch_logw_split(const float *W, const int32_t *idx, const uint8_t *mask, int n_pix,
                             int n_rot, __half *planes, int ld_p, float *S, cudaStream_t st, bool gauss) {
    dim3 grid(n_rot, ceil_div(n_pix, kPixPerBlock));
    logw_split_kernel<<<grid, kThreads, 0, st>>>(W, idx, mask, n_pix, planes, ld_p,
                                                 (size_t)n_rot * ld_p, S, gauss ? 1 : 0);
    EMC_LAUNCHED();
    return EMC_OK;
}

}  // namespace emc
