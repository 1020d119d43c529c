// Stage 1, Expand (e-step), eq. (2.9), and the log-slice planes that feed the
// log-likelihood contraction (north_star stage 2).
//
//   W[r,p] = sum over the 8 voxels around x = R_r q_p + c of (trilinear weight) * model[voxel]
//
// Fused into the same pass: logW = log(max(W,1e-30)) split into two fp16 planes
// (hi, lo) with masked / outside samples zeroed, and S[r] = sum_{p:mask} W[r,p].
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
__device__ __forceinline__ void split_logw(float w, bool live, __half &hi, __half &lo, int gauss = 0) {
    float lw = live ? (gauss ? w : logf(fmaxf(w, 1e-30f))) : 0.f;
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

// ---- blocked, staggered copies of the model (n even) -----------------------------------------
// A sample reads the 2x2x2 voxels at its base corner b.  In the plain [n][n][n] layout these are 8
// gathers on 4 different cache lines.  Here the model is re-laid as 8 copies, one per parity
// (b_x&1, b_y&1, b_z&1) of the base; copy c holds, for every base of that parity, the 8 corner values
// as one aligned 32-byte block (corner order 4*dx + 2*dy + dz), blocks ordered [b_x/2][b_y/2][b_z/2].
// One sample = two 16-byte loads from one sector-aligned block; z-adjacent bases share a cache line.
// Cost: 32 G bytes written once per iteration (8 MB at 64^3), L2-resident up to n = 128.
__global__ void __launch_bounds__(256)
build_blocked_kernel(const float *__restrict__ model, int n, float4 *__restrict__ blocked) {
    const int h = n >> 1;
    const size_t per_copy = (size_t)h * h * h;
    const size_t t = (size_t)blockIdx.x * 256 + threadIdx.x;
    if (t >= 8 * per_copy) return;
    const int c = (int)(t / per_copy);
    size_t i = t - (size_t)c * per_copy;
    const int bk = 2 * (int)(i % h) + (c & 1);
    i /= h;
    const int bj = 2 * (int)(i % h) + ((c >> 1) & 1);
    const int bi = 2 * (int)(i / h) + ((c >> 2) & 1);
    float v[8];
#pragma unroll
    for (int d = 0; d < 8; ++d) {
        const int x = bi + (d >> 2), y = bj + ((d >> 1) & 1), z = bk + (d & 1);
        v[d] = (x < n && y < n && z < n) ? model[((size_t)x * n + y) * n + z] : 0.f;
    }
    blocked[2 * t] = make_float4(v[0], v[1], v[2], v[3]);
    blocked[2 * t + 1] = make_float4(v[4], v[5], v[6], v[7]);
}

// One 32-byte corner block in one request (LDG.256): a divergent gather costs the L1 one tag lookup per lane and
// instruction, so two 16-byte loads of the same block cost twice as much as this.
__device__ __forceinline__ void ldg256(const float4 *p, float4 &a, float4 &b) {
    asm volatile("ld.global.nc.v8.f32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                 : "=f"(a.x), "=f"(a.y), "=f"(a.z), "=f"(a.w), "=f"(b.x), "=f"(b.y), "=f"(b.z), "=f"(b.w)
                 : "l"(p));
}

// q and the mask as one float4 per pixel (x, y, z, use ? 1 : 0): one coalesced 16-byte load per sample
__global__ void __launch_bounds__(256)
pack_geometry_kernel(const float *__restrict__ q, const uint8_t *__restrict__ mask, int n_pix, float4 *__restrict__ qm) {
    const int p = blockIdx.x * 256 + threadIdx.x;
    if (p >= n_pix) return;
    qm[p] = make_float4(q[3 * p], q[3 * p + 1], q[3 * p + 2], (mask && mask[p] == 0) ? 0.f : 1.f);
}

// The kernel is bound by instruction issue (about 180 warp instructions per 32 samples before this version,
// ncu r01_v2), not by memory, so it is specialised on the outputs it has to write, reads its geometry as one
// float4 per pixel and has no divergent control flow: a lane past the end of the detector repeats the last
// pixel and only its stores are predicated.
template <bool W_OUT, bool IDX_OUT, bool PLANES>
__global__ void __launch_bounds__(kThreads)
expand_blocked_kernel(const float4 *__restrict__ blocked, int n, const float4 *__restrict__ qm, int n_pix,
                      const float *__restrict__ quat, float *__restrict__ W, int32_t *__restrict__ idx,
                      __half *__restrict__ planes, int ld_p, size_t plane_stride, float *__restrict__ S, int gauss) {
    __shared__ float rm_s[9];
    __shared__ float red[kThreads / 32];
    const int r = blockIdx.x;
    if (threadIdx.x == 0) {
        RotMat m = rotation_matrix(quat + 4 * (size_t)r);
#pragma unroll
        for (int i = 0; i < 9; ++i) rm_s[i] = m.m[i];
    }
    __syncthreads();
    float rm[9];
#pragma unroll
    for (int i = 0; i < 9; ++i) rm[i] = rm_s[i];
    const unsigned h = (unsigned)n >> 1;
    const unsigned per_copy = h * h * h;                    // 8 * per_copy <= 2^30 for n <= 1024
    float part = 0.f;
#pragma unroll
    for (int j = 0; j < kPixPerThread; ++j) {
        const int p = blockIdx.y * kPixPerBlock + j * kThreads + threadIdx.x;
        const bool in = p < n_pix;
        const float4 g = qm[in ? p : n_pix - 1];
        const Sample s = locate(rm, g.x, g.y, g.z, n);
        const bool inside = s.base >= 0;
        // outside samples read block 0 (any valid address) and are zeroed afterwards
        const unsigned bx = inside ? (unsigned)s.bx : 0u, by = inside ? (unsigned)s.by : 0u, bz = inside ? (unsigned)s.bz : 0u;
        const unsigned c = ((bx & 1u) << 2) | ((by & 1u) << 1) | (bz & 1u);
        const unsigned blk = c * per_copy + ((bx >> 1) * h + (by >> 1)) * h + (bz >> 1);
        float4 lo4, hi4;
        ldg256(blocked + 2 * (size_t)blk, lo4, hi4);
        const float z0 = 1.f - s.tz, y0 = 1.f - s.ty, x0 = 1.f - s.tx;
        const float c00 = lo4.x * z0 + lo4.y * s.tz;
        const float c01 = lo4.z * z0 + lo4.w * s.tz;
        const float c10 = hi4.x * z0 + hi4.y * s.tz;
        const float c11 = hi4.z * z0 + hi4.w * s.tz;
        float w = (c00 * y0 + c01 * s.ty) * x0 + (c10 * y0 + c11 * s.ty) * s.tx;
        w = inside ? w : 0.f;
        const size_t o = (size_t)r * n_pix + p;
        if (W_OUT && in) W[o] = w;
        if (IDX_OUT && in) idx[o] = s.base;
        const bool use = in && g.w != 0.f;
        if (PLANES && in) {
            __half hi, lo;
            split_logw(w, use && inside, hi, lo, gauss);
            const size_t po = (size_t)r * ld_p + p;
            planes[po] = hi;
            planes[plane_stride + po] = lo;
        }
        part += use ? (gauss ? w * w : w) : 0.f;
    }
    if (PLANES) {                                            // S accompanies the planes (log-likelihood operands)
        const float t = block_sum(part, red);
        if (threadIdx.x == 0) atomicAdd(S + r, t);
    }
}

__global__ void __launch_bounds__(kThreads)
logw_split_kernel(const float *__restrict__ W, const int32_t *__restrict__ idx,
                  const uint8_t *__restrict__ mask, int n_pix, __half *__restrict__ planes, int ld_p,
                  size_t plane_stride, float *__restrict__ S) {
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
        split_logw(w, use && inside, hi, lo);
        const size_t po = (size_t)r * ld_p + p;
        planes[po] = hi;
        planes[plane_stride + po] = lo;
        if (use) part += w;
    }
    const float t = block_sum(part, red);
    if (threadIdx.x == 0) atomicAdd(S + r, t);
}

}  // namespace

static size_t expand_blocked_floats(int n) { return (size_t)8 * n * n * n; }
// blocked model copies + one float4 of geometry per pixel
emc_status launch_pack_geometry(const float *q, const uint8_t *mask, int n_pix, float4 *qm, cudaStream_t st) {
    pack_geometry_kernel<<<ceil_div(n_pix, 256), 256, 0, st>>>(q, mask, n_pix, qm);
    EMC_LAUNCHED();
    return EMC_OK;
}

size_t expand_scratch_floats(int n, int n_pix) { return (n & 1) ? 0 : expand_blocked_floats(n) + (size_t)4 * n_pix; }

emc_status launch_expand(const float *model, int n, const float *q, const uint8_t *mask, int n_pix,
                         const float *quat, int n_rot, float *W, int32_t *idx, __half *planes,
                         int ld_p, float *S, float *blocked, cudaStream_t st, bool gauss) {
    dim3 grid(n_rot, ceil_div(n_pix, kPixPerBlock));
    const int g = gauss ? 1 : 0;
    if (planes && !S) return EMC_ERR_ARG;
    if (blocked && (n & 1) == 0) {
        const size_t blocks = (size_t)n * n * n;              // 8 copies x (n/2)^3 blocks
        float4 *qm = reinterpret_cast<float4 *>(blocked + expand_blocked_floats(n));
        build_blocked_kernel<<<(unsigned)((blocks + 255) / 256), 256, 0, st>>>(model, n, (float4 *)blocked);
        EMC_LAUNCHED();
        pack_geometry_kernel<<<ceil_div(n_pix, 256), 256, 0, st>>>(q, mask, n_pix, qm);
        EMC_LAUNCHED();
        const float4 *b4 = (const float4 *)blocked;
        const size_t ps = (size_t)n_rot * ld_p;
#define EMC_EXPAND_CASE(w_, i_, p_)                                                                                   \
    expand_blocked_kernel<w_, i_, p_><<<grid, kThreads, 0, st>>>(b4, n, qm, n_pix, quat, W, idx, planes, ld_p, ps, S, g)
        const int sel = (W ? 4 : 0) | (idx ? 2 : 0) | (planes ? 1 : 0);
        switch (sel) {
            case 1: EMC_EXPAND_CASE(false, false, true); break;
            case 2: EMC_EXPAND_CASE(false, true, false); break;
            case 4: EMC_EXPAND_CASE(true, false, false); break;
            case 6: EMC_EXPAND_CASE(true, true, false); break;
            default: return EMC_ERR_ARG;                         // no caller asks for slices and operand planes at once
        }
#undef EMC_EXPAND_CASE
        EMC_LAUNCHED();
        return EMC_OK;
    }
    expand_kernel<<<grid, kThreads, 0, st>>>(model, n, q, mask, n_pix, quat, W, idx, planes, ld_p,
                                             (size_t)n_rot * ld_p, S, g);
    EMC_LAUNCHED();
    return EMC_OK;
}

emc_status launch_logw_split(const float *W, const int32_t *idx, const uint8_t *mask, int n_pix,
                             int n_rot, __half *planes, int ld_p, float *S, cudaStream_t st) {
    dim3 grid(n_rot, ceil_div(n_pix, kPixPerBlock));
    logw_split_kernel<<<grid, kThreads, 0, st>>>(W, idx, mask, n_pix, planes, ld_p,
                                                 (size_t)n_rot * ld_p, S);
    EMC_LAUNCHED();
    return EMC_OK;
}

}  // namespace emc
