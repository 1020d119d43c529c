// Stage 3: normalisation of the likelihoods over the rotation space (reconstructed eq. (2.4),
// PAPER.md:78-80; "normalization ... in a separate final sweep"; "only maximal
// rotational probabilities and sums are necessary"):
//
//   a[r,d] = L[r,d] + log w_r;   m_d = max_r a;   P[r,d] = exp(a - m_d) / sum_r exp(a - m_d)
//
// Two sweeps over L (column-wise reductions on a row-major matrix): (1) per-column online
// (max, sum) in warp-shuffle-free lane-per-column form, split over row ranges for parallelism;
// (2) write P, its three bf16 planes for the update GEMM, s[r] = sum_d P[r,d] and the total
// log-likelihood.  HBM-bound: 8 algorithmic bytes per (r,d).
#include "emc_internal.cuh"

namespace emc {

namespace {

// One thread owns 4 adjacent columns (a float4 of a row): a warp reads 512 contiguous bytes of a row,
// a block of 8 warps walks down the rows, kBatch rows of independent loads in flight per thread.
constexpr int kVec = 4;
constexpr int kColsPerBlock = 32 * kVec;      // 128
constexpr int kWarps = 8;
constexpr int kThreads = 32 * kWarps;
constexpr int kBatch = 4;

__host__ __device__ inline int row_splits_for(int n_rot, int n_col_blocks) {
    int want = (6 * 148 + n_col_blocks - 1) / n_col_blocks;
    int cap = (n_rot + 127) / 128;
    if (cap > 64) cap = 64;
    if (want > cap) want = cap;
    return want < 1 ? 1 : want;
}

__device__ __forceinline__ float log_weight(const float *__restrict__ weight, int r, float log_uniform) {
    return weight ? logf(weight[r]) : log_uniform;
}

__device__ __forceinline__ void online(float a, float &m, float &z) {
    if (a > m) {
        z = z * expf(m - a) + 1.f;
        m = a;
    } else {
        z += expf(a - m);
    }
}

// sweep 1: partial (max, sum) of every column over the rows of one split
__global__ void __launch_bounds__(kThreads)
colstats_kernel(const float *__restrict__ L, const float *__restrict__ weight, int n_rot, int n_pat,
                int ld_n, int rows_per_split, float *__restrict__ part_m, float *__restrict__ part_z) {
    __shared__ float4 sm_m[kWarps][32], sm_z[kWarps][32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int d = blockIdx.x * kColsPerBlock + lane * kVec;
    const int r_lo = blockIdx.y * rows_per_split;
    const int r_hi = min(n_rot, r_lo + rows_per_split);
    const float log_uniform = -logf((float)n_rot);
    float m[kVec], z[kVec];
#pragma unroll
    for (int j = 0; j < kVec; ++j) { m[j] = -INFINITY; z[j] = 0.f; }
    if (d < n_pat) {                                   // ld_n is a multiple of 4: the float4 stays inside the row
        for (int r0 = r_lo + warp; r0 < r_hi; r0 += kWarps * kBatch) {
            float4 v[kBatch];
            float lw[kBatch];
#pragma unroll
            for (int b = 0; b < kBatch; ++b) {
                const int r = r0 + b * kWarps;
                if (r < r_hi) {
                    v[b] = *reinterpret_cast<const float4 *>(L + (size_t)r * ld_n + d);
                    lw[b] = log_weight(weight, r, log_uniform);
                }
            }
#pragma unroll
            for (int b = 0; b < kBatch; ++b) {
                if (r0 + b * kWarps < r_hi) {
                    online(v[b].x + lw[b], m[0], z[0]);
                    online(v[b].y + lw[b], m[1], z[1]);
                    online(v[b].z + lw[b], m[2], z[2]);
                    online(v[b].w + lw[b], m[3], z[3]);
                }
            }
        }
    }
    sm_m[warp][lane] = make_float4(m[0], m[1], m[2], m[3]);
    sm_z[warp][lane] = make_float4(z[0], z[1], z[2], z[3]);
    __syncthreads();
    if (warp == 0 && d < n_pat) {
        float mt[kVec], zt[kVec];
#pragma unroll
        for (int j = 0; j < kVec; ++j) { mt[j] = -INFINITY; zt[j] = 0.f; }
#pragma unroll
        for (int w = 0; w < kWarps; ++w) {
            const float4 a = sm_m[w][lane];
            mt[0] = fmaxf(mt[0], a.x); mt[1] = fmaxf(mt[1], a.y); mt[2] = fmaxf(mt[2], a.z); mt[3] = fmaxf(mt[3], a.w);
        }
#pragma unroll
        for (int w = 0; w < kWarps; ++w) {
            const float4 a = sm_m[w][lane], b = sm_z[w][lane];
            if (b.x > 0.f) zt[0] += b.x * expf(a.x - mt[0]);
            if (b.y > 0.f) zt[1] += b.y * expf(a.y - mt[1]);
            if (b.z > 0.f) zt[2] += b.z * expf(a.z - mt[2]);
            if (b.w > 0.f) zt[3] += b.w * expf(a.w - mt[3]);
        }
        *reinterpret_cast<float4 *>(part_m + (size_t)blockIdx.y * ld_n + d) = make_float4(mt[0], mt[1], mt[2], mt[3]);
        *reinterpret_cast<float4 *>(part_z + (size_t)blockIdx.y * ld_n + d) = make_float4(zt[0], zt[1], zt[2], zt[3]);
    }
}

// p -> hi + mid (+ lo) bf16 planes, four columns at a time (8-byte stores)
__device__ __forceinline__ void split4_bf16(const float (&p)[kVec], int n_planes, __nv_bfloat16 *__restrict__ planes,
                                            size_t plane_stride, size_t o) {
    float rem[kVec];
    __nv_bfloat16 h[kVec];
#pragma unroll
    for (int j = 0; j < kVec; ++j) { h[j] = __float2bfloat16_rn(p[j]); rem[j] = p[j] - __bfloat162float(h[j]); }
    *reinterpret_cast<uint2 *>(planes + o) = *reinterpret_cast<const uint2 *>(h);
#pragma unroll
    for (int j = 0; j < kVec; ++j) { h[j] = __float2bfloat16_rn(rem[j]); rem[j] -= __bfloat162float(h[j]); }
    *reinterpret_cast<uint2 *>(planes + plane_stride + o) = *reinterpret_cast<const uint2 *>(h);
    if (n_planes > 2) {
#pragma unroll
        for (int j = 0; j < kVec; ++j) h[j] = __float2bfloat16_rn(rem[j]);
        *reinterpret_cast<uint2 *>(planes + 2 * plane_stride + o) = *reinterpret_cast<const uint2 *>(h);
    }
}

__device__ __forceinline__ void split_bf16(float p, int n_planes, __nv_bfloat16 *__restrict__ planes,
                                           size_t plane_stride, size_t o) {
    const __nv_bfloat16 h = __float2bfloat16_rn(p);
    planes[o] = h;
    float rem = p - __bfloat162float(h);
    const __nv_bfloat16 m = __float2bfloat16_rn(rem);
    planes[plane_stride + o] = m;
    if (n_planes > 2) {
        rem -= __bfloat162float(m);
        planes[2 * plane_stride + o] = __float2bfloat16_rn(rem);
    }
}

// sweep 2: combine the partials, write P / planes / s / LL
__global__ void __launch_bounds__(kThreads)
normalize_kernel(const float *__restrict__ L, const float *__restrict__ weight, int n_rot, int n_pat,
                 int ld_n, int rows_per_split, int n_splits, const float *__restrict__ part_m,
                 const float *__restrict__ part_z, float *__restrict__ P,
                 __nv_bfloat16 *__restrict__ planes, int n_planes, size_t plane_stride,
                 float *__restrict__ s, double *__restrict__ loglik) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int d = blockIdx.x * kColsPerBlock + lane * kVec;
    const int r_lo = blockIdx.y * rows_per_split;
    const int r_hi = min(n_rot, r_lo + rows_per_split);
    const float log_uniform = -logf((float)n_rot);
    const bool col_ok = d < n_pat;
    // every warp combines the split partials of its own 4 columns (L2-resident, n_splits <= 64)
    float mt[kVec], iz[kVec];
    double ll = 0.0;
#pragma unroll
    for (int j = 0; j < kVec; ++j) { mt[j] = -INFINITY; iz[j] = 0.f; }
    if (col_ok) {
        float zt[kVec] = {0.f, 0.f, 0.f, 0.f};
        for (int k = 0; k < n_splits; ++k) {
            const float4 a = *reinterpret_cast<const float4 *>(part_m + (size_t)k * ld_n + d);
            mt[0] = fmaxf(mt[0], a.x); mt[1] = fmaxf(mt[1], a.y); mt[2] = fmaxf(mt[2], a.z); mt[3] = fmaxf(mt[3], a.w);
        }
        for (int k = 0; k < n_splits; ++k) {
            const float4 a = *reinterpret_cast<const float4 *>(part_m + (size_t)k * ld_n + d);
            const float4 b = *reinterpret_cast<const float4 *>(part_z + (size_t)k * ld_n + d);
            if (b.x > 0.f) zt[0] += b.x * expf(a.x - mt[0]);
            if (b.y > 0.f) zt[1] += b.y * expf(a.y - mt[1]);
            if (b.z > 0.f) zt[2] += b.z * expf(a.z - mt[2]);
            if (b.w > 0.f) zt[3] += b.w * expf(a.w - mt[3]);
        }
#pragma unroll
        for (int j = 0; j < kVec; ++j) {
            iz[j] = 1.f / zt[j];
            if (d + j < n_pat) ll += (double)mt[j] + (double)logf(zt[j]);
        }
    }
    if (loglik && blockIdx.y == 0 && warp == 0) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) ll += __shfl_xor_sync(0xffffffffu, ll, o);
        if (lane == 0) atomicAdd(loglik, ll);
    }
    for (int r0 = r_lo + warp; r0 < r_hi; r0 += kWarps * kBatch) {
        float4 v[kBatch];
        float lw[kBatch];
#pragma unroll
        for (int b = 0; b < kBatch; ++b) {
            const int r = r0 + b * kWarps;
            if (r < r_hi && col_ok) {
                v[b] = *reinterpret_cast<const float4 *>(L + (size_t)r * ld_n + d);
                lw[b] = log_weight(weight, r, log_uniform);
            }
        }
#pragma unroll
        for (int b = 0; b < kBatch; ++b) {
            const int r = r0 + b * kWarps;
            if (r >= r_hi) break;                       // warp-uniform
            float p[kVec] = {0.f, 0.f, 0.f, 0.f};
            if (col_ok) {
                const float a[kVec] = {v[b].x + lw[b], v[b].y + lw[b], v[b].z + lw[b], v[b].w + lw[b]};
#pragma unroll
                for (int j = 0; j < kVec; ++j) {
                    float pj = expf(a[j] - mt[j]) * iz[j];
                    if (pj < EMC_P_MIN || d + j >= n_pat) pj = 0.f;      // DESIGN.md §3 G20
                    p[j] = pj;
                }
                const size_t o = (size_t)r * ld_n + d;
                if (P) *reinterpret_cast<float4 *>(P + o) = make_float4(p[0], p[1], p[2], p[3]);
                if (planes) split4_bf16(p, n_planes, planes, plane_stride, o);
            }
            if (s) {
                float t = (p[0] + p[1]) + (p[2] + p[3]);
#pragma unroll
                for (int off = 16; off > 0; off >>= 1) t += __shfl_xor_sync(0xffffffffu, t, off);
                if (lane == 0) atomicAdd(s + r, t);
            }
        }
    }
}

__global__ void __launch_bounds__(256)
p_split_kernel(const float *__restrict__ P, int n_pat, int ld_n, __nv_bfloat16 *__restrict__ planes,
               int ld_pl, int n_planes, size_t plane_stride) {
    const int d = blockIdx.y * 256 + threadIdx.x;
    if (d >= n_pat) return;
    float p = P[(size_t)blockIdx.x * ld_n + d];
    if (p < EMC_P_MIN) p = 0.f;
    split_bf16(p, n_planes, planes, plane_stride, (size_t)blockIdx.x * ld_pl + d);
}

__global__ void __launch_bounds__(256)
div_rows_kernel(float *__restrict__ Wn, const float *__restrict__ s, int n_pix) {
    const int p = blockIdx.y * 256 + threadIdx.x;
    if (p >= n_pix) return;
    const float sr = s[blockIdx.x];
    const size_t o = (size_t)blockIdx.x * n_pix + p;
    Wn[o] = sr > 0.f ? Wn[o] / sr : 0.f;
}

}  // namespace

size_t normalize_scratch_floats(int n_rot, int ld_n) {
    (void)n_rot;
    return (size_t)2 * 64 * (size_t)ld_n;
}

emc_status launch_normalize(const float *L, const float *weight, int n_rot, int n_pat, int ld_n,
                            float *P, __nv_bfloat16 *planes, int n_planes, size_t plane_stride,
                            float *s, double *loglik, bool accumulate, float *scratch,
                            cudaStream_t st) {
    const int col_blocks = ceil_div(n_pat, kColsPerBlock);
    const int splits = row_splits_for(n_rot, col_blocks);
    const int rows_per_split = ceil_div(n_rot, splits);
    const int n_splits = ceil_div(n_rot, rows_per_split);
    float *part_m = scratch, *part_z = scratch + (size_t)64 * ld_n;
    if (!accumulate) {
        if (s) EMC_TRY_CUDA(cudaMemsetAsync(s, 0, sizeof(float) * n_rot, st));
        if (loglik) EMC_TRY_CUDA(cudaMemsetAsync(loglik, 0, sizeof(double), st));
    }
    dim3 grid(col_blocks, n_splits);
    colstats_kernel<<<grid, kThreads, 0, st>>>(L, weight, n_rot, n_pat, ld_n, rows_per_split, part_m, part_z);
    EMC_LAUNCHED();
    normalize_kernel<<<grid, kThreads, 0, st>>>(L, weight, n_rot, n_pat, ld_n, rows_per_split, n_splits, part_m,
                                                part_z, P, planes, n_planes, plane_stride, s, loglik);
    EMC_LAUNCHED();
    return EMC_OK;
}

emc_status launch_p_split(const float *P, int n_rot, int n_pat, int ld_n, __nv_bfloat16 *planes,
                          int ld_pl, int n_planes, size_t plane_stride, cudaStream_t st) {
    dim3 grid(n_rot, ceil_div(n_pat, 256));
    p_split_kernel<<<grid, 256, 0, st>>>(P, n_pat, ld_n, planes, ld_pl, n_planes, plane_stride);
    EMC_LAUNCHED();
    return EMC_OK;
}

emc_status launch_div_rows(float *Wnew, const float *s, int n_rot, int n_pix, cudaStream_t st) {
    dim3 grid(n_rot, ceil_div(n_pix, 256));
    div_rows_kernel<<<grid, 256, 0, st>>>(Wnew, s, n_pix);
    EMC_LAUNCHED();
    return EMC_OK;
}

}  // namespace emc
