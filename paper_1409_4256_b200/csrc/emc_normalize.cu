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

constexpr int kCols = 32;        // one lane per column: a warp reads 128 contiguous bytes of a row
constexpr int kWarps = 8;
constexpr int kThreads = kCols * kWarps;

__host__ __device__ inline int row_splits_for(int n_rot, int n_col_blocks) {
    int want = (4 * 148 + n_col_blocks - 1) / n_col_blocks;
    int cap = (n_rot + 63) / 64;
    if (cap > 64) cap = 64;
    if (want > cap) want = cap;
    return want < 1 ? 1 : want;
}

__device__ __forceinline__ float log_weight(const float *__restrict__ weight, int r, float log_uniform) {
    return weight ? logf(weight[r]) : log_uniform;
}

// sweep 1: partial (max, sum) of every column over the rows of one split
__global__ void __launch_bounds__(kThreads)
colstats_kernel(const float *__restrict__ L, const float *__restrict__ weight, int n_rot, int n_pat,
                int ld_n, int rows_per_split, float *__restrict__ part_m, float *__restrict__ part_z) {
    __shared__ float sm_m[kWarps][kCols], sm_z[kWarps][kCols];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int d = blockIdx.x * kCols + lane;
    const int r_lo = blockIdx.y * rows_per_split;
    const int r_hi = min(n_rot, r_lo + rows_per_split);
    const float log_uniform = -logf((float)n_rot);
    float m = -INFINITY, z = 0.f;
    if (d < n_pat) {
#pragma unroll 4
        for (int r = r_lo + warp; r < r_hi; r += kWarps) {
            const float a = L[(size_t)r * ld_n + d] + log_weight(weight, r, log_uniform);
            if (a > m) {
                z = z * expf(m - a) + 1.f;
                m = a;
            } else {
                z += expf(a - m);
            }
        }
    }
    sm_m[warp][lane] = m;
    sm_z[warp][lane] = z;
    __syncthreads();
    if (warp == 0 && d < n_pat) {
        float mt = sm_m[0][lane];
#pragma unroll
        for (int w = 1; w < kWarps; ++w) mt = fmaxf(mt, sm_m[w][lane]);
        float zt = 0.f;
#pragma unroll
        for (int w = 0; w < kWarps; ++w)
            if (sm_z[w][lane] > 0.f) zt += sm_z[w][lane] * expf(sm_m[w][lane] - mt);
        part_m[(size_t)blockIdx.y * ld_n + d] = mt;
        part_z[(size_t)blockIdx.y * ld_n + d] = zt;
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
    __shared__ float sm_m[kCols], sm_iz[kCols];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int d = blockIdx.x * kCols + lane;
    const int r_lo = blockIdx.y * rows_per_split;
    const int r_hi = min(n_rot, r_lo + rows_per_split);
    const float log_uniform = -logf((float)n_rot);
    if (warp == 0) {
        float mt = -INFINITY, zt = 1.f;
        double ll = 0.0;
        if (d < n_pat) {
            for (int k = 0; k < n_splits; ++k) mt = fmaxf(mt, part_m[(size_t)k * ld_n + d]);
            zt = 0.f;
            for (int k = 0; k < n_splits; ++k) {
                const float zk = part_z[(size_t)k * ld_n + d];
                if (zk > 0.f) zt += zk * expf(part_m[(size_t)k * ld_n + d] - mt);
            }
            ll = (double)mt + (double)logf(zt);
        }
        sm_m[lane] = mt;
        sm_iz[lane] = 1.f / zt;
        if (loglik && blockIdx.y == 0) {
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) ll += __shfl_xor_sync(0xffffffffu, ll, o);
            if (lane == 0) atomicAdd(loglik, ll);
        }
    }
    __syncthreads();
    const float mt = sm_m[lane], iz = sm_iz[lane];
    const bool col_ok = d < n_pat;
#pragma unroll 2
    for (int r = r_lo + warp; r < r_hi; r += kWarps) {
        float p = 0.f;
        const size_t o = (size_t)r * ld_n + d;
        if (col_ok) {
            const float a = L[o] + log_weight(weight, r, log_uniform);
            p = expf(a - mt) * iz;
            if (p < EMC_P_MIN) p = 0.f;          // DESIGN.md §3 G20
            if (P) P[o] = p;
            if (planes) split_bf16(p, n_planes, planes, plane_stride, o);
        }
        if (s) {
            float t = p;
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) t += __shfl_xor_sync(0xffffffffu, t, off);
            if (lane == 0) atomicAdd(s + r, t);
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
    const int col_blocks = ceil_div(n_pat, kCols);
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
