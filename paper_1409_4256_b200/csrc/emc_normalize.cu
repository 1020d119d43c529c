// Stage 3: normalisation of the likelihoods over the rotation space (reconstructed eq. (2.4),
// PAPER.md:78-80; "normalization ... in a separate final sweep"; "only maximal
// rotational probabilities and sums are necessary"):
//
//   a[r,d] = L[r,d] + log w_r;   m_d = max_r a;   P[r,d] = exp(a - m_d) / sum_r exp(a - m_d)
//
// Two sweeps (column-wise reductions on a row-major matrix):
// (1) per-column statistics (ColStat below) as partials over row ranges.  Inside emc_iterate they come from the
//     log-likelihood GEMM's epilogue, one partial per 32 rotations, and L is never read for them; the stage API
//     emc_normalize, which is handed an arbitrary L, uses colstats_kernel.  colstats_combine_kernel merges the
//     partials per column and adds up the total log-likelihood.
// (2) normalize_kernel reads L once and writes P, its operand planes for the update GEMM and s[r] = sum_d P[r,d].
// HBM-bound: 8 algorithmic bytes per (r,d).
#include <atomic>

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

// Column statistics are kept as a REFERENCE PAIR (mL, mw) = (L, log w) of the row with the largest a = L + log w seen
// so far, and z = sum exp((L - mL) + (log w - mw)).  Subtracting L from L and log w from log w before adding keeps
// the exponent accurate to its own magnitude; forming a = L + log w first would round it to ulp(|L|), which at
// |L| of a few thousand moves P by 1e-4 relative (T2 asks 1e-6 absolute).  With uniform weights the second
// difference is exactly 0.
struct ColStat {
    float mL, mw, z;
};
__device__ __forceinline__ float rel_exponent(float L, float lw, float mL, float mw) { return (L - mL) + (lw - mw); }
__device__ __forceinline__ void online(float L, float lw, ColStat &c) {
    if (!(L + lw > -INFINITY)) return;                 // w_r = 0 (log w = -inf) or L = -inf: the row takes no part
    if (L + lw > c.mL + c.mw) {
        c.z = c.z * expf(rel_exponent(c.mL, c.mw, L, lw)) + 1.f;      // z = 0 while the pair is (-inf, 0): 0 * 0
        c.mL = L;
        c.mw = lw;
    } else {
        c.z += expf(rel_exponent(L, lw, c.mL, c.mw));
    }
}
// merge b into a
__device__ __forceinline__ void merge(ColStat &a, const ColStat &b) {
    if (!(b.z > 0.f)) return;
    if (b.mL + b.mw > a.mL + a.mw) {
        a.z = a.z * expf(rel_exponent(a.mL, a.mw, b.mL, b.mw)) + b.z;
        a.mL = b.mL;
        a.mw = b.mw;
    } else {
        a.z += b.z * expf(rel_exponent(b.mL, b.mw, a.mL, a.mw));
    }
}

// sweep 1: partial statistics of every column over the rows of one split (stage API; inside emc_iterate the
// log-likelihood GEMM's epilogue writes the same partials, one per 32 rows)
__global__ void __launch_bounds__(kThreads)
colstats_kernel(const float *__restrict__ L, const float *__restrict__ weight, float log_uniform, int n_rot, int n_pat,
                int ld_n, int rows_per_split, float *__restrict__ part_m, float *__restrict__ part_w,
                float *__restrict__ part_z) {
    __shared__ float sm_m[kWarps][kColsPerBlock], sm_w[kWarps][kColsPerBlock], sm_z[kWarps][kColsPerBlock];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int d = blockIdx.x * kColsPerBlock + lane * kVec;
    const int r_lo = blockIdx.y * rows_per_split;
    const int r_hi = min(n_rot, r_lo + rows_per_split);
    ColStat c[kVec];
#pragma unroll
    for (int j = 0; j < kVec; ++j) c[j] = ColStat{-INFINITY, 0.f, 0.f};
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
                    online(v[b].x, lw[b], c[0]);
                    online(v[b].y, lw[b], c[1]);
                    online(v[b].z, lw[b], c[2]);
                    online(v[b].w, lw[b], c[3]);
                }
            }
        }
    }
#pragma unroll
    for (int j = 0; j < kVec; ++j) {
        sm_m[warp][lane * kVec + j] = c[j].mL;
        sm_w[warp][lane * kVec + j] = c[j].mw;
        sm_z[warp][lane * kVec + j] = c[j].z;
    }
    __syncthreads();
    if (warp == 0 && d < n_pat) {
#pragma unroll
        for (int j = 0; j < kVec; ++j) {
            ColStat t = ColStat{-INFINITY, 0.f, 0.f};
#pragma unroll
            for (int w = 0; w < kWarps; ++w) merge(t, ColStat{sm_m[w][lane * kVec + j], sm_w[w][lane * kVec + j], sm_z[w][lane * kVec + j]});
            const size_t o = (size_t)blockIdx.y * ld_n + d + j;
            part_m[o] = t.mL;
            part_w[o] = t.mw;
            part_z[o] = t.z;
        }
    }
}

// ---- operand planes of P for the update contraction -------------------------------------------
// Two fp16 planes with one power-of-two scale per (row, 512-column chunk): the chunk is scaled so
// that its largest value lies in [2^14, 2^15), then hi = fp16(v), lo = fp16(v - hi).  The update
// GEMM accumulates each 512-element K chunk separately and applies the inverse scale when it drains
// the chunk (exact), so fp16's narrow exponent only has to span one chunk of one row: 22
// significand bits for every value within 2^-17 of the chunk maximum and an absolute error below
// 2^-40 of the chunk maximum for the rest.  P covers float32's whole normal range
// [2^-126, 1] (EMC_P_MIN), so the scale 2^k, k = 14 - floor(log2 max) <= 140, is applied as two exact
// factors 2^(k/2) 2^(k - k/2) and its inverse 2^-k (a float32 subnormal below 2^-126, still an exact
// power of two down to 2^-149) multiplies the chunk's sum in the GEMM's drain.
constexpr int kChunkCols = 512;               // = the GEMM's K chunk (kChunkKBlocks * 64)
constexpr int kGroups = kChunkCols / kColsPerBlock;   // float4 groups per lane per row

__device__ __forceinline__ float warp_max(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}
__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// exact 2^e for -149 <= e <= 127 (subnormal below -126)
__device__ __forceinline__ float pow2_exact(int e) {
    return e >= -126 ? __uint_as_float((uint32_t)(e + 127) << 23) : __uint_as_float(1u << (e + 149));
}
// 2^k = s1 * s2 with k = 14 - floor(log2 mx), and inv = 2^-k; mx = 0 gives 1, 1, 1.  mx is a float32 in
// [2^-126, 2^15) here (P >= EMC_P_MIN; the Gaussian operand P / phi may be a subnormal: its exponent field reads
// -127 and the chunk simply keeps fewer bits).
__device__ __forceinline__ void chunk_scale_of(float mx, float &s1, float &s2, float &inv) {
    if (mx > 0.f) {
        const int k = 14 - ((int)((__float_as_uint(mx) >> 23) & 0xffu) - 127);      // -1 <= k <= 141
        const int k1 = k / 2;
        s1 = pow2_exact(k1);
        s2 = pow2_exact(k - k1);
        inv = pow2_exact(-k);
    } else {
        s1 = s2 = inv = 1.f;
    }
}

__device__ __forceinline__ void store4_f16_pair(const float (&v)[4], __half *__restrict__ planes, size_t plane_stride,
                                                size_t o) {
    __half h[4], l[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        h[j] = __float2half_rn(v[j]);
        l[j] = __float2half_rn(v[j] - __half2float(h[j]));
    }
    *reinterpret_cast<uint2 *>(planes + o) = *reinterpret_cast<const uint2 *>(h);
    *reinterpret_cast<uint2 *>(planes + plane_stride + o) = *reinterpret_cast<const uint2 *>(l);
}

// One row x one 512-column chunk held by a warp (p[g][4] = columns d0 + g*128 + lane*4 ..+3): writes the
// operand planes and the chunk's inverse scale.
__device__ __forceinline__ void write_planes(float (&p)[kGroups][4], int d0, int lane, int ld_pl, size_t row_off,
                                             __half *__restrict__ planes, size_t plane_stride,
                                             float *__restrict__ inv_scale_out) {
    float mx = 0.f;
#pragma unroll
    for (int g = 0; g < kGroups; ++g)
        mx = fmaxf(mx, fmaxf(fmaxf(p[g][0], p[g][1]), fmaxf(p[g][2], p[g][3])));
    mx = warp_max(mx);
    float s1, s2, inv;
    chunk_scale_of(mx, s1, s2, inv);
    if (lane == 0) *inv_scale_out = inv;
#pragma unroll
    for (int g = 0; g < kGroups; ++g) {
        const int d = d0 + g * kColsPerBlock + lane * kVec;
        if (d < ld_pl) {
            const float v[4] = {(p[g][0] * s1) * s2, (p[g][1] * s1) * s2, (p[g][2] * s1) * s2, (p[g][3] * s1) * s2};
            store4_f16_pair(v, planes, plane_stride, row_off + d);
        }
    }
}

// between the sweeps: per column, combine the split partials into (max, 1/sum) and add up the total
// log-likelihood  LL = sum_d (m_d + log z_d).  block = 32 columns x 8 row lanes; row lane y merges the
// partials k = y, y + 8, ... online, then the 8 are merged through shared memory.
__global__ void __launch_bounds__(256)
colstats_combine_kernel(float *__restrict__ part_m, float *__restrict__ part_w,
                        float *__restrict__ part_z, int n_pat, int ld_n, int n_store, int n_splits,
                        float *__restrict__ col_m, float *__restrict__ col_w, float *__restrict__ col_iz,
                        double *__restrict__ loglik, int carry_row, int carry_in) {
    __shared__ float sm_m[8][32], sm_w[8][32], sm_z[8][32];
    const int x = threadIdx.x & 31, y = threadIdx.x >> 5;
    const int d = blockIdx.x * 32 + x;
    ColStat t = ColStat{-INFINITY, 0.f, 0.f};
    if (d < n_pat) {
        for (int k0 = y; k0 < n_splits; k0 += 8 * 4) {               // 4 independent partials in flight
            ColStat c[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int k = k0 + 8 * u;
                const size_t o = (size_t)k * ld_n + d;
                c[u] = k < n_splits ? ColStat{part_m[o], part_w[o], part_z[o]} : ColStat{-INFINITY, 0.f, 0.f};
            }
#pragma unroll
            for (int u = 0; u < 4; ++u) merge(t, c[u]);
        }
    }
    sm_m[y][x] = t.mL;
    sm_w[y][x] = t.mw;
    sm_z[y][x] = t.z;
    __syncthreads();
    if (y != 0) return;
    double ll = 0.0;
    if (d < n_pat) {
#pragma unroll
        for (int k = 1; k < 8; ++k) merge(t, ColStat{sm_m[k][x], sm_w[k][x], sm_z[k][x]});
        // rotation chunks: row `carry_row` of the partial arrays holds the statistics of the chunks seen
        // so far; merge them in and hand the result on
        if (carry_row >= 0) {
            const size_t o = (size_t)carry_row * ld_n + d;
            if (carry_in) merge(t, ColStat{part_m[o], part_w[o], part_z[o]});
            part_m[o] = t.mL;
            part_w[o] = t.mw;
            part_z[o] = t.z;
        }
        col_m[d] = t.mL;
        col_w[d] = t.mw;
        col_iz[d] = 1.f / t.z;
        ll = ((double)t.mL + (double)t.mw) + (double)logf(t.z);
    } else if (d < n_store) {
        col_m[d] = 0.f;
        col_w[d] = 0.f;
        col_iz[d] = 0.f;
    }
    if (loglik) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) ll += __shfl_xor_sync(0xffffffffu, ll, o);
        if (x == 0) atomicAdd(loglik, ll);
    }
}

// sweep 2: write P / planes / s.  grid = (ceil(N/512), row splits); a warp owns one row x 512 columns at a
// time and prefetches the next row while it works on the current one.
// UNIFORM = no weight array: log w is the same for every row and drops out of (L - mL) + (log w - mw).
template <bool UNIFORM>
__global__ void __launch_bounds__(kThreads, UNIFORM ? 3 : 2)
normalize_kernel(const float *__restrict__ L, const float *__restrict__ weight, int n_rot, int n_pat,
                 int ld_n, int n_store, int rows_per_split, const float *__restrict__ col_m, const float *__restrict__ col_w,
                 const float *__restrict__ col_iz, float *__restrict__ P, __half *__restrict__ planes, size_t plane_stride,
                 float *__restrict__ chunk_inv_scale, float *__restrict__ s) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int d0 = blockIdx.x * kChunkCols;
    const int r_lo = blockIdx.y * rows_per_split;
    const int r_hi = min(n_rot, r_lo + rows_per_split);
    float4 mt[kGroups], mw[UNIFORM ? 1 : kGroups], iz[kGroups];
    bool ok[kGroups];
#pragma unroll
    for (int g = 0; g < kGroups; ++g) {
        const int d = d0 + g * kColsPerBlock + lane * kVec;
        ok[g] = d < n_pat;                              // col_m / col_w / col_iz are defined (0) up to ld_n
        mt[g] = ok[g] ? *reinterpret_cast<const float4 *>(col_m + d) : make_float4(0.f, 0.f, 0.f, 0.f);
        iz[g] = ok[g] ? *reinterpret_cast<const float4 *>(col_iz + d) : make_float4(0.f, 0.f, 0.f, 0.f);
        if (!UNIFORM) mw[g] = ok[g] ? *reinterpret_cast<const float4 *>(col_w + d) : make_float4(0.f, 0.f, 0.f, 0.f);
    }
    float4 nxt[kGroups];
    int r = r_lo + warp;
    if (r < r_hi) {
#pragma unroll
        for (int g = 0; g < kGroups; ++g)
            if (ok[g]) nxt[g] = *reinterpret_cast<const float4 *>(L + (size_t)r * ld_n + d0 + g * kColsPerBlock + lane * kVec);
    }
    for (; r < r_hi; r += kWarps) {
        float4 v[kGroups];
#pragma unroll
        for (int g = 0; g < kGroups; ++g) v[g] = nxt[g];
        if (r + kWarps < r_hi) {
#pragma unroll
            for (int g = 0; g < kGroups; ++g)
                if (ok[g])
                    nxt[g] = *reinterpret_cast<const float4 *>(L + (size_t)(r + kWarps) * ld_n + d0 + g * kColsPerBlock + lane * kVec);
        }
        const float lw = UNIFORM ? 0.f : logf(weight[r]);
        const size_t row_off = (size_t)r * ld_n;
        float p[kGroups][4];
        float sum = 0.f;
#pragma unroll
        for (int g = 0; g < kGroups; ++g) {
            const int d = d0 + g * kColsPerBlock + lane * kVec;
            const float a[4] = {v[g].x, v[g].y, v[g].z, v[g].w};
            const float m4[4] = {mt[g].x, mt[g].y, mt[g].z, mt[g].w};
            const float z4[4] = {iz[g].x, iz[g].y, iz[g].z, iz[g].w};
            float w4[4] = {0.f, 0.f, 0.f, 0.f};
            if (!UNIFORM) { w4[0] = lw - mw[g].x; w4[1] = lw - mw[g].y; w4[2] = lw - mw[g].z; w4[3] = lw - mw[g].w; }
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                float pj = 0.f;
                if (d + j < n_pat) {
                    pj = expf(UNIFORM ? a[j] - m4[j] : (a[j] - m4[j]) + w4[j]) * z4[j];
                    if (pj < EMC_P_MIN) pj = 0.f;                      // DESIGN.md §3 G20
                }
                p[g][j] = pj;
                sum += pj;
            }
            if (P && ok[g]) *reinterpret_cast<float4 *>(P + row_off + d) = make_float4(p[g][0], p[g][1], p[g][2], p[g][3]);
        }
        if (planes)
            write_planes(p, d0, lane, n_store, row_off, planes, plane_stride,
                         chunk_inv_scale + (size_t)blockIdx.x * n_rot + r);
        if (s) {
            sum = warp_sum(sum);
            if (lane == 0) atomicAdd(s + r, sum);
        }
    }
}

// Second sweep for the paper's Gaussian model (NEXT-3): the "L" buffer holds B[r,d] = sum_p W K.
//   Q = B^2 g_d + (log w_r - C_r / (2 sigma^2))   (same two terms, bit for bit, as the GEMM's statistics),
//   P = exp((B^2 g_d - mL_d) + (lw'_r - mw_d)) / z_d,   update operand = P / phi = P B / A_d   (eq. 2.11).
// Same thread layout as normalize_kernel; column data is re-read per row (L1-resident) to keep registers free.
__global__ void __launch_bounds__(kThreads, 2)
normalize_gauss_kernel(const float *__restrict__ B, const float *__restrict__ weight, const float *__restrict__ c_row,
                       const float *__restrict__ g_col, const float *__restrict__ ia_col, float inv2s2, float log_uniform,
                       int n_rot, int n_pat, int ld_n, int n_store, int rows_per_split,
                       const float *__restrict__ col_m, const float *__restrict__ col_w, const float *__restrict__ col_iz,
                       float *__restrict__ P, __half *__restrict__ planes, size_t plane_stride,
                       float *__restrict__ chunk_inv_scale, float *__restrict__ s) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int d0 = blockIdx.x * kChunkCols;
    const int r_lo = blockIdx.y * rows_per_split;
    const int r_hi = min(n_rot, r_lo + rows_per_split);
    // the column statistics stay in registers for the whole row range; the two Gaussian column factors are re-read per
    // row (L1-resident); the next row of B is fetched while the current one is worked on
    const float4 z4 = make_float4(0.f, 0.f, 0.f, 0.f);
    float4 cm[kGroups], cw[kGroups], ci[kGroups], nxt[kGroups];
    bool okg[kGroups];
#pragma unroll
    for (int g = 0; g < kGroups; ++g) {
        const int d = d0 + g * kColsPerBlock + lane * kVec;
        okg[g] = d < n_pat;                             // ld_n is a multiple of 4: whole float4s
        cm[g] = okg[g] ? *reinterpret_cast<const float4 *>(col_m + d) : z4;
        cw[g] = okg[g] ? *reinterpret_cast<const float4 *>(col_w + d) : z4;
        ci[g] = okg[g] ? *reinterpret_cast<const float4 *>(col_iz + d) : z4;
        nxt[g] = z4;
    }
    int r = r_lo + warp;
    if (r < r_hi) {
#pragma unroll
        for (int g = 0; g < kGroups; ++g)
            if (okg[g]) nxt[g] = *reinterpret_cast<const float4 *>(B + (size_t)r * ld_n + d0 + g * kColsPerBlock + lane * kVec);
    }
    for (; r < r_hi; r += kWarps) {
        float4 cur[kGroups];
#pragma unroll
        for (int g = 0; g < kGroups; ++g) cur[g] = nxt[g];
        if (r + kWarps < r_hi) {
#pragma unroll
            for (int g = 0; g < kGroups; ++g)
                if (okg[g])
                    nxt[g] = *reinterpret_cast<const float4 *>(B + (size_t)(r + kWarps) * ld_n + d0 + g * kColsPerBlock + lane * kVec);
        }
        const float lw = gauss_row_term(weight ? logf(weight[r]) : log_uniform, c_row[r], inv2s2);
        const size_t row_off = (size_t)r * ld_n;
        float p[kGroups][4], q[kGroups][4];
        float sum = 0.f;
#pragma unroll
        for (int g = 0; g < kGroups; ++g) {
            const int d = d0 + g * kColsPerBlock + lane * kVec;
            const bool ok = okg[g];
            const float4 b4 = cur[g], m4 = cm[g], w4 = cw[g], i4 = ci[g];
            const float4 a4 = ok ? __ldg(reinterpret_cast<const float4 *>(ia_col + d)) : z4;
            const float4 g4 = ok ? __ldg(reinterpret_cast<const float4 *>(g_col + d)) : z4;
            const float bb[4] = {b4.x, b4.y, b4.z, b4.w}, mm[4] = {m4.x, m4.y, m4.z, m4.w};
            const float ww[4] = {w4.x, w4.y, w4.z, w4.w}, ii[4] = {i4.x, i4.y, i4.z, i4.w};
            const float aa[4] = {a4.x, a4.y, a4.z, a4.w}, gg[4] = {g4.x, g4.y, g4.z, g4.w};
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                float pj = 0.f, qj = 0.f;
                if (d + j < n_pat) {
                    const float e = gauss_elem_term(bb[j], gg[j]);
                    pj = expf((e - mm[j]) + (lw - ww[j])) * ii[j];
                    if (pj < EMC_P_MIN) pj = 0.f;                      // DESIGN.md §3 G20
                    qj = pj * (bb[j] * aa[j]);                         // P / phi = P B / A (GA3: 1/A = 0 without photons)
                }
                p[g][j] = pj;
                q[g][j] = qj;
                sum += pj;
            }
            if (P && ok) *reinterpret_cast<float4 *>(P + row_off + d) = make_float4(p[g][0], p[g][1], p[g][2], p[g][3]);
        }
        if (planes)
            write_planes(q, d0, lane, n_store, row_off, planes, plane_stride,
                         chunk_inv_scale + (size_t)blockIdx.x * n_rot + r);
        if (s) {
            sum = warp_sum(sum);
            if (lane == 0) atomicAdd(s + r, sum);
        }
    }
}

// operand planes of a given P (stage API of emc_update).  grid = (ceil(N/512), ceil(R/8)); warp per row.
__global__ void __launch_bounds__(kThreads)
p_split_kernel(const float *__restrict__ P, int n_rot, int n_pat, int ld_n, __half *__restrict__ planes, int ld_pl,
               size_t plane_stride, float *__restrict__ chunk_inv_scale) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int r = blockIdx.y * kWarps + warp;
    if (r >= n_rot) return;
    const int d0 = blockIdx.x * kChunkCols;
    float p[kGroups][4];
#pragma unroll
    for (int g = 0; g < kGroups; ++g) {
        const int d = d0 + g * kColsPerBlock + lane * kVec;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            float pj = (d + j < n_pat) ? P[(size_t)r * ld_n + d + j] : 0.f;
            if (pj < EMC_P_MIN) pj = 0.f;
            p[g][j] = pj;
        }
    }
    write_planes(p, d0, lane, ld_pl, (size_t)r * ld_pl, planes, plane_stride,
                 chunk_inv_scale + (size_t)blockIdx.x * n_rot + r);
}

// stage API of the Gaussian model: the E-step's exponent and the fluence themselves
__global__ void __launch_bounds__(256)
gauss_q_kernel(const float *__restrict__ B, const float *__restrict__ c_row, const float *__restrict__ g_col,
               const float *__restrict__ ia_col, float inv2s2, int n_pat, int ld_b, float *__restrict__ Q,
               float *__restrict__ phi, int ld_out) {
    const int d = blockIdx.y * 256 + threadIdx.x, r = blockIdx.x;
    if (d >= n_pat) return;
    const float b = B[(size_t)r * ld_b + d];
    // the same two terms, formed the same way, as the GEMM epilogue's statistics and the second sweep (emc_internal.cuh)
    if (Q) Q[(size_t)r * ld_out + d] = __fadd_rn(gauss_elem_term(b, g_col[d]), gauss_row_term(0.f, c_row[r], inv2s2));
    if (phi) {
        const float ia = ia_col[d];
        phi[(size_t)r * ld_out + d] = (b > 0.f && ia > 0.f) ? 1.f / (b * ia) : INFINITY;      // GA3: K / phi = 0
    }
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

// rows of the partial-statistics arrays: the column sweep uses at most 64 row splits, the fused GEMM epilogue
// (emc_gemm.cu store_row_and_col_stats) one per 32 rotations
int normalize_stat_rows(int n_rot) {
    const int fused = ceil_div(n_rot, 32);
    return (fused > 64 ? fused : 64) + 1;              // + the carry row of rotation chunks
}

size_t normalize_scratch_floats(int n_rot, int ld_n) {
    return (size_t)(3 * normalize_stat_rows(n_rot) + 3) * (size_t)ld_n;   // partials (mL, mw, z) + combined (mL, mw, 1/z)
}

emc_status launch_normalize(const float *L, const float *weight, int n_rot, int n_pat, int ld_n,
                            float *P, __half *planes, size_t plane_stride, float *chunk_inv_scale,
                            float *s, double *loglik, bool accumulate, float *scratch, bool stats_ready,
                            cudaStream_t st, const GaussTerms *gauss, int n_store, float log_uniform, int chunk_mode,
                            bool carry_in, int layout_rot) {
    if (n_store <= 0 || n_store > ld_n) n_store = ld_n;          // columns of a row this call may write
    if (log_uniform == 0.f) log_uniform = log_uniform_of(n_rot);
    if (gauss && !stats_ready) return EMC_ERR_UNSUPPORTED;       // the Gaussian model's statistics come from the GEMM
    const int stat_rows = normalize_stat_rows(layout_rot > 0 ? layout_rot : n_rot);
    float *part_m = scratch, *part_w = part_m + (size_t)stat_rows * ld_n, *part_z = part_w + (size_t)stat_rows * ld_n;
    if (!accumulate) {
        if (s) EMC_TRY_CUDA(cudaMemsetAsync(s, 0, sizeof(float) * n_rot, st));
        if (loglik) EMC_TRY_CUDA(cudaMemsetAsync(loglik, 0, sizeof(double), st));
    }
    float *col_m = scratch + (size_t)3 * stat_rows * ld_n, *col_w = col_m + ld_n, *col_iz = col_w + ld_n;
    int n_splits = 0;
    if (chunk_mode == 2) {
        // second sweep of a rotation chunk: the final column statistics are in place
    } else if (stats_ready) {
        n_splits = ceil_div(n_rot, 32);               // written by the log-likelihood GEMM's epilogue
    } else {
        const int col_blocks = ceil_div(n_pat, kColsPerBlock);
        const int splits = row_splits_for(n_rot, col_blocks);
        const int rows_per_split = ceil_div(n_rot, splits);
        n_splits = ceil_div(n_rot, rows_per_split);
        colstats_kernel<<<dim3(col_blocks, n_splits), kThreads, 0, st>>>(L, weight, log_uniform, n_rot, n_pat, ld_n,
                                                                         rows_per_split, part_m, part_w, part_z);
        EMC_LAUNCHED();
    }
    if (chunk_mode != 2) {
        colstats_combine_kernel<<<ceil_div(n_store, 32), 256, 0, st>>>(part_m, part_w, part_z, n_pat, ld_n, n_store, n_splits, col_m,
                                                                     col_w, col_iz, chunk_mode == 2 ? nullptr : loglik,
                                                                     chunk_mode == 1 ? stat_rows - 1 : -1, carry_in ? 1 : 0);
        EMC_LAUNCHED();
    }
    if (chunk_mode == 1) return EMC_OK;                 // first sweep of a rotation chunk: statistics only
    // second sweep: 512-column chunks; row splits so that the grid is at most 6 x 148 blocks = whole waves of the 2 or 3
    // blocks per SM the kernels run at (one block more is a wave more: a quarter of the time at C2)
    const int chunks = ceil_div(n_pat, kChunkCols);
    int splits2 = (6 * 148) / chunks;
    const int cap2 = ceil_div(n_rot, 4 * kWarps);
    if (splits2 > cap2) splits2 = cap2;
    if (splits2 < 1) splits2 = 1;
    const int rows2 = ceil_div(n_rot, splits2);
    const dim3 grid2(chunks, ceil_div(n_rot, rows2));
    if (gauss)
        normalize_gauss_kernel<<<grid2, kThreads, 0, st>>>(L, weight, gauss->c_row, gauss->g_col, gauss->ia_col, gauss->inv2s2,
                                                           gauss->log_uniform, n_rot, n_pat, ld_n, n_store, rows2, col_m, col_w,
                                                           col_iz, P, planes, plane_stride, chunk_inv_scale, s);
    else if (weight)
        normalize_kernel<false><<<grid2, kThreads, 0, st>>>(L, weight, n_rot, n_pat, ld_n, n_store, rows2, col_m, col_w, col_iz, P,
                                                            planes, plane_stride, chunk_inv_scale, s);
    else
        normalize_kernel<true><<<grid2, kThreads, 0, st>>>(L, weight, n_rot, n_pat, ld_n, n_store, rows2, col_m, col_w, col_iz, P,
                                                           planes, plane_stride, chunk_inv_scale, s);
    EMC_LAUNCHED();
    return EMC_OK;
}

void normalize_stat_row(float *scratch, int layout_rot, int ld_n, int row, float **m, float **w, float **z) {
    const size_t stat_rows = (size_t)normalize_stat_rows(layout_rot);
    if (row < 0) row = (int)stat_rows - 1;                       // the carry row
    *m = scratch + (size_t)row * ld_n;
    *w = *m + stat_rows * ld_n;
    *z = *w + stat_rows * ld_n;
}

emc_status launch_colstats_combine_rows(float *scratch, int layout_rot, int n_rows, int n_pat, int ld_n, double *loglik,
                                        cudaStream_t st) {
    const int stat_rows = normalize_stat_rows(layout_rot);
    if (n_rows > stat_rows) return EMC_ERR_UNSUPPORTED;
    float *part_m = scratch, *part_w = part_m + (size_t)stat_rows * ld_n, *part_z = part_w + (size_t)stat_rows * ld_n;
    float *col_m = scratch + (size_t)3 * stat_rows * ld_n, *col_w = col_m + ld_n, *col_iz = col_w + ld_n;
    colstats_combine_kernel<<<ceil_div(ld_n, 32), 256, 0, st>>>(part_m, part_w, part_z, n_pat, ld_n, ld_n, n_rows, col_m, col_w, col_iz,
                                                               loglik, -1, 0);
    EMC_LAUNCHED();
    return EMC_OK;
}

emc_status launch_p_split(const float *P, int n_rot, int n_pat, int ld_n, __half *planes, int ld_pl,
                          size_t plane_stride, float *chunk_inv_scale, cudaStream_t st) {
    dim3 grid(ceil_div(n_pat, kChunkCols), ceil_div(n_rot, kWarps));
    p_split_kernel<<<grid, kThreads, 0, st>>>(P, n_rot, n_pat, ld_n, planes, ld_pl, plane_stride, chunk_inv_scale);
    EMC_LAUNCHED();
    return EMC_OK;
}

emc_status launch_gauss_q(const float *B, const float *c_row, const float *g_col, const float *ia_col, float inv2s2, int n_rot,
                          int n_pat, int ld_b, float *Q, float *phi, int ld_out, cudaStream_t st) {
    gauss_q_kernel<<<dim3(n_rot, ceil_div(n_pat, 256)), 256, 0, st>>>(B, c_row, g_col, ia_col, inv2s2, n_pat, ld_b, Q, phi, ld_out);
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

// ---------------------------------------------------------------- emc_normalize_static (include/emc.h)
// Stage 3 for callers that cannot allocate device memory (a plug-in with fixed buffers, an acquisition loop that must
// stay off the allocator's device-wide lock, a process whose pool is spent): the partial column statistics of the
// first sweep live in an array that is part of the library image instead of the caller's workspace.  The array costs
// EMC_STATIC_SCRATCH_BYTES on every GPU that loads libemc, for the life of the process.  The kernels are the ones
// emc_normalize runs (colstats_kernel, colstats_combine_kernel, normalize_kernel), with the same row splits.
//
// `emc_static_scratch` below is a device object.  On the host its name is only a handle for the runtime's symbol
// table -- passing it to a kernel would hand the kernel a host address -- so the host asks the runtime once per device
// where the object lives (cudaGetSymbolAddress, that device current) and passes THAT pointer.
static __device__ __align__(256) float emc_static_scratch[EMC_STATIC_SCRATCH_BYTES / sizeof(float)];

namespace emc {
namespace {

constexpr int kMaxDevices = 64;
std::atomic<float *> g_static_scratch_addr[kMaxDevices];   // device address of emc_static_scratch, per device ordinal

// Address of the array on the current device.  The first call on a device does the look-up (the documented set-up
// step: outside stream capture); two threads racing here both obtain the same address, so a plain store suffices.
emc_status static_scratch_on_current_device(float **out) {
    int dev = -1;
    EMC_TRY_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices) return EMC_ERR_UNSUPPORTED;
    float *p = g_static_scratch_addr[dev].load(std::memory_order_acquire);
    if (!p) {
        void *sym = nullptr;
        EMC_TRY_CUDA(cudaGetSymbolAddress(&sym, emc_static_scratch));
        if (!sym || ((uintptr_t)sym & 255)) return EMC_ERR_CUDA;
        p = (float *)sym;
        g_static_scratch_addr[dev].store(p, std::memory_order_release);
    }
    *out = p;
    return EMC_OK;
}

// the row splits launch_normalize takes when the statistics do not come from the GEMM, and the floats they need:
// three partial arrays [n_splits][ld_n] and the three combined column arrays [ld_n]
struct StaticPlan {
    int col_blocks, rows_per_split, n_splits;
    size_t floats;
};
bool static_plan(int n_rot, int n_pat, int ld_n, StaticPlan *pl) {
    if (n_rot <= 0 || n_pat <= 0 || ld_n < n_pat || (ld_n & 3)) return false;
    pl->col_blocks = ceil_div(n_pat, kColsPerBlock);
    const int splits = row_splits_for(n_rot, pl->col_blocks);
    pl->rows_per_split = ceil_div(n_rot, splits);
    pl->n_splits = ceil_div(n_rot, pl->rows_per_split);
    pl->floats = (size_t)(3 * pl->n_splits + 3) * (size_t)ld_n;
    return true;
}

}  // namespace
}  // namespace emc

extern "C" {

size_t emc_normalize_static_bytes(int n_rot, int n_pat, int ld_n) {
    emc::StaticPlan pl;
    return emc::static_plan(n_rot, n_pat, ld_n, &pl) ? pl.floats * sizeof(float) : 0;
}

emc_status emc_normalize_static(const float *L, const emc_rotations *rot, int n_pat, int ld_n, float *P, float *s,
                                double *loglik, unsigned flags, void *stream) {
    using namespace emc;
    StaticPlan pl;
    if (!L || !rot || !P || ((uintptr_t)L & 15) || ((uintptr_t)P & 15) || !static_plan(rot->n_rot, n_pat, ld_n, &pl))
        return EMC_ERR_ARG;
    if (pl.floats * sizeof(float) > EMC_STATIC_SCRATCH_BYTES) return EMC_ERR_STATIC_SCRATCH;   // nothing enqueued
    float *scratch = nullptr;
    EMC_TRY(static_scratch_on_current_device(&scratch));
    cudaStream_t st = (cudaStream_t)stream;
    const int n_rot = rot->n_rot;
    const float *weight = rot->weight;
    const size_t plane = (size_t)pl.n_splits * ld_n;
    float *part_m = scratch, *part_w = part_m + plane, *part_z = part_w + plane;
    float *col_m = part_z + plane, *col_w = col_m + ld_n, *col_iz = col_w + ld_n;
    // results the kernels add into start at zero; the scratch needs no clearing (every element read below is written
    // by the kernel before it: partials for d < n_pat and k < n_splits, column arrays up to ld_n)
    if (!(flags & EMC_ACCUMULATE)) {
        if (s) EMC_TRY_CUDA(cudaMemsetAsync(s, 0, sizeof(float) * n_rot, st));
        if (loglik) EMC_TRY_CUDA(cudaMemsetAsync(loglik, 0, sizeof(double), st));
    }
    colstats_kernel<<<dim3(pl.col_blocks, pl.n_splits), kThreads, 0, st>>>(L, weight, log_uniform_of(n_rot), n_rot, n_pat, ld_n,
                                                                           pl.rows_per_split, part_m, part_w, part_z);
    EMC_LAUNCHED();
    colstats_combine_kernel<<<ceil_div(ld_n, 32), 256, 0, st>>>(part_m, part_w, part_z, n_pat, ld_n, ld_n, pl.n_splits, col_m, col_w,
                                                               col_iz, loglik, -1, 0);
    EMC_LAUNCHED();
    // second sweep: the grid emc_normalize uses (512-column chunks, at most 6 x 148 blocks)
    const int chunks = ceil_div(n_pat, kChunkCols);
    int splits2 = (6 * 148) / chunks;
    const int cap2 = ceil_div(n_rot, 4 * kWarps);
    if (splits2 > cap2) splits2 = cap2;
    if (splits2 < 1) splits2 = 1;
    const int rows2 = ceil_div(n_rot, splits2);
    const dim3 grid2(chunks, ceil_div(n_rot, rows2));
    if (weight)
        normalize_kernel<false><<<grid2, kThreads, 0, st>>>(L, weight, n_rot, n_pat, ld_n, ld_n, rows2, col_m, col_w, col_iz, P,
                                                            nullptr, 0, nullptr, s);
    else
        normalize_kernel<true><<<grid2, kThreads, 0, st>>>(L, weight, n_rot, n_pat, ld_n, ld_n, rows2, col_m, col_w, col_iz, P,
                                                           nullptr, 0, nullptr, s);
    EMC_LAUNCHED();
    return EMC_OK;
}

}  // extern "C"
