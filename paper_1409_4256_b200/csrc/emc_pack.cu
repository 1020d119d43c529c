// Photon counts K[d][p] -> the exact 16-bit operands of the two contractions:
//   Kc [N][ld_p] fp16, row = pattern  (B operand of the log-likelihood GEMM, K-dim = pixels)
//   KT [P][ld_n] fp16, row = pixel    (B operand of the update GEMM,         K-dim = patterns)
// Masked pixels become 0 in both (G16).  Small integers are exact in fp16 up to 2048 = EMC_MAX_COUNT; an unmasked
// count above that is recorded in the workspace header: emc_check() reports it and the call's results are
// overwritten with NaN (poison_kernel) so that they cannot be consumed unnoticed.
#include "emc_internal.cuh"

namespace emc {

namespace {

constexpr int kTile = 64;

template <class T>
__global__ void __launch_bounds__(256)
pack_kernel(const T *__restrict__ counts, int n_pat, int n_pix, const uint8_t *__restrict__ mask,
            __half *__restrict__ Kc, int ld_p, __half *__restrict__ KT, int ld_n,
            WsHeader *__restrict__ hdr) {
    __shared__ float tile[kTile][kTile + 1];
    const int p0 = blockIdx.x * kTile, d0 = blockIdx.y * kTile;
    const int tx = threadIdx.x & 63, ty = threadIdx.x >> 6;   // 64 x 4
    int vmax = 0;
#pragma unroll 4
    for (int j = ty; j < kTile; j += 4) {
        const int d = d0 + j, p = p0 + tx;
        float v = 0.f;
        if (d < n_pat && p < n_pix) {
            const bool use = mask ? (mask[p] != 0) : true;
            if (use) {
                long long c = (long long)counts[(size_t)d * n_pix + p];
                if (c < 0) c = 0;
                vmax = max(vmax, (int)min(c, (long long)0x7fffffff));
                v = (float)min(c, (long long)65504);
            }
            if (Kc) Kc[(size_t)d * ld_p + p] = __float2half_rn(v);
        }
        tile[j][tx] = v;
    }
    __syncthreads();
    if (KT) {
#pragma unroll 4
        for (int j = ty; j < kTile; j += 4) {
            const int p = p0 + j, d = d0 + tx;
            if (p < n_pix && d < n_pat) {
                const size_t o = (size_t)p * ld_n + d;
                KT[o] = __float2half_rn(tile[tx][j]);
            }
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) vmax = max(vmax, __shfl_xor_sync(0xffffffffu, vmax, o));
    if ((threadIdx.x & 31) == 0 && vmax > EMC_MAX_COUNT) atomicMax(&hdr->max_count, vmax);
}

// uint16 counts with an even number of pixels (the configs' case): the same 64 x 64 tile, but every global access is
// 4 bytes per lane (two adjacent pixels in, half2 out; two adjacent patterns per half2 on the transposed side), which
// halves the instruction count of the 2-byte version above (it ran at 50 % issue, 22 % DRAM).
__global__ void __launch_bounds__(256)
pack_u16x2_kernel(const uint16_t *__restrict__ counts, int n_pat, int n_pix, const uint8_t *__restrict__ mask,
                  __half *__restrict__ Kc, int ld_p, __half *__restrict__ KT, int ld_n, WsHeader *__restrict__ hdr) {
    __shared__ float tile[kTile][kTile + 1];
    const int p0 = blockIdx.x * kTile, d0 = blockIdx.y * kTile;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;   // 32 lanes x 2 pixels, 8 rows at a time
    const int p = p0 + 2 * tx;
    bool use0 = false, use1 = false;
    if (p < n_pix) {                                           // n_pix even: p + 1 < n_pix too
        use0 = mask ? mask[p] != 0 : true;
        use1 = mask ? mask[p + 1] != 0 : true;
    }
    int vmax = 0;
#pragma unroll
    for (int j = ty; j < kTile; j += 8) {
        const int d = d0 + j;
        float v0 = 0.f, v1 = 0.f;
        if (d < n_pat && p < n_pix) {
            const uint32_t two = *reinterpret_cast<const uint32_t *>(counts + (size_t)d * n_pix + p);
            const int c0 = (int)(two & 0xffffu), c1 = (int)(two >> 16);
            if (use0) { vmax = max(vmax, c0); v0 = (float)c0; }
            if (use1) { vmax = max(vmax, c1); v1 = (float)c1; }
            if (Kc) *reinterpret_cast<__half2 *>(Kc + (size_t)d * ld_p + p) = __floats2half2_rn(v0, v1);
        }
        tile[j][2 * tx] = v0;
        tile[j][2 * tx + 1] = v1;
    }
    __syncthreads();
    if (KT) {
        const int d = d0 + 2 * tx;
#pragma unroll
        for (int j = ty; j < kTile; j += 8) {
            const int pp = p0 + j;
            if (pp < n_pix && d < n_pat)                       // ld_n is even: the half2 stays inside the row
                *reinterpret_cast<__half2 *>(KT + (size_t)pp * ld_n + d) =
                    __floats2half2_rn(tile[2 * tx][j], d + 1 < n_pat ? tile[2 * tx + 1][j] : 0.f);
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) vmax = max(vmax, __shfl_xor_sync(0xffffffffu, vmax, o));
    if ((threadIdx.x & 31) == 0 && vmax > EMC_MAX_COUNT) atomicMax(&hdr->max_count, vmax);
}

// A[d] = sum_{p: mask} K[d,p]^2 from the packed counts (masked pixels are already 0): the numerator of the
// fluence, eq. (2.6); stored as the two factors the Gaussian model's kernels use per column.  One warp per pattern; counts <= 2048 are exact in float and so are the squares.
__global__ void __launch_bounds__(256)
rowsq_kernel(const __half *__restrict__ Kc, int n_pat, int n_pix, int ld_p, float inv2s2, float *__restrict__ g_col,
             float *__restrict__ ia_col) {
    const int d = blockIdx.x * 8 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (d >= n_pat) return;
    const __half *row = Kc + (size_t)d * ld_p;
    float t = 0.f;
    for (int p = lane * 8; p < n_pix; p += 256) {              // ld_p is a multiple of 64: 16-byte loads stay in the row
        const uint4 v = *reinterpret_cast<const uint4 *>(row + p);
        const __half2 *h = reinterpret_cast<const __half2 *>(&v);
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const float2 f = __half22float2(h[j]);
            if (p + 2 * j < n_pix) t += f.x * f.x;
            if (p + 2 * j + 1 < n_pix) t += f.y * f.y;
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
    if (lane == 0) {                                          // the two per-column factors every (r, d) needs
        g_col[d] = gauss_col_factor(t, inv2s2);               // 1 / (2 sigma^2 A_d), 0 for a frame without photons
        ia_col[d] = t > 0.f ? 1.f / t : 0.f;                  // 1 / A_d
    }
}

// out[i] = NaN for every i if a count was out of range (grid-stride; a no-op launch otherwise)
__global__ void __launch_bounds__(256)
poison_kernel(const WsHeader *__restrict__ hdr, float *__restrict__ out, size_t n, double *__restrict__ out64, int n64) {
    if (hdr->max_count == 0 && hdr->shard_mismatch == 0) return;
    const float nan = __int_as_float(0x7fc00000);
    for (size_t i = (size_t)blockIdx.x * 256 + threadIdx.x; i < n; i += (size_t)gridDim.x * 256) out[i] = nan;
    if (blockIdx.x == 0 && (int)threadIdx.x < n64) out64[threadIdx.x] = (double)nan;
}

__global__ void shard_stamp_kernel(WsHeader *__restrict__ hdr, int n_rot, int n_pat, int n_pix, int verify) {
    if (threadIdx.x != 0) return;
    if (verify) {
        if (hdr->shard_stamp[0] != n_rot || hdr->shard_stamp[1] != n_pat || hdr->shard_stamp[2] != n_pix ||
            hdr->shard_stamp[3] != kShardTag)
            hdr->shard_mismatch = 1;
    } else {
        hdr->shard_stamp[0] = n_rot;
        hdr->shard_stamp[1] = n_pat;
        hdr->shard_stamp[2] = n_pix;
        hdr->shard_stamp[3] = kShardTag;
    }
}

}  // namespace

emc_status launch_shard_stamp(WsHeader *hdr, int n_rot, int n_pat, int n_pix, bool verify, cudaStream_t st) {
    shard_stamp_kernel<<<1, 32, 0, st>>>(hdr, n_rot, n_pat, n_pix, verify ? 1 : 0);
    EMC_LAUNCHED();
    return EMC_OK;
}

emc_status launch_poison(const WsHeader *hdr, float *out, size_t n, double *out64, int n64, cudaStream_t st) {
    if (n64 > 256) return EMC_ERR_UNSUPPORTED;
    poison_kernel<<<148, 256, 0, st>>>(hdr, out, out ? n : 0, out64, out64 ? n64 : 0);
    EMC_LAUNCHED();
    return EMC_OK;
}

emc_status launch_rowsq(const __half *Kc, int n_pat, int n_pix, int ld_p, float inv2s2, float *g_col, float *ia_col,
                        cudaStream_t st) {
    rowsq_kernel<<<ceil_div(n_pat, 8), 256, 0, st>>>(Kc, n_pat, n_pix, ld_p, inv2s2, g_col, ia_col);
    EMC_LAUNCHED();
    return EMC_OK;
}

emc_status launch_pack(const void *counts, emc_count_type type, int n_pat, int n_pix,
                       const uint8_t *mask, __half *Kc, int ld_p, __half *KT, int ld_n,
                       WsHeader *hdr, cudaStream_t st) {
    dim3 grid(ceil_div(n_pix, kTile), ceil_div(n_pat, kTile));
    switch (type) {
        case EMC_I32:
            pack_kernel<int32_t><<<grid, 256, 0, st>>>((const int32_t *)counts, n_pat, n_pix, mask, Kc, ld_p, KT, ld_n, hdr);
            break;
        case EMC_U16:
            if ((n_pix & 1) == 0 && (((uintptr_t)counts) & 3) == 0) {
                pack_u16x2_kernel<<<grid, 256, 0, st>>>((const uint16_t *)counts, n_pat, n_pix, mask, Kc, ld_p, KT, ld_n, hdr);
                break;
            }
            pack_kernel<uint16_t><<<grid, 256, 0, st>>>((const uint16_t *)counts, n_pat, n_pix, mask, Kc, ld_p, KT, ld_n, hdr);
            break;
        case EMC_U8:
            pack_kernel<uint8_t><<<grid, 256, 0, st>>>((const uint8_t *)counts, n_pat, n_pix, mask, Kc, ld_p, KT, ld_n, hdr);
            break;
        default:
            return EMC_ERR_ARG;
    }
    EMC_LAUNCHED();
    return EMC_OK;
}

}  // namespace emc
