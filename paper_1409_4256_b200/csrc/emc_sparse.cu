// Photon-list (sparse) form of stages 2 and 4 for frames that are almost empty (BASELINE.json config 4: 0.01 photons
// per pixel, > 99 % zeros).  EMC_SPARSE_PHOTONS selects it inside emc_iterate; the
// dense tensor-core contractions stay the default (DESIGN.md section 11 has the measured comparison).
//
//   L[r,d]  = sum_{(p,c) in frame d} c logW[r,p] - S[r]          (the zero pixels only contribute -W[r,p] = -S[r])
//   W'[r,p] = sum_{(d,c) in pixel p} c P[r,d] / s[r]
//
// Both are Y = A X with A sparse (frames x pixels, resp. pixels x frames) and X dense with the ROTATIONS along its
// rows: the work is done in the transposed world, X = logW^T [P][R] resp. P^T [N][R], Y = L^T [N][R] resp. W'^T [P][R],
// so that a warp reads and writes runs of consecutive rotations.  One kernel serves both.  The lists by frame are
// made straight from the raw counts, the lists by pixel from those; stage 3 is a soft-max along the contiguous rows of
// L^T (in place: P^T); only log W (from Expand) and W' (for Compress) cross a tiled transpose.
#include "emc_internal.cuh"

namespace emc {

namespace {

// ---------------------------------------------------------------- photon lists
// CSR: row_ptr [rows + 1], entries = column | count << 20.  Built by: nonzeros per row, exclusive scan, fill.
constexpr int kColBits = 20;

// exclusive scan of row_nnz [rows] into row_ptr [rows + 1] by one block (rows is at most about a million)
__global__ void __launch_bounds__(1024)
scan_kernel(const int *__restrict__ row_nnz, int rows, int *__restrict__ row_ptr) {
    __shared__ int warp_tot[32];
    __shared__ int carry;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int base = 0; base < rows; base += 1024) {
        const int i = base + threadIdx.x;
        const int v = i < rows ? row_nnz[i] : 0;
        int x = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int y = __shfl_up_sync(0xffffffffu, x, o);
            if (lane >= o) x += y;
        }
        if (lane == 31) warp_tot[warp] = x;
        __syncthreads();
        if (warp == 0) {
            int t = warp_tot[lane];
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int y = __shfl_up_sync(0xffffffffu, t, o);
                if (lane >= o) t += y;
            }
            warp_tot[lane] = t;                       // inclusive totals of the warps
        }
        __syncthreads();
        const int before = carry + (warp ? warp_tot[warp - 1] : 0) + x - v;
        if (i < rows) row_ptr[i] = before;
        __syncthreads();
        if (threadIdx.x == 1023) carry = before + v;
        __syncthreads();
    }
    if (threadIdx.x == 0) row_ptr[rows] = carry;
}

// CSR by frame from counts [N][P] of the caller's type (masked pixels skipped, counts clamped as the pack kernel clamps
// them and the largest recorded in the header); frame order inside a list = pixel order (deterministic).
template <class T>
__device__ __forceinline__ int live_count(const T *__restrict__ row, const uint8_t *__restrict__ mask, int c, int cols) {
    if (c >= cols || (mask && mask[c] == 0)) return 0;
    long long v = (long long)row[c];
    return v <= 0 ? 0 : (int)(v > 0x7fffffffLL ? 0x7fffffffLL : v);
}

template <class T>
__global__ void __launch_bounds__(256)
count_raw_kernel(const T *__restrict__ counts, int rows, int cols, const uint8_t *__restrict__ mask, int *__restrict__ row_nnz,
                 WsHeader *__restrict__ hdr) {
    const int row = blockIdx.x * 8 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (row >= rows) return;
    const T *a = counts + (size_t)row * cols;
    int n = 0, vmax = 0;
    for (int c0 = 0; c0 < cols; c0 += 32) {
        const int v = live_count(a, mask, c0 + lane, cols);
        vmax = max(vmax, v);
        n += __popc(__ballot_sync(0xffffffffu, v != 0));
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) vmax = max(vmax, __shfl_xor_sync(0xffffffffu, vmax, o));
    if (lane == 0) {
        row_nnz[row] = n;
        if (vmax > EMC_MAX_COUNT) atomicMax(&hdr->max_count, vmax);
    }
}

// fills the frame lists and counts the entries of every pixel (col_nnz zeroed by the caller)
template <class T>
__global__ void __launch_bounds__(256)
fill_raw_kernel(const T *__restrict__ counts, int rows, int cols, const uint8_t *__restrict__ mask,
                const int *__restrict__ row_ptr, uint32_t *__restrict__ entries, int *__restrict__ col_nnz) {
    const int row = blockIdx.x * 8 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (row >= rows) return;
    const T *a = counts + (size_t)row * cols;
    int at = row_ptr[row];
    for (int c0 = 0; c0 < cols; c0 += 32) {
        const int c = c0 + lane;
        const int v = live_count(a, mask, c, cols);
        const unsigned m = __ballot_sync(0xffffffffu, v != 0);
        if (v != 0) {
            entries[at + __popc(m & ((1u << lane) - 1u))] = (uint32_t)c | ((uint32_t)min(v, 4095) << kColBits);
            atomicAdd(col_nnz + c, 1);
        }
        at += __popc(m);
    }
}

// uint16 counts with rows that are whole 16-byte vectors (the configs' case): a lane takes 8 adjacent pixels per step, one
// 16-byte load of counts and one 8-byte load of the mask (the scalar kernels above move 64 bytes per warp-load and ran
// at a fifth of the memory rate).  Same lists, same order.
__device__ __forceinline__ void load8_u16(const uint16_t *__restrict__ row, const uint8_t *__restrict__ mask, int c, int cols, int (&v)[8]) {
    if (c >= cols) {
#pragma unroll
        for (int j = 0; j < 8; ++j) v[j] = 0;
        return;
    }
    const uint4 raw = *reinterpret_cast<const uint4 *>(row + c);
    uint2 mk = make_uint2(0x01010101u, 0x01010101u);
    if (mask) mk = *reinterpret_cast<const uint2 *>(mask + c);
    const uint32_t w[4] = {raw.x, raw.y, raw.z, raw.w};
#pragma unroll
    for (int j = 0; j < 8; ++j) {
        const uint32_t m = ((j < 4 ? mk.x : mk.y) >> (8 * (j & 3))) & 0xffu;
        v[j] = m ? (int)((w[j >> 1] >> (16 * (j & 1))) & 0xffffu) : 0;
    }
}

__global__ void __launch_bounds__(256)
count_u16x8_kernel(const uint16_t *__restrict__ counts, int rows, int cols, const uint8_t *__restrict__ mask,
                   int *__restrict__ row_nnz, WsHeader *__restrict__ hdr) {
    const int row = blockIdx.x * 8 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (row >= rows) return;
    const uint16_t *a = counts + (size_t)row * cols;
    int n = 0, vmax = 0;
    for (int c0 = 0; c0 < cols; c0 += 256) {
        int v[8];
        load8_u16(a, mask, c0 + 8 * lane, cols, v);
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            n += v[j] != 0;
            vmax = max(vmax, v[j]);
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        n += __shfl_xor_sync(0xffffffffu, n, o);
        vmax = max(vmax, __shfl_xor_sync(0xffffffffu, vmax, o));
    }
    if (lane == 0) {
        row_nnz[row] = n;
        if (vmax > EMC_MAX_COUNT) atomicMax(&hdr->max_count, vmax);
    }
}

__global__ void __launch_bounds__(256)
fill_u16x8_kernel(const uint16_t *__restrict__ counts, int rows, int cols, const uint8_t *__restrict__ mask,
                  const int *__restrict__ row_ptr, uint32_t *__restrict__ entries, int *__restrict__ col_nnz) {
    const int row = blockIdx.x * 8 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (row >= rows) return;
    const uint16_t *a = counts + (size_t)row * cols;
    int at = row_ptr[row];
    for (int c0 = 0; c0 < cols; c0 += 256) {
        int v[8];
        const int c = c0 + 8 * lane;
        load8_u16(a, mask, c, cols, v);
        int cnt = 0;
#pragma unroll
        for (int j = 0; j < 8; ++j) cnt += v[j] != 0;
        int incl = cnt;                                             // inclusive scan over the lanes
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int y = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += y;
        }
        int pos = at + incl - cnt;
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            if (v[j] != 0) {
                entries[pos++] = (uint32_t)(c + j) | ((uint32_t)min(v[j], 4095) << kColBits);
                atomicAdd(col_nnz + c + j, 1);
            }
        }
        at += __shfl_sync(0xffffffffu, incl, 31);
    }
}

// the lists by pixel from the lists by frame: entry (frame d, pixel p, count c) goes to pixel p's list as d | c << 20.
// cursor [cols] zeroed by the caller; the order inside a pixel's list is the order the atomics happen to take (the sums of
// the update then vary in their last bits from run to run, as Compress's do).
__global__ void __launch_bounds__(256)
transpose_lists_kernel(const int *__restrict__ row_ptr, const uint32_t *__restrict__ entries, int rows,
                       const int *__restrict__ col_ptr, int *__restrict__ cursor, uint32_t *__restrict__ out) {
    const int row = blockIdx.x * 8 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (row >= rows) return;
    const uint32_t col_mask = (1u << kColBits) - 1u;
    for (int e = row_ptr[row] + lane; e < row_ptr[row + 1]; e += 32) {
        const uint32_t en = entries[e];
        const int p = (int)(en & col_mask);
        const int at = col_ptr[p] + atomicAdd(cursor + p, 1);
        out[at] = (uint32_t)row | (en & ~col_mask);
    }
}

// ---------------------------------------------------------------- Y = A X (+ epilogue), rotations along the rows
// A: CSR (row_ptr, entries).  X [K][ld] fp32, Y [rows][ld] fp32, R valid columns (rotations).
// One warp = one row of A x 128 consecutive rotations (a float4 per lane); the entry is the same address in every lane
// (one broadcast load), the X row a 512-byte run.  Blocks are ordered rotation-tile-major so that the blocks running
// at any one time read the same 128-rotation slab of X (K x 512 bytes: 8 MB for 16384 pixels), which stays in L2.
// sub_row (optional, [R]): Y = A X - sub_row (the log-likelihood's -S[r]).  accumulate: Y += A X (pattern chunks).
__global__ void __launch_bounds__(256)
spmm_rot_kernel(const int *__restrict__ row_ptr, const uint32_t *__restrict__ entries, int rows,
                const float *__restrict__ X, float *__restrict__ Y, int ld, int n_rot,
                const float *__restrict__ sub_row, int accumulate) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int row_blocks = (rows + 7) >> 3;
    const int tile = blockIdx.x / row_blocks;                       // rotation tile (slow index)
    const int row = (blockIdx.x - tile * row_blocks) * 8 + warp;
    const int r = tile * 128 + 4 * lane;
    if (row >= rows || r >= ld) return;                             // ld is a multiple of 4: whole float4s
    const int e0 = row_ptr[row], e1 = row_ptr[row + 1];
    // four partial sums (one per slot of the unrolled loop): independent dependency chains, and the rounding error of a
    // sum of n terms grows like n / 4
    float4 part[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) part[u] = make_float4(0.f, 0.f, 0.f, 0.f);
    const uint32_t col_mask = (1u << kColBits) - 1u;
    int e = e0;
    for (; e + 4 <= e1; e += 4) {                                   // four independent X rows in flight
        uint32_t en[4];
        float4 x[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) en[u] = __ldg(entries + e + u);
#pragma unroll
        for (int u = 0; u < 4; ++u) x[u] = __ldg(reinterpret_cast<const float4 *>(X + (size_t)(en[u] & col_mask) * ld + r));
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const float c = (float)(en[u] >> kColBits);
            part[u].x = fmaf(c, x[u].x, part[u].x);
            part[u].y = fmaf(c, x[u].y, part[u].y);
            part[u].z = fmaf(c, x[u].z, part[u].z);
            part[u].w = fmaf(c, x[u].w, part[u].w);
        }
    }
    for (int u = 0; e < e1; ++e, ++u) {
        const uint32_t en = __ldg(entries + e);
        const float4 x = __ldg(reinterpret_cast<const float4 *>(X + (size_t)(en & col_mask) * ld + r));
        const float c = (float)(en >> kColBits);
        part[u & 3].x = fmaf(c, x.x, part[u & 3].x);
        part[u & 3].y = fmaf(c, x.y, part[u & 3].y);
        part[u & 3].z = fmaf(c, x.z, part[u & 3].z);
        part[u & 3].w = fmaf(c, x.w, part[u & 3].w);
    }
    float4 acc;
    acc.x = (part[0].x + part[1].x) + (part[2].x + part[3].x);
    acc.y = (part[0].y + part[1].y) + (part[2].y + part[3].y);
    acc.z = (part[0].z + part[1].z) + (part[2].z + part[3].z);
    acc.w = (part[0].w + part[1].w) + (part[2].w + part[3].w);
    float4 *y = reinterpret_cast<float4 *>(Y + (size_t)row * ld + r);
    if (sub_row) {
        const float4 sr = *reinterpret_cast<const float4 *>(sub_row + r);     // padded to ld by the caller
        acc.x -= sr.x; acc.y -= sr.y; acc.z -= sr.z; acc.w -= sr.w;
    }
    if (accumulate) {
        const float4 o = *y;
        acc.x += o.x; acc.y += o.y; acc.z += o.z; acc.w += o.w;
    }
    *y = acc;
}

// ---------------------------------------------------------------- transposes
// out [cols][ld_out] = in [rows][ld_in]^T through 32 x 32 shared-memory tiles; columns >= rows of out are left alone.
// MODE 0: plain.  MODE 1 (log-slices): in = W [R][P]; out = logW^T [P][ld_r] with log(max(W, 1e-30)), 0 for masked
// pixels and samples outside the grid (idx < 0); also S[r] += sum_{p:mask} W.  MODE 2: out = in^T / s[col of out]
// (eq. 2.5: W' = numerator / s[r], 0 where s[r] = 0).
template <int MODE>
__global__ void __launch_bounds__(256)
transpose_kernel(const float *__restrict__ in, int rows, int cols, int ld_in, float *__restrict__ out, int ld_out,
                 const int32_t *__restrict__ idx, const uint8_t *__restrict__ mask, float *__restrict__ S,
                 const float *__restrict__ s_div) {
    __shared__ float tile[32][33];
    const int c0 = blockIdx.x * 32, r0 = blockIdx.y * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;         // 32 x 8
#pragma unroll
    for (int j = ty; j < 32; j += 8) {
        const int r = r0 + j, c = c0 + tx;
        float v = 0.f;
        const bool live = r < rows && c < cols;
        if (live) v = in[(size_t)r * ld_in + c];
        if (MODE == 1) {                                            // warp-uniform branch; r is the same in every lane
            const bool use = live && (mask ? mask[c] != 0 : true);
            const bool inside = live && (idx ? idx[(size_t)r * ld_in + c] >= 0 : true);
            float part = use ? v : 0.f;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
            if (tx == 0 && r < rows) atomicAdd(S + r, part);
            v = (use && inside) ? logf(fmaxf(v, 1e-30f)) : 0.f;
        }
        tile[j][tx] = v;
    }
    __syncthreads();
#pragma unroll
    for (int j = ty; j < 32; j += 8) {
        const int c = c0 + j, r = r0 + tx;                          // out row = in column
        if (c < cols && r < rows) {
            float v = tile[tx][j];
            if (MODE == 2) {
                const float sr = s_div[c];
                v = sr > 0.f ? v / sr : 0.f;
            }
            out[(size_t)c * ld_out + r] = v;
        }
    }
}

// ---------------------------------------------------------------- stage 3 in the transposed world
// One block per frame d: the row L^T[d][0..R) becomes P^T[d][0..R) in place (soft-max over the rotations with the prior
// weights, evaluated against the reference pair (L*, log w*) of the row's largest L + log w, as everywhere else: emc_normalize.cu
// ColStat), values below EMC_P_MIN flushed (G20); loglik += (L* + log w*) + log z.
__global__ void __launch_bounds__(256)
softmax_rows_kernel(float *__restrict__ LT, int n_rot, int ld, const float *__restrict__ logw, float log_uniform,
                    double *__restrict__ loglik) {
    __shared__ float sk[8];
    __shared__ int si[8];
    __shared__ float sz[8];
    float *x = LT + (size_t)blockIdx.x * ld;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    float bk = -INFINITY;
    int bi = 0;
    for (int r = threadIdx.x; r < n_rot; r += 256) {
        const float k = x[r] + (logw ? logw[r] : 0.f);
        if (k > bk) { bk = k; bi = r; }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const float k2 = __shfl_xor_sync(0xffffffffu, bk, o);
        const int i2 = __shfl_xor_sync(0xffffffffu, bi, o);
        if (k2 > bk || (k2 == bk && i2 < bi)) { bk = k2; bi = i2; }
    }
    if (lane == 0) { sk[warp] = bk; si[warp] = bi; }
    __syncthreads();
    bk = sk[0]; bi = si[0];
#pragma unroll
    for (int w = 1; w < 8; ++w)
        if (sk[w] > bk || (sk[w] == bk && si[w] < bi)) { bk = sk[w]; bi = si[w]; }
    const float mL = x[bi], mw = logw ? logw[bi] : 0.f;
    float z = 0.f;
    for (int r = threadIdx.x; r < n_rot; r += 256) z += expf((x[r] - mL) + ((logw ? logw[r] : 0.f) - mw));
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) z += __shfl_xor_sync(0xffffffffu, z, o);
    if (lane == 0) sz[warp] = z;
    __syncthreads();
    z = ((sz[0] + sz[1]) + (sz[2] + sz[3])) + ((sz[4] + sz[5]) + (sz[6] + sz[7]));
    const float iz = 1.f / z;
    __syncthreads();                                                // everyone has read x[bi] before it is overwritten
    for (int r = threadIdx.x; r < n_rot; r += 256) {
        float p = expf((x[r] - mL) + ((logw ? logw[r] : 0.f) - mw)) * iz;
        if (p < EMC_P_MIN) p = 0.f;                                 // DESIGN.md section 3 G20
        x[r] = p;
    }
    // uniform weights: log w = log_uniform drops out of every difference above and enters the total only
    if (threadIdx.x == 0 && loglik) atomicAdd(loglik, ((double)mL + (double)(logw ? mw : log_uniform)) + (double)logf(z));
}

__global__ void __launch_bounds__(256)
logw_kernel(const float *__restrict__ weight, int n_rot, float *__restrict__ out) {
    const int r = blockIdx.x * 256 + threadIdx.x;
    if (r < n_rot) out[r] = logf(weight[r]);
}

// s[r] += sum over the frames of P^T[d][r]: a thread per rotation, the frames cut into blockDim.y ranges
__global__ void __launch_bounds__(256)
colsum_rows_kernel(const float *__restrict__ PT, int rows, int n_rot, int ld, int rows_per_split, float *__restrict__ s) {
    const int r = blockIdx.x * 256 + threadIdx.x;
    if (r >= n_rot) return;
    const int d0 = blockIdx.y * rows_per_split, d1 = min(rows, d0 + rows_per_split);
    float a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f;
    int d = d0;
    for (; d + 4 <= d1; d += 4) {
        a0 += PT[(size_t)d * ld + r];
        a1 += PT[(size_t)(d + 1) * ld + r];
        a2 += PT[(size_t)(d + 2) * ld + r];
        a3 += PT[(size_t)(d + 3) * ld + r];
    }
    for (; d < d1; ++d) a0 += PT[(size_t)d * ld + r];
    atomicAdd(s + r, (a0 + a1) + (a2 + a3));
}

}  // namespace

emc_status launch_lists_raw(const void *counts, emc_count_type type, int rows, int cols, const uint8_t *mask, int *list_pat,
                            int *list_pix, WsHeader *hdr, SparseList *by_frame, SparseList *by_pixel, cudaStream_t st) {
    if (cols >= (1 << kColBits) || rows >= (1 << kColBits)) return EMC_ERR_UNSUPPORTED;
    int *row_nnz = list_pat, *row_ptr = list_pat + rows + 64;
    uint32_t *entries = reinterpret_cast<uint32_t *>(list_pat + 2 * ((size_t)rows + 64));
    int *col_nnz = list_pix, *col_ptr = list_pix + cols + 64;
    uint32_t *entries_pix = reinterpret_cast<uint32_t *>(list_pix + 2 * ((size_t)cols + 64));
    EMC_TRY_CUDA(cudaMemsetAsync(col_nnz, 0, sizeof(int) * cols, st));
    const int grid = ceil_div(rows, 8);
#define EMC_RAW(T)                                                                                                   \
    count_raw_kernel<T><<<grid, 256, 0, st>>>((const T *)counts, rows, cols, mask, row_nnz, hdr);                    \
    EMC_LAUNCHED();                                                                                                  \
    scan_kernel<<<1, 1024, 0, st>>>(row_nnz, rows, row_ptr);                                                         \
    EMC_LAUNCHED();                                                                                                  \
    fill_raw_kernel<T><<<grid, 256, 0, st>>>((const T *)counts, rows, cols, mask, row_ptr, entries, col_nnz);        \
    EMC_LAUNCHED();
    const bool vec16 = type == EMC_U16 && cols % 8 == 0 && (((uintptr_t)counts) & 15) == 0 && (!mask || (((uintptr_t)mask) & 7) == 0);
    switch (type) {
        case EMC_I32: { EMC_RAW(int32_t) break; }
        case EMC_U16: {
            if (vec16) {
                count_u16x8_kernel<<<grid, 256, 0, st>>>((const uint16_t *)counts, rows, cols, mask, row_nnz, hdr);
                EMC_LAUNCHED();
                scan_kernel<<<1, 1024, 0, st>>>(row_nnz, rows, row_ptr);
                EMC_LAUNCHED();
                fill_u16x8_kernel<<<grid, 256, 0, st>>>((const uint16_t *)counts, rows, cols, mask, row_ptr, entries, col_nnz);
                EMC_LAUNCHED();
                break;
            }
            EMC_RAW(uint16_t) break;
        }
        case EMC_U8: { EMC_RAW(uint8_t) break; }
        default: return EMC_ERR_ARG;
    }
#undef EMC_RAW
    scan_kernel<<<1, 1024, 0, st>>>(col_nnz, cols, col_ptr);
    EMC_LAUNCHED();
    EMC_TRY_CUDA(cudaMemsetAsync(col_nnz, 0, sizeof(int) * cols, st));       // now the cursors
    transpose_lists_kernel<<<grid, 256, 0, st>>>(row_ptr, entries, rows, col_ptr, col_nnz, entries_pix);
    EMC_LAUNCHED();
    *by_frame = SparseList{row_ptr, entries, rows};
    *by_pixel = SparseList{col_ptr, entries_pix, cols};
    return EMC_OK;
}

emc_status launch_softmax_rows(float *LT, int rows, int n_rot, int ld, const float *logw, float log_uniform, float *s,
                               double *loglik, cudaStream_t st) {
    softmax_rows_kernel<<<rows, 256, 0, st>>>(LT, n_rot, ld, logw, log_uniform, loglik);
    EMC_LAUNCHED();
    if (s) {
        const int splits = rows >= 4096 ? 32 : (rows >= 256 ? 8 : 1);
        const int per = ceil_div(rows, splits);
        colsum_rows_kernel<<<dim3(ceil_div(n_rot, 256), ceil_div(rows, per)), 256, 0, st>>>(LT, rows, n_rot, ld, per, s);
        EMC_LAUNCHED();
    }
    return EMC_OK;
}

emc_status launch_logw(const float *weight, int n_rot, float *out, cudaStream_t st) {
    logw_kernel<<<ceil_div(n_rot, 256), 256, 0, st>>>(weight, n_rot, out);
    EMC_LAUNCHED();
    return EMC_OK;
}

size_t sparse_list_ints(int rows, size_t max_entries) { return 2 * ((size_t)rows + 64) + max_entries; }

emc_status launch_spmm_rot(const SparseList &a, const float *X, float *Y, int ld, int n_rot, const float *sub_row,
                           bool accumulate, cudaStream_t st) {
    if (ld % 4 || ((uintptr_t)X & 15) || ((uintptr_t)Y & 15)) return EMC_ERR_ARG;
    const long long blocks = (long long)ceil_div(a.rows, 8) * ceil_div(n_rot, 128);
    if (blocks > 0x7fffffffLL) return EMC_ERR_UNSUPPORTED;
    spmm_rot_kernel<<<(unsigned)blocks, 256, 0, st>>>(a.row_ptr, a.entries, a.rows, X, Y, ld, n_rot, sub_row, accumulate ? 1 : 0);
    EMC_LAUNCHED();
    return EMC_OK;
}

emc_status launch_transpose(const float *in, int rows, int cols, int ld_in, float *out, int ld_out, cudaStream_t st) {
    transpose_kernel<0><<<dim3(ceil_div(cols, 32), ceil_div(rows, 32)), 256, 0, st>>>(in, rows, cols, ld_in, out, ld_out,
                                                                                      nullptr, nullptr, nullptr, nullptr);
    EMC_LAUNCHED();
    return EMC_OK;
}

emc_status launch_logw_transposed(const float *W, const int32_t *idx, const uint8_t *mask, int n_rot, int n_pix, float *logWT,
                                  int ld_r, float *S, cudaStream_t st) {
    transpose_kernel<1><<<dim3(ceil_div(n_pix, 32), ceil_div(n_rot, 32)), 256, 0, st>>>(W, n_rot, n_pix, n_pix, logWT, ld_r, idx,
                                                                                        mask, S, nullptr);
    EMC_LAUNCHED();
    return EMC_OK;
}

emc_status launch_transpose_div(const float *WT, int n_pix, int n_rot, int ld_r, float *Wnew, const float *s, cudaStream_t st) {
    // in = W'^T [P][ld_r] (rows = pixels, cols = rotations); out = W' [R][P]; out row = in column = rotation
    transpose_kernel<2><<<dim3(ceil_div(n_rot, 32), ceil_div(n_pix, 32)), 256, 0, st>>>(WT, n_pix, n_rot, ld_r, Wnew, n_pix,
                                                                                        nullptr, nullptr, nullptr, s);
    EMC_LAUNCHED();
    return EMC_OK;
}

}  // namespace emc
