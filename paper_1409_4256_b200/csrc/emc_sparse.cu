// Photon-list (sparse) form of stages 2 and 4 for frames that are almost empty (BASELINE.json config 4: 0.01 photons
// per pixel, > 99 % zeros).  EMC_SPARSE_PHOTONS selects it inside emc_iterate; the
// dense tensor-core contractions stay the default (DESIGN.md section 11 has the measured comparison).
//
//   L[r,d]  = sum_{(p,c) in frame d} c logW[r,p] - S[r]          (the zero pixels only contribute -W[r,p] = -S[r])
//   W'[r,p] = sum_{(d,c) in pixel p} c P[r,d] / s[r]
//
// Both are Y = A X with A sparse (frames x pixels, resp. pixels x frames) and X dense with the ROTATIONS along its
// rows: the work is done in the transposed world, X = logW^T [P][R] resp. P^T [N][R], Y = L^T [N][R] resp. W'^T [P][R],
// so that a warp reads and writes runs of consecutive rotations.  One kernel serves both.  The operands are made
// from the dense path's own buffers: the lists from the packed fp16 count matrices (their rows are frames resp.
// pixels), the transposes by a tiled transpose kernel.
#include "emc_internal.cuh"

namespace emc {

namespace {

// ---------------------------------------------------------------- lists from the packed count matrices
// A [rows][ld] fp16 (exact small integers, masked pixels already 0) -> CSR: row_ptr [rows + 1], entries = column |
// count << 20 in row order (deterministic).  Three kernels: nonzeros per row, exclusive scan, fill.
constexpr int kColBits = 20;

__global__ void __launch_bounds__(256)
count_nonzeros_kernel(const __half *__restrict__ A, int rows, int cols, int ld, int *__restrict__ row_nnz) {
    const int row = blockIdx.x * 8 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (row >= rows) return;
    const __half *a = A + (size_t)row * ld;
    int n = 0;
    for (int c0 = 0; c0 < cols; c0 += 32) {
        const int c = c0 + lane;
        const bool nz = c < cols && __half2float(a[c]) != 0.f;
        n += __popc(__ballot_sync(0xffffffffu, nz));
    }
    if (lane == 0) row_nnz[row] = n;
}

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

__global__ void __launch_bounds__(256)
fill_entries_kernel(const __half *__restrict__ A, int rows, int cols, int ld, const int *__restrict__ row_ptr,
                    uint32_t *__restrict__ entries) {
    const int row = blockIdx.x * 8 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (row >= rows) return;
    const __half *a = A + (size_t)row * ld;
    int at = row_ptr[row];
    for (int c0 = 0; c0 < cols; c0 += 32) {
        const int c = c0 + lane;
        const float v = c < cols ? __half2float(a[c]) : 0.f;
        const unsigned m = __ballot_sync(0xffffffffu, v != 0.f);
        if (v != 0.f) entries[at + __popc(m & ((1u << lane) - 1u))] = (uint32_t)c | ((uint32_t)fminf(v, 4095.f) << kColBits);   // counts above EMC_MAX_COUNT poison the call anyway
        at += __popc(m);
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

}  // namespace

size_t sparse_list_ints(int rows, size_t max_entries) { return 2 * ((size_t)rows + 64) + max_entries; }

emc_status launch_sparsify(const __half *A, int rows, int cols, int ld, int *lists, size_t max_entries, SparseList *out,
                           cudaStream_t st) {
    if (cols >= (1 << kColBits)) return EMC_ERR_UNSUPPORTED;
    int *row_nnz = lists, *row_ptr = lists + rows + 64;
    uint32_t *entries = reinterpret_cast<uint32_t *>(lists + 2 * ((size_t)rows + 64));
    (void)max_entries;                                              // sized for rows x cols by the caller: cannot overflow
    count_nonzeros_kernel<<<ceil_div(rows, 8), 256, 0, st>>>(A, rows, cols, ld, row_nnz);
    EMC_LAUNCHED();
    scan_kernel<<<1, 1024, 0, st>>>(row_nnz, rows, row_ptr);
    EMC_LAUNCHED();
    fill_entries_kernel<<<ceil_div(rows, 8), 256, 0, st>>>(A, rows, cols, ld, row_ptr, entries);
    EMC_LAUNCHED();
    *out = SparseList{row_ptr, entries, rows};
    return EMC_OK;
}

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
