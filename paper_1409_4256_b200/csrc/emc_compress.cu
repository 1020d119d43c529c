// Stage 5, Compress (c-step), eq. (2.10) / (2.12), PAPER.md:118-130:
//
//   num[l] += f om_r W'[r,p],   den[l] += f om_r     over unmasked samples inside the grid,
//   model'[l] = den > 0 ? num/den : 0                ("division as a final step")
//
// with the same trilinear weights f and the same pinned sample geometry as Expand.
//
// Measured on B200 (DESIGN.md §7 "Compress"): what bounds the scatter is the chip's rate of fp32 reductions into
// L2, which depends on how the bytes are grouped: 64 bytes per sample as four unrelated 16-byte reductions cost
// 347 us per 2e7 samples, as ONE contiguous 64-byte group issued by four adjacent lanes 224 us (and a
// cp.reduce.async.bulk of the same 64 bytes, or any mix of the two, the same 225 us); shared-memory atomics are
// slower than all of them.  So the design (a) moves a sample's 8 corners x (num, den) = 64 bytes in four 16-byte
// red.global.add.v4.f32 (16 bytes per lane is the widest reduction there is), and (b) makes those 64 bytes
// CONTIGUOUS and lets four adjacent lanes issue them in
// one instruction: the accumulator is not a voxel grid but 8 staggered grids of 2x2x2 blocks, one per parity
// (b_x&1, b_y&1, b_z&1) of the base corner; grid c holds, for every base of that parity, one aligned 64-byte
// block {num, den} x corner (4 dx + 2 dy + dz), blocks ordered [b_x/2][b_y/2][b_z/2].  After computing its
// own sample a lane hands (block, t_x, t_y, t_z, W') to its group of four by shuffles, and the group adds the
// four samples' blocks one after the other, each lane carrying the corner pair (dx, dy, dz = 0..1) it owns.
// The divide kernel gathers a voxel's 8 contributions.  64 G bytes of accumulators (16 MB at 64^3, 134 MB at
// 128^3); n odd falls back to 8-byte reductions on a plain (num, den) grid.
#include "emc_geometry.cuh"
#include "emc_internal.cuh"

namespace emc {

namespace {

constexpr int kThreads = 256;
constexpr int kPixPerThread = 4;
constexpr int kPixPerBlock = kThreads * kPixPerThread;

__device__ __forceinline__ void red_add_v2(float2 *addr, float a, float b) {
    asm volatile("red.global.add.v2.f32 [%0], {%1, %2};" ::"l"(addr), "f"(a), "f"(b) : "memory");
}

__device__ __forceinline__ void red_add_v4(float4 *addr, float a, float b, float c, float d) {
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(addr), "f"(a), "f"(b), "f"(c), "f"(d) : "memory");
}

// Block layout: 16 floats = num of the 8 corners (order 4 dx + 2 dy + dz), then den of the 8 corners; as float4s:
// 0 = num dx 0, 1 = num dx 1, 2 = den dx 0, 3 = den dx 1.
//
// den does not depend on W': with eq. (2.10) (weight 1 per slice) it only depends on the rotation list and on WHICH
// slices are skipped (s[r] = 0).  Inside emc_iterate the iterations after the first therefore run NUM_ONLY (32 bytes
// per sample, two lanes per sample) as long as the set of skipped slices is the one den was accumulated for;
// active_check_kernel decides that on the device and the scatter kernel branches on its flag, so no host
// synchronisation is needed (probe: 153 us against 224 us per 2e7 samples).

// One thread per rotation, one warp per word: bits[r / 32] = mask of slices with s[r] > 0; *changed = 1 if it differs
// from the stored mask (or force), else left as the caller zeroed it.
__global__ void __launch_bounds__(256)
active_check_kernel(const float *__restrict__ s, int n_rot, uint32_t *__restrict__ bits, int *__restrict__ changed,
                    int force) {
    const int r = blockIdx.x * 256 + threadIdx.x;
    const uint32_t m = __ballot_sync(0xffffffffu, r < n_rot && s[r] > 0.f);
    if ((threadIdx.x & 31) == 0 && r < n_rot) {
        if (force || bits[r >> 5] != m) *changed = 1;
        bits[r >> 5] = m;
    }
}

// zero the accumulators: everything if *changed, else only the num halves of the blocks
__global__ void __launch_bounds__(256)
compress_clear_kernel(float4 *__restrict__ acc, size_t n_blocks, const int *__restrict__ changed) {
    const size_t t = (size_t)blockIdx.x * 256 + threadIdx.x;           // one float4
    if (t >= 4 * n_blocks) return;
    if (*changed != 0 || (t & 2) == 0) acc[t] = make_float4(0.f, 0.f, 0.f, 0.f);
}

// FULL: four rounds, the four lanes of a group add the 64-byte block of the sample of lane grp + k.
// NUM_ONLY: two rounds, lanes 0-1 add the 32 num bytes of the sample of lane grp + 2k, lanes 2-3 of grp + 2k + 1.
// A lane carries the four corners (dx, dy, dz), dy, dz = 0..1, of num (or den).  Warp-wide: every lane calls it.
template <bool NUM_ONLY>
__device__ __forceinline__ void scatter_rounds(float4 *__restrict__ acc, int blk, float stx, float sty, float stz, float v,
                                               float om, unsigned lane) {
    const unsigned sub = lane & 3u, grp = lane & ~3u;
    const bool dx1 = (sub & 1u) != 0;
    const bool is_den = !NUM_ONLY && (sub & 2u) != 0;
    const unsigned slot = NUM_ONLY ? (sub & 1u) : sub;         // float4 index inside the block
    constexpr int kRounds = NUM_ONLY ? 2 : 4;
#pragma unroll
    for (int k = 0; k < kRounds; ++k) {
        const int src = NUM_ONLY ? (int)grp + 2 * k + (int)(sub >> 1) : (int)grp + k;
        const int b = __shfl_sync(0xffffffffu, blk, src);
        const float tx = __shfl_sync(0xffffffffu, stx, src);
        const float ty = __shfl_sync(0xffffffffu, sty, src);
        const float tz = __shfl_sync(0xffffffffu, stz, src);
        const float vv = __shfl_sync(0xffffffffu, v, src);
        if (b >= 0) {
            const float wx = (dx1 ? tx : 1.f - tx) * om;
            const float a0 = wx * (1.f - ty), a1 = wx * ty;
            const float z0 = 1.f - tz;
            const float sc = is_den ? 1.f : vv;
            red_add_v4(acc + 4 * (size_t)b + slot, (a0 * z0) * sc, (a0 * tz) * sc, (a1 * z0) * sc, (a1 * tz) * sc);
        }
    }
}

// grid = (R, ceil(P / kPixPerBlock)); n even.  acc = [8][(n/2)^3] blocks of 4 float4.  changed: device flag of
// active_check_kernel, 0 = den is still valid, add num only; null = add both.
__global__ void __launch_bounds__(kThreads)
compress_scatter_blocked_kernel(const float *__restrict__ Wn, const float *__restrict__ slice_w, int weighted,
                                const float4 *__restrict__ qm, int n_pix,
                                const float *__restrict__ quat, int n, float4 *__restrict__ acc,
                                const int *__restrict__ changed) {
    __shared__ float rm[9];
    const bool num_only = changed && *changed == 0;   // uniform over the grid
    const int r = blockIdx.x;
    float om = 1.f;
    if (slice_w) {
        const float sw = slice_w[r];
        if (!(sw > 0.f)) return;                 // slice skipped (G17); uniform over the block
        if (weighted) om = sw;
    }
    if (threadIdx.x == 0) {
        RotMat m = rotation_matrix(quat + 4 * (size_t)r);
#pragma unroll
        for (int i = 0; i < 9; ++i) rm[i] = m.m[i];
    }
    __syncthreads();
    const unsigned h = (unsigned)n >> 1;
    const unsigned per_copy = h * h * h;
    const unsigned lane = threadIdx.x & 31u;
#pragma unroll
    for (int j = 0; j < kPixPerThread; ++j) {
        const int p = blockIdx.y * kPixPerBlock + j * kThreads + threadIdx.x;
        // every lane stays in the loop (the exchange below is warp-wide); a lane without a sample carries blk = -1
        const int pc = p < n_pix ? p : n_pix - 1;
        const float4 g = qm[pc];                               // (q, mask) in one 16-byte load
        const Sample s = locate(rm, g.x, g.y, g.z, n);
        const bool ok = p < n_pix && s.base >= 0 && g.w != 0.f;
        const float v = ok ? Wn[(size_t)r * n_pix + pc] : 0.f;
        int blk = -1;
        if (ok) {
            const unsigned c = ((s.bx & 1u) << 2) | ((s.by & 1u) << 1) | (s.bz & 1u);
            blk = (int)(c * per_copy + (((unsigned)s.bx >> 1) * h + ((unsigned)s.by >> 1)) * h + ((unsigned)s.bz >> 1));
        }
        if (num_only) scatter_rounds<true>(acc, blk, s.tx, s.ty, s.tz, v, om, lane);
        else scatter_rounds<false>(acc, blk, s.tx, s.ty, s.tz, v, om, lane);
    }
}

// model'[l] = num/den, (num, den) gathered from the (up to) 8 blocks whose 2x2x2 corner set contains voxel l
__global__ void __launch_bounds__(256)
compress_divide_blocked_kernel(const float *__restrict__ acc, int n, float *__restrict__ model_out,
                               float *__restrict__ den_out) {
    const size_t l = (size_t)blockIdx.x * 256 + threadIdx.x;
    const size_t g = (size_t)n * n * n;
    if (l >= g) return;
    const int z = (int)(l % n), y = (int)((l / n) % n), x = (int)(l / ((size_t)n * n));
    const unsigned h = (unsigned)n >> 1;
    const size_t per_copy = (size_t)h * h * h;
    float num = 0.f, den = 0.f;
#pragma unroll
    for (int d = 0; d < 8; ++d) {
        const int bx = x - (d >> 2), by = y - ((d >> 1) & 1), bz = z - (d & 1);
        if (bx < 0 || by < 0 || bz < 0 || bx > n - 2 || by > n - 2 || bz > n - 2) continue;
        const unsigned c = ((bx & 1u) << 2) | ((by & 1u) << 1) | (bz & 1u);
        const size_t blk = c * per_copy + (((size_t)(bx >> 1) * h + (by >> 1)) * h + (bz >> 1));
        num += acc[16 * blk + d];
        den += acc[16 * blk + 8 + d];
    }
    model_out[l] = den > 0.f ? num / den : 0.f;
    if (den_out) den_out[l] = den;
}

// grid = (R, ceil(P / kPixPerBlock))
__global__ void __launch_bounds__(kThreads)
compress_scatter_kernel(const float *__restrict__ Wn, const float *__restrict__ slice_w, int weighted,
                        const float *__restrict__ q, const uint8_t *__restrict__ mask, int n_pix,
                        const float *__restrict__ quat, int n, float2 *__restrict__ acc) {
    __shared__ float rm[9];
    const int r = blockIdx.x;
    float om = 1.f;
    if (slice_w) {
        const float sw = slice_w[r];
        if (!(sw > 0.f)) return;                 // slice skipped (G17); uniform over the block
        if (weighted) om = sw;
    }
    if (threadIdx.x == 0) {
        RotMat m = rotation_matrix(quat + 4 * (size_t)r);
#pragma unroll
        for (int i = 0; i < 9; ++i) rm[i] = m.m[i];
    }
    __syncthreads();
    const int nn = n * n;
#pragma unroll
    for (int j = 0; j < kPixPerThread; ++j) {
        const int p = blockIdx.y * kPixPerBlock + j * kThreads + threadIdx.x;
        if (p >= n_pix) continue;
        if (mask && mask[p] == 0) continue;
        const Sample s = locate(rm, q[3 * p], q[3 * p + 1], q[3 * p + 2], n);
        if (s.base < 0) continue;
        const float v = Wn[(size_t)r * n_pix + p];
        const float x1 = s.tx * om, x0 = (1.f - s.tx) * om;
        const float y1 = s.ty, y0 = 1.f - s.ty, z1 = s.tz, z0 = 1.f - s.tz;
        float2 *b = acc + s.base;
        float f;
        f = x0 * y0 * z0; red_add_v2(b, f * v, f);
        f = x0 * y0 * z1; red_add_v2(b + 1, f * v, f);
        f = x0 * y1 * z0; red_add_v2(b + n, f * v, f);
        f = x0 * y1 * z1; red_add_v2(b + n + 1, f * v, f);
        f = x1 * y0 * z0; red_add_v2(b + nn, f * v, f);
        f = x1 * y0 * z1; red_add_v2(b + nn + 1, f * v, f);
        f = x1 * y1 * z0; red_add_v2(b + nn + n, f * v, f);
        f = x1 * y1 * z1; red_add_v2(b + nn + n + 1, f * v, f);
    }
}

__global__ void __launch_bounds__(256)
compress_divide_kernel(const float2 *__restrict__ acc, size_t g, float *__restrict__ model_out,
                       float *__restrict__ den_out) {
    const size_t l = (size_t)blockIdx.x * 256 + threadIdx.x;
    if (l >= g) return;
    const float2 a = acc[l];
    model_out[l] = a.y > 0.f ? a.x / a.y : 0.f;
    if (den_out) den_out[l] = a.y;
}

}  // namespace

size_t compress_scratch_float2(int n, int n_pix) { return (size_t)8 * n * n * n + (size_t)2 * n_pix; }

emc_status launch_compress(const float *Wnew, const float *slice_w, bool weighted, const float *q,
                           const uint8_t *mask, int n_pix, const float *quat, int n_rot, int n,
                           float2 *acc, float *model_out, float *den_out, cudaStream_t st, const DenCache *cache) {
    const size_t g = (size_t)n * n * n;
    dim3 grid(n_rot, ceil_div(n_pix, kPixPerBlock));
    if ((n & 1) == 0) {
        float4 *acc4 = reinterpret_cast<float4 *>(acc);          // 8 grids x (n/2)^3 blocks x 64 B = 8 G float2
        const float *accf = reinterpret_cast<const float *>(acc);
        const int w = weighted ? 1 : 0;
        float4 *qm = reinterpret_cast<float4 *>(acc + 8 * g);     // after the accumulators
        EMC_TRY(launch_pack_geometry(q, mask, n_pix, qm, st));
        if (cache && slice_w && !weighted) {
            // den is reused while the set of skipped slices stays the one it was accumulated for (decided on the device)
            EMC_TRY_CUDA(cudaMemsetAsync(cache->changed, 0, sizeof(int), st));
            active_check_kernel<<<ceil_div(n_rot, 256), 256, 0, st>>>(slice_w, n_rot, cache->active,
                                                                                 cache->changed, cache->force ? 1 : 0);
            EMC_LAUNCHED();
            compress_clear_kernel<<<(unsigned)((4 * g + 255) / 256), 256, 0, st>>>(acc4, g, cache->changed);   // g blocks of 64 B
            EMC_LAUNCHED();
            compress_scatter_blocked_kernel<<<grid, kThreads, 0, st>>>(Wnew, slice_w, w, qm, n_pix, quat, n, acc4,
                                                                       cache->changed);
            EMC_LAUNCHED();
        } else {
            EMC_TRY_CUDA(cudaMemsetAsync(acc4, 0, g * 8 * sizeof(float2), st));
            compress_scatter_blocked_kernel<<<grid, kThreads, 0, st>>>(Wnew, slice_w, w, qm, n_pix, quat, n, acc4, nullptr);
            EMC_LAUNCHED();
        }
        compress_divide_blocked_kernel<<<(unsigned)((g + 255) / 256), 256, 0, st>>>(accf, n, model_out, den_out);
        EMC_LAUNCHED();
        return EMC_OK;
    }
    EMC_TRY_CUDA(cudaMemsetAsync(acc, 0, g * sizeof(float2), st));
    compress_scatter_kernel<<<grid, kThreads, 0, st>>>(Wnew, slice_w, weighted ? 1 : 0, q, mask, n_pix, quat, n, acc);
    EMC_LAUNCHED();
    compress_divide_kernel<<<(unsigned)((g + 255) / 256), 256, 0, st>>>(acc, g, model_out, den_out);
    EMC_LAUNCHED();
    return EMC_OK;
}

}  // namespace emc
