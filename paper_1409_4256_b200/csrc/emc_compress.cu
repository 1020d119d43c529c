// Stage 5, Compress (c-step), eq. (2.10) / (2.12), PAPER.md:118-130:
//
//   num[l] += f om_r W'[r,p],   den[l] += f om_r     over unmasked samples inside the grid,
//   model'[l] = den > 0 ? num/den : 0                ("division as a final step")
//
// with the same trilinear weights f and the same pinned sample geometry as Expand.
//
// Measured on B200 (DESIGN.md section 7 "Compress"): what bounds the scatter is the chip's rate of fp32 reductions
// into L2, which depends on how the bytes are grouped: 64 bytes per sample as four unrelated 16-byte reductions cost
// 347 us per 2e7 samples, as ONE contiguous 64-byte group issued by four adjacent lanes 224 us; shared-memory
// atomics on fp32 are CAS loops (ATOMS.CAST.SPIN) at 2 cycles per lane and slower than all of them.  So the design
// (a) moves a sample's 8 corners x (num, den) = 64 bytes in four 16-byte red.global.add.v4.f32 (16 bytes per lane is
// the widest reduction there is), and (b) makes those 64 bytes CONTIGUOUS and lets four adjacent lanes issue them in
// one instruction: the accumulator is not a voxel grid but one aligned 64-byte block {num, den} x corner
// (4 dx + 2 dy + dz) per BASE CORNER, acc[(b_x n + b_y) n + b_z] (the block index is the index map itself).
// After computing its own sample a lane hands (block, t_x, t_y, t_z, W') to its group of four by shuffles, and the
// group adds the four samples' blocks one after the other, each lane carrying the corner quad (dx; num or den) it owns.
// A warp works on a 4 x 8 tile of detector pixels at a time (emc_geometry.cuh TileMap).
// The divide kernel gathers a voxel's 8 contributions.  64 G bytes of accumulators (16 MB at 64^3, 134 MB at 128^3).
#include <algorithm>

#include "emc_geometry.cuh"
#include "emc_internal.cuh"

namespace emc {

namespace {

constexpr int kThreads = 256;
constexpr int kWarps = kThreads / 32;

__device__ __forceinline__ void red_add_v4(float4 *addr, const float4 v) {
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(addr), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}

// Block layout: 16 floats = num of the 8 corners (order 4 dx + 2 dy + dz), then den of the 8 corners; as float4s:
// 0 = num dx 0, 1 = num dx 1, 2 = den dx 0, 3 = den dx 1.
//
// den does not depend on W': with eq. (2.10) (weight 1 per slice) it only depends on the rotation list and on WHICH
// slices are skipped (s[r] = 0).  Inside emc_iterate the iterations after the first therefore run NUM_ONLY (32 bytes
// per sample, two lanes per sample) as long as the set of skipped slices is the one den was accumulated for;
// active_check_kernel decides that on the device and the scatter kernel branches on its flag, so no host
// synchronisation is needed.

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

// Warp-wide: every lane calls it with its own sample (blk < 0: none).
// FULL: four rounds, the four lanes of a group add the 64-byte block of the sample of lane grp + k.
// NUM_ONLY: two rounds, lanes 0-1 add the 32 num bytes of the sample of lane grp + 2k, lanes 2-3 of grp + 2k + 1.
// A lane carries the four corners (dx, dy, dz), dy, dz = 0..1, of num (or den); it gets the sample by shuffles and forms
// its own four products.  (Measured against parking each lane's 16 products in shared memory and reading them back
// transposed: 232 us against 240 us per C2 stage; the shared-memory traffic costs more L1 wavefronts than the
// shuffles, and the multiplier has room: issue slots 36 % busy.)
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
            red_add_v4(acc + 4 * (size_t)b + slot, make_float4((a0 * z0) * sc, (a0 * tz) * sc, (a1 * z0) * sc, (a1 * tz) * sc));
        }
    }
}

// One warp per (rotation, band) work item (a stride loop covers item counts beyond the grid limit); it walks along its
// band kTilesPerStep tiles at a time (emc_geometry.cuh).  acc = [n^3] blocks of 4 float4.  changed: device flag
// of active_check_kernel, 0 = den is still valid, add num only; null = add both.
__global__ void __launch_bounds__(kThreads, 4)
compress_scatter_blocked_kernel(const float *__restrict__ Wn, const float *__restrict__ slice_w, int weighted,
                                const float4 *__restrict__ qm, const TileMap tm, int n_rot, int n_pix,
                                const float4 *__restrict__ rotm, int n, float4 *__restrict__ acc,
                                const int *__restrict__ changed) {
    const bool num_only = changed && *changed == 0;   // uniform over the grid
    const unsigned lane = threadIdx.x & 31u;
    const int n_items = n_rot * tm.n_bands;
    for (int item = blockIdx.x * kWarps + (threadIdx.x >> 5); item < n_items; item += gridDim.x * kWarps) {
        const int r = item / tm.n_bands;
        float om = 1.f;
        if (slice_w) {
            const float sw = slice_w[r];
            if (!(sw > 0.f)) continue;           // slice skipped (G17); uniform over the warp
            if (weighted) om = sw;
        }
        float rm[9];
        load_rotation(rotm, r, rm);
        const Band band(tm, item - r * tm.n_bands, (int)lane);
        const float *const w_row = Wn + (size_t)r * n_pix;
        for (int t0 = 0; t0 < band.n_tiles; t0 += kTilesPerStep) {
            // the geometry and the loads of four tiles first (independent), then the four exchanges
            Sample smp[kTilesPerStep];
            float val[kTilesPerStep];
            int blk[kTilesPerStep];
            float4 g[kTilesPerStep];
            int pix[kTilesPerStep];
#pragma unroll
            for (int j = 0; j < kTilesPerStep; ++j) {
                pix[j] = band.pixel(t0 + j);
                g[j] = qm[max(pix[j], 0)];                     // (q, mask) in one 16-byte load
                val[j] = w_row[max(pix[j], 0)];
            }
#pragma unroll
            for (int j = 0; j < kTilesPerStep; ++j) {
                // every lane stays in the loop (the exchange is warp-wide); a lane without a sample carries blk = -1
                smp[j] = locate(rm, g[j].x, g[j].y, g[j].z, n);
                const bool ok = pix[j] >= 0 && smp[j].base >= 0 && g[j].w != 0.f;
                blk[j] = ok ? smp[j].base : -1;
            }
#pragma unroll
            for (int j = 0; j < kTilesPerStep; ++j) {
                if (__all_sync(0xffffffffu, blk[j] < 0)) continue;     // warp-uniform: nothing to send (ragged edge, masked tile)
                if (num_only) scatter_rounds<true>(acc, blk[j], smp[j].tx, smp[j].ty, smp[j].tz, val[j], om, lane);
                else scatter_rounds<false>(acc, blk[j], smp[j].tx, smp[j].ty, smp[j].tz, val[j], om, lane);
            }
        }
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
    float num = 0.f, den = 0.f;
#pragma unroll
    for (int d = 0; d < 8; ++d) {
        const int bx = x - (d >> 2), by = y - ((d >> 1) & 1), bz = z - (d & 1);
        if (bx < 0 || by < 0 || bz < 0 || bx > n - 2 || by > n - 2 || bz > n - 2) continue;
        const size_t blk = ((size_t)bx * n + by) * n + bz;
        num += acc[16 * blk + d];
        den += acc[16 * blk + 8 + d];
    }
    model_out[l] = den > 0.f ? num / den : 0.f;
    if (den_out) den_out[l] = den;
}

// num and den of every voxel, gathered from the corner blocks, undivided
__global__ void __launch_bounds__(256)
compress_export_kernel(const float *__restrict__ acc, int n, float *__restrict__ numden) {
    const size_t l = (size_t)blockIdx.x * 256 + threadIdx.x;
    const size_t g = (size_t)n * n * n;
    if (l >= g) return;
    const int z = (int)(l % n), y = (int)((l / n) % n), x = (int)(l / ((size_t)n * n));
    float num = 0.f, den = 0.f;
#pragma unroll
    for (int d = 0; d < 8; ++d) {
        const int bx = x - (d >> 2), by = y - ((d >> 1) & 1), bz = z - (d & 1);
        if (bx < 0 || by < 0 || bz < 0 || bx > n - 2 || by > n - 2 || bz > n - 2) continue;
        const size_t blk = ((size_t)bx * n + by) * n + bz;
        num += acc[16 * blk + d];
        den += acc[16 * blk + 8 + d];
    }
    numden[l] = num;
    numden[g + l] = den;
}

__global__ void __launch_bounds__(256)
numden_divide_kernel(const float *__restrict__ numden, size_t g, float *__restrict__ model_out) {
    const size_t l = (size_t)blockIdx.x * 256 + threadIdx.x;
    if (l >= g) return;
    const float num = numden[l], den = numden[g + l];
    model_out[l] = den > 0.f ? num / den : 0.f;
}

}  // namespace

emc_status launch_compress_export(const float2 *acc, int n, float *numden, cudaStream_t st) {
    const size_t g = (size_t)n * n * n;
    compress_export_kernel<<<(unsigned)((g + 255) / 256), 256, 0, st>>>(reinterpret_cast<const float *>(acc), n, numden);
    EMC_LAUNCHED();
    return EMC_OK;
}

emc_status launch_numden_divide(const float *numden, int n, float *model_out, cudaStream_t st) {
    const size_t g = (size_t)n * n * n;
    numden_divide_kernel<<<(unsigned)((g + 255) / 256), 256, 0, st>>>(numden, g, model_out);
    EMC_LAUNCHED();
    return EMC_OK;
}

size_t compress_scratch_float2(int n) { return (size_t)8 * n * n * n; }

emc_status launch_compress(const float *Wnew, const float *slice_w, bool weighted, const Geometry &geo, int n,
                           float2 *acc, float *model_out, float *den_out, cudaStream_t st, const DenCache *cache, int phases) {
    const size_t g = (size_t)n * n * n;
    const int n_pix = geo.n_pix, n_rot = geo.n_rot;
    float4 *acc4 = reinterpret_cast<float4 *>(acc);          // n^3 blocks x 64 B = 8 G float2
    const float *accf = reinterpret_cast<const float *>(acc);
    const int w = weighted ? 1 : 0;
    const TileMap tm = make_tile_map(n_pix, geo.row_len);
    const long long items = (long long)n_rot * tm.n_bands;
    if (items > 0x7fffffffLL) return EMC_ERR_UNSUPPORTED;          // the kernel counts work items in 32 bits
    const int grid = (int)std::min<long long>((items + kWarps - 1) / kWarps, (long long)1 << 30);
    if (phases != COMPRESS_ALL) {
        if (phases & COMPRESS_CLEAR) EMC_TRY_CUDA(cudaMemsetAsync(acc4, 0, g * 8 * sizeof(float2), st));
        if (phases & COMPRESS_SCATTER) {
            compress_scatter_blocked_kernel<<<grid, kThreads, 0, st>>>(Wnew, slice_w, w, geo.qm, tm, n_rot, n_pix, geo.rotm, n, acc4, nullptr);
            EMC_LAUNCHED();
        }
        if (phases & COMPRESS_DIVIDE) {
            compress_divide_blocked_kernel<<<(unsigned)((g + 255) / 256), 256, 0, st>>>(accf, n, model_out, den_out);
            EMC_LAUNCHED();
        }
        return EMC_OK;
    }
    if (cache && slice_w && !weighted) {
        // den is reused while the set of skipped slices stays the one it was accumulated for (decided on the device)
        EMC_TRY_CUDA(cudaMemsetAsync(cache->changed, 0, sizeof(int), st));
        active_check_kernel<<<ceil_div(n_rot, 256), 256, 0, st>>>(slice_w, n_rot, cache->active, cache->changed,
                                                                  cache->force ? 1 : 0);
        EMC_LAUNCHED();
        compress_clear_kernel<<<(unsigned)((4 * g + 255) / 256), 256, 0, st>>>(acc4, g, cache->changed);   // g blocks of 64 B
        EMC_LAUNCHED();
        compress_scatter_blocked_kernel<<<grid, kThreads, 0, st>>>(Wnew, slice_w, w, geo.qm, tm, n_rot, n_pix, geo.rotm, n, acc4,
                                                                   cache->changed);
        EMC_LAUNCHED();
    } else {
        EMC_TRY_CUDA(cudaMemsetAsync(acc4, 0, g * 8 * sizeof(float2), st));
        compress_scatter_blocked_kernel<<<grid, kThreads, 0, st>>>(Wnew, slice_w, w, geo.qm, tm, n_rot, n_pix, geo.rotm, n, acc4, nullptr);
        EMC_LAUNCHED();
    }
    compress_divide_blocked_kernel<<<(unsigned)((g + 255) / 256), 256, 0, st>>>(accf, n, model_out, den_out);
    EMC_LAUNCHED();
    return EMC_OK;
}

}  // namespace emc
