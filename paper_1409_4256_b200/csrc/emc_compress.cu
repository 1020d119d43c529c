// Stage 5, Compress (c-step), eq. (2.10) / (2.12), PAPER.md:118-130:
//
//   num[l] += f om_r W'[r,p],   den[l] += f om_r     over unmasked samples inside the grid,
//   model'[l] = den > 0 ? num/den : 0                ("division as a final step")
//
// with the same trilinear weights f and the same pinned sample geometry as Expand.
//
// The scatter is bound by the rate at which an SM issues global reductions (about one lane-operation
// per 1.3 cycles), so the design minimises lane-operations: numerator and denominator
// of a voxel are interleaved, and the two z-neighbours of a corner pair are adjacent in memory, so
// one 16-byte red.global.add.v4.f32 carries {num,den}(z), {num,den}(z+1): 4 reductions per sample
// instead of 16 scalar atomics.  A 16-byte reduction must be 16-byte aligned, which a pair starting
// at an odd z is not; hence TWO accumulator grids, one holding pairs (2k,2k+1) and one holding pairs
// (2k+1,2k+2); a sample uses the grid that matches the parity of its base z, and the final divide
// kernel adds the two.  (n odd falls back to 8-byte reductions on a single grid.)
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

// grid = (R, ceil(P / kPixPerBlock)); n even.  acc = [2][n][n][n/2] float4 (even-z pairs, odd-z pairs).
__global__ void __launch_bounds__(kThreads)
compress_scatter_pairs_kernel(const float *__restrict__ Wn, const float *__restrict__ slice_w, int weighted,
                              const float *__restrict__ q, const uint8_t *__restrict__ mask, int n_pix,
                              const float *__restrict__ quat, int n, float4 *__restrict__ acc) {
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
    const int h = n >> 1;                        // float4 per z row
    const size_t layer = (size_t)n * n * h;      // float4 per grid
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
        const int bz = s.bz, row = s.bx * n + s.by;
        float4 *b = acc + (bz & 1 ? layer : 0) + (size_t)row * h + (bz >> 1);
        float f0, f1;
        f0 = x0 * y0 * z0; f1 = x0 * y0 * z1; red_add_v4(b, f0 * v, f0, f1 * v, f1);
        f0 = x0 * y1 * z0; f1 = x0 * y1 * z1; red_add_v4(b + h, f0 * v, f0, f1 * v, f1);
        f0 = x1 * y0 * z0; f1 = x1 * y0 * z1; red_add_v4(b + (size_t)n * h, f0 * v, f0, f1 * v, f1);
        f0 = x1 * y1 * z0; f1 = x1 * y1 * z1; red_add_v4(b + (size_t)n * h + h, f0 * v, f0, f1 * v, f1);
    }
}

// model'[l] = num/den with (num, den) = even-grid entry + odd-grid entry of voxel l
__global__ void __launch_bounds__(256)
compress_divide_pairs_kernel(const float4 *__restrict__ acc, int n, float *__restrict__ model_out,
                             float *__restrict__ den_out) {
    const int h = n >> 1;
    const size_t rows = (size_t)n * n;
    const size_t t = (size_t)blockIdx.x * 256 + threadIdx.x;   // one thread per even-grid float4 = voxels (2k, 2k+1)
    if (t >= rows * h) return;
    const int k2 = (int)(t % h);
    const float4 e = acc[t];
    const float4 *odd = acc + rows * h;
    // odd grid entry m holds voxels (2m+1, 2m+2): voxel 2k is .zw of entry k-1, voxel 2k+1 is .xy of entry k
    float n0 = e.x, d0 = e.y, n1 = e.z, d1 = e.w;
    const float4 ok = odd[t];
    n1 += ok.x; d1 += ok.y;
    if (k2 > 0) {
        const float4 om1 = odd[t - 1];
        n0 += om1.z; d0 += om1.w;
    }
    const size_t l = (t / h) * n + 2 * (size_t)k2;
    model_out[l] = d0 > 0.f ? n0 / d0 : 0.f;
    model_out[l + 1] = d1 > 0.f ? n1 / d1 : 0.f;
    if (den_out) { den_out[l] = d0; den_out[l + 1] = d1; }
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

emc_status launch_compress(const float *Wnew, const float *slice_w, bool weighted, const float *q,
                           const uint8_t *mask, int n_pix, const float *quat, int n_rot, int n,
                           float2 *acc, float *model_out, float *den_out, cudaStream_t st) {
    const size_t g = (size_t)n * n * n;
    dim3 grid(n_rot, ceil_div(n_pix, kPixPerBlock));
    if ((n & 1) == 0) {
        float4 *acc4 = reinterpret_cast<float4 *>(acc);          // 2 grids x G/2 float4 = 2 G float2
        EMC_TRY_CUDA(cudaMemsetAsync(acc4, 0, g * sizeof(float4), st));
        compress_scatter_pairs_kernel<<<grid, kThreads, 0, st>>>(Wnew, slice_w, weighted ? 1 : 0, q, mask, n_pix,
                                                                 quat, n, acc4);
        EMC_LAUNCHED();
        compress_divide_pairs_kernel<<<(unsigned)((g / 2 + 255) / 256), 256, 0, st>>>(acc4, n, model_out, den_out);
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
