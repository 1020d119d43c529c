// Stage 5, Compress (c-step), eq. (2.10) / (2.12), PAPER.md:118-130:
//
//   num[l] += f om_r W'[r,p],   den[l] += f om_r     over unmasked samples inside the grid,
//   model'[l] = den > 0 ? num/den : 0                ("division as a final step")
//
// with the same trilinear weights f and the same pinned sample geometry as Expand.  Numerator and
// denominator of a voxel are interleaved as one float2 so that each corner costs ONE 8-byte vector
// reduction (red.global.add.v2.f32) instead of two scalar atomics.
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
    EMC_TRY_CUDA(cudaMemsetAsync(acc, 0, g * sizeof(float2), st));
    dim3 grid(n_rot, ceil_div(n_pix, kPixPerBlock));
    compress_scatter_kernel<<<grid, kThreads, 0, st>>>(Wnew, slice_w, weighted ? 1 : 0, q, mask, n_pix, quat, n, acc);
    EMC_LAUNCHED();
    compress_divide_kernel<<<(unsigned)((g + 255) / 256), 256, 0, st>>>(acc, g, model_out, den_out);
    EMC_LAUNCHED();
    return EMC_OK;
}

}  // namespace emc
