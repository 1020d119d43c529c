// Sample geometry shared by Expand and Compress: rotation matrix, grid coordinate, base corner.
// The arithmetic sequence is PINNED (DESIGN.md §3 G4) so that the rotation -> voxel index map is
// bit-exact against the oracle: explicit round-to-nearest intrinsics, no FMA contraction.
#pragma once

#include <cuda_runtime.h>

namespace emc {

struct RotMat {
    float m[9];   // row-major 3x3
};

// Active rotation matrix of the unit quaternion (w,x,y,z): textbook formula in
// float64 from the float32 components, every entry rounded once to float32.
__device__ __forceinline__ RotMat rotation_matrix(const float *__restrict__ quat) {
    const double w = (double)quat[0], x = (double)quat[1], y = (double)quat[2], z = (double)quat[3];
    const double xx = __dmul_rn(x, x), yy = __dmul_rn(y, y), zz = __dmul_rn(z, z);
    const double xy = __dmul_rn(x, y), xz = __dmul_rn(x, z), yz = __dmul_rn(y, z);
    const double wx = __dmul_rn(w, x), wy = __dmul_rn(w, y), wz = __dmul_rn(w, z);
    RotMat r;
    r.m[0] = __double2float_rn(__dsub_rn(1.0, __dmul_rn(2.0, __dadd_rn(yy, zz))));
    r.m[1] = __double2float_rn(__dmul_rn(2.0, __dsub_rn(xy, wz)));
    r.m[2] = __double2float_rn(__dmul_rn(2.0, __dadd_rn(xz, wy)));
    r.m[3] = __double2float_rn(__dmul_rn(2.0, __dadd_rn(xy, wz)));
    r.m[4] = __double2float_rn(__dsub_rn(1.0, __dmul_rn(2.0, __dadd_rn(xx, zz))));
    r.m[5] = __double2float_rn(__dmul_rn(2.0, __dsub_rn(yz, wx)));
    r.m[6] = __double2float_rn(__dmul_rn(2.0, __dsub_rn(xz, wy)));
    r.m[7] = __double2float_rn(__dmul_rn(2.0, __dadd_rn(yz, wx)));
    r.m[8] = __double2float_rn(__dsub_rn(1.0, __dmul_rn(2.0, __dadd_rn(xx, yy))));
    return r;
}

struct Sample {
    int base;          // linear index of the base corner, -1 outside the grid
    int bx, by, bz;    // the base corner itself (meaningful when base >= 0)
    float tx, ty, tz;  // fractional offsets in [0,1)
};

// x_a = ((R_a0 q_x + R_a1 q_y) + R_a2 q_z) + c, every operation one float32 rounding; b = floor(x),
// t = x - b (exact); valid iff 0 <= b_a <= n-2 on every axis (G7).
__device__ __forceinline__ Sample locate(const float *__restrict__ m, float qx, float qy, float qz,
                                         int n) {
    const float c = 0.5f * (float)n;   // exact: n <= 1024
    float x[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const float t0 = __fmul_rn(m[3 * a + 0], qx);
        const float t1 = __fmul_rn(m[3 * a + 1], qy);
        const float t2 = __fmul_rn(m[3 * a + 2], qz);
        x[a] = __fadd_rn(__fadd_rn(__fadd_rn(t0, t1), t2), c);
    }
    const float bx = floorf(x[0]), by = floorf(x[1]), bz = floorf(x[2]);
    const float hi = (float)(n - 2);
    Sample s;
    s.tx = __fsub_rn(x[0], bx);
    s.ty = __fsub_rn(x[1], by);
    s.tz = __fsub_rn(x[2], bz);
    const bool valid = (bx >= 0.f) && (bx <= hi) && (by >= 0.f) && (by <= hi) && (bz >= 0.f) && (bz <= hi);
    s.bx = (int)bx;
    s.by = (int)by;
    s.bz = (int)bz;
    s.base = valid ? (s.bx * n + s.by) * n + s.bz : -1;
    return s;
}

}  // namespace emc
