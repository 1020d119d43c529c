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

// rows of R_r from the table launch_geometry() wrote (three 16-byte loads, the same address in every lane)
__device__ __forceinline__ void load_rotation(const float4 *__restrict__ rotm, int r, float (&m)[9]) {
    const float4 a = __ldg(rotm + 3 * (size_t)r), b = __ldg(rotm + 3 * (size_t)r + 1), c = __ldg(rotm + 3 * (size_t)r + 2);
    m[0] = a.x; m[1] = a.y; m[2] = a.z;
    m[3] = b.x; m[4] = b.y; m[5] = b.z;
    m[6] = c.x; m[7] = c.y; m[8] = c.z;
}

struct Sample {
    int base;          // linear index of the base corner, -1 outside the grid
    int bx, by, bz;    // the base corner itself (meaningful when base >= 0)
    float tx, ty, tz;  // fractional offsets in [0,1)
};

// x_a = ((R_a0 q_x + R_a1 q_y) + R_a2 q_z) + c, every operation one float32 rounding; b = floor(x),
// t = x - b (one float32 subtraction); valid iff 0 <= b_a <= n-2 on every axis (G7).
//
// floor(x) without the conversion unit (FRND / F2I issue at a quarter of the FADD rate): for |x| < 2^22,
// u = x + 1.5 * 2^23 rounded DOWN is the integer floor(x) + 1.5 * 2^23 exactly (the float32 grid has spacing 1 in
// [2^23, 2^24)), so floor(x) = u - 1.5 * 2^23 (exact) and, as an integer, bits(u) - bits(1.5 * 2^23).  For |x| >= 2^22 or
// NaN the integer lands outside [0, n-2] (n <= 1024) and the sample is invalid, as it is by the plain definition.
__device__ __forceinline__ Sample locate(const float *__restrict__ m, float qx, float qy, float qz,
                                         int n) {
    const float c = 0.5f * (float)n;   // exact: n <= 1024
    constexpr float kMagic = 12582912.f;             // 1.5 * 2^23 = 0x4B400000
    float x[3], bf[3];
    int bi[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const float t0 = __fmul_rn(m[3 * a + 0], qx);
        const float t1 = __fmul_rn(m[3 * a + 1], qy);
        const float t2 = __fmul_rn(m[3 * a + 2], qz);
        x[a] = __fadd_rn(__fadd_rn(__fadd_rn(t0, t1), t2), c);
        const float u = __fadd_rd(x[a], kMagic);
        bf[a] = __fsub_rn(u, kMagic);
        bi[a] = __float_as_int(u) - 0x4B400000;
    }
    const unsigned hi = (unsigned)(n - 2);
    Sample s;
    s.tx = __fsub_rn(x[0], bf[0]);
    s.ty = __fsub_rn(x[1], bf[1]);
    s.tz = __fsub_rn(x[2], bf[2]);
    const bool valid = ((unsigned)bi[0] <= hi) && ((unsigned)bi[1] <= hi) && ((unsigned)bi[2] <= hi);
    s.bx = bi[0];
    s.by = bi[1];
    s.bz = bi[2];
    s.base = valid ? (s.bx * n + s.by) * n + s.bz : -1;
    return s;
}

// Detector pixels as 2-D tiles (emc_detector.row_len): a warp works on TH x TW pixels at a time (4 x 8 when the row
// length is known, 1 x 32 otherwise), so that its 32 samples cover a compact patch of the slice.  Work is handed out
// to warps in BANDS: one tile row (TH detector rows), cut into segments of at most kMaxTilesPerBand tiles; a warp walks
// along its band kTilesPerStep tiles at a time.  Any row_len gives the same results; only locality changes.
constexpr int kTilesPerStep = 4;           // measured at C2: 4 tiles per step (64 registers) 130 us, 2 (40-48 registers) 137-139 us, 1: 178 us
constexpr int kMaxTilesPerBand = 4;        // measured at C2: 4 (one step per item) 127-130 us, 8: 207 us, 32 with 6 blocks per SM: 258 us
struct TileMap {
    int row_len, n_rows, n_tx, n_seg, n_bands, tw_shift, th;
};
static inline TileMap make_tile_map(int n_pix, int row_len) {
    TileMap t;
    const bool tiled = row_len >= 8 && n_pix % row_len == 0 && n_pix / row_len >= 4;
    t.row_len = tiled ? row_len : n_pix;
    t.n_rows = tiled ? n_pix / row_len : 1;
    t.tw_shift = tiled ? 3 : 5;
    t.th = tiled ? 4 : 1;
    t.n_tx = (t.row_len + (1 << t.tw_shift) - 1) >> t.tw_shift;
    t.n_seg = (t.n_tx + kMaxTilesPerBand - 1) / kMaxTilesPerBand;
    t.n_bands = t.n_seg * ((t.n_rows + t.th - 1) / t.th);
    return t;
}
// The lane's pixels in one band: pixel(t) of tile t of the band (t may run past the end: -1), or -1 in a row that does
// not exist.
struct Band {
    int row_off, col0, step, row_len, n_tiles;
    __device__ __forceinline__ Band(const TileMap &tm, int band, int lane) {
        const int ty = band / tm.n_seg, seg = band - ty * tm.n_seg;
        const int row = ty * tm.th + (lane >> tm.tw_shift);
        step = 1 << tm.tw_shift;
        col0 = seg * kMaxTilesPerBand * step + (lane & (step - 1));
        n_tiles = min(kMaxTilesPerBand, tm.n_tx - seg * kMaxTilesPerBand);
        row_len = row < tm.n_rows ? tm.row_len : 0;      // 0: no column passes the test below
        row_off = row * tm.row_len;
    }
    __device__ __forceinline__ int pixel(int t) const {
        const int col = col0 + t * step;
        return (t < n_tiles && col < row_len) ? row_off + col : -1;
    }
};

}  // namespace emc
