// sampler.cuh — O5 trilinear sampling of the tiled cube with a per-ray register cache of x-rows.
//
// ncu of the first caster (profiles/r01_cast_full.md) showed the L1TEX data stage at 96 %: eight scalar
// corner loads per sample, each a warp request over ~20-32 distinct lines.  Here a ray keeps, in
// registers, the four 16-byte x-chunks (4 voxels each) that hold its current 2x2 (y,z) rows, loads a row
// only when the ray has moved off it, and re-uses rows across steps:
//   * x0 and x0+1 come out of ONE 128-bit load per row (plus one scalar load only when x0 is the last
//     voxel of its chunk),
//   * a step that keeps (chunk, y0, z0) loads nothing; a step that advances y0 or z0 by one voxel in
//     the ray's direction of travel moves the leading rows to the trailing slots and loads only the new
//     leading rows.
// Rows are indexed trailing/leading (T/L) along the ray's direction of travel per axis, so the shift is
// the same code for either sign.  Values and weights are those of O5 exactly (same voxels, same f).
#pragma once
#include <cuda_runtime.h>

namespace vr {

struct RowCache {
    float4 r[2][2];     // [y: T,L][z: T,L] chunk of 4 voxels along x
    float e[2][2];      // voxel after the chunk (valid while the ray sits on the chunk's last voxel)
    unsigned cx, iy, iz;
    bool have, prev_straddle;
};

__device__ __forceinline__ float pick4(const float4& v, unsigned c, float last) {
    // element c of (v.x, v.y, v.z, v.w, last), c in 0..4
    const float lo = (c & 1) ? v.y : v.x;
    const float hi = (c & 1) ? v.w : v.z;
    const float q = (c & 2) ? hi : lo;
    return (c & 4) ? last : q;
}

// Returns the trilinear value at (qx,qy,qz) = position - 1/2.  ypos/zpos: the ray travels towards +y/+z.
__device__ __forceinline__ float sample_cached(const float* __restrict__ vol, unsigned ty_stride,
                                               unsigned slab_stride, float nxm1, float nym1, float nzm1,
                                               float qx, float qy, float qz, bool ypos, bool zpos,
                                               RowCache& K) {
    qx = fminf(fmaxf(qx, 0.0f), nxm1);
    qy = fminf(fmaxf(qy, 0.0f), nym1);
    qz = fminf(fmaxf(qz, 0.0f), nzm1);
    const float rx = __fadd_rd(qx, 8388608.0f), ry = __fadd_rd(qy, 8388608.0f), rz = __fadd_rd(qz, 8388608.0f);
    const unsigned ix = __float_as_uint(rx) & 0x7fffffu, iy = __float_as_uint(ry) & 0x7fffffu,
                   iz = __float_as_uint(rz) & 0x7fffffu;
    const float fx = qx - (rx - 8388608.0f), fy = qy - (ry - 8388608.0f), fz = qz - (rz - 8388608.0f);
    const unsigned cx = ix >> 2, c = ix & 3;
    const bool straddle = (c == 3);

    // ---- which rows survive from the previous sample ----
    bool all = !K.have || cx != K.cx;
    const int dy = (int)iy - (int)K.iy, dz = (int)iz - (int)K.iz;
    const bool my = (dy == (ypos ? 1 : -1)), mz = (dz == (zpos ? 1 : -1));
    all = all || (dy != 0 && !my) || (dz != 0 && !mz);
    if (my) {            // trailing rows <- leading rows (y)
        K.r[0][0] = K.r[1][0]; K.r[0][1] = K.r[1][1];
        K.e[0][0] = K.e[1][0]; K.e[0][1] = K.e[1][1];
    }
    if (mz) {            // trailing rows <- leading rows (z)
        K.r[0][0] = K.r[0][1]; K.r[1][0] = K.r[1][1];
        K.e[0][0] = K.e[0][1]; K.e[1][0] = K.e[1][1];
    }
    const bool e_all = all || !K.prev_straddle;

    // ---- addresses: rows T/L in y and z, chunk base in x ----
    const unsigned yT = ypos ? iy : iy + 1, yL = ypos ? iy + 1 : iy;
    const unsigned zT = zpos ? iz : iz + 1, zL = zpos ? iz + 1 : iz;
    const unsigned exc = (cx >> 1) * TILE_ELEMS + ((cx & 1) << 2);
    const unsigned ix1 = ix + 1;
    const unsigned exe = (ix1 >> 3) * TILE_ELEMS + (ix1 & 7);
    const unsigned eyv[2] = {(yT >> 3) * ty_stride + ((yT & 7) << 3), (yL >> 3) * ty_stride + ((yL & 7) << 3)};
    const float* __restrict__ pzv[2] = {vol + (size_t)(zT >> 3) * slab_stride + ((zT & 7) << 6),
                                        vol + (size_t)(zL >> 3) * slab_stride + ((zL & 7) << 6)};
#pragma unroll
    for (int a = 0; a < 2; ++a)
#pragma unroll
        for (int b = 0; b < 2; ++b) {
            const bool need = all || (a == 1 && my) || (b == 1 && mz);
            if (need) K.r[a][b] = __ldg(reinterpret_cast<const float4*>(pzv[b] + (exc + eyv[a])));
            if (straddle && (need || e_all)) K.e[a][b] = __ldg(pzv[b] + (exe + eyv[a]));
        }
    K.cx = cx; K.iy = iy; K.iz = iz; K.have = true; K.prev_straddle = straddle;

    // ---- O5 blend: x inside each row, then y, then z (weights in T/L order) ----
    const float gy = ypos ? fy : 1.0f - fy, gz = zpos ? fz : 1.0f - fz;
    float row[2][2];
#pragma unroll
    for (int a = 0; a < 2; ++a)
#pragma unroll
        for (int b = 0; b < 2; ++b) {
            const float v0 = pick4(K.r[a][b], c, 0.0f);
            const float v1 = pick4(K.r[a][b], c + 1, K.e[a][b]);
            row[a][b] = fmaf(fx, v1 - v0, v0);
        }
    const float c0 = fmaf(gy, row[1][0] - row[0][0], row[0][0]);
    const float c1 = fmaf(gy, row[1][1] - row[0][1], row[0][1]);
    return fmaf(gz, c1 - c0, c0);
}

}  // namespace vr
