// sampler.cuh — O5 trilinear sampling of the tiled cube with a per-ray register cache of x-rows.
//
// ncu of the first caster (profiles/r01_cast_full.md) showed the L1TEX data stage at 96 %: eight scalar
// corner loads per sample, each a warp request over ~20-32 distinct lines.  Here a ray keeps, in
// registers, the four 16-byte x-chunks (4 voxels each) that hold its current 2x2 (y,z) rows and loads a
// row only when the ray has moved off it:
//   * x0 and x0+1 come out of ONE 128-bit load per row (plus one scalar load only when x0 is the last
//     voxel of its chunk),
//   * rows live in slots chosen by the PARITY of their y and z index: the two rows a sample needs along an
//     axis always have different parity, and when the ray advances by one voxel the row it keeps stays in
//     its slot while the new row replaces the one left behind — no data movement, no dependence on the
//     direction of travel, and any step length is handled (a slot is reloaded whenever the row index it
//     should hold differs from the one it holds).
// Values and weights are those of O5 exactly (same voxels, same fractions).
#pragma once
#include <cuda_runtime.h>

namespace vr {

struct RowCache {
    float4 r[2][2];          // [y parity][z parity] chunk of 4 voxels along x
    float e[2][2];           // voxel after the chunk (valid while the ray sits on the chunk's last voxel)
    unsigned cx;             // chunk index the slots hold
    unsigned hy[2], hz[2];   // row indices the slots hold
    bool straddle;           // the previous sample sat on the last voxel of its chunk (e[][] valid)
};

__device__ __forceinline__ void cache_init(RowCache& K) {
    K.cx = 0xffffffffu; K.hy[0] = K.hy[1] = K.hz[0] = K.hz[1] = 0xffffffffu; K.straddle = false;
#pragma unroll
    for (int a = 0; a < 2; ++a)
#pragma unroll
        for (int b = 0; b < 2; ++b) { K.r[a][b] = make_float4(0.f, 0.f, 0.f, 0.f); K.e[a][b] = 0.f; }
}

__device__ __forceinline__ float pick4(const float4& v, unsigned c, float last) {
    // element c of (v.x, v.y, v.z, v.w, last), c in 0..4
    const float lo = (c & 1) ? v.y : v.x;
    const float hi = (c & 1) ? v.w : v.z;
    const float q = (c & 2) ? hi : lo;
    return (c & 4) ? last : q;
}

// base + 4*e as ONE instruction (IMAD.WIDE.U32); e is an element offset below 2^30
__device__ __forceinline__ const float* elem_ptr(unsigned long long base, unsigned e) {
    unsigned long long a;
    asm("mad.wide.u32 %0, %1, 4, %2;" : "=l"(a) : "r"(e), "l"(base));
    return reinterpret_cast<const float*>(a);
}

// Returns the trilinear value at (qx,qy,qz) = position - 1/2.
// vol_base: address of the tiled cube; ty_stride in elements; slab_bytes = bytes between z-tile slabs.
__device__ __forceinline__ float sample_cached(unsigned long long vol_base, unsigned ty_stride, unsigned slab_bytes,
                                               float nxm1, float nym1, float nzm1, float qx, float qy, float qz,
                                               RowCache& K) {
    qx = fminf(fmaxf(qx, 0.0f), nxm1);
    qy = fminf(fmaxf(qy, 0.0f), nym1);
    qz = fminf(fmaxf(qz, 0.0f), nzm1);
    // floor of a non-negative float < 2^22 without F2I/I2F: add 2^23 rounding down; the integer is the low
    // mantissa bits and (r - 2^23) is that integer as a float, exactly.
    const float rx = __fadd_rd(qx, 8388608.0f), ry = __fadd_rd(qy, 8388608.0f), rz = __fadd_rd(qz, 8388608.0f);
    const unsigned ix = __float_as_uint(rx) & 0x7fffffu, iy = __float_as_uint(ry) & 0x7fffffu,
                   iz = __float_as_uint(rz) & 0x7fffffu;
    const float fx = qx - (rx - 8388608.0f), fy = qy - (ry - 8388608.0f), fz = qz - (rz - 8388608.0f);
    const unsigned cx = ix >> 2, c = ix & 3;
    const bool straddle = (c == 3);

    // rows the two parity slots must hold: the even one and the odd one of {i, i+1}
    const unsigned wy[2] = {(iy + 1) & ~1u, iy | 1u};
    const unsigned wz[2] = {(iz + 1) & ~1u, iz | 1u};
    const bool xchg = cx != K.cx;
    const bool ychg[2] = {wy[0] != K.hy[0], wy[1] != K.hy[1]};
    const bool zchg[2] = {wz[0] != K.hz[0], wz[1] != K.hz[1]};
    const bool e_all = !K.straddle;

    const unsigned exc = (cx >> 1) * TILE_ELEMS + ((cx & 1) << 2);
    const unsigned ix1 = ix + 1;
    const unsigned exe = (ix1 >> 3) * TILE_ELEMS + (ix1 & 7);
    const unsigned ey[2] = {(wy[0] >> 3) * ty_stride + ((wy[0] & 7) << 3),
                            (wy[1] >> 3) * ty_stride + ((wy[1] & 7) << 3)};
    unsigned long long pz[2];
    unsigned ez[2];
#pragma unroll
    for (int b = 0; b < 2; ++b) {
        asm("mad.wide.u32 %0, %1, %2, %3;" : "=l"(pz[b]) : "r"(wz[b] >> 3), "r"(slab_bytes), "l"(vol_base));
        ez[b] = (wz[b] & 7) << 6;
    }
#pragma unroll
    for (int a = 0; a < 2; ++a)
#pragma unroll
        for (int b = 0; b < 2; ++b) {
            const bool need = xchg || ychg[a] || zchg[b];
            if (need) K.r[a][b] = __ldg(reinterpret_cast<const float4*>(elem_ptr(pz[b], exc + ey[a] + ez[b])));
            if (straddle && (need || e_all)) K.e[a][b] = __ldg(elem_ptr(pz[b], exe + ey[a] + ez[b]));
        }
    K.cx = cx; K.hy[0] = wy[0]; K.hy[1] = wy[1]; K.hz[0] = wz[0]; K.hz[1] = wz[1]; K.straddle = straddle;

    // O5 blend: x inside each row, then y, then z.  Slot 0 holds the even row: it is row i when i is even
    // (weight 1-f) and row i+1 when i is odd (weight f).
    const float gy = (iy & 1) ? 1.0f - fy : fy, gz = (iz & 1) ? 1.0f - fz : fz;
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
