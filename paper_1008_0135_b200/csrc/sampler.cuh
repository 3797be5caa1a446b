// sampler.cuh — O5 trilinear sampling of the tiled cube: segment-anchored positions, a per-ray register
// cache of x-rows, and the occupancy-mask test of empty-space skipping.
//
// Positions.  A ray's samples are t_i = t_near + (i + 1/2) step (O4).  Absolute fp32 coordinates reach 2048
// on the headline cube, where half an ulp is 6e-5 voxel: against noise with voxel-to-voxel differences of
// several units that is ~3e-4 in the interpolated value — inside the 1e-4 RGBA gate (each sample carries a
// small alpha) but not inside the 1e-4 gate on raw MIP maxima.  So the march is cut into SEGMENTS of
// P.seg_len samples; at the start of a segment the position is evaluated in double (the oracle's expression),
// split into an integer origin O and a remainder rel in [0, seg span], and inside the segment
// q_rel(j') = rel + j' h in fp32 with |q_rel| <= ~65: rounding <= 4e-6 voxel.  Voxel index = O + floor(q_rel).
//
// Row cache.  ncu of the round-1 caster showed the L1TEX data stage at 96 %: eight
// scalar corner loads per sample, each a warp request over ~20-32 distinct lines.  Here a ray keeps, in
// registers, the four 16-byte x-chunks (4 voxels each) that hold its current 2x2 (y,z) rows and loads a
// row only when the ray has moved off it:
//   * x0 and x0+1 come out of ONE 128-bit load per row (plus one scalar load only when x0 is the last
//     voxel of its chunk),
//   * rows live in slots chosen by the PARITY of their y and z index: the two rows a sample needs along an
//     axis always have different parity, and when the ray advances by one voxel the row it keeps stays in
//     its slot while the new row replaces the one left behind — no data movement, no dependence on the
//     direction of travel, and any step length is handled (a slot is reloaded whenever the row index it
//     should hold differs from the one it holds), including the jumps empty-space skipping makes.
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

// Segment anchor: integer origin and remainder of the segment's first sample, in PADDED coordinates
// u = q + PAD = p - 1/2 + PAD (kernels.cuh, re-layout): no clamp is needed, the replicated layers do O5's clamp-to-edge.
struct Anchor {
    int O[3];
    float rel[3];
};

// Anchor of the segment whose first sample has lattice index i0 (double precision; O2-O4's expressions).
// span >= seg_len * |h_a| + 1 is subtracted on axes the ray descends, so that u_rel stays non-negative over
// the whole segment (the magic-add floor below needs that).
__device__ __forceinline__ void set_anchor(const double o[3], const double d[3], double t_near, double step,
                                           long long i0, const float h[3], int span, Anchor& A) {
    const double ta = t_near + ((double)i0 + 0.5) * step;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const double ud = o[a] + ta * d[a] + ((a == 0 ? PAD_X : a == 1 ? PAD_Y : PAD_Z) - 0.5);
        const double base = floor(ud) - (h[a] < 0.0f ? (double)span : 0.0);
        A.O[a] = (int)base;
        A.rel[a] = (float)(ud - base);
    }
}

struct Cell {                // padded cell of one sample: low corner and fractions
    unsigned ix, iy, iz;
    float fx, fy, fz;
};

// Sample jl of the segment: u_rel = rel + jl h, floor by the 2^23 magic add (no F2I/I2F), index = O + floor.
__device__ __forceinline__ void locate(const Anchor& A, int jl, const float h[3], Cell& c) {
    const float jf = (float)jl;
    float q[3], r[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        q[a] = fmaf(jf, h[a], A.rel[a]);
        r[a] = __fadd_rd(q[a], 8388608.0f);       // 0 <= q < 2^22: the integer is the low mantissa bits
    }
    c.ix = (unsigned)(A.O[0] + (int)(__float_as_uint(r[0]) & 0x7fffffu));
    c.iy = (unsigned)(A.O[1] + (int)(__float_as_uint(r[1]) & 0x7fffffu));
    c.iz = (unsigned)(A.O[2] + (int)(__float_as_uint(r[2]) & 0x7fffffu));
    c.fx = q[0] - (r[0] - 8388608.0f);
    c.fy = q[1] - (r[1] - 8388608.0f);
    c.fz = q[2] - (r[2] - 8388608.0f);
}

// The same cell without the fractions (occupancy pass of empty-space skipping).
__device__ __forceinline__ void locate_cell(const Anchor& A, int jl, const float h[3], unsigned& ix, unsigned& iy,
                                            unsigned& iz) {
    const float jf = (float)jl;
    ix = (unsigned)(A.O[0] + (int)(__float_as_uint(__fadd_rd(fmaf(jf, h[0], A.rel[0]), 8388608.0f)) & 0x7fffffu));
    iy = (unsigned)(A.O[1] + (int)(__float_as_uint(__fadd_rd(fmaf(jf, h[1], A.rel[1]), 8388608.0f)) & 0x7fffffu));
    iz = (unsigned)(A.O[2] + (int)(__float_as_uint(__fadd_rd(fmaf(jf, h[2], A.rel[2]), 8388608.0f)) & 0x7fffffu));
}

// Empty-space skipping (NEXT-2): one bit per padded cell, set when a sample inside the cell can be non-transparent
// (build_mask_kernel).  Words of 64 bits = 4x4x4 cells, word index ((bz*NBY + by)*NBX + bx); the ray keeps the
// word of its current block in registers and reloads it only when it enters another block.
struct MaskCursor {
    unsigned lo, hi;         // the 64-bit word: lo = cells with (iz & 3) < 2
    unsigned tag;
};
__device__ __forceinline__ bool cell_occupied(const unsigned long long* __restrict__ mask, unsigned nbx, unsigned nbxy,
                                              unsigned ix, unsigned iy, unsigned iz, MaskCursor& mc) {
    const unsigned tag = (iz >> 2) * nbxy + (iy >> 2) * nbx + (ix >> 2);
    if (tag != mc.tag) {
        const uint2 w = __ldg(reinterpret_cast<const uint2*>(mask + tag));
        mc.lo = w.x; mc.hi = w.y; mc.tag = tag;
    }
    const unsigned half = (iz & 2u) ? mc.hi : mc.lo;
    const unsigned bit = ((iz & 1u) << 4) | ((iy & 3u) << 2) | (ix & 3u);
    return (half >> bit) & 1u;
}

// The 16-byte row-chunk load (read-only path).  Larger L2 fill sizes (ld.global.nc.L2::NNNB) were measured in round 2:
// no gain (profiles/r02_experiments.md).
__device__ __forceinline__ float4 load_row_chunk(unsigned long long addr) {
    return __ldg(reinterpret_cast<const float4*>(addr));
}

// Trilinear value of the cell (O5) through the row cache.
// vol_base: address of the tiled cube; ty_stride in elements; slab_bytes = bytes between z-tile slabs.
__device__ __forceinline__ float sample_cached(unsigned long long vol_base, unsigned ty_stride, unsigned slab_bytes,
                                               const Cell& s, RowCache& K) {
    const unsigned ix = s.ix, iy = s.iy, iz = s.iz;
    const unsigned cx = ix >> 2, c = ix & 3;
    const bool straddle = (c == 3);

    // rows the two parity slots must hold: the even one and the odd one of {i, i+1}
    const unsigned wy[2] = {(iy + 1) & ~1u, iy | 1u};
    const unsigned wz[2] = {(iz + 1) & ~1u, iz | 1u};
    const bool xchg = cx != K.cx;
    const bool ychg[2] = {wy[0] != K.hy[0], wy[1] != K.hy[1]};
    const bool zchg[2] = {wz[0] != K.hz[0], wz[1] != K.hz[1]};
    const bool e_all = !K.straddle;

    const unsigned exc = tile_fx(cx << 2);
    const unsigned ey[2] = {tile_fy(wy[0], ty_stride), tile_fy(wy[1], ty_stride)};
    // Row addresses are formed ONCE, unconditionally (volatile: ptxas otherwise re-derives the whole offset inside
    // each predicated load, +80 instructions per sample); the loads themselves stay predicated.
    unsigned long long rp[2][2];
#pragma unroll
    for (int b = 0; b < 2; ++b) {
        unsigned long long pz;
        asm("mad.wide.u32 %0, %1, %2, %3;" : "=l"(pz) : "r"(wz[b] >> 3), "r"(slab_bytes), "l"(vol_base));
        const unsigned ez = ((wz[b] & 7) << 6) + exc;
#pragma unroll
        for (int a = 0; a < 2; ++a)
            asm volatile("mad.wide.u32 %0, %1, 4, %2;" : "=l"(rp[a][b]) : "r"(ez + ey[a]), "l"(pz));
    }
    // byte distance from the chunk to voxel ix + 1 when ix is the chunk's last voxel: the next chunk of the same tile
    // row (16 B on) or, from a tile's second chunk, the first voxel of the next tile in x ((512 - 4) * 4 B on)
    const unsigned de = (ix & 4u) ? (TILE_ELEMS - 4) * 4u : 16u;
#pragma unroll
    for (int a = 0; a < 2; ++a)
#pragma unroll
        for (int b = 0; b < 2; ++b) {
            const bool need = xchg || ychg[a] || zchg[b];
            if (need) K.r[a][b] = load_row_chunk(rp[a][b]);
            if (straddle && (need || e_all)) K.e[a][b] = __ldg(reinterpret_cast<const float*>(rp[a][b] + de));
        }
    K.cx = cx; K.hy[0] = wy[0]; K.hy[1] = wy[1]; K.hz[0] = wz[0]; K.hz[1] = wz[1]; K.straddle = straddle;

    // O5 blend: x inside each row, then y, then z.  Slot 0 holds the even row: it is row i when i is even
    // (weight 1-f) and row i+1 when i is odd (weight f).
    const float gy = (iy & 1) ? 1.0f - s.fy : s.fy, gz = (iz & 1) ? 1.0f - s.fz : s.fz;
    float row[2][2];
#pragma unroll
    for (int a = 0; a < 2; ++a)
#pragma unroll
        for (int b = 0; b < 2; ++b) {
            const float v0 = pick4(K.r[a][b], c, 0.0f);
            const float v1 = pick4(K.r[a][b], c + 1, K.e[a][b]);
            row[a][b] = fmaf(s.fx, v1 - v0, v0);
        }
    const float c0 = fmaf(gy, row[1][0] - row[0][0], row[0][0]);
    const float c1 = fmaf(gy, row[1][1] - row[0][1], row[0][1]);
    return fmaf(gz, c1 - c0, c0);
}

}  // namespace vr
