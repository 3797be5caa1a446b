// slab.cuh — the slab-staged caster (north_star kernel (2): "brick slabs staged through shared memory via TMA
// where the view is near axis-aligned"; section 2.4).
//
// When the pixel pitch times the step is small, many samples fall into every voxel cell and the caster is bound by
// instruction issue, not by HBM (the ridge at ~14 B per sample).  The row-cache sampler of sampler.cuh
// spends ~140 of its ~220 instructions per sample on address formation, slot bookkeeping and selects.  Here a CTA
// instead marches its 16x8-pixel tile through the brick SLAB BY SLAB along the dominant axis of the view direction: a
// slab is D cell layers thick; the box of voxels all its rays can touch inside the slab (window, D + 1 layers with the
// far neighbours) is copied by ONE bulk tensor copy (cp.async.bulk.tensor.3d, SASS UTMALDG) from a LINEAR padded copy of
// the cube into shared memory, double-buffered with mbarriers, and the eight corners of a sample are eight LDS from
// one base address plus three adds.  Orthographic frames: one window size per frame; perspective frames: the window
// follows the diverging rays (up to four sizes per frame).  Views whose dominant axis is x read a second linear copy
// with z fastest, so that a slab is always thin along the SLOWEST axis of its source.
// Positions, cells and fractions come from the same segment-anchored arithmetic as the row-cache caster
// (sampler.cuh: set_anchor / locate), the lattice, ownership and termination rules are unchanged (O4, O7, O9).
// Host side (window sizing, choice per frame, tensor maps): vr_api.cu plan_slab / choose_caster; measurements:
// profiles/r02_slab.md.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace vr {

// Linear padded copy: float lin[LZ][LY][LX] in the PADDED coordinates of the tiled copy (u = voxel + PAD), so the
// replicated layers are O5's clamp-to-edge here too.  LX is a multiple of 4 (row pitch a multiple of 16 B for TMA).
struct LinearDims {
    int LX, LY, LZ;
};
__host__ __device__ inline LinearDims linear_dims(int nx, int ny, int nz) {
    LinearDims L;
    L.LX = (nx + PAD_X + 1 + 3) & ~3;
    L.LY = ny + PAD_Y + 1;
    L.LZ = nz + PAD_Z + 1;
    return L;
}

// tiled copy -> linear padded copy: one thread per 16-byte chunk (4 voxels along x); reads whole 32-byte tile rows
// per pair of lanes, writes 512 contiguous bytes per warp.
__global__ void __launch_bounds__(256)
linearize_kernel(const float* __restrict__ tiled, float* __restrict__ lin, int LX, int LY, int LZ, unsigned ty_stride,
                 unsigned slab_stride) {
    const int cx = blockIdx.x * 64 + (threadIdx.x & 63);        // chunk index along x
    const int y = blockIdx.y * 4 + (threadIdx.x >> 6);
    const int z = blockIdx.z;
    if (cx * 4 >= LX || y >= LY) return;
    const float4 v = __ldcs(reinterpret_cast<const float4*>(tiled + tiled_index(cx * 4, y, z, ty_stride, slab_stride)));
    *reinterpret_cast<float4*>(lin + ((size_t)z * LY + y) * LX + cx * 4) = v;
}

// Second linear copy for views whose dominant axis is x: float linT[LXT][LY][LZT] with z FASTEST (LZT a multiple of 4),
// same padded coordinates.  A slab thin along x is then thin along the slowest dimension of its source, as a slab thin
// along z is for lin[][][].  One CTA transposes a 32(x) x 32(z) patch at one y through shared memory.
__host__ __device__ inline LinearDims linear_dims_t(int nx, int ny, int nz) {
    LinearDims L;
    L.LX = nx + PAD_X + 1;
    L.LY = ny + PAD_Y + 1;
    L.LZ = (nz + PAD_Z + 1 + 3) & ~3;
    return L;
}
__global__ void __launch_bounds__(256)
transpose_kernel(const float* __restrict__ tiled, float* __restrict__ linT, int LX, int LY, int LZ, int z_last,
                 unsigned ty_stride, unsigned slab_stride) {
    __shared__ float sm[32][33];
    const int x0 = blockIdx.x * 32, z0 = blockIdx.z * 32, y = blockIdx.y;
    const int tx = threadIdx.x & 31, tr = threadIdx.x >> 5;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const int zz = tr + 8 * k;
        const int x = min(x0 + tx, LX - 1), z = min(z0 + zz, z_last);      // z beyond the padded cube: copies of the last layer
        sm[zz][tx] = __ldg(tiled + tiled_index(x, y, z, ty_stride, slab_stride));
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const int xx = tr + 8 * k;
        if (x0 + xx < LX && z0 + tx < LZ) linT[((size_t)(x0 + xx) * LY + y) * LZ + z0 + tx] = sm[tx][xx];
    }
}

#ifndef VR_SLAB_WARP_W
#define VR_SLAB_WARP_W 16
#endif

constexpr double SLAB_FUZZ = 1e-3;
constexpr int SLAB_MAPS = 4;      // window sizes (tensor maps) a frame may use: perspective windows grow with depth

struct SlabParams {
    int logD;                 // slab thickness D = 1 << logD cell layers along the dominant axis
    int n_maps;               // orthographic: 1; perspective: up to SLAB_MAPS, largest first
    int w[SLAB_MAPS][3];      // window extent in voxels per axis (dominant axis: D + 1; the source's fastest axis — x, or z for
                              // x-dominant views — + 3 for the aligned start, a multiple of 4)
    int box_floats[SLAB_MAPS];// w[k][0]*w[k][1]*w[k][2]: what one bulk tensor copy with map k delivers
    int slot_floats;          // floats per buffer: box_floats[0] rounded up to a multiple of 32 (buffers stay 128-byte aligned)
    // The ray of pixel (px,py) in PADDED coordinates, both projections: it passes through Q = q0 + px*dqx + py*dqy with
    // direction V = v0 + px*dvx + py*dvy (orthographic: Q = the pixel's origin, V = fwd; perspective: Q = the eye,
    // V = fwd + u T asp right + v T up).  Where its dominant coordinate is c it is at U_a(c) = Q_a + (c - Q_dom) V_a / V_dom.
    double q0[3], dqx[3], dqy[3], v0[3], dvx[3], dvy[3];
};

struct SlabMaps {
    CUtensorMap m[SLAB_MAPS];
};

// ---- mbarrier / TMA primitives (PTX ISA: mbarrier, cp.async.bulk.tensor) ----
__device__ __forceinline__ unsigned smem_addr(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_addr(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_addr(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_addr(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_load_3d(void* dst, const CUtensorMap* map, unsigned long long* bar, int c0, int c1, int c2) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
        ::"r"(smem_addr(dst)), "l"(reinterpret_cast<unsigned long long>(map)), "r"(smem_addr(bar)), "r"(c0), "r"(c1), "r"(c2)
        : "memory");
}


// ------------------------------------------------------------------------------------------------
// a1 + a3 + a4/a5, slab-staged.  Same grid and CTA shape as cast_kernel (16x8-pixel tiles per brick rectangle).
// DOM = the dominant axis of the view direction; DOM = x reads the z-fastest copy (window laid out [x][y][z]).
// Dynamic shared memory: [2 window buffers][256 float4 table]
// [2 mbarriers][corner rays][origins].
// ------------------------------------------------------------------------------------------------
template <int MODE, int DOM>
__global__ void __launch_bounds__(CTA_THREADS)
cast_slab_kernel(const __grid_constant__ FrameParams P, const __grid_constant__ SlabParams S,
                 const __grid_constant__ SlabMaps maps, const BrickRec* __restrict__ bricks, int n_bricks,
                 const float4* __restrict__ tf_global, float* __restrict__ img) {
    extern __shared__ unsigned char smem_raw[];
    // carve: windows first (128-byte aligned for the bulk tensor copy)
    unsigned char* sb = smem_raw + ((128u - (smem_addr(smem_raw) & 127u)) & 127u);
    float* win = reinterpret_cast<float*>(sb);
    float4* tf = reinterpret_cast<float4*>(sb + (size_t)2 * S.slot_floats * 4);
    unsigned long long* bar = reinterpret_cast<unsigned long long*>(tf + 256);
    double* s_ray = reinterpret_cast<double*>(bar + 2);    // [4 tile corners][5]: Q_a1, Q_a2, Q_dom, slope_a1, slope_a2
    int* s_org = reinterpret_cast<int*>(s_ray + 20);       // [2][8]: window origin (3), x pitch, layer pitch per buffer
    int* s_misc = s_org + 16;                              // [0] brick, [1] min slab, [2] max slab

    const int tid = threadIdx.x;
    if (MODE == MODE_EA)
        for (int i = tid; i < 256; i += CTA_THREADS) tf[i] = tf_global[i];
    if (tid == 0) {
        int lo = 0, hi = n_bricks - 1;
        while (lo < hi) {
            const int mid = (lo + hi + 1) >> 1;
            if (bricks[mid].tile0 <= (int)blockIdx.x) lo = mid; else hi = mid - 1;
        }
        s_misc[0] = lo; s_misc[1] = 0x7fffffff; s_misc[2] = -0x7fffffff;
        mbar_init(&bar[0], 1); mbar_init(&bar[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const BrickRec* __restrict__ br = bricks + s_misc[0];
    const int tloc = (int)blockIdx.x - br->tile0;
    const int tiles_x = br->tiles_x;
    const int tyi = tloc / tiles_x, txi = tloc - tyi * tiles_x;
    const int warp = tid >> 5, lane = tid & 31;
    // warp patch SLAB_WARP_W x (32 / SLAB_WARP_W) pixels: a wide patch spreads the lanes of one pixel row over many
    // banks of the window (measured 16x2 vs 8x4 in profiles/r02_slab.md)
    constexpr int WW = VR_SLAB_WARP_W, WH = 32 / VR_SLAB_WARP_W, WPR = CTA_W / WW;
    const int lx = txi * CTA_W + (warp % WPR) * WW + (lane % WW);
    const int ly = tyi * CTA_H + (warp / WPR) * WH + (lane / WW);
    const bool inside = lx < br->rw && ly < br->rh;
    const int px = br->rx0 + lx, py = br->ry0 + ly;

    double o[3], d[3];
    make_ray(P, px, py, o, d);
    long long i_lo = 0;
    double t_near = 0.0;
    const int n = inside ? owned_samples(P, br, o, d, t_near, i_lo) : 0;
    const float h[3] = {(float)(P.step * d[0]), (float)(P.step * d[1]), (float)(P.step * d[2])};
    const int logD = S.logD;

    Anchor An;
    int js = 0;                                            // first sample of the current segment
    if (n > 0) {                                           // slab range of this ray: its first and its last sample
        // Both with the arithmetic the march below places them with (anchor of the sample's segment + locate): an
        // anchor of its own at the last sample may disagree with the march by ~5e-6 voxel and, on a slab face, name a
        // slab the sample is not marched in; that slab would never be staged and the sample dropped.
        Cell c;
        const int js_last = ((n - 1) / P.seg_len) * P.seg_len;
        set_anchor(o, d, t_near, P.step, i_lo + js_last, h, P.seg_span, An);
        locate(An, (n - 1) - js_last, h, c);
        const int c_last = (int)(DOM == 0 ? c.ix : DOM == 1 ? c.iy : c.iz) >> logD;
        set_anchor(o, d, t_near, P.step, i_lo, h, P.seg_span, An);
        locate(An, 0, h, c);
        const int c_first = (int)(DOM == 0 ? c.ix : DOM == 1 ? c.iy : c.iz) >> logD;
        atomicMin(&s_misc[1], min(c_first, c_last));
        atomicMax(&s_misc[2], max(c_first, c_last));
    }
    __syncthreads();
    const int s_min = s_misc[1], s_max = s_misc[2];
    const int ns = s_max >= s_min ? s_max - s_min + 1 : 0;
    const int sgn = P.fwd[DOM] >= 0.0 ? 1 : -1;            // every ray of the frame advances this way along DOM (host check)
    const int s_begin = sgn > 0 ? s_min : s_max;

    // Window of a slab on the two other axes: bounding box of the tile's rays between the slab's faces.  U_a(c) is
    // linear-fractional in (px,py) and linear in c, so its extremes over the tile are taken by a corner ray on a face.
    constexpr int A1 = (DOM + 1) % 3, A2 = (DOM + 2) % 3;
    constexpr int FAST = DOM == 0 ? 2 : 0, SLOW = DOM == 0 ? 0 : 2;       // fastest / slowest axis of the window and its source
    if (tid == 0) {
        const int px0 = br->rx0 + txi * CTA_W, py0 = br->ry0 + tyi * CTA_H;
#pragma unroll
        for (int cnr = 0; cnr < 4; ++cnr) {
            const double fx = (double)(px0 + ((cnr & 1) ? CTA_W - 1 : 0)), fy = (double)(py0 + ((cnr & 2) ? CTA_H - 1 : 0));
            const double vd = S.v0[DOM] + fx * S.dvx[DOM] + fy * S.dvy[DOM];
            s_ray[cnr * 5 + 0] = S.q0[A1] + fx * S.dqx[A1] + fy * S.dqy[A1];
            s_ray[cnr * 5 + 1] = S.q0[A2] + fx * S.dqx[A2] + fy * S.dqy[A2];
            s_ray[cnr * 5 + 2] = S.q0[DOM] + fx * S.dqx[DOM] + fy * S.dqy[DOM];
            s_ray[cnr * 5 + 3] = (S.v0[A1] + fx * S.dvx[A1] + fy * S.dvy[A1]) / vd;
            s_ray[cnr * 5 + 4] = (S.v0[A2] + fx * S.dvx[A2] + fy * S.dvy[A2]) / vd;
        }
    }
    auto issue = [&](int k) {                              // thread 0: start the copy of slab k into buffer k & 1
        const int s = s_begin + sgn * k, slot = k & 1;
        const double c0 = (double)(s << logD), c1 = c0 + (double)(1 << logD);
        double lo1 = INFINITY, lo2 = INFINITY, hi1 = -INFINITY, hi2 = -INFINITY;
#pragma unroll
        for (int cnr = 0; cnr < 4; ++cnr) {
            const double q1 = s_ray[cnr * 5 + 0], q2 = s_ray[cnr * 5 + 1], qd = s_ray[cnr * 5 + 2];
            const double m1 = s_ray[cnr * 5 + 3], m2 = s_ray[cnr * 5 + 4];
            const double a0 = q1 + (c0 - qd) * m1, a1 = q1 + (c1 - qd) * m1;
            const double b0 = q2 + (c0 - qd) * m2, b1 = q2 + (c1 - qd) * m2;
            lo1 = fmin(lo1, fmin(a0, a1)); hi1 = fmax(hi1, fmax(a0, a1));
            lo2 = fmin(lo2, fmin(b0, b1)); hi2 = fmax(hi2, fmax(b0, b1));
        }
        int org[3], ext[3];
        org[DOM] = s << logD; ext[DOM] = 0;
        // voxels floor(lo) .. floor(hi) + 1; SLAB_FUZZ covers the difference between these fp64 corner rays and the
        // fp32 segment arithmetic that places the samples (<= 1e-5 voxel)
        org[A1] = (int)floor(lo1 - SLAB_FUZZ); ext[A1] = (int)floor(hi1 + SLAB_FUZZ) + 2 - org[A1];
        org[A2] = (int)floor(lo2 - SLAB_FUZZ); ext[A2] = (int)floor(hi2 + SLAB_FUZZ) + 2 - org[A2];
        ext[FAST] += org[FAST] & 3;
        org[FAST] &= ~3;                                   // the copy must start 16-byte aligned (measured: a start
                                                           // coordinate that is not a multiple of 4 floats faults)
        int m = 0;                                         // the smallest window that holds the box (map 0 always does)
        for (int q = 1; q < S.n_maps; ++q)
            if (ext[A1] <= S.w[q][A1] && ext[A2] <= S.w[q][A2]) m = q;
        int* so = s_org + slot * 8;
        so[0] = org[0]; so[1] = org[1]; so[2] = org[2]; so[3] = S.w[m][FAST]; so[4] = S.w[m][FAST] * S.w[m][1];
        mbar_expect_tx(&bar[slot], (unsigned)S.box_floats[m] * 4u);
        tma_load_3d(win + (size_t)slot * S.slot_floats, &maps.m[m], &bar[slot], org[FAST], org[1], org[SLOW]);
    };
    if (tid == 0 && ns > 0) issue(0);

    float Cr = 0.f, Cg = 0.f, Cb = 0.f, A = 0.f, M = -INFINITY;
    int j = 0;
    for (int k = 0; k < ns; ++k) {
        const int slot = k & 1;
        const int any = __syncthreads_or(j < n);           // every thread is done with slab k - 1 (buffer (k + 1) & 1)
        if (any && tid == 0 && k + 1 < ns) issue(k + 1);
        mbar_wait(&bar[slot], (unsigned)(k >> 1) & 1u);    // slab k has landed (it was issued in any case)
        if (!any) break;
        const int s = s_begin + sgn * k;
        const int w0 = s_org[slot * 8 + 3], w01 = s_org[slot * 8 + 4];
        const float* __restrict__ wbase = win + (size_t)slot * S.slot_floats
                                          - (s_org[slot * 8 + FAST] + s_org[slot * 8 + 1] * w0 + s_org[slot * 8 + SLOW] * w01);
        // The segment origin O is folded into the window base, and the slab test runs on the integer part m of the
        // position relative to O (cell = O + m): cell_dom in [s D, s D + D)  <=>  (unsigned)(m_dom - (s D - O_dom)) < D.
        const int D = 1 << logD;
        const float* __restrict__ sbase = wbase + (An.O[FAST] + An.O[1] * w0 + An.O[SLOW] * w01);
        int lo_m = (s << logD) - An.O[DOM];
        while (j < n) {
            int jl = j - js;
            if (jl == P.seg_len) {
                js = j; jl = 0;
                set_anchor(o, d, t_near, P.step, i_lo + js, h, P.seg_span, An);
                sbase = wbase + (An.O[FAST] + An.O[1] * w0 + An.O[SLOW] * w01);
                lo_m = (s << logD) - An.O[DOM];
            }
            const float jf = (float)jl;
            float q[3], r[3];
            int m[3];
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                q[a] = fmaf(jf, h[a], An.rel[a]);
                r[a] = __fadd_rd(q[a], 8388608.0f);       // 0 <= q < 2^22: the integer part is the low mantissa bits
                m[a] = (int)(__float_as_uint(r[a]) & 0x7fffffu);
            }
            if ((unsigned)(m[DOM] - lo_m) >= (unsigned)D) break;
            Cell c;                                        // fractions only: the cell itself is O + m
            c.fx = q[0] - (r[0] - 8388608.0f);
            c.fy = q[1] - (r[1] - 8388608.0f);
            c.fz = q[2] - (r[2] - 8388608.0f);
            const float* __restrict__ p0 = sbase + (m[FAST] + m[1] * w0 + m[SLOW] * w01);
            const float* __restrict__ p1 = p0 + w0;
            const float* __restrict__ p2 = p0 + w01;
            const float* __restrict__ p3 = p2 + w0;
            // corners v[dz][dy][dx]: the +1 neighbour along the window's fastest axis is the next float
            const float v000 = p0[0], v010 = p1[0];
            const float v100 = DOM == 0 ? p0[1] : p2[0], v110 = DOM == 0 ? p1[1] : p3[0];
            const float v001 = DOM == 0 ? p2[0] : p0[1], v011 = DOM == 0 ? p3[0] : p1[1];
            const float v101 = DOM == 0 ? p2[1] : p2[1], v111 = p3[1];
            const float c00 = fmaf(c.fx, v001 - v000, v000);
            const float c10 = fmaf(c.fx, v011 - v010, v010);
            const float c01 = fmaf(c.fx, v101 - v100, v100);
            const float c11 = fmaf(c.fx, v111 - v110, v110);
            const float c0 = fmaf(c.fy, c10 - c00, c00);
            const float c1 = fmaf(c.fy, c11 - c01, c01);
            const float v = fmaf(c.fz, c1 - c0, c0);
            ++j;
            if (MODE == MODE_EA) {
                classify_blend(tf, P, v, Cr, Cg, Cb, A);
                if (P.ert_on && A >= P.ert) j = n;
            } else {
                M = fmaxf(M, v);
            }
        }
    }
    if (!inside) return;
    const size_t pix = (size_t)br->img_base + (size_t)(py - br->oy) * br->img_stride + (size_t)(px - br->ox);
    if (MODE == MODE_EA) reinterpret_cast<float4*>(img)[pix] = make_float4(Cr, Cg, Cb, A);
    else img[pix] = M;
}

}  // namespace vr
