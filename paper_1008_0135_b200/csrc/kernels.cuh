// kernels.cuh — the sm_100a kernels of the hot path.
//
//   relayout_kernel   a0  linear cube -> 8x8x8-voxel tiles
//   cast_kernel<EA>   a1,a3,a4  per-brick ray caster, emission-absorption
//   cast_kernel<MIP>  a1,a3,a5  maximum-intensity variant
//   composite_kernel  a7  depth-ordered "over" / max of the brick images
//
// Per-ray set-up (ray, slab clips, sample index ranges) is double precision and follows DESIGN.md
// O2-O4 and O9 term by term; per-sample work is fp32.  No code is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string.h>

namespace vr {

constexpr int TILE = 8;                 // voxels per tile edge
constexpr int TILE_ELEMS = 512;         // 8^3 floats = 2 KB, x-rows of 32 B = one DRAM sector
// Padded coordinates of the tiled copy: u = voxel index + PAD.  y and z carry one replicated layer below index 0;
// x carries a whole tile (8) so that the re-layout's row reads stay 32-byte aligned with the source rows.
constexpr int PAD_X = 8, PAD_Y = 1, PAD_Z = 1;
// CTA shape of the caster, chosen by measurement on the config-3 orbit (B200): 16x8 pixels (4 warps) with 7
// CTAs per SM (72 registers) gave 5.88 ms mean cast time; 16x16 with 3 CTAs 6.08 ms; forcing 64 registers for
// 8 CTAs (32 warps) 7.6 ms - more resident rays thrash the L1 that carries the sector re-use between rays.
#ifndef VR_WARP_W
#define VR_WARP_W 8
#endif
#ifndef VR_CTA_H
#define VR_CTA_H 8
#endif
#ifndef VR_CAST_MINBLOCKS
#define VR_CAST_MINBLOCKS 7
#endif
#ifndef VR_CTA_W
#define VR_CTA_W 16
#endif
#ifndef VR_OCC_GROUP
#define VR_OCC_GROUP 16     // samples per group of the occupancy pass (power of two <= 32; measured 2: 4.43, 4: 4.38, 8: 4.35, 16: 4.34 ms)
#endif
constexpr int CTA_W = VR_CTA_W;               // a CTA renders a CTA_W x CTA_H pixel tile: warps of 8x4 pixels, 2 across
constexpr int CTA_H = VR_CTA_H;
constexpr int CTA_THREADS = CTA_W * CTA_H;
constexpr int MODE_EA = 0, MODE_MIP = 1;
constexpr int MAX_RUNS = 16;                  // VR_MAX_CHANNEL_RUNS of include/vr.h

struct FrameParams {
    double eye[3], right[3], up[3], fwd[3];   // O1
    double h, asp, tanhalf;                   // O2: ortho half height, W/H, tan(fovy/2)
    double step;                              // O4: Delta in voxels
    int proj, W, H;
    int nx, ny, nz;
    unsigned ty_stride;                       // elements between tiles adjacent in y  = TX*512
    unsigned slab_stride;                     // elements between tiles adjacent in z  = TX*TY*512
    float vmin, inv_range;                    // O6
    float ert;                                // O7 threshold
    float x_zero_below;                       // table position below which alpha is exactly 0 (-1: nowhere)
    int ert_on;
    int seg_len, seg_span;                    // samples per anchored segment; ceil(seg_len*step)+1 (sampler.cuh)
    int nbx, nby;                             // occupancy-mask words (4^3 cells) per row / per column
    int n_runs;                               // S2 channel mask: runs of enabled channels (0 = no mask)
    int run_z[2 * MAX_RUNS];                  // [za, zb) per run, ascending
};

struct BrickRec {
    int lo[3], hi[3];         // brick box (voxels)
    int rx0, ry0, rw, rh;     // rendering rectangle (pixels)
    int tile0, tiles_x;       // first CTA index of this brick, CTAs per rectangle row
    long long img_base;       // pixel offset of this brick's image in the image buffer
    int img_stride, ox, oy;   // row stride (pixels) and pixel coordinates of image element (0,0)
    int pad;
};

// Tile order: plain row-major, tile (tx,ty,tz) at ((tz*TY + ty)*TX + tx); the address is separable,
// off = fx(x) + fy(y) + fz(z).  (north_star kernel (1) also names a Morton order of the tiles: measured in round 2 as a
// build switch and rejected, +6-7 % frame time; profiles/r02_experiments.md names the commit that still carries it.)
__host__ __device__ __forceinline__ unsigned tile_fx(unsigned x) { return (x >> 3) * TILE_ELEMS + (x & 7u); }
__host__ __device__ __forceinline__ unsigned tile_fy(unsigned y, unsigned ty_stride) { return (y >> 3) * ty_stride + ((y & 7u) << 3); }
__host__ __device__ __forceinline__ size_t tile_fz(unsigned z, unsigned slab_stride) { return (size_t)(z >> 3) * slab_stride + ((z & 7u) << 6); }

// ------------------------------------------------------------------------------------------------
// a0  re-layout.  The tiled copy holds the cube in PADDED coordinates u = voxel index + PAD_a (8, 1, 1): replicated
// layers below index 0 and at least one above index n-1 on every axis (T_a = ceil((n_a + PAD_a + 1)/8) tiles).  Trilinear
// interpolation between an edge voxel and its replica returns the edge value exactly (fma(f, v-v, v) = v), which is
// O5's clamp-to-edge without a clamp, a floor of a negative number or a bounds test in the sample loop: a sample
// at q = p - 1/2 in [-1/2, n - 1/2] reads padded voxels floor(q) + PAD (>= PAD - 1) and floor(q) + PAD + 1 (<= n + PAD).
// (An infinite voxel on a face would give inf - inf = NaN where the clamp gives inf; survey cubes blank with NaN.)
// One CTA moves an 8(z) x 8(y) x 64(x) block: coalesced row reads -> shared memory -> 8 whole tiles written as
// one contiguous 16 KB run of float4 stores.
// ------------------------------------------------------------------------------------------------
constexpr int RANGE_SLOTS = 256;
// order-preserving map float -> unsigned (so atomicMin/atomicMax on the key order the floats)
__host__ __device__ __forceinline__ unsigned float_key(float f) {
#ifdef __CUDA_ARCH__
    const unsigned u = __float_as_uint(f);
#else
    unsigned u; memcpy(&u, &f, 4);
#endif
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__host__ __device__ __forceinline__ float key_float(unsigned k) {
    const unsigned u = (k & 0x80000000u) ? (k & 0x7fffffffu) : ~k;
#ifdef __CUDA_ARCH__
    return __uint_as_float(u);
#else
    float f; memcpy(&f, &u, 4); return f;
#endif
}

__global__ void __launch_bounds__(256)
relayout_kernel(const float* __restrict__ src, float* __restrict__ dst, int nx, int ny, int nz,
                int TX, int TY, unsigned* __restrict__ range_slots) {
    __shared__ __align__(16) float sm[64][72];   // row = lz*8+ly; 72-float pitch: conflict-free float4 reads
    const int tx0 = blockIdx.x * 8, ty = blockIdx.y, tz = blockIdx.z;
    const int t = threadIdx.x;
    const int xo = t & 63;
    const int xs = min(max(tx0 * 8 + xo - PAD_X, 0), nx - 1);  // padded -> voxel, replicated at both ends
    float vmin = INFINITY, vmax = -INFINITY;
#pragma unroll
    for (int k = 0; k < 16; ++k) {
        const int row = (t >> 6) + 4 * k;
        const int z = min(max(tz * 8 + (row >> 3) - PAD_Z, 0), nz - 1);
        const int y = min(max(ty * 8 + (row & 7) - PAD_Y, 0), ny - 1);
        const float val = __ldcs(src + ((size_t)z * ny + y) * nx + xs);
        sm[row][xo] = val;
        vmin = fminf(vmin, val);      // fminf/fmaxf ignore NaN (blanked voxels)
        vmax = fmaxf(vmax, val);
    }
    // min/max of the cube, fused into the one pass that reads it (each GPU computes the
    // minimum and maximum of its portion).  Order-preserving unsigned keys, RANGE_SLOTS slot pairs to keep the
    // atomics uncontended; the host reduces the slots.
    for (int sft = 16; sft > 0; sft >>= 1) {
        vmin = fminf(vmin, __shfl_xor_sync(0xffffffffu, vmin, sft));
        vmax = fmaxf(vmax, __shfl_xor_sync(0xffffffffu, vmax, sft));
    }
    __shared__ float s_min[8], s_max[8];
    if ((t & 31) == 0) { s_min[t >> 5] = vmin; s_max[t >> 5] = vmax; }
    __syncthreads();
    if (t == 0 && range_slots) {      // one candidate per CTA; the atomic is issued only if it would change the slot
        float lo = s_min[0], hi = s_max[0];
#pragma unroll
        for (int w = 1; w < 8; ++w) { lo = fminf(lo, s_min[w]); hi = fmaxf(hi, s_max[w]); }
        if (lo <= hi) {               // false only if every voxel seen was NaN
            unsigned* slot = range_slots + 2 * ((blockIdx.x + 7u * blockIdx.y + 13u * blockIdx.z) & (RANGE_SLOTS - 1));
            const unsigned klo = float_key(lo), khi = float_key(hi);
            if (klo < *(volatile unsigned*)slot) atomicMin(slot, klo);
            if (khi > *(volatile unsigned*)(slot + 1)) atomicMax(slot + 1, khi);
        }
    }
    const int ntile = min(8, TX - tx0);
    float4* out = reinterpret_cast<float4*>(dst + ((size_t)((size_t)tz * TY + ty) * TX + tx0) * TILE_ELEMS);
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const int j = t + 256 * k;           // float4 index inside the 8-tile run
        const int tile = j >> 7, r = j & 127;
        if (tile < ntile) {
            const int row = r >> 1, lxq = r & 1;
            const float4 v = *reinterpret_cast<const float4*>(&sm[row][tile * 8 + lxq * 4]);
            out[j] = v;
        }
    }
}

// element offset of PADDED position (x,y,z) = voxel index + (PAD_X, PAD_Y, PAD_Z) in the tiled copy
__device__ __forceinline__ size_t tiled_index(int x, int y, int z, unsigned ty_stride, unsigned slab_stride) {
    return tile_fz((unsigned)z, slab_stride) + (size_t)tile_fy((unsigned)y, ty_stride) + (size_t)tile_fx((unsigned)x);
}

// NEXT-1  histogram of the cube (the data range and distribution the colour map is built on).
// One pass over the tiled copy; padding replicas are not counted.  bin = floor((v - lo) * scale) in fp32, clamped to
// [0, n_bins - 1]; NaN voxels are counted in nan_count only.  Per-CTA shared-memory bins, then one global add per bin.
constexpr int HIST_MAX_BINS = 4096;
__global__ void __launch_bounds__(256)
histogram_kernel(const float* __restrict__ tiled, size_t n_tiles, int TX, int TY, int nx, int ny, int nz, float lo,
                 float scale, int n_bins, unsigned long long* __restrict__ bins, unsigned long long* __restrict__ nan_count) {
    extern __shared__ unsigned sh_bins[];
    for (int i = threadIdx.x; i < n_bins; i += 256) sh_bins[i] = 0u;
    __syncthreads();
    unsigned nans = 0;
    for (size_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        const int tx = (int)(tile % TX), ty = (int)((tile / TX) % TY), tz = (int)(tile / ((size_t)TX * TY));
        const float4* src = reinterpret_cast<const float4*>(tiled + tile * TILE_ELEMS);
        for (int q = threadIdx.x; q < TILE_ELEMS / 4; q += 256) {
            const float4 v4 = __ldcs(src + q);
            const int lx = (q & 1) * 4, ly = (q >> 1) & 7, lz = q >> 4;
            const int y = ty * 8 + ly - PAD_Y, z = tz * 8 + lz - PAD_Z;
            if (y < 0 || y >= ny || z < 0 || z >= nz) continue;
            const float v[4] = {v4.x, v4.y, v4.z, v4.w};
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const int x = tx * 8 + lx + k - PAD_X;
                if (x < 0 || x >= nx) continue;
                if (v[k] != v[k]) { ++nans; continue; }
                const float b = floorf((v[k] - lo) * scale);
                const int bi = (int)fminf(fmaxf(b, 0.0f), (float)(n_bins - 1));
                atomicAdd(&sh_bins[bi], 1u);
            }
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < n_bins; i += 256)
        if (sh_bins[i]) atomicAdd(&bins[i], (unsigned long long)sh_bins[i]);
    if (nans) atomicAdd(nan_count, (unsigned long long)nans);
}

// inverse of a0 (round-trip test only)
__global__ void export_linear_kernel(const float* __restrict__ tiled, float* __restrict__ dst, int nx, int ny,
                                     int nz, unsigned ty_stride, unsigned slab_stride) {
    const size_t n = (size_t)nx * ny * nz;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const int x = (int)(i % nx);
        const size_t r = i / nx;
        const int y = (int)(r % ny), z = (int)(r / ny);
        dst[i] = tiled[tiled_index(x + PAD_X, y + PAD_Y, z + PAD_Z, ty_stride, slab_stride)];
    }
}

__global__ void fill_kernel(float* __restrict__ p, size_t n, float v) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
        p[i] = v;
}

// ------------------------------------------------------------------------------------------------
// per-ray set-up in double (O2, O3, O4, O9)
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void make_ray(const FrameParams& P, int px, int py, double o[3], double d[3]) {
    const double u = 2.0 * ((double)px + 0.5) / (double)P.W - 1.0;
    const double v = 2.0 * ((double)py + 0.5) / (double)P.H - 1.0;
    if (P.proj == 0) {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            o[c] = P.eye[c] + u * P.h * P.asp * P.right[c] + v * P.h * P.up[c];
            d[c] = P.fwd[c];
        }
    } else {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            o[c] = P.eye[c];
            d[c] = P.fwd[c] + u * P.tanhalf * P.asp * P.right[c] + v * P.tanhalf * P.up[c];
        }
        const double l = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
        d[0] /= l; d[1] /= l; d[2] /= l;
    }
}

// O3 slab clip against [lo,hi]; t0 is not clamped to >= 0 here.
__device__ __forceinline__ bool slab_clip(const double o[3], const double d[3], const double lo[3],
                                          const double hi[3], double& tn, double& tf) {
    tn = -INFINITY; tf = INFINITY;
    bool ok = true;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        if (d[a] == 0.0) {
            if (!(lo[a] <= o[a] && o[a] < hi[a])) ok = false;
        } else {
            const double t0 = (lo[a] - o[a]) / d[a];
            const double t1 = (hi[a] - o[a]) / d[a];
            const double tmin = t0 < t1 ? t0 : t1;
            const double tmax = t0 < t1 ? t1 : t0;
            if (tmin > tn) tn = tmin;
            if (tmax < tf) tf = tmax;
        }
    }
    return ok;
}

// O4: I(t) = max(0, ceil((t - t_near)/step - 1/2))
__device__ __forceinline__ long long lattice_index(double t, double t_near, double step) {
    const double x = ceil((t - t_near) / step - 0.5);
    return x > 0.0 ? (long long)x : 0ll;
}

// O3 + O4 + O9 for one (ray, brick): global clip, t_near, and the range [i_lo, i_lo + n) of the global lattice the
// brick owns.  Returns n (0: miss or nothing owned).
__device__ __forceinline__ int owned_samples(const FrameParams& P, const BrickRec* __restrict__ br, const double o[3],
                                             const double d[3], double& t_near, long long& i_lo) {
    const double glo[3] = {0.0, 0.0, 0.0};
    const double ghi[3] = {(double)P.nx, (double)P.ny, (double)P.nz};
    double tn, tf_;
    bool hit = slab_clip(o, d, glo, ghi, tn, tf_);
    if (tn < 0.0) tn = 0.0;
    hit = hit && (tf_ > tn);
    long long i_hi = 0;
    i_lo = 0; t_near = 0.0;
    if (hit) {
        t_near = tn;
        const double blo[3] = {(double)br->lo[0], (double)br->lo[1], (double)br->lo[2]};
        const double bhi[3] = {(double)br->hi[0], (double)br->hi[1], (double)br->hi[2]};
        double t0, t1;
        bool bh = slab_clip(o, d, blo, bhi, t0, t1);
        if (t0 < tn) t0 = tn;
        if (t1 > tf_) t1 = tf_;
        if (bh && t1 > t0) {
            i_lo = lattice_index(t0, tn, P.step);
            i_hi = lattice_index(t1, tn, P.step);
        }
    }
    return (i_hi > i_lo) ? (int)(i_hi - i_lo) : 0;
}

// ------------------------------------------------------------------------------------------------
// O5  plain 8-corner trilinear sample of one cell (measuring build only: marks the 32-byte sectors it reads).
// ------------------------------------------------------------------------------------------------
struct Footprint {           // the 8 voxels of one sample
    float v[8];
};

}  // namespace vr
#include "sampler.cuh"
namespace vr {

__device__ __forceinline__ void fetch_marked(const float* __restrict__ vol, const FrameParams& P, const Cell& c,
                                             Footprint& F, unsigned* __restrict__ bitmap) {
    const unsigned ix = c.ix, iy = c.iy, iz = c.iz;
    // separable tiled offsets; +1 neighbours always exist (padding), see relayout_kernel
    const unsigned ix1 = ix + 1, iy1 = iy + 1, iz1 = iz + 1;
    const unsigned ex0 = tile_fx(ix), ex1 = tile_fx(ix1);
    const unsigned ey0 = tile_fy(iy, P.ty_stride), ey1 = tile_fy(iy1, P.ty_stride);
    const float* __restrict__ pz0 = vol + tile_fz(iz, P.slab_stride);
    const float* __restrict__ pz1 = vol + tile_fz(iz1, P.slab_stride);
    const unsigned e00 = ex0 + ey0, e10 = ex1 + ey0, e01 = ex0 + ey1, e11 = ex1 + ey1;
    F.v[0] = __ldg(pz0 + e00); F.v[1] = __ldg(pz0 + e10);
    F.v[2] = __ldg(pz0 + e01); F.v[3] = __ldg(pz0 + e11);
    F.v[4] = __ldg(pz1 + e00); F.v[5] = __ldg(pz1 + e10);
    F.v[6] = __ldg(pz1 + e01); F.v[7] = __ldg(pz1 + e11);
    // mark the 32-byte sectors (8 consecutive floats) of the footprint
    const size_t b0 = (size_t)(pz0 - vol), b1 = (size_t)(pz1 - vol);
    const size_t s[8] = {(b0 + e00) >> 3, (b0 + e10) >> 3, (b0 + e01) >> 3, (b0 + e11) >> 3,
                         (b1 + e00) >> 3, (b1 + e10) >> 3, (b1 + e01) >> 3, (b1 + e11) >> 3};
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        const unsigned bit = 1u << (unsigned)(s[k] & 31);
        unsigned* w = bitmap + (s[k] >> 5);
        if (!(*(volatile unsigned*)w & bit)) atomicOr(w, bit);
    }
}

__device__ __forceinline__ float trilerp(const Footprint& F, const Cell& c) {
    const float c00 = fmaf(c.fx, F.v[1] - F.v[0], F.v[0]);
    const float c10 = fmaf(c.fx, F.v[3] - F.v[2], F.v[2]);
    const float c01 = fmaf(c.fx, F.v[5] - F.v[4], F.v[4]);
    const float c11 = fmaf(c.fx, F.v[7] - F.v[6], F.v[6]);
    const float c0 = fmaf(c.fy, c10 - c00, c00);
    const float c1 = fmaf(c.fy, c11 - c01, c01);
    return fmaf(c.fz, c1 - c0, c0);
}

// O6 + O7: classify through the shared-memory table (256 float4 entries) and blend.
// Transparent-sample skip: x_zero_below = (index of the first table entry with alpha > 0) - 1.  For x below it both
// entries the lookup would blend have alpha exactly 0, so the sample adds exactly nothing to C and A (as in
// the oracle) and the table reads and the blend are skipped — with a noise-suppressing table
// that is most samples of a survey cube, and the shared-memory lookups are a fifth of the L1 data-pipe load.
__device__ __forceinline__ void classify_blend(const float4* __restrict__ tf, const FrameParams& P, float value,
                                               float& Cr, float& Cg, float& Cb, float& A) {
    const float x = __saturatef((value - P.vmin) * P.inv_range) * 255.0f;    // NaN -> 0
    if (x < P.x_zero_below) return;
    const float r = fminf(__fadd_rd(x, 8388608.0f), 8388608.0f + 254.0f);   // 2^23 + min(floor(x),254)
    const unsigned m = __float_as_uint(r) & 0xffu;
    const float w = x - (r - 8388608.0f);
    const float4 t0 = tf[m], t1 = tf[m + 1];
    const float4 dt = make_float4(t1.x - t0.x, t1.y - t0.y, t1.z - t0.z, t1.w - t0.w);
    float a = fmaf(w, dt.w, t0.w);
    a = (value == value) ? a : 0.0f;                                         // O5/A14: NaN sample skipped
    const float wgt = (1.0f - A) * a;
    Cr = fmaf(wgt, fmaf(w, dt.x, t0.x), Cr);
    Cg = fmaf(wgt, fmaf(w, dt.y, t0.y), Cg);
    Cb = fmaf(wgt, fmaf(w, dt.z, t0.z), Cb);
    A += wgt;
}

// ------------------------------------------------------------------------------------------------
// NEXT-2  occupancy mask for empty-space skipping (PAPER.md:144 balanced work, PAPER.md:205 finding 2: the work
// depends on the data, PAPER.md:294 noise-suppressing transfer functions).  One bit per PADDED cell (i,j,k), i in
// [0, n_x + PAD_X) etc. = the unit cube between padded voxels i..i+1, j..j+1, k..k+1 in which O5 interpolates (cell 0 and
// cell n_a are the half-voxel rims where the replicated layer stands in for the clamp).  The bit is CLEAR when
// every sample in the cell contributes exactly nothing under the current table:
//   * a corner is NaN  -> the blend is NaN -> the sample is skipped (O5/A14), or
//   * all 8 corners classify more than MASK_MARGIN table entries below the first entry with alpha > 0: the
//     blend is a convex combination of the corners (up to a few ulp), so its table position x is below
//     x_zero_below and both entries the lookup blends have alpha = 0 (O6) -> C and A unchanged (O7).
// A clear bit therefore never changes a pixel: the oracle needs no rule for it, and parity gates stay as they are.
// Layout: 64-bit words of 4x4x4 cells, word ((bz*NBY + by)*NBX + bx), bit (lz*4 + ly)*4 + lx.
// One CTA = 32 x 8 x 8 cells (8 x 2 x 2 words): each warp classifies rows of 33 corner voxels into two bit sets
// (ballot), a cell row of 32 cells is then four ORs, a shift and an AND-NOT on 64-bit words.
// ------------------------------------------------------------------------------------------------
constexpr float MASK_MARGIN = 0.01f;       // in table entries (x units): far above fp32 rounding of the blend

__global__ void __launch_bounds__(256)
build_mask_kernel(const float* __restrict__ vol, unsigned ty_stride, unsigned slab_stride, int nx, int ny, int nz,
                  float vmin, float inv_range, float x_zero_below, unsigned long long* __restrict__ mask, int NBX,
                  int NBY, unsigned long long* __restrict__ n_occupied) {
    // per (z,y) row of the 33 x 9 x 9 corner voxels: bit x set when the voxel may be visible / is NaN
    __shared__ unsigned long long vis[9][9], nanb[9][9];
    __shared__ unsigned rowbits[8][8];          // [lz][ly]: the 32 cell bits of one cell row
    const int x0 = blockIdx.x * 32, y0 = blockIdx.y * 8, z0 = blockIdx.z * 8;
    const int t = threadIdx.x;
    const int x_last = (int)(ty_stride >> 9) * 8 - 1;            // last padded x that exists (TX * 8 - 1)
    const float thr = x_zero_below - MASK_MARGIN;
    if (t < 81) { (&vis[0][0])[t] = 0ull; (&nanb[0][0])[t] = 0ull; }
    __syncthreads();
    // 81 rows x (8 aligned 16-byte chunks + the 33rd voxel) = 729 items, three per thread: all loads first
    float4 q[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const int i = t + 256 * k;
        q[k] = make_float4(0.f, 0.f, 0.f, 0.f);
        if (i < 729) {
            const int row = i / 9, ch = i - row * 9;
            const int y = min(y0 + row % 9, ny + PAD_Y), z = min(z0 + row / 9, nz + PAD_Z);
            if (ch < 8) q[k] = __ldg(reinterpret_cast<const float4*>(vol + tiled_index(min(x0 + 4 * ch, x_last - 3), y, z, ty_stride, slab_stride)));
            else q[k].x = __ldg(vol + tiled_index(min(x0 + 32, x_last), y, z, ty_stride, slab_stride));
        }
    }
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const int i = t + 256 * k;
        if (i < 729) {
            const int row = i / 9, ch = i - row * 9;
            const float v[4] = {q[k].x, q[k].y, q[k].z, q[k].w};
            unsigned long long bv = 0ull, bn = 0ull;
            const int nv = ch < 8 ? 4 : 1;
            for (int e = 0; e < nv; ++e) {
                const float xt = __saturatef((v[e] - vmin) * inv_range) * 255.0f;
                if (v[e] != v[e]) bn |= 1ull << e;
                else if (!(xt < thr)) bv |= 1ull << e;
            }
            if (bv) atomicOr(&vis[row / 9][row % 9], bv << (4 * ch));
            if (bn) atomicOr(&nanb[row / 9][row % 9], bn << (4 * ch));
        }
    }
    __syncthreads();
    if (t < 64) {                                                // one thread per cell row: 32 cells bit-parallel
        const int ly = t & 7, lz = t >> 3;
        const unsigned long long V = vis[lz][ly] | vis[lz][ly + 1] | vis[lz + 1][ly] | vis[lz + 1][ly + 1];
        const unsigned long long N = nanb[lz][ly] | nanb[lz][ly + 1] | nanb[lz + 1][ly] | nanb[lz + 1][ly + 1];
        unsigned occ = (unsigned)(V | (V >> 1)) & ~(unsigned)(N | (N >> 1));      // any corner visible, no corner NaN
        const int n_in = nx + PAD_X - x0;                         // cells x0 + lx < nx + PAD_X exist
        if (n_in < 32) occ &= n_in > 0 ? ((1u << n_in) - 1u) : 0u;
        if (y0 + ly >= ny + PAD_Y || z0 + lz >= nz + PAD_Z) occ = 0u;
        rowbits[lz][ly] = occ;
    }
    __syncthreads();
    if (t < 32) {                                                // one thread per 64-bit word of 4x4x4 cells
        const int wx = t & 7, wyy = (t >> 3) & 1, wzz = t >> 4;
        unsigned long long w = 0ull;
#pragma unroll
        for (int lz4 = 0; lz4 < 4; ++lz4)
#pragma unroll
            for (int ly4 = 0; ly4 < 4; ++ly4) {
                const unsigned long long nib = (rowbits[wzz * 4 + lz4][wyy * 4 + ly4] >> (4 * wx)) & 15u;
                w |= nib << ((lz4 * 4 + ly4) * 4);
            }
        const int bx = blockIdx.x * 8 + wx, by = blockIdx.y * 2 + wyy, bz = blockIdx.z * 2 + wzz;
        const bool in = bx < NBX && by < NBY && bz * 4 < nz + PAD_Z;
        if (in) mask[((size_t)bz * NBY + by) * NBX + bx] = w;
        unsigned long long cnt = in ? (unsigned long long)__popcll(w) : 0ull;
        for (int sft = 16; sft > 0; sft >>= 1) cnt += __shfl_xor_sync(0xffffffffu, cnt, sft);
        if (t == 0 && cnt) atomicAdd(n_occupied, cnt);
    }
}

// MIP skipping: an upper bound of every sample value inside a block of 4x4x4 cells (5x5x5 voxels: the cells' far corners
// included), NaN ignored; same block grid as the occupancy mask.  One thread per block; once per volume, at the first MIP
// frame.  The bound is the block's largest voxel plus a margin for the rounding of the fp32 blend: a lerp
// fmaf(w, x - y, y) can pass max(x, y) by the rounding of the difference (<= 2^-24 of the block's value range; at w = 1
// exactly, which voxel-centred samples of axis-aligned views hit, it returns y + rnd(x - y), not x) and by half an ulp of
// the result; three nested lerps.  With max + 2^-21 (max - min) + 2^-21 |max| as the stored value a skipped block
// provably holds no sample above the running maximum, so frames are bit-identical with skipping on and off.
__global__ void __launch_bounds__(256)
build_blockmax_kernel(const float* __restrict__ vol, unsigned ty_stride, unsigned slab_stride, int x_last, int y_last,
                      int z_last, float* __restrict__ bmax, int NBX, int NBY, int NBZ) {
    const int bx = blockIdx.x * 64 + (threadIdx.x & 63), by = blockIdx.y * 4 + (threadIdx.x >> 6), bz = blockIdx.z;
    if (bx >= NBX || by >= NBY || bz >= NBZ) return;
    float m = -INFINITY, lo = INFINITY;
    for (int dz = 0; dz < 5; ++dz)
        for (int dy = 0; dy < 5; ++dy) {
            const int y = min(by * 4 + dy, y_last), z = min(bz * 4 + dz, z_last);
#pragma unroll
            for (int dx = 0; dx < 5; ++dx) {
                const float v = __ldg(vol + tiled_index(min(bx * 4 + dx, x_last), y, z, ty_stride, slab_stride));
                m = fmaxf(m, v);
                lo = fminf(lo, v);
            }
        }
    if (lo <= m)          // false only when every voxel of the block is NaN (m stays -inf: nothing to find there)
        m = __fadd_ru(m, __fadd_ru(__fmul_ru(m - lo, 4.76837158203125e-7f), __fmul_ru(fabsf(m), 4.76837158203125e-7f)));
    bmax[((size_t)bz * NBY + by) * NBX + bx] = m;
}

// bits [lo, hi) of a 64-bit set kept as two words, 0 <= lo, hi <= 64
__device__ __forceinline__ void range_bits(int lo, int hi, unsigned& b_lo, unsigned& b_hi) {
    const unsigned long long m_hi = hi >= 64 ? ~0ull : ((1ull << hi) - 1ull);
    const unsigned long long m_lo = lo >= 64 ? ~0ull : ((1ull << lo) - 1ull);
    const unsigned long long m = hi > lo ? (m_hi & ~m_lo) : 0ull;
    b_lo = (unsigned)m; b_hi = (unsigned)(m >> 32);
}

// S2 channel mask: samples jl in [0, je) of the segment starting at lattice index i_seg that are owned
// (O9's rule, double precision, the oracle's expressions) by the slab [za, zb] of some run of enabled channels.
// Only runs that can reach the segment's z-range cost the two divisions.
__device__ __forceinline__ void channel_bits(const FrameParams& P, const double o[3], const double d[3], double t_near,
                                             long long i_seg, int je, unsigned& b_lo, unsigned& b_hi) {
    b_lo = b_hi = 0u;
    const double z_a = o[2] + (t_near + ((double)i_seg + 0.5) * P.step) * d[2];
    const double z_b = o[2] + (t_near + ((double)(i_seg + je - 1) + 0.5) * P.step) * d[2];
    const double z_min = fmin(z_a, z_b) - 1.0, z_max = fmax(z_a, z_b) + 1.0;
    for (int r = 0; r < P.n_runs; ++r) {
        const double za = (double)P.run_z[2 * r], zb = (double)P.run_z[2 * r + 1];
        if (zb < z_min || za > z_max) continue;
        int lo = 0, hi = je;
        if (d[2] == 0.0) {
            if (!(za <= o[2] && o[2] < zb)) continue;                       // O3's rule for a ray parallel to the planes
        } else {
            const double t0 = (za - o[2]) / d[2], t1 = (zb - o[2]) / d[2];
            const double ta = t0 < t1 ? t0 : t1, tb = t0 < t1 ? t1 : t0;
            const long long ia = lattice_index(ta, t_near, P.step) - i_seg, ib = lattice_index(tb, t_near, P.step) - i_seg;
            lo = (int)(ia < 0 ? 0 : (ia > je ? je : ia));
            hi = (int)(ib < 0 ? 0 : (ib > je ? je : ib));
        }
        unsigned m_lo, m_hi;
        range_bits(lo, hi, m_lo, m_hi);
        b_lo |= m_lo; b_hi |= m_hi;
    }
}

// ------------------------------------------------------------------------------------------------
// a1 + a3 + a4/a5  the caster.  grid.x = sum over bricks of the CTA_W x CTA_H pixel tiles (16x8) of their
// rendering rectangles; block = 128 threads = 4 warps, each an 8x4-pixel patch.
// SKIP = 1 consults the occupancy mask (EA only); CHAN = 1 applies the channel mask (S2).  INSTR = 1 is the measuring build (samples, sector bitmaps),
// never the product path; it walks the same cells and takes the same skip and termination decisions.
// counters (INSTR): [0] lattice samples visited (the oracle's count), [1] samples evaluated (not skipped).
// ------------------------------------------------------------------------------------------------
template <int MODE, int INSTR, int SKIP, int CHAN>
__global__ void __launch_bounds__(CTA_THREADS, VR_CAST_MINBLOCKS)
cast_kernel(const __grid_constant__ FrameParams P, const BrickRec* __restrict__ bricks, int n_bricks,
            const float* __restrict__ vol, const float4* __restrict__ tf_global, const unsigned long long* __restrict__ mask,
            float* __restrict__ img, unsigned long long* __restrict__ counters, unsigned* __restrict__ bitmap,
            unsigned* __restrict__ mask_bitmap) {
    __shared__ __align__(16) float4 tf[MODE == MODE_EA ? 256 : 1];   // 4 KB: keeps the L1 share of the SM large
    __shared__ int s_brick;
    if (MODE == MODE_EA) {
        for (int i = threadIdx.x; i < 256; i += CTA_THREADS) tf[i] = tf_global[i];
    }
    if (threadIdx.x == 0) {               // which brick owns this CTA: last brick with tile0 <= blockIdx.x
        int lo = 0, hi = n_bricks - 1;
        while (lo < hi) {
            const int mid = (lo + hi + 1) >> 1;
            if (bricks[mid].tile0 <= (int)blockIdx.x) lo = mid; else hi = mid - 1;
        }
        s_brick = lo;
    }
    __syncthreads();
    const BrickRec* __restrict__ br = bricks + s_brick;
    const int tloc = (int)blockIdx.x - br->tile0;
    const int tiles_x = br->tiles_x;
    const int tyi = tloc / tiles_x, txi = tloc - tyi * tiles_x;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    constexpr int WW = VR_WARP_W, WH = 32 / VR_WARP_W, WPR = CTA_W / WW;   // warp patch WW x WH pixels, WPR patches per row
    const int lx = txi * CTA_W + (warp % WPR) * WW + (lane % WW);
    const int ly = tyi * CTA_H + (warp / WPR) * WH + (lane / WW);
    if (lx >= br->rw || ly >= br->rh) return;
    const int px = br->rx0 + lx, py = br->ry0 + ly;

    // ---- per-ray set-up, double precision (O2-O4, O9) ----
    double o[3], d[3];
    make_ray(P, px, py, o, d);
    long long i_lo = 0;
    double t_near = 0.0;
    const int n = owned_samples(P, br, o, d, t_near, i_lo);

    const size_t pix = (size_t)br->img_base + (size_t)(py - br->oy) * br->img_stride + (size_t)(px - br->ox);
    if (n == 0) {
        if (MODE == MODE_EA) reinterpret_cast<float4*>(img)[pix] = make_float4(0.f, 0.f, 0.f, 0.f);
        else img[pix] = -INFINITY;
        return;
    }
    // The march: segments of P.seg_len (<= 64) samples, each anchored in double (sampler.cuh); inside a segment
    // u_rel(j') = rel + j' h in fp32.  With empty-space skipping a segment is walked twice: an occupancy pass
    // that only locates each sample's cell and collects one bit per sample from the mask, then the sampling pass
    // over the set bits — lanes of a warp then work on different samples of the SAME segment, which compacts the
    // occupied samples of 32 rays into full warp instructions without letting the rays drift apart.
    const float h[3] = {(float)(P.step * d[0]), (float)(P.step * d[1]), (float)(P.step * d[2])};
    const unsigned nbx = (unsigned)P.nbx, nbxy = (unsigned)P.nbx * (unsigned)P.nby;

    float Cr = 0.f, Cg = 0.f, Cb = 0.f, A = 0.f, M = -INFINITY;
    MaskCursor mc;
    mc.lo = mc.hi = 0u; mc.tag = 0xffffffffu;
    if (INSTR) {
        unsigned long long visited = 0, evaluated = 0;
        bool done = false;
        for (int js = 0; js < n && !done; js += P.seg_len) {
            Anchor An;
            set_anchor(o, d, t_near, P.step, i_lo + js, h, P.seg_span, An);
            const int je = min(n - js, P.seg_len);
            unsigned en_lo = 0xffffffffu, en_hi = 0xffffffffu;
            if (CHAN) channel_bits(P, o, d, t_near, i_lo + js, je, en_lo, en_hi);
            const float M_seg = M;                 // MIP skipping decides per segment, with the maximum reached before it
            for (int jl = 0; jl < je; ++jl) {
                if (CHAN && !(((jl < 32 ? en_lo : en_hi) >> (jl & 31)) & 1u)) continue;   // S2: channel disabled
                Cell c;
                locate(An, jl, h, c);
                ++visited;
                if (SKIP) {
                    const unsigned tag = (c.iz >> 2) * nbxy + (c.iy >> 2) * nbx + (c.ix >> 2);
                    if (mask_bitmap) {             // 32-byte sectors: 4 mask words (EA) or 8 block maxima (MIP)
                        const unsigned sct = MODE == MODE_EA ? tag >> 2 : tag >> 3, bit = 1u << (sct & 31);
                        if (!(*(volatile unsigned*)(mask_bitmap + (sct >> 5)) & bit)) atomicOr(mask_bitmap + (sct >> 5), bit);
                    }
                    if (MODE == MODE_EA) {
                        if (!cell_occupied(mask, nbx, nbxy, c.ix, c.iy, c.iz, mc)) continue;
                    } else {
                        if (!(__ldg(reinterpret_cast<const float*>(mask) + tag) > M_seg)) continue;   // cannot raise the maximum
                    }
                }
                Footprint F;
                fetch_marked(vol, P, c, F, bitmap);
                const float v = trilerp(F, c);
                ++evaluated;
                if (MODE == MODE_EA) {
                    classify_blend(tf, P, v, Cr, Cg, Cb, A);
                    if (P.ert_on && A >= P.ert) { done = true; break; }
                } else {
                    M = fmaxf(M, v);
                }
            }
        }
        if (counters) { atomicAdd(counters, visited); atomicAdd(counters + 1, evaluated); }
    } else {
        // Row-cached sampler (sampler.cuh); the blend of the previous evaluated sample is issued after the loads
        // of the current one so that classification and blending overlap the load latency.
        RowCache K;
        cache_init(K);
        const unsigned long long vol_base = reinterpret_cast<unsigned long long>(vol);
        const unsigned slab_bytes = P.slab_stride * 4u;
        float vprev = 0.f;
        bool have = false, done = false;
        for (int js = 0; js < n && !done; js += P.seg_len) {
            // In the two-pass variants the ray is re-derived from the pixel here (same expressions, same doubles)
            // rather than kept: twelve live double registers across both passes spilled to local memory (measured:
            // -2.5 % with skipping; the plain loop is 1.5 % faster keeping them).
            double o2[3], d2[3];
            const double *os = o, *ds = d;
            if (SKIP || CHAN) { make_ray(P, px, py, o2, d2); os = o2; ds = d2; }
            Anchor An;
            set_anchor(os, ds, t_near, P.step, i_lo + js, h, P.seg_span, An);
            const int je = min(n - js, P.seg_len);
            if (SKIP || CHAN) {
                unsigned todo_lo, todo_hi;                     // bit jl: sample jl of this segment is to be evaluated
                range_bits(0, je, todo_lo, todo_hi);
                if (CHAN) {                                    // S2: channels the user disabled
                    unsigned en_lo, en_hi;
                    channel_bits(P, os, ds, t_near, i_lo + js, je, en_lo, en_hi);
                    todo_lo &= en_lo; todo_hi &= en_hi;
                }
                if (SKIP && MODE == MODE_MIP) {
                    // MIP: a sample cannot raise the running maximum M when the largest voxel of its 4x4x4-cell block
                    // (5x5x5 voxels, build_blockmax_kernel) is not above M (the stored bound covers the rounding of the blend).
                    // Decided per segment with the M reached before it (M only grows, so the test stays valid).
                    if (have) { M = fmaxf(M, vprev); have = false; }
                    const float* __restrict__ bmax = reinterpret_cast<const float*>(mask);
                    unsigned occ_lo = 0u, occ_hi = 0u;
                    constexpr int G = 8;
                    for (int jb = 0; jb < je; jb += G) {
                        float bm[G];
#pragma unroll
                        for (int k = 0; k < G; ++k) {
                            unsigned ix, iy, iz;
                            locate_cell(An, min(jb + k, je - 1), h, ix, iy, iz);
                            bm[k] = __ldg(bmax + ((iz >> 2) * nbxy + (iy >> 2) * nbx + (ix >> 2)));
                        }
                        unsigned nib = 0u;
#pragma unroll
                        for (int k = 0; k < G; ++k) nib |= (bm[k] > M ? 1u : 0u) << k;
                        if (jb < 32) occ_lo |= nib << jb; else occ_hi |= nib << (jb - 32);
                    }
                    todo_lo &= occ_lo; todo_hi &= occ_hi;
                }
                if (SKIP && MODE == MODE_EA) {                 // NEXT-2: cells that cannot contribute
                    unsigned occ_lo = 0u, occ_hi = 0u;
                    // VR_OCC_GROUP samples at a time: tags, then the (rare) word loads back to back into registers of
                    // their own, then the bit tests — the loads of a group are in flight together instead of one L2/HBM
                    // latency per new block.  Samples at or beyond je are located as copies of sample je - 1 and
                    // dropped by the AND with todo below.
                    constexpr int G = VR_OCC_GROUP;
                    for (int jb = 0; jb < je; jb += G) {
                        unsigned tg[G], bp[G];
#pragma unroll
                        for (int k = 0; k < G; ++k) {
                            unsigned ix, iy, iz;
                            locate_cell(An, min(jb + k, je - 1), h, ix, iy, iz);
                            tg[k] = (iz >> 2) * nbxy + (iy >> 2) * nbx + (ix >> 2);
                            bp[k] = ((iz & 3u) << 4) | ((iy & 3u) << 2) | (ix & 3u);
                        }
                        uint2 w[G];
#pragma unroll
                        for (int k = 0; k < G; ++k) {
                            const unsigned prev = k ? tg[k - 1] : mc.tag;
                            w[k] = make_uint2(0u, 0u);
                            if (tg[k] != prev) w[k] = __ldg(reinterpret_cast<const uint2*>(mask + tg[k]));
                        }
                        uint2 cur = make_uint2(mc.lo, mc.hi);
                        unsigned nib = 0u;
#pragma unroll
                        for (int k = 0; k < G; ++k) {
                            const unsigned prev = k ? tg[k - 1] : mc.tag;
                            if (tg[k] != prev) cur = w[k];
                            const unsigned half = (bp[k] & 32u) ? cur.y : cur.x;
                            nib |= ((half >> (bp[k] & 31u)) & 1u) << k;
                        }
                        mc.lo = cur.x; mc.hi = cur.y; mc.tag = tg[G - 1];
                        if (jb < 32) occ_lo |= nib << jb; else occ_hi |= nib << (jb - 32);
                    }
                    todo_lo &= occ_lo; todo_hi &= occ_hi;
                }
                cache_init(K);      // the row cache does not survive a segment: its 25 registers are then dead during the
                                    // occupancy pass, which lets ptxas keep a group's mask loads in flight (measured
                                    // -3.6 % on config 3, -6 % on config 2; profiles/r02_experiments.md)
                while (todo_lo | todo_hi) {
                    int jl;
                    if (todo_lo) { jl = __ffs((int)todo_lo) - 1; todo_lo &= todo_lo - 1u; }
                    else { jl = 31 + __ffs((int)todo_hi); todo_hi &= todo_hi - 1u; }
                    Cell c;
                    locate(An, jl, h, c);
                    const float v = sample_cached(vol_base, P.ty_stride, slab_bytes, c, K);
                    if (have) {
                        if (MODE == MODE_EA) {
                            classify_blend(tf, P, vprev, Cr, Cg, Cb, A);
                            if (P.ert_on && A >= P.ert) { done = true; break; }
                        } else {
                            M = fmaxf(M, vprev);
                        }
                    }
                    vprev = v; have = true;
                }
            } else {
                for (int jl = 0; jl < je; ++jl) {
                    Cell c;
                    locate(An, jl, h, c);
                    const float v = sample_cached(vol_base, P.ty_stride, slab_bytes, c, K);
                    if (have) {
                        if (MODE == MODE_EA) {
                            classify_blend(tf, P, vprev, Cr, Cg, Cb, A);
                            if (P.ert_on && A >= P.ert) { done = true; break; }
                        } else {
                            M = fmaxf(M, vprev);
                        }
                    }
                    vprev = v; have = true;
                }
            }
        }
        if (have && !done) {
            if (MODE == MODE_EA) classify_blend(tf, P, vprev, Cr, Cg, Cb, A);
            else M = fmaxf(M, vprev);
        }
    }
    if (MODE == MODE_EA) reinterpret_cast<float4*>(img)[pix] = make_float4(Cr, Cg, Cb, A);
    else img[pix] = M;
}

// number of set bits of the sector bitmap (measuring build only): out[0] = distinct 32-byte sectors, out[1] = distinct
// 64-byte units (sector pairs s, s^1) and out[2] = distinct 128-byte lines (sector quads) holding a touched sector —
// what a memory system that fetches 64 or 128 bytes per miss would have to move for the same samples.
__global__ void popcount_kernel(const unsigned* __restrict__ bitmap, size_t n_words, unsigned long long* out) {
    unsigned long long c32 = 0, c64 = 0, c128 = 0;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_words; i += (size_t)gridDim.x * blockDim.x) {
        const unsigned w = bitmap[i];
        const unsigned p = (w | (w >> 1)) & 0x55555555u;          // bit 2k: pair k touched
        const unsigned q = (p | (p >> 2)) & 0x11111111u;          // bit 4k: quad k touched
        c32 += __popc(w); c64 += __popc(p); c128 += __popc(q);
    }
    for (int s = 16; s > 0; s >>= 1) {
        c32 += __shfl_xor_sync(0xffffffffu, c32, s);
        c64 += __shfl_xor_sync(0xffffffffu, c64, s);
        c128 += __shfl_xor_sync(0xffffffffu, c128, s);
    }
    if ((threadIdx.x & 31) == 0 && c32) { atomicAdd(out, c32); atomicAdd(out + 1, c64); atomicAdd(out + 2, c128); }
}

// ------------------------------------------------------------------------------------------------
// a7  sort-last composite.  One thread per pixel walks the bricks front to back
// (order[] from the host, A11) and applies "over" (EA) or max (MIP, then the O8 colour lookup in the
// uncorrected table).  A brick is skipped by the whole warp when none of its 32 pixels lies inside
// the brick's rendering rectangle (warp vote), so the cost per pixel is the depth complexity, not B.
// ------------------------------------------------------------------------------------------------
template <int MODE>
__global__ void __launch_bounds__(256)
composite_kernel(const BrickRec* __restrict__ bricks, const int* __restrict__ order, int n_bricks,
                 const float* __restrict__ img, int W, int H, const float4* __restrict__ tf_raw, float vmin,
                 float inv_range, float* __restrict__ out_rgba, float* __restrict__ out_scalar) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int px = blockIdx.x * 16 + (warp & 1) * 8 + (lane & 7);
    const int py = blockIdx.y * 16 + (warp >> 1) * 4 + (lane >> 3);
    const bool live = px < W && py < H;
    float Cr = 0.f, Cg = 0.f, Cb = 0.f, Tr = 1.f, M = -INFINITY;
    for (int k = 0; k < n_bricks; ++k) {
        const BrickRec* __restrict__ br = bricks + order[k];
        const bool in = live && px >= br->rx0 && px < br->rx0 + br->rw && py >= br->ry0 && py < br->ry0 + br->rh;
        if (!__any_sync(0xffffffffu, in)) continue;
        if (in) {
            const size_t pix = (size_t)br->img_base + (size_t)(py - br->oy) * br->img_stride + (size_t)(px - br->ox);
            if (MODE == MODE_EA) {
                const float4 v = __ldcs(reinterpret_cast<const float4*>(img) + pix);
                Cr = fmaf(Tr, v.x, Cr); Cg = fmaf(Tr, v.y, Cg); Cb = fmaf(Tr, v.z, Cb);
                Tr *= (1.0f - v.w);
            } else {
                M = fmaxf(M, __ldcs(img + pix));
            }
        }
    }
    if (!live) return;
    const size_t o = (size_t)py * W + px;
    if (MODE == MODE_EA) {
        reinterpret_cast<float4*>(out_rgba)[o] = make_float4(Cr, Cg, Cb, 1.0f - Tr);
    } else {
        if (out_scalar) out_scalar[o] = M;
        float4 e = make_float4(0.f, 0.f, 0.f, 0.f);
        if (M != -INFINITY) {       // O8: colour of the maximum, uncorrected table, un-premultiplied
            const float x = __saturatef((M - vmin) * inv_range) * 255.0f;
            const int m = min((int)x, 254);
            const float w = x - (float)m;
            const float4 t0 = tf_raw[m], t1 = tf_raw[m + 1];
            e = make_float4(fmaf(w, t1.x - t0.x, t0.x), fmaf(w, t1.y - t0.y, t0.y), fmaf(w, t1.z - t0.z, t0.z),
                            fmaf(w, t1.w - t0.w, t0.w));
        }
        reinterpret_cast<float4*>(out_rgba)[o] = e;
    }
}

}  // namespace vr
