// vr_api.cu — the C ABI of include/vr.h (and the measurement aids of include/vr_measure.h): argument checks, per-frame planning on the host (plan.h)
// and kernel launches (kernels.cuh).  Every step of the path runs in the kernels; this file only
// validates, plans and enqueues.  There is no CPU fallback.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "../../include/vr.h"
#include "../../include/vr_measure.h"
#include "kernels.cuh"
#include "slab.cuh"
#include "plan.h"

// Tuning constants of measurement builds (VR_DEFINES="-DVR_SEG_MAX=32" python -m paper_1008_0135_b200.build, which
// writes a library file of its own; profiles/r02_experiments.md, r02_slab.md).  Product values:
#ifndef VR_SEG_MAX
#define VR_SEG_MAX 64        // samples per double-precision anchor, 1..64
#endif
#ifndef VR_SLAB_LOGD
#define VR_SLAB_LOGD (-1)    // slab thickness chosen per frame
#endif
static_assert(VR_SEG_MAX >= 1 && VR_SEG_MAX <= 64 && VR_SLAB_LOGD >= -1 && VR_SLAB_LOGD <= 3, "tuning constants out of range");

namespace {

thread_local std::string g_err;

vr_status fail(vr_status s, const std::string& msg) {
    g_err = msg;
    return s;
}
vr_status cuda_fail(cudaError_t e, const char* what) {
    vr_status s = (e == cudaErrorMemoryAllocation) ? VR_ERR_OOM : VR_ERR_CUDA;
    return fail(s, std::string(what) + ": " + cudaGetErrorString(e));
}
#define VR_CUDA(call, what)                                   \
    do {                                                      \
        cudaError_t e_ = (call);                              \
        if (e_ != cudaSuccess) return cuda_fail(e_, what);    \
    } while (0)

}  // namespace

struct vr_volume {
    int dims[3] = {0, 0, 0};
    int TX = 0, TY = 0, TZ = 0;
    size_t tiled_elems = 0;
    float* d_tiled = nullptr;
    cudaStream_t stream = nullptr;
    float relayout_ms = 0.f;
    unsigned* d_range = nullptr;      // RANGE_SLOTS x (min key, max key), written by the re-layout pass
    float data_min = 0.f, data_max = 0.f;
    bool has_range = false;

    bool has_tf = false;
    float tf_host[1024];
    float vmin = 0.f, vmax = 1.f;
    double tf_step = -1.0;            // step the device EA table is currently corrected for
    float4* d_tf_ea = nullptr;        // 256 float4: the table corrected for the current step (O6)
    float4* d_tf_raw = nullptr;       // 256 float4: table as given (MIP colour, O8)

    int bricks[3] = {1, 1, 1};
    int sub_lo[3] = {0, 0, 0}, sub_hi[3] = {0, 0, 0};   // sub-cube (S1); set to the whole cube at create
    vr::BrickRec* d_bricks = nullptr; // VR_MAX_BRICKS records
    int* d_order = nullptr;

    float* d_pool = nullptr;          // rect-cropped brick images of vr_render
    size_t pool_floats = 0;
    float* d_frame[2] = {nullptr, nullptr};   // internal frames of vr_render_to_host(_async), used alternately
    size_t frame_floats = 0;
    cudaStream_t copy_stream = nullptr;        // device->host copies of finished frames
    cudaEvent_t frame_done[2] = {nullptr, nullptr}, copy_done[2] = {nullptr, nullptr};
    unsigned frame_idx = 0;

    // NEXT-2 empty-space skipping: occupancy mask (one bit per voxel cell), built for the current table on demand
    int n_runs = 0;                   // S2 channel mask as runs of enabled channels; 0 = every channel enabled
    int run_z[2 * vr::MAX_RUNS] = {0};
    int seg_max = VR_SEG_MAX;         // samples (and voxels of path) per anchored segment
    bool debug = false;               // env VR_DEBUG=1 at vr_create_volume: wait for and check every kernel of a frame
    bool skip_enabled = true;
    unsigned long long* d_mask = nullptr;
    float* d_blockmax = nullptr;      // MIP skipping: largest voxel per block of 4x4x4 cells (same grid as the mask words)
    float blockmax_build_ms = 0.f;
    unsigned long long* d_mask_count = nullptr;
    int NBX = 0, NBY = 0, NBZ = 0;
    size_t mask_words = 0;
    bool mask_valid = false;
    float mask_key[3] = {0.f, 0.f, 0.f};   // vmin, inv_range, x_zero_below the mask was built for
    float mask_build_ms = 0.f;
    long long mask_occupied = 0;
    // slab-staged caster (slab.cuh): linear padded copy, made on first use
    int slab_mode = 1;                // 0 off, 1 auto (dense orthographic frames), 2 whenever the window fits
    int slab_logd = VR_SLAB_LOGD;     // >= 0 forces the slab thickness 2^k cell layers (tuning builds), -1 = heuristic
    float* d_linear = nullptr;        // x fastest: views whose dominant axis is y or z
    float* d_linear_t = nullptr;      // z fastest: views whose dominant axis is x
    bool linear_failed = false;       // allocation failed once: stay on the row-cache caster
    float linearize_ms = 0.f, transpose_ms = 0.f;
    int last_slab[6] = {0, 0, 0, 0, 0, 0};   // last frame: used, dominant axis, D, window x, y, z
    cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};   // cast begin/end, composite begin/end
    bool timed_cast = false, timed_comp = false;
};

namespace {

// element strides between tiles adjacent in y / z
unsigned ty_stride_of(const vr_volume* v);
unsigned slab_stride_of(const vr_volume* v);

struct Frame {                         // everything one frame needs, built on the host
    vr::FrameParams P;
    std::vector<vr::BrickRec> recs;
    std::vector<int> order;
    int total_tiles = 0;
    size_t pool_pixels = 0;
};

unsigned ty_stride_of(const vr_volume* v) { return (unsigned)v->TX * vr::TILE_ELEMS; }
unsigned slab_stride_of(const vr_volume* v) { return (unsigned)v->TX * (unsigned)v->TY * vr::TILE_ELEMS; }

vr_status check_render_args(const vr_volume* vol, const vr_camera* cam, int W, int H, float step, int mode) {
    if (!vol) return fail(VR_ERR_INVALID_ARG, "volume is NULL");
    if (!cam) return fail(VR_ERR_INVALID_ARG, "camera is NULL");
    if (W <= 0 || H <= 0 || W > 32768 || H > 32768) return fail(VR_ERR_INVALID_ARG, "W and H must be in [1,32768]");
    if (!(step > 0.0f) || !std::isfinite(step)) return fail(VR_ERR_INVALID_ARG, "step_voxels must be positive and finite");
    if (mode != VR_MODE_EA && mode != VR_MODE_MIP) return fail(VR_ERR_INVALID_ARG, "unknown mode");
    if (const char* why = vr::check_camera(*cam)) return fail(VR_ERR_INVALID_ARG, why);
    const double diag = std::sqrt((double)vol->dims[0] * vol->dims[0] + (double)vol->dims[1] * vol->dims[1] +
                                  (double)vol->dims[2] * vol->dims[2]);
    if (diag / (double)step > 8.0e6) return fail(VR_ERR_INVALID_ARG, "step_voxels too small for this volume (> 8e6 samples per ray)");
    if (!vol->has_tf) return fail(VR_ERR_STATE, "no transfer function set (vr_set_transfer_function)");
    return VR_OK;
}

// VR_DEBUG=1: wait for the kernel just launched and report its failure at the call that caused it (otherwise an
// asynchronous fault surfaces at some later call).  Off by default: the frame path never synchronises.
vr_status debug_sync(const vr_volume* vol, const char* what) {
    if (!vol->debug) return VR_OK;
    VR_CUDA(cudaStreamSynchronize(vol->stream), what);
    return VR_OK;
}

// x_zero_below of the current table: (index of the first entry with alpha > 0) - 1
float table_zero_below(const vr_volume* vol) {
    int j0 = 0;
    while (j0 < 256 && !(vol->tf_host[4 * j0 + 3] > 0.0f)) ++j0;
    return (float)(j0 - 1);
}

// Empty-space skipping applies to emission-absorption frames whose table starts with at least two transparent
// entries (otherwise no cell can be proven empty and the mask would be all ones).
bool skip_applies(const vr_volume* vol, int mode) {
    if (mode == VR_MODE_MIP) return vol->skip_enabled;        // MIP: blocks whose largest voxel cannot raise the maximum
    return vol->skip_enabled && mode == VR_MODE_EA && table_zero_below(vol) - vr::MASK_MARGIN > 0.0f;
}

// cropped = true: brick images are rect-sized and packed (vr_render); false: full W x H frames.
vr_status build_frame(const vr_volume* vol, const vr_camera* cam, int W, int H, float step, float ert, bool cropped,
                      bool direct, Frame& f) {
    const vr::Basis bs = vr::make_basis(*cam);
    vr::FrameParams& P = f.P;
    for (int c = 0; c < 3; ++c) {
        P.eye[c] = bs.eye[c]; P.right[c] = bs.right[c]; P.up[c] = bs.up[c]; P.fwd[c] = bs.fwd[c];
    }
    P.h = (double)cam->ortho_half_h;
    P.asp = (double)W / (double)H;
    P.tanhalf = cam->projection == VR_PROJ_PERSP ? vr::tan_half_fov(*cam) : 0.0;
    P.step = (double)step;
    P.proj = cam->projection; P.W = W; P.H = H;
    P.nx = vol->dims[0]; P.ny = vol->dims[1]; P.nz = vol->dims[2];
    P.ty_stride = ty_stride_of(vol);
    P.slab_stride = slab_stride_of(vol);
    P.vmin = vol->vmin;
    P.inv_range = 1.0f / (vol->vmax - vol->vmin);
    P.ert_on = (ert > 0.0f && ert < 1.0f) ? 1 : 0;
    P.ert = ert;
    // segments of <= 64 voxels of path (sampler.cuh): fp32 positions stay within ~65 of their anchor
    P.seg_len = std::max(1, std::min(vol->seg_max, (int)((double)vol->seg_max / (double)step)));
    P.seg_span = (int)std::ceil((double)P.seg_len * (double)step) + 1;
    P.nbx = vol->NBX; P.nby = vol->NBY;
    P.n_runs = vol->n_runs;
    for (int k = 0; k < 2 * vr::MAX_RUNS; ++k) P.run_z[k] = vol->run_z[k];
    P.x_zero_below = table_zero_below(vol);   // the per-step opacity correction keeps zeros zero

    std::vector<vr::BrickPlan> plan;
    vr::plan_bricks(vol->dims, vol->bricks, *cam, W, H, plan, f.order, vol->sub_lo, vol->sub_hi);
    const int B = (int)plan.size();
    f.recs.assign(B, vr::BrickRec());
    long long tiles = 0;                  // 64-bit: 512 full-frame rectangles at 32768^2 overflow an int
    size_t pool = 0;
    // CTAs are laid out brick by brick, front to back
    for (int k = 0; k < B; ++k) {
        const int b = f.order[k];
        vr::BrickPlan bp = plan[b];
        if (direct) { bp.rx0 = 0; bp.ry0 = 0; bp.rw = W; bp.rh = H; }   // one brick writes the frame itself
        vr::BrickRec& r = f.recs[b];
        for (int a = 0; a < 3; ++a) { r.lo[a] = bp.lo[a]; r.hi[a] = bp.hi[a]; }
        r.rx0 = bp.rx0; r.ry0 = bp.ry0; r.rw = bp.rw; r.rh = bp.rh;
        r.tile0 = (int)std::min<long long>(tiles, 2147483647ll);
        r.tiles_x = (bp.rw + vr::CTA_W - 1) / vr::CTA_W;
        const int tiles_y = (bp.rh + vr::CTA_H - 1) / vr::CTA_H;
        tiles += (long long)r.tiles_x * tiles_y;
        if (cropped && !direct) {
            r.img_base = (long long)pool; r.img_stride = bp.rw; r.ox = bp.rx0; r.oy = bp.ry0;
            pool += (size_t)bp.rw * bp.rh;
        } else {
            r.img_base = direct ? 0 : (long long)b * W * H; r.img_stride = W; r.ox = 0; r.oy = 0;
        }
        r.pad = 0;
    }
    if (tiles > 2147483647ll)
        return fail(VR_ERR_INVALID_ARG, "image x bricks too large: more than 2^31-1 pixel tiles in one frame");
    if (pool > ((size_t)1 << 34))         // 16 Gi pixels of brick images = 256 GB of float4: cannot be meant
        return fail(VR_ERR_INVALID_ARG, "image x bricks too large: brick images would exceed 2^34 pixels");
    f.total_tiles = (int)tiles;
    f.pool_pixels = pool;
    return VR_OK;
}

// The cast kernel looks its brick up by tile0 with a binary search over records in FRONT-TO-BACK order;
// recs[] is indexed by brick id, so upload a copy sorted by order[] for the caster and keep ids for
// the compositor: simplest is to store records in order[] sequence and make order[] the identity.
vr_status upload_plan(vr_volume* vol, Frame& f) {
    const int B = (int)f.recs.size();
    std::vector<vr::BrickRec> sorted(B);
    std::vector<int> ident(B);
    for (int k = 0; k < B; ++k) { sorted[k] = f.recs[f.order[k]]; ident[k] = k; }
    VR_CUDA(cudaMemcpyAsync(vol->d_bricks, sorted.data(), sizeof(vr::BrickRec) * B, cudaMemcpyHostToDevice, vol->stream),
            "upload brick table");
    VR_CUDA(cudaMemcpyAsync(vol->d_order, ident.data(), sizeof(int) * B, cudaMemcpyHostToDevice, vol->stream),
            "upload brick order");
    return VR_OK;
}

// O6: per-entry opacity correction for this step, in double.
vr_status upload_tf_for_step(vr_volume* vol, double step) {
    if (vol->tf_step == step) return VR_OK;
    std::vector<float> t(256 * 4);
    for (int j = 0; j < 256; ++j) {
        for (int c = 0; c < 3; ++c) t[4 * j + c] = vol->tf_host[4 * j + c];
        const double a = (double)vol->tf_host[4 * j + 3];
        t[4 * j + 3] = (float)((step == 1.0) ? a : 1.0 - std::pow(1.0 - a, step));
    }
    VR_CUDA(cudaMemcpyAsync(vol->d_tf_ea, t.data(), sizeof(float) * 1024, cudaMemcpyHostToDevice, vol->stream),
            "upload transfer function");
    vol->tf_step = step;
    return VR_OK;
}

// Cells the occupancy mask holds a bit for (and build_mask_kernel counts over): the padded cells, n_a + PAD_a per axis.
double mask_cells(const vr_volume* vol) {
    return (double)(vol->dims[0] + vr::PAD_X) * (double)(vol->dims[1] + vr::PAD_Y) * (double)(vol->dims[2] + vr::PAD_Z);
}

// Build (or reuse) the occupancy mask for the current table.  One pass over the tiled cube.
vr_status ensure_mask(vr_volume* vol) {
    const float key[3] = {vol->vmin, 1.0f / (vol->vmax - vol->vmin), table_zero_below(vol)};
    if (vol->mask_valid && std::memcmp(key, vol->mask_key, sizeof(key)) == 0) return VR_OK;
    if (!vol->d_mask) {
        VR_CUDA(cudaMalloc(&vol->d_mask, vol->mask_words * sizeof(unsigned long long)), "allocate occupancy mask");
        VR_CUDA(cudaMalloc(&vol->d_mask_count, sizeof(unsigned long long)), "allocate occupancy counter");
    }
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    VR_CUDA(cudaEventCreate(&e0), "create event");
    cudaError_t e = cudaEventCreate(&e1);
    if (e == cudaSuccess) e = cudaMemsetAsync(vol->d_mask_count, 0, sizeof(unsigned long long), vol->stream);
    if (e == cudaSuccess) e = cudaEventRecord(e0, vol->stream);
    if (e == cudaSuccess) {
        dim3 grid((vol->dims[0] + vr::PAD_X + 31) / 32, (vol->dims[1] + vr::PAD_Y + 7) / 8, (vol->dims[2] + vr::PAD_Z + 7) / 8);
        vr::build_mask_kernel<<<grid, 256, 0, vol->stream>>>(
            vol->d_tiled, ty_stride_of(vol), slab_stride_of(vol),
            vol->dims[0], vol->dims[1], vol->dims[2], key[0], key[1], key[2], vol->d_mask, vol->NBX, vol->NBY,
            vol->d_mask_count);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaEventRecord(e1, vol->stream);
    unsigned long long cnt = 0;
    if (e == cudaSuccess) e = cudaMemcpyAsync(&cnt, vol->d_mask_count, sizeof(cnt), cudaMemcpyDeviceToHost, vol->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(vol->stream);
    if (e == cudaSuccess) e = cudaEventElapsedTime(&vol->mask_build_ms, e0, e1);
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    if (e != cudaSuccess) return cuda_fail(e, "build occupancy mask");
    vol->mask_occupied = (long long)cnt;
    std::memcpy(vol->mask_key, key, sizeof(key));
    vol->mask_valid = true;
    return VR_OK;
}

// MIP skipping: block maxima, once per volume (independent of the table).
vr_status ensure_blockmax(vr_volume* vol) {
    if (vol->d_blockmax) return VR_OK;
    VR_CUDA(cudaMalloc(&vol->d_blockmax, vol->mask_words * sizeof(float)), "allocate block maxima");
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    cudaError_t e = cudaEventCreate(&e0);
    if (e == cudaSuccess) e = cudaEventCreate(&e1);
    if (e == cudaSuccess) e = cudaEventRecord(e0, vol->stream);
    if (e == cudaSuccess) {
        dim3 grid((vol->NBX + 63) / 64, (vol->NBY + 3) / 4, vol->NBZ);
        vr::build_blockmax_kernel<<<grid, 256, 0, vol->stream>>>(vol->d_tiled, ty_stride_of(vol), slab_stride_of(vol),
                                                                 vol->TX * 8 - 1, vol->dims[1] + vr::PAD_Y, vol->dims[2] + vr::PAD_Z,
                                                                 vol->d_blockmax, vol->NBX, vol->NBY, vol->NBZ);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaEventRecord(e1, vol->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(vol->stream);
    if (e == cudaSuccess) e = cudaEventElapsedTime(&vol->blockmax_build_ms, e0, e1);
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    if (e != cudaSuccess) { cudaFree(vol->d_blockmax); vol->d_blockmax = nullptr; return cuda_fail(e, "build block maxima"); }
    return VR_OK;
}

// the per-table (EA) or per-volume (MIP) structure empty-space skipping consults
vr_status ensure_skip_structure(vr_volume* vol, int mode) {
    return mode == VR_MODE_MIP ? ensure_blockmax(vol) : ensure_mask(vol);
}

template <int INSTR>
vr_status launch_cast(vr_volume* vol, const Frame& f, int mode, float* d_img, unsigned long long* d_counter,
                      unsigned* d_bitmap, unsigned* d_mask_bitmap) {
    if (f.total_tiles == 0) return VR_OK;
    const int B = (int)f.recs.size();
    // callers run ensure_skip_structure first
    const bool skip = skip_applies(vol, mode) && (mode == VR_MODE_MIP ? vol->d_blockmax != nullptr : vol->mask_valid);
    const unsigned long long* d_skip = mode == VR_MODE_MIP ? reinterpret_cast<const unsigned long long*>(vol->d_blockmax) : vol->d_mask;
#define VR_LAUNCH(MODE_, SKIP_, CHAN_)                                                                       \
    vr::cast_kernel<MODE_, INSTR, SKIP_, CHAN_><<<f.total_tiles, vr::CTA_THREADS, 0, vol->stream>>>(         \
        f.P, vol->d_bricks, B, vol->d_tiled, vol->d_tf_ea, d_skip, d_img, d_counter, d_bitmap, d_mask_bitmap)
    const bool chan = f.P.n_runs > 0;
    if (mode == VR_MODE_EA) {
        if (skip) { if (chan) VR_LAUNCH(vr::MODE_EA, 1, 1); else VR_LAUNCH(vr::MODE_EA, 1, 0); }
        else { if (chan) VR_LAUNCH(vr::MODE_EA, 0, 1); else VR_LAUNCH(vr::MODE_EA, 0, 0); }
    } else {
        if (skip) { if (chan) VR_LAUNCH(vr::MODE_MIP, 1, 1); else VR_LAUNCH(vr::MODE_MIP, 1, 0); }
        else { if (chan) VR_LAUNCH(vr::MODE_MIP, 0, 1); else VR_LAUNCH(vr::MODE_MIP, 0, 0); }
    }
#undef VR_LAUNCH
    VR_CUDA(cudaGetLastError(), "cast kernel launch");
    return debug_sync(vol, "cast kernel (VR_DEBUG)");
}

// ---- slab-staged caster (slab.cuh): eligibility, window sizing, tensor maps, launch ----
struct SlabPlan {
    bool use = false;
    int dom = 2;
    vr::SlabParams S;
    size_t smem = 0;
    double bytes_per_sample = 0.0;
    vr::SlabMaps maps;
};

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn encode_tiled_fn() {
    static EncodeTiledFn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
    }
    return fn;
}

constexpr size_t SLAB_SMEM_EXTRA = 4096 + 16 + 160 + 64 + 16 + 128;   // table, barriers, corner rays, origins, misc, slack

// Largest extent (voxels, before margins) of a slab window on the two non-dominant axes over every CTA tile of the
// frame and every slab of its brick, for slabs of D cell layers.  false: some ray of the frame does not advance along
// the dominant axis in the direction of fwd, or is too oblique to it (perspective), or there are too many tiles to scan.
bool slab_extents(const Frame& f, const vr::SlabParams& S, int dom, int D, double ext[3]) {
    const vr::FrameParams& P = f.P;
    const int a1 = (dom + 1) % 3, a2 = (dom + 2) % 3;
    const double pad[3] = {(double)vr::PAD_X, (double)vr::PAD_Y, (double)vr::PAD_Z};
    const double sg = P.fwd[dom] >= 0.0 ? 1.0 : -1.0;
    ext[0] = ext[1] = ext[2] = 0.0;
    if (P.proj == VR_PROJ_PERSP && f.total_tiles > 400000) return false;
    for (const vr::BrickRec& r : f.recs) {
        if (r.rw <= 0 || r.rh <= 0) continue;
        const double cmin = (double)r.lo[dom] + pad[dom] - 1.0, cmax = (double)r.hi[dom] + pad[dom] + 1.0;
        const int tiles_x = (r.rw + vr::CTA_W - 1) / vr::CTA_W, tiles_y = (r.rh + vr::CTA_H - 1) / vr::CTA_H;
        const int nty = P.proj == VR_PROJ_PERSP ? tiles_y : 1, ntx = P.proj == VR_PROJ_PERSP ? tiles_x : 1;   // orthographic: every tile alike
        for (int ty = 0; ty < nty; ++ty)
            for (int tx = 0; tx < ntx; ++tx) {
                double q[4][3], m[4][2];
                for (int c = 0; c < 4; ++c) {
                    const double fx = (double)(r.rx0 + tx * vr::CTA_W + ((c & 1) ? vr::CTA_W - 1 : 0));
                    const double fy = (double)(r.ry0 + ty * vr::CTA_H + ((c & 2) ? vr::CTA_H - 1 : 0));
                    const double vd = S.v0[dom] + fx * S.dvx[dom] + fy * S.dvy[dom];
                    if (!(vd * sg > 1e-9)) return false;
                    q[c][0] = S.q0[a1] + fx * S.dqx[a1] + fy * S.dqy[a1];
                    q[c][1] = S.q0[a2] + fx * S.dqx[a2] + fy * S.dqy[a2];
                    q[c][2] = S.q0[dom] + fx * S.dqx[dom] + fy * S.dqy[dom];
                    m[c][0] = (S.v0[a1] + fx * S.dvx[a1] + fy * S.dvy[a1]) / vd;
                    m[c][1] = (S.v0[a2] + fx * S.dvx[a2] + fy * S.dvy[a2]) / vd;
                    if (std::fabs(m[c][0]) > 4.0 || std::fabs(m[c][1]) > 4.0) return false;
                }
                // the extent is convex in the slab position: its maximum over the brick is at the first or the last slab
                for (int end = 0; end < 2; ++end) {
                    const double c0 = end == 0 ? cmin - D + 1.0 : cmax - 1.0, c1 = c0 + D;    // slabs overhanging the brick's ends
                    for (int k = 0; k < 2; ++k) {
                        double lo = INFINITY, hi = -INFINITY;
                        for (int c = 0; c < 4; ++c) {
                            const double u0 = q[c][k] + (c0 - q[c][2]) * m[c][k], u1 = q[c][k] + (c1 - q[c][2]) * m[c][k];
                            lo = std::min(lo, std::min(u0, u1)); hi = std::max(hi, std::max(u0, u1));
                        }
                        const int a = k == 0 ? a1 : a2;
                        ext[a] = std::max(ext[a], hi - lo);
                    }
                }
            }
    }
    return true;
}

// Decide whether this frame can run on the slab-staged caster and size its windows.
void plan_slab(const vr_volume* vol, const Frame& f, double limit_bytes_per_sample, size_t max_smem, SlabPlan& sp) {
    const vr::FrameParams& P = f.P;
    sp.use = false;
    if (vol->slab_mode == 0 || P.n_runs > 0 || vol->linear_failed || f.total_tiles == 0) return;
    int dom = 0;
    for (int a = 1; a < 3; ++a) if (std::fabs(P.fwd[a]) > std::fabs(P.fwd[dom])) dom = a;
    const double pad[3] = {(double)vr::PAD_X, (double)vr::PAD_Y, (double)vr::PAD_Z};
    vr::SlabParams& S = sp.S;
    for (int a = 0; a < 3; ++a) {
        if (P.proj == VR_PROJ_ORTHO) {
            S.q0[a] = P.eye[a] + (1.0 / P.W - 1.0) * P.h * P.asp * P.right[a] + (1.0 / P.H - 1.0) * P.h * P.up[a] + pad[a] - 0.5;
            S.dqx[a] = 2.0 * P.h * P.asp * P.right[a] / P.W;
            S.dqy[a] = 2.0 * P.h * P.up[a] / P.H;
            S.v0[a] = P.fwd[a]; S.dvx[a] = 0.0; S.dvy[a] = 0.0;
        } else {
            S.q0[a] = P.eye[a] + pad[a] - 0.5; S.dqx[a] = 0.0; S.dqy[a] = 0.0;
            S.v0[a] = P.fwd[a] + (1.0 / P.W - 1.0) * P.tanhalf * P.asp * P.right[a] + (1.0 / P.H - 1.0) * P.tanhalf * P.up[a];
            S.dvx[a] = 2.0 * P.tanhalf * P.asp * P.right[a] / P.W;
            S.dvy[a] = 2.0 * P.tanhalf * P.up[a] / P.H;
        }
    }
    if (P.proj == VR_PROJ_PERSP && std::isfinite(limit_bytes_per_sample)) {
        // Quick reject before the scan over all tiles (a frame of the headline has ~10^4 of them): the tile at the image
        // centre, half way through the cube, in a slab one cell layer thick, already stages more bytes per sample than
        // the limit (d(V_a/V_dom)/dpx = (dvx_a V_dom - dvx_dom V_a) / V_dom^2).
        const double fx = 0.5 * P.W, fy = 0.5 * P.H;
        const double vd = S.v0[dom] + fx * S.dvx[dom] + fy * S.dvy[dom];
        const double dims[3] = {(double)P.nx, (double)P.ny, (double)P.nz};
        const double depth = std::fabs(0.5 * dims[dom] + pad[dom] - S.q0[dom]);
        double e[3] = {0.0, 0.0, 0.0};
        for (int a = 0; a < 3; ++a) {
            const double va = S.v0[a] + fx * S.dvx[a] + fy * S.dvy[a];
            e[a] = depth * (std::fabs(S.dvx[a] * vd - S.dvx[dom] * va) * (vr::CTA_W - 1) +
                            std::fabs(S.dvy[a] * vd - S.dvy[dom] * va) * (vr::CTA_H - 1)) / (vd * vd);
        }
        double wq[3];
        for (int a = 0; a < 3; ++a) wq[a] = e[a] + (a == (dom == 0 ? 2 : 0) ? 5.0 : 2.0);             // the margins of window_scan
        const double layer = wq[(dom + 1) % 3] * wq[(dom + 2) % 3] * 4.0;            // bytes per cell layer of the window
        const double layers = std::floor((double)max_smem / (2.0 * layer));          // what two buffers can hold
        if (layers < 2.0) return;
        const double Dq = layers >= 9.0 ? 8.0 : layers >= 5.0 ? 4.0 : layers >= 3.0 ? 2.0 : 1.0;
        const double low = layer * (Dq + 1.0) / Dq * std::fabs(P.fwd[dom]) * P.step / (double)vr::CTA_THREADS;
        if (low > limit_bytes_per_sample) return;
    }
    auto window_scan = [&](int logd, int w[3]) -> bool {
        const int D = 1 << logd;
        double ext[3];
        if (!slab_extents(f, S, dom, D, ext)) return false;
        for (int a = 0; a < 3; ++a) {
            w[a] = a == dom ? D + 1 : (int)std::ceil(ext[a] + 2.0 * vr::SLAB_FUZZ) + 2;   // the kernel's floor(hi + fuzz) + 2 - floor(lo - fuzz)
            if (a == (dom == 0 ? 2 : 0)) w[a] = (w[a] + 3 + 3) & ~3;   // the source's fastest axis: + 3, the copy starts at a multiple of 4 voxels
            if (w[a] > 256) return false;
        }
        return true;
    };
    bool have[4] = {false, false, false, false}, okw[4] = {false, false, false, false};
    int wc[4][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
    auto window = [&](int logd, int w[3]) -> bool {           // one scan per slab thickness
        if (!have[logd]) { have[logd] = true; okw[logd] = window_scan(logd, wc[logd]); }
        for (int a = 0; a < 3; ++a) w[a] = wc[logd][a];
        return okw[logd];
    };
    int best = -1, w[3] = {0, 0, 0};
    for (int pass = 0; pass < 2 && best < 0; ++pass) {
        const size_t budget = std::min(max_smem, pass == 0 ? (size_t)56 * 1024 : (size_t)113 * 1024);   // 4 or 2 CTAs per SM
        for (int logd = 3; logd >= 0; --logd) {
            if (vol->slab_logd >= 0 && logd != vol->slab_logd) continue;
            if (!window(logd, w)) continue;
            const long long fl = (long long)w[0] * w[1] * w[2];
            const size_t smem = (size_t)2 * (size_t)((fl + 31) & ~31ll) * 4 + SLAB_SMEM_EXTRA;
            if (smem <= budget) { best = logd; break; }
        }
    }
    if (best < 0) return;
    const int D = 1 << best;
    S.logD = best;
    S.n_maps = P.proj == VR_PROJ_PERSP ? vr::SLAB_MAPS : 1;
    const int a1 = (dom + 1) % 3, a2 = (dom + 2) % 3;
    for (int k = 0; k < vr::SLAB_MAPS; ++k) {
        const double fk = std::pow(0.8, (double)k);          // perspective: windows near the eye are smaller
        for (int a = 0; a < 3; ++a) S.w[k][a] = w[a];
        if (k > 0 && k < S.n_maps) {
            S.w[k][a1] = std::max(8, (int)std::ceil(w[a1] * fk));
            S.w[k][a2] = std::max(8, (int)std::ceil(w[a2] * fk));
            const int fa = dom == 0 ? 2 : 0;
            S.w[k][fa] = std::min(w[fa], (S.w[k][fa] + 3) & ~3);
        }
        S.box_floats[k] = S.w[k][0] * S.w[k][1] * S.w[k][2];
    }
    S.slot_floats = (S.box_floats[0] + 31) & ~31;
    sp.smem = (size_t)2 * S.slot_floats * 4 + SLAB_SMEM_EXTRA;
    sp.dom = dom;
    // window bytes a CTA tile stages per sample it takes (a ray takes about D / (|fwd_dom| step) samples per slab)
    sp.bytes_per_sample = (double)S.box_floats[0] * 4.0 * std::fabs(P.fwd[dom]) * P.step / ((double)vr::CTA_THREADS * D);
    sp.use = true;
}

vr_status ensure_linear(vr_volume* vol, bool transposed) {
    float*& dst = transposed ? vol->d_linear_t : vol->d_linear;
    if (dst) return VR_OK;
    const vr::LinearDims L = transposed ? vr::linear_dims_t(vol->dims[0], vol->dims[1], vol->dims[2])
                                        : vr::linear_dims(vol->dims[0], vol->dims[1], vol->dims[2]);
    cudaError_t e = cudaMalloc(&dst, (size_t)L.LX * L.LY * L.LZ * sizeof(float));
    if (e != cudaSuccess) { dst = nullptr; vol->linear_failed = true; cudaGetLastError(); return cuda_fail(e, "allocate linear copy"); }
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    e = cudaEventCreate(&e0);
    if (e == cudaSuccess) e = cudaEventCreate(&e1);
    if (e == cudaSuccess) e = cudaEventRecord(e0, vol->stream);
    if (e == cudaSuccess) {
        if (transposed) {
            dim3 grid((L.LX + 31) / 32, L.LY, (L.LZ + 31) / 32);
            vr::transpose_kernel<<<grid, 256, 0, vol->stream>>>(vol->d_tiled, dst, L.LX, L.LY, L.LZ, vol->dims[2] + vr::PAD_Z,
                                                                ty_stride_of(vol), slab_stride_of(vol));
        } else {
            dim3 grid((L.LX / 4 + 63) / 64, (L.LY + 3) / 4, L.LZ);
            vr::linearize_kernel<<<grid, 256, 0, vol->stream>>>(vol->d_tiled, dst, L.LX, L.LY, L.LZ, ty_stride_of(vol),
                                                                slab_stride_of(vol));
        }
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaEventRecord(e1, vol->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(vol->stream);
    if (e == cudaSuccess) e = cudaEventElapsedTime(transposed ? &vol->transpose_ms : &vol->linearize_ms, e0, e1);
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    if (e != cudaSuccess) { cudaFree(dst); dst = nullptr; vol->linear_failed = true; return cuda_fail(e, "linearize"); }
    return VR_OK;
}

vr_status encode_slab_map(vr_volume* vol, SlabPlan& sp) {
    EncodeTiledFn enc = encode_tiled_fn();
    if (!enc) return fail(VR_ERR_CUDA, "cuTensorMapEncodeTiled is not available from this driver");
    const bool tr = sp.dom == 0;                      // x-dominant views read the z-fastest copy: tensor dims (z, y, x)
    const vr::LinearDims L = tr ? vr::linear_dims_t(vol->dims[0], vol->dims[1], vol->dims[2])
                                : vr::linear_dims(vol->dims[0], vol->dims[1], vol->dims[2]);
    const int d0 = tr ? L.LZ : L.LX, d2 = tr ? L.LX : L.LZ;
    const cuuint64_t gdim[3] = {(cuuint64_t)d0, (cuuint64_t)L.LY, (cuuint64_t)d2};
    const cuuint64_t gstr[2] = {(cuuint64_t)d0 * 4, (cuuint64_t)d0 * L.LY * 4};
    const cuuint32_t estr[3] = {1, 1, 1};
    const int fa = tr ? 2 : 0, sl = tr ? 0 : 2;
    for (int k = 0; k < vr::SLAB_MAPS; ++k) {
        const int kk = k < sp.S.n_maps ? k : 0;
        const cuuint32_t box[3] = {(cuuint32_t)sp.S.w[kk][fa], (cuuint32_t)sp.S.w[kk][1], (cuuint32_t)sp.S.w[kk][sl]};
        const CUresult r = enc(&sp.maps.m[k], CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, tr ? vol->d_linear_t : vol->d_linear, gdim, gstr, box, estr,
                               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) return fail(VR_ERR_CUDA, "cuTensorMapEncodeTiled failed (code " + std::to_string((int)r) + ")");
    }
    return VR_OK;
}

template <int MODE, int DOM>
vr_status launch_slab_t(vr_volume* vol, const Frame& f, const SlabPlan& sp, float* d_img) {
    // the opt-in above 48 KB of dynamic shared memory is a per-device attribute of the function: set on every launch
    // (a host-side call of about a microsecond) rather than remembered per process, so that volumes on several GPUs work
    VR_CUDA(cudaFuncSetAttribute(vr::cast_slab_kernel<MODE, DOM>, cudaFuncAttributeMaxDynamicSharedMemorySize, 113 * 1024),
            "cudaFuncSetAttribute(slab caster)");
    vr::cast_slab_kernel<MODE, DOM><<<f.total_tiles, vr::CTA_THREADS, sp.smem, vol->stream>>>(
        f.P, sp.S, sp.maps, vol->d_bricks, (int)f.recs.size(), vol->d_tf_ea, d_img);
    VR_CUDA(cudaGetLastError(), "slab caster launch");
    return debug_sync(vol, "slab caster (VR_DEBUG)");
}

vr_status launch_slab(vr_volume* vol, const Frame& f, const SlabPlan& sp, int mode, float* d_img) {
    if (f.total_tiles == 0) return VR_OK;
    if (mode == VR_MODE_EA) {
        if (sp.dom == 0) return launch_slab_t<vr::MODE_EA, 0>(vol, f, sp, d_img);
        if (sp.dom == 1) return launch_slab_t<vr::MODE_EA, 1>(vol, f, sp, d_img);
        return launch_slab_t<vr::MODE_EA, 2>(vol, f, sp, d_img);
    }
    if (sp.dom == 0) return launch_slab_t<vr::MODE_MIP, 0>(vol, f, sp, d_img);
    if (sp.dom == 1) return launch_slab_t<vr::MODE_MIP, 1>(vol, f, sp, d_img);
    return launch_slab_t<vr::MODE_MIP, 2>(vol, f, sp, d_img);
}

// Which caster renders this frame, and its per-table / per-volume preparations (mask, linear copy) — called before the
// frame's timed region.  Measured on config 4 (profiles/r02_slab.md): staging pays when the window bytes per sample
// are below ~80 against the dense row-cache walk, and below ~130 x (occupied cell fraction) against the skipping
// caster (40 B per sample for config 3's table, where 31 % of the cells are occupied).
vr_status choose_caster(vr_volume* vol, const Frame& f, int mode, SlabPlan& sp) {
    const bool skip = skip_applies(vol, mode);
    if (skip) {
        vr_status s = ensure_skip_structure(vol, mode);                   // builds only after a table change (EA) / once (MIP)
        if (s != VR_OK) return s;
    }
    double limit = INFINITY;                                              // mode 2: whenever the window fits
    if (vol->slab_mode == 1) {
        limit = !skip ? 80.0 : mode == VR_MODE_MIP ? 20.0 : 130.0 * (double)vol->mask_occupied / mask_cells(vol);
    }
    // Perspective frames: the windows must hold the far corner tiles and the host has to scan every tile of the frame
    // for their size (milliseconds at 2048^2); measured on config 3's cube and on config 1 the slab caster never beat
    // the row-cache caster there (profiles/r02_slab.md).  Automatic choice: orthographic frames only.
    if (vol->slab_mode == 1 && f.P.proj == VR_PROJ_PERSP) { sp.use = false; vol->last_slab[0] = 0; return VR_OK; }
    plan_slab(vol, f, limit, (size_t)113 * 1024, sp);
    if (sp.use && sp.bytes_per_sample > limit) sp.use = false;
    if (sp.use && ensure_linear(vol, sp.dom == 0) != VR_OK) sp.use = false;            // no memory for the second copy: row-cache caster
    if (sp.use) {
        vr_status s = encode_slab_map(vol, sp);
        if (s != VR_OK) return s;
    }
    vol->last_slab[0] = sp.use ? 1 : 0;
    if (sp.use) {
        vol->last_slab[1] = sp.dom; vol->last_slab[2] = 1 << sp.S.logD;
        for (int a = 0; a < 3; ++a) vol->last_slab[3 + a] = sp.S.w[0][a];
    }
    return VR_OK;
}

vr_status cast_frame(vr_volume* vol, const Frame& f, const SlabPlan& sp, int mode, float* d_img) {
    if (sp.use) return launch_slab(vol, f, sp, mode, d_img);
    return launch_cast<0>(vol, f, mode, d_img, nullptr, nullptr, nullptr);
}

vr_status launch_composite(vr_volume* vol, const Frame& f, int mode, const float* d_img, int W, int H, float* d_out,
                           float* d_scalar) {
    const int B = (int)f.recs.size();
    dim3 grid((W + 15) / 16, (H + 15) / 16);
    if (mode == VR_MODE_EA)
        vr::composite_kernel<vr::MODE_EA><<<grid, 256, 0, vol->stream>>>(vol->d_bricks, vol->d_order, B, d_img, W, H,
                                                                         vol->d_tf_raw, f.P.vmin, f.P.inv_range, d_out, d_scalar);
    else
        vr::composite_kernel<vr::MODE_MIP><<<grid, 256, 0, vol->stream>>>(vol->d_bricks, vol->d_order, B, d_img, W, H,
                                                                          vol->d_tf_raw, f.P.vmin, f.P.inv_range, d_out, d_scalar);
    VR_CUDA(cudaGetLastError(), "composite kernel launch");
    return debug_sync(vol, "composite kernel (VR_DEBUG)");
}

// Brick images of vr_render live in one grow-only pool.  The rectangles change with the view, so the request is
// rounded up to the most a frame of this size can need (every brick a full frame) when that is modest (<= 1 GiB),
// else doubled: a camera orbit then never reallocates inside a frame sequence (cudaFree synchronises the device).
vr_status ensure_pool(vr_volume* vol, size_t floats, size_t full_frames_floats = 0) {
    if (floats <= vol->pool_floats) return VR_OK;
    if (vol->d_pool) { cudaFree(vol->d_pool); vol->d_pool = nullptr; vol->pool_floats = 0; }
    size_t want = floats * 2;
    if (full_frames_floats >= floats && full_frames_floats * sizeof(float) <= ((size_t)1 << 30)) want = full_frames_floats;
    VR_CUDA(cudaMalloc(&vol->d_pool, want * sizeof(float)), "allocate brick images");
    vol->pool_floats = want;
    return VR_OK;
}

}  // namespace

extern "C" {

const char* vr_last_error(void) { return g_err.c_str(); }

vr_status vr_create_volume(const int dims[3], const float* d_data, vr_volume** out) {
    if (!dims || !d_data || !out) return fail(VR_ERR_INVALID_ARG, "vr_create_volume: NULL argument");
    *out = nullptr;
    for (int a = 0; a < 3; ++a)
        if (dims[a] <= 0 || dims[a] > 65528) return fail(VR_ERR_INVALID_ARG, "vr_create_volume: each dim must be in [1,65528]");
    vr_volume* v = new (std::nothrow) vr_volume();
    if (!v) return fail(VR_ERR_OOM, "vr_create_volume: host allocation failed");
    for (int a = 0; a < 3; ++a) { v->dims[a] = dims[a]; v->sub_hi[a] = dims[a]; }
    if (const char* e_ = std::getenv("VR_DEBUG")) v->debug = e_[0] != '\0' && e_[0] != '0';   // the library's only environment variable
    // padded: PAD_a replicated layers below, at least one above
    v->TX = (dims[0] + vr::PAD_X + 1 + 7) / 8; v->TY = (dims[1] + vr::PAD_Y + 1 + 7) / 8; v->TZ = (dims[2] + vr::PAD_Z + 1 + 7) / 8;
    if ((double)v->TX * v->TY * vr::TILE_ELEMS >= 1073741824.0) {   // slab bytes and in-slab offsets stay 32-bit
        delete v;
        return fail(VR_ERR_INVALID_ARG, "vr_create_volume: nx*ny too large for 32-bit in-slab offsets");
    }
    v->tiled_elems = (size_t)v->TX * v->TY * v->TZ * vr::TILE_ELEMS;
    v->NBX = (dims[0] + vr::PAD_X + 3) / 4; v->NBY = (dims[1] + vr::PAD_Y + 3) / 4; v->NBZ = (dims[2] + vr::PAD_Z + 3) / 4;   // n_a + PAD_a padded cells
    v->mask_words = (size_t)v->NBX * v->NBY * v->NBZ;
    cudaError_t e = cudaMalloc(&v->d_tiled, v->tiled_elems * sizeof(float));
    if (e == cudaSuccess) e = cudaMalloc(&v->d_range, 2 * vr::RANGE_SLOTS * sizeof(unsigned));
    if (e == cudaSuccess) e = cudaMalloc(&v->d_tf_ea, 256 * sizeof(float4));
    if (e == cudaSuccess) e = cudaMalloc(&v->d_tf_raw, 256 * sizeof(float4));
    if (e == cudaSuccess) e = cudaMalloc(&v->d_bricks, VR_MAX_BRICKS * sizeof(vr::BrickRec));
    if (e == cudaSuccess) e = cudaMalloc(&v->d_order, VR_MAX_BRICKS * sizeof(int));
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (e == cudaSuccess) e = cudaEventCreate(&e0);
    if (e == cudaSuccess) e = cudaEventCreate(&e1);
    for (int k = 0; k < 4 && e == cudaSuccess; ++k) e = cudaEventCreate(&v->ev[k]);
    if (e == cudaSuccess) {
        dim3 grid((v->TX + 7) / 8, v->TY, v->TZ);
        std::vector<unsigned> init(2 * vr::RANGE_SLOTS);
        for (int k = 0; k < vr::RANGE_SLOTS; ++k) { init[2 * k] = 0xffffffffu; init[2 * k + 1] = 0u; }
        e = cudaMemcpyAsync(v->d_range, init.data(), init.size() * sizeof(unsigned), cudaMemcpyHostToDevice, v->stream);
        if (e == cudaSuccess) e = cudaEventRecord(e0, v->stream);
        if (e == cudaSuccess) {
            vr::relayout_kernel<<<grid, 256, 0, v->stream>>>(d_data, v->d_tiled, dims[0], dims[1], dims[2], v->TX, v->TY,
                                                             v->d_range);
            e = cudaGetLastError();
        }
        if (e == cudaSuccess) e = cudaEventRecord(e1, v->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(v->stream);
        if (e == cudaSuccess) e = cudaEventElapsedTime(&v->relayout_ms, e0, e1);
        if (e == cudaSuccess) {
            std::vector<unsigned> slots(2 * vr::RANGE_SLOTS);
            e = cudaMemcpy(slots.data(), v->d_range, slots.size() * sizeof(unsigned), cudaMemcpyDeviceToHost);
            unsigned kmin = 0xffffffffu, kmax = 0u;
            for (int k = 0; k < vr::RANGE_SLOTS; ++k) {
                kmin = std::min(kmin, slots[2 * k]); kmax = std::max(kmax, slots[2 * k + 1]);
            }
            if (kmin <= kmax) {
                v->data_min = vr::key_float(kmin); v->data_max = vr::key_float(kmax); v->has_range = true;
            }
        }
    }
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    if (e != cudaSuccess) {
        vr_status s = cuda_fail(e, "vr_create_volume");
        vr_destroy_volume(v);
        return s;
    }
    *out = v;
    return VR_OK;
}

void vr_destroy_volume(vr_volume* v) {
    if (!v) return;
    if (v->d_tiled) cudaFree(v->d_tiled);
    if (v->d_range) cudaFree(v->d_range);
    if (v->d_tf_ea) cudaFree(v->d_tf_ea);
    if (v->d_tf_raw) cudaFree(v->d_tf_raw);
    if (v->d_bricks) cudaFree(v->d_bricks);
    if (v->d_order) cudaFree(v->d_order);
    if (v->d_pool) cudaFree(v->d_pool);
    for (int k = 0; k < 2; ++k) {
        if (v->d_frame[k]) cudaFree(v->d_frame[k]);
        if (v->frame_done[k]) cudaEventDestroy(v->frame_done[k]);
        if (v->copy_done[k]) cudaEventDestroy(v->copy_done[k]);
    }
    if (v->copy_stream) cudaStreamDestroy(v->copy_stream);
    if (v->d_mask) cudaFree(v->d_mask);
    if (v->d_blockmax) cudaFree(v->d_blockmax);
    if (v->d_linear) cudaFree(v->d_linear);
    if (v->d_linear_t) cudaFree(v->d_linear_t);
    if (v->d_mask_count) cudaFree(v->d_mask_count);
    for (int k = 0; k < 4; ++k)
        if (v->ev[k]) cudaEventDestroy(v->ev[k]);
    delete v;
}

vr_status vr_set_stream(vr_volume* vol, void* cuda_stream) {
    if (!vol) return fail(VR_ERR_INVALID_ARG, "vr_set_stream: volume is NULL");
    vol->stream = (cudaStream_t)cuda_stream;
    return VR_OK;
}

vr_status vr_set_transfer_function(vr_volume* vol, const float rgba[1024], float vmin, float vmax) {
    if (!vol || !rgba) return fail(VR_ERR_INVALID_ARG, "vr_set_transfer_function: NULL argument");
    if (!std::isfinite(vmin) || !std::isfinite(vmax) || !(vmax > vmin))
        return fail(VR_ERR_INVALID_ARG, "vr_set_transfer_function: need finite vmin < vmax");
    for (int i = 0; i < 1024; ++i)
        if (!(rgba[i] >= 0.0f && rgba[i] <= 1.0f))
            return fail(VR_ERR_INVALID_ARG, "vr_set_transfer_function: table entries must be in [0,1]");
    std::memcpy(vol->tf_host, rgba, sizeof(float) * 1024);
    vol->vmin = vmin; vol->vmax = vmax;
    vol->tf_step = -1.0;
    VR_CUDA(cudaMemcpyAsync(vol->d_tf_raw, vol->tf_host, sizeof(float) * 1024, cudaMemcpyHostToDevice, vol->stream),
            "upload transfer function");
    vol->has_tf = true;
    return VR_OK;
}

vr_status vr_set_bricks(vr_volume* vol, int bx, int by, int bz) {
    if (!vol) return fail(VR_ERR_INVALID_ARG, "vr_set_bricks: volume is NULL");
    const int b[3] = {bx, by, bz};
    for (int a = 0; a < 3; ++a)
        if (b[a] < 1 || b[a] > vol->dims[a]) return fail(VR_ERR_INVALID_ARG, "vr_set_bricks: need 1 <= b_a <= n_a");
    if ((long long)bx * by * bz > VR_MAX_BRICKS) return fail(VR_ERR_INVALID_ARG, "vr_set_bricks: more than VR_MAX_BRICKS bricks");
    for (int a = 0; a < 3; ++a) vol->bricks[a] = b[a];
    return VR_OK;
}

vr_status vr_set_subcube(vr_volume* vol, const int lo[3], const int hi[3]) {
    if (!vol) return fail(VR_ERR_INVALID_ARG, "vr_set_subcube: volume is NULL");
    if (!lo || !hi) {                                  // NULL, NULL: back to the whole cube
        if (lo || hi) return fail(VR_ERR_INVALID_ARG, "vr_set_subcube: pass both corners or neither");
        for (int a = 0; a < 3; ++a) { vol->sub_lo[a] = 0; vol->sub_hi[a] = vol->dims[a]; }
        return VR_OK;
    }
    for (int a = 0; a < 3; ++a)
        if (lo[a] < 0 || hi[a] > vol->dims[a] || hi[a] < lo[a])
            return fail(VR_ERR_INVALID_ARG, "vr_set_subcube: need 0 <= lo_a <= hi_a <= n_a");
    for (int a = 0; a < 3; ++a) { vol->sub_lo[a] = lo[a]; vol->sub_hi[a] = hi[a]; }
    return VR_OK;
}

vr_status vr_set_channel_mask(vr_volume* vol, const unsigned char* enabled) {
    if (!vol) return fail(VR_ERR_INVALID_ARG, "vr_set_channel_mask: volume is NULL");
    if (!enabled) { vol->n_runs = 0; return VR_OK; }                 // NULL: every channel enabled
    static_assert(vr::MAX_RUNS == VR_MAX_CHANNEL_RUNS, "run limit of the kernels and of the header differ");
    int runs[2 * vr::MAX_RUNS], n = 0;
    const int nz = vol->dims[2];
    for (int z = 0; z < nz;) {
        if (!enabled[z]) { ++z; continue; }
        int z1 = z;
        while (z1 < nz && enabled[z1]) ++z1;
        if (n == vr::MAX_RUNS)
            return fail(VR_ERR_INVALID_ARG, "vr_set_channel_mask: more than VR_MAX_CHANNEL_RUNS runs of enabled channels");
        runs[2 * n] = z; runs[2 * n + 1] = z1; ++n;
        z = z1;
    }
    if (n == 1 && runs[0] == 0 && runs[1] == nz) { vol->n_runs = 0; return VR_OK; }   // all enabled = no mask
    if (n == 0) { runs[0] = 0; runs[1] = 0; n = 1; }                 // nothing enabled: one empty run
    vol->n_runs = n;
    for (int k = 0; k < 2 * n; ++k) vol->run_z[k] = runs[k];
    return VR_OK;
}

vr_status vr_render(vr_volume* vol, const vr_camera* cam, int W, int H, float step, int mode, float ert,
                    float* d_out_rgba, float* d_out_scalar) {
    vr_status s = check_render_args(vol, cam, W, H, step, mode);
    if (s != VR_OK) return s;
    if (!d_out_rgba) return fail(VR_ERR_INVALID_ARG, "vr_render: d_out_rgba is NULL");
    const int B = vol->bricks[0] * vol->bricks[1] * vol->bricks[2];
    const bool direct = (B == 1 && mode == VR_MODE_EA);
    Frame f;
    if ((s = build_frame(vol, cam, W, H, step, ert, true, direct, f)) != VR_OK) return s;
    if ((s = upload_plan(vol, f)) != VR_OK) return s;
    if (mode == VR_MODE_EA && (s = upload_tf_for_step(vol, (double)step)) != VR_OK) return s;
    vol->timed_cast = vol->timed_comp = false;
    if (!direct && (s = ensure_pool(vol, f.pool_pixels * (mode == VR_MODE_EA ? 4 : 1),
                                    (size_t)B * W * H * (mode == VR_MODE_EA ? 4 : 1))) != VR_OK) return s;
    SlabPlan sp;
    if ((s = choose_caster(vol, f, mode, sp)) != VR_OK) return s;
    VR_CUDA(cudaEventRecord(vol->ev[0], vol->stream), "record event");
    s = cast_frame(vol, f, sp, mode, direct ? d_out_rgba : vol->d_pool);
    if (s != VR_OK) return s;
    VR_CUDA(cudaEventRecord(vol->ev[1], vol->stream), "record event");
    vol->timed_cast = true;
    if (direct) return VR_OK;
    VR_CUDA(cudaEventRecord(vol->ev[2], vol->stream), "record event");
    s = launch_composite(vol, f, mode, vol->d_pool, W, H, d_out_rgba, d_out_scalar);
    if (s != VR_OK) return s;
    VR_CUDA(cudaEventRecord(vol->ev[3], vol->stream), "record event");
    vol->timed_comp = true;
    return VR_OK;
}

vr_status vr_get_stage_ms(vr_volume* vol, float* h_cast_ms, float* h_composite_ms) {
    if (!vol) return fail(VR_ERR_INVALID_ARG, "vr_get_stage_ms: volume is NULL");
    if (!vol->timed_cast) return fail(VR_ERR_STATE, "vr_get_stage_ms: no frame rendered yet");
    float c = 0.f, m = 0.f;
    VR_CUDA(cudaEventSynchronize(vol->ev[vol->timed_comp ? 3 : 1]), "vr_get_stage_ms");
    VR_CUDA(cudaEventElapsedTime(&c, vol->ev[0], vol->ev[1]), "vr_get_stage_ms");
    if (vol->timed_comp) VR_CUDA(cudaEventElapsedTime(&m, vol->ev[2], vol->ev[3]), "vr_get_stage_ms");
    if (h_cast_ms) *h_cast_ms = c;
    if (h_composite_ms) *h_composite_ms = m;
    return VR_OK;
}

vr_status vr_render_to_host_async(vr_volume* vol, const vr_camera* cam, int W, int H, float step, int mode, float ert,
                                  float* h_out_rgba) {
    if (!h_out_rgba) return fail(VR_ERR_INVALID_ARG, "vr_render_to_host: h_out_rgba is NULL");
    if (!vol) return fail(VR_ERR_INVALID_ARG, "volume is NULL");
    if (W <= 0 || H <= 0 || W > 32768 || H > 32768) return fail(VR_ERR_INVALID_ARG, "W and H must be in [1,32768]");
    const size_t floats = (size_t)W * H * 4;
    if (!vol->copy_stream) {
        VR_CUDA(cudaStreamCreateWithFlags(&vol->copy_stream, cudaStreamNonBlocking), "create copy stream");
        for (int k = 0; k < 2; ++k) {
            VR_CUDA(cudaEventCreateWithFlags(&vol->frame_done[k], cudaEventDisableTiming), "create event");
            VR_CUDA(cudaEventCreateWithFlags(&vol->copy_done[k], cudaEventDisableTiming), "create event");
        }
    }
    if (floats > vol->frame_floats) {
        VR_CUDA(cudaStreamSynchronize(vol->copy_stream), "vr_render_to_host");       // no copy may be reading a frame
        for (int k = 0; k < 2; ++k) {
            if (vol->d_frame[k]) { cudaFree(vol->d_frame[k]); vol->d_frame[k] = nullptr; }
        }
        vol->frame_floats = 0;
        for (int k = 0; k < 2; ++k) VR_CUDA(cudaMalloc(&vol->d_frame[k], floats * sizeof(float)), "allocate frame");
        vol->frame_floats = floats;
    }
    const int slot = (int)(vol->frame_idx & 1u);
    // the copy that last read this device frame must be over before the compositor overwrites it
    if (vol->frame_idx >= 2) VR_CUDA(cudaStreamWaitEvent(vol->stream, vol->copy_done[slot], 0), "wait for copy");
    vr_status s = vr_render(vol, cam, W, H, step, mode, ert, vol->d_frame[slot], nullptr);
    if (s != VR_OK) return s;
    VR_CUDA(cudaEventRecord(vol->frame_done[slot], vol->stream), "record event");
    VR_CUDA(cudaStreamWaitEvent(vol->copy_stream, vol->frame_done[slot], 0), "wait for frame");
    VR_CUDA(cudaMemcpyAsync(h_out_rgba, vol->d_frame[slot], floats * sizeof(float), cudaMemcpyDeviceToHost, vol->copy_stream),
            "copy frame to host");
    VR_CUDA(cudaEventRecord(vol->copy_done[slot], vol->copy_stream), "record event");
    ++vol->frame_idx;
    return VR_OK;
}

vr_status vr_wait_frames(vr_volume* vol) {
    if (!vol) return fail(VR_ERR_INVALID_ARG, "vr_wait_frames: volume is NULL");
    if (vol->copy_stream) VR_CUDA(cudaStreamSynchronize(vol->copy_stream), "vr_wait_frames");
    return VR_OK;
}

vr_status vr_render_to_host(vr_volume* vol, const vr_camera* cam, int W, int H, float step, int mode, float ert,
                            float* h_out_rgba) {
    vr_status s = vr_render_to_host_async(vol, cam, W, H, step, mode, ert, h_out_rgba);
    if (s != VR_OK) return s;
    return vr_wait_frames(vol);
}

vr_status vr_render_bricks(vr_volume* vol, const vr_camera* cam, int W, int H, float step, int mode, float ert,
                           float* d_brick_images) {
    vr_status s = check_render_args(vol, cam, W, H, step, mode);
    if (s != VR_OK) return s;
    if (!d_brick_images) return fail(VR_ERR_INVALID_ARG, "vr_render_bricks: d_brick_images is NULL");
    Frame f;
    if ((s = build_frame(vol, cam, W, H, step, ert, false, false, f)) != VR_OK) return s;
    if ((s = upload_plan(vol, f)) != VR_OK) return s;
    if (mode == VR_MODE_EA && (s = upload_tf_for_step(vol, (double)step)) != VR_OK) return s;
    const size_t B = f.recs.size();
    // full frames: pixels outside a brick's rectangle hold "nothing" (0 / -inf)
    const size_t n = B * (size_t)W * H * (mode == VR_MODE_EA ? 4 : 1);
    vr::fill_kernel<<<1184, 256, 0, vol->stream>>>(d_brick_images, n, mode == VR_MODE_EA ? 0.0f : -INFINITY);
    VR_CUDA(cudaGetLastError(), "fill kernel launch");
    SlabPlan sp;
    if ((s = choose_caster(vol, f, mode, sp)) != VR_OK) return s;
    return cast_frame(vol, f, sp, mode, d_brick_images);
}

vr_status vr_composite(vr_volume* vol, const vr_camera* cam, int W, int H, int mode, const float* d_brick_images,
                       float* d_out_rgba, float* d_out_scalar) {
    vr_status s = check_render_args(vol, cam, W, H, 1.0f, mode);
    if (s != VR_OK) return s;
    if (!d_brick_images || !d_out_rgba) return fail(VR_ERR_INVALID_ARG, "vr_composite: NULL image pointer");
    Frame f;
    if ((s = build_frame(vol, cam, W, H, 1.0f, 0.0f, false, false, f)) != VR_OK) return s;
    // a stack of full frames may hold anything anywhere: composite every brick at every pixel
    for (auto& r : f.recs) { r.rx0 = 0; r.ry0 = 0; r.rw = W; r.rh = H; }
    if ((s = upload_plan(vol, f)) != VR_OK) return s;
    return launch_composite(vol, f, mode, d_brick_images, W, H, d_out_rgba, d_out_scalar);
}

vr_status vr_plan_bricks(const int dims[3], const int bricks[3], const vr_camera* cam, int W, int H,
                         int out_rect[][4], int out_order[]) {
    if (!dims || !bricks || !cam || !out_rect || !out_order) return fail(VR_ERR_INVALID_ARG, "vr_plan_bricks: NULL argument");
    if (W <= 0 || H <= 0) return fail(VR_ERR_INVALID_ARG, "vr_plan_bricks: W and H must be positive");
    for (int a = 0; a < 3; ++a)
        if (dims[a] <= 0 || bricks[a] < 1 || bricks[a] > dims[a])
            return fail(VR_ERR_INVALID_ARG, "vr_plan_bricks: need dims > 0 and 1 <= b_a <= n_a");
    if ((long long)bricks[0] * bricks[1] * bricks[2] > VR_MAX_BRICKS)
        return fail(VR_ERR_INVALID_ARG, "vr_plan_bricks: more than VR_MAX_BRICKS bricks");
    if (const char* why = vr::check_camera(*cam)) return fail(VR_ERR_INVALID_ARG, why);
    std::vector<vr::BrickPlan> plan;
    std::vector<int> order;
    vr::plan_bricks(dims, bricks, *cam, W, H, plan, order);
    for (size_t b = 0; b < plan.size(); ++b) {
        out_rect[b][0] = plan[b].rx0; out_rect[b][1] = plan[b].ry0;
        out_rect[b][2] = plan[b].rw; out_rect[b][3] = plan[b].rh;
        out_order[b] = order[b];
    }
    return VR_OK;
}

vr_status vr_plan_slab(const int dims[3], const int bricks[3], const vr_camera* cam, int W, int H, float step,
                       int h_plan[8], double* h_bytes_per_sample, double h_ray[18]) {
    if (!dims || !bricks || !cam || !h_plan) return fail(VR_ERR_INVALID_ARG, "vr_plan_slab: NULL argument");
    if (W <= 0 || H <= 0 || W > 32768 || H > 32768) return fail(VR_ERR_INVALID_ARG, "vr_plan_slab: W and H must be in [1,32768]");
    if (!(step > 0.0f) || !std::isfinite(step)) return fail(VR_ERR_INVALID_ARG, "vr_plan_slab: step_voxels must be positive and finite");
    for (int a = 0; a < 3; ++a)
        if (dims[a] <= 0 || dims[a] > 65528 || bricks[a] < 1 || bricks[a] > dims[a])
            return fail(VR_ERR_INVALID_ARG, "vr_plan_slab: need 0 < dims <= 65528 and 1 <= b_a <= n_a");
    if ((long long)bricks[0] * bricks[1] * bricks[2] > VR_MAX_BRICKS) return fail(VR_ERR_INVALID_ARG, "vr_plan_slab: more than VR_MAX_BRICKS bricks");
    if (const char* why = vr::check_camera(*cam)) return fail(VR_ERR_INVALID_ARG, why);
    vr_volume v;                                   // host fields only: nothing is allocated, nothing touches a device
    for (int a = 0; a < 3; ++a) { v.dims[a] = dims[a]; v.sub_hi[a] = dims[a]; v.bricks[a] = bricks[a]; }
    v.TX = (dims[0] + vr::PAD_X + 1 + 7) / 8; v.TY = (dims[1] + vr::PAD_Y + 1 + 7) / 8; v.TZ = (dims[2] + vr::PAD_Z + 1 + 7) / 8;
    v.slab_mode = 2;
    Frame f;
    vr_status s = build_frame(&v, cam, W, H, step, 0.0f, true, false, f);
    if (s != VR_OK) return s;
    SlabPlan sp;
    plan_slab(&v, f, INFINITY, (size_t)113 * 1024, sp);
    h_plan[0] = sp.use ? 1 : 0;
    h_plan[1] = sp.use ? sp.dom : 0; h_plan[2] = sp.use ? 1 << sp.S.logD : 0;
    for (int a = 0; a < 3; ++a) h_plan[3 + a] = sp.use ? sp.S.w[0][a] : 0;
    h_plan[6] = sp.use ? sp.S.n_maps : 0; h_plan[7] = sp.use ? (int)sp.smem : 0;
    if (h_bytes_per_sample) *h_bytes_per_sample = sp.use ? sp.bytes_per_sample : 0.0;
    if (h_ray && sp.use)
        for (int a = 0; a < 3; ++a) {
            h_ray[a] = sp.S.q0[a]; h_ray[3 + a] = sp.S.dqx[a]; h_ray[6 + a] = sp.S.dqy[a];
            h_ray[9 + a] = sp.S.v0[a]; h_ray[12 + a] = sp.S.dvx[a]; h_ray[15 + a] = sp.S.dvy[a];
        }
    return VR_OK;
}

vr_status vr_measure_units(vr_volume* vol, const vr_camera* cam, int W, int H, float step, int mode, float ert,
                           long long h_samples[2], long long h_units[4]) {
    vr_status s = check_render_args(vol, cam, W, H, step, mode);
    if (s != VR_OK) return s;
    Frame f;
    if ((s = build_frame(vol, cam, W, H, step, ert, true, false, f)) != VR_OK) return s;
    if ((s = upload_plan(vol, f)) != VR_OK) return s;
    if (mode == VR_MODE_EA && (s = upload_tf_for_step(vol, (double)step)) != VR_OK) return s;
    if ((s = ensure_pool(vol, f.pool_pixels * (mode == VR_MODE_EA ? 4 : 1))) != VR_OK) return s;
    if (skip_applies(vol, mode) && (s = ensure_skip_structure(vol, mode)) != VR_OK) return s;
    const size_t n_words = (vol->tiled_elems / 8 + 31) / 32;
    const size_t m_words = (vol->mask_words / 4 + 31) / 32 + 1;      // one bit per 32-byte sector (4 words) of the mask
    unsigned *d_bitmap = nullptr, *d_mbitmap = nullptr;
    unsigned long long* d_cnt = nullptr;                              // [0..1] samples, [2..4] cube units, [5..7] mask units
    cudaError_t e = cudaMalloc(&d_bitmap, n_words * sizeof(unsigned));
    if (e == cudaSuccess) e = cudaMalloc(&d_mbitmap, m_words * sizeof(unsigned));
    if (e == cudaSuccess) e = cudaMalloc(&d_cnt, 8 * sizeof(unsigned long long));
    if (e == cudaSuccess) e = cudaMemsetAsync(d_bitmap, 0, n_words * sizeof(unsigned), vol->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(d_mbitmap, 0, m_words * sizeof(unsigned), vol->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(d_cnt, 0, 8 * sizeof(unsigned long long), vol->stream);
    if (e != cudaSuccess) s = cuda_fail(e, "vr_measure: allocate / clear counters");
    if (s == VR_OK) s = launch_cast<1>(vol, f, mode, vol->d_pool, d_cnt, d_bitmap, d_mbitmap);
    unsigned long long h[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    if (s == VR_OK) {
        vr::popcount_kernel<<<1184, 256, 0, vol->stream>>>(d_bitmap, n_words, d_cnt + 2);
        vr::popcount_kernel<<<148, 256, 0, vol->stream>>>(d_mbitmap, m_words, d_cnt + 5);
        e = cudaGetLastError();
        if (e == cudaSuccess) e = cudaMemcpyAsync(h, d_cnt, sizeof(h), cudaMemcpyDeviceToHost, vol->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(vol->stream);
        if (e != cudaSuccess) s = cuda_fail(e, "vr_measure");
    }
    if (d_bitmap) cudaFree(d_bitmap);
    if (d_mbitmap) cudaFree(d_mbitmap);
    if (d_cnt) cudaFree(d_cnt);
    if (s != VR_OK) return s;
    if (h_samples) { h_samples[0] = (long long)h[0]; h_samples[1] = (long long)h[1]; }
    if (h_units) { for (int k = 0; k < 3; ++k) h_units[k] = (long long)h[2 + k]; h_units[3] = (long long)h[5]; }
    return VR_OK;
}

vr_status vr_measure(vr_volume* vol, const vr_camera* cam, int W, int H, float step, int mode, float ert,
                     long long* h_samples, long long* h_sectors) {
    long long c[2] = {0, 0}, u[4] = {0, 0, 0, 0};
    vr_status s = vr_measure_units(vol, cam, W, H, step, mode, ert, c, u);
    if (s == VR_OK && h_samples) *h_samples = c[0];
    if (s == VR_OK && h_sectors) *h_sectors = u[0];
    return s;
}

vr_status vr_set_empty_space_skipping(vr_volume* vol, int enabled) {
    if (!vol) return fail(VR_ERR_INVALID_ARG, "vr_set_empty_space_skipping: volume is NULL");
    vol->skip_enabled = enabled != 0;
    return VR_OK;
}

vr_status vr_get_skip_info(vr_volume* vol, int* h_active, float* h_build_ms, long long* h_mask_bytes,
                           double* h_occupied_fraction) {
    if (!vol) return fail(VR_ERR_INVALID_ARG, "vr_get_skip_info: volume is NULL");
    const bool active = vol->has_tf && skip_applies(vol, VR_MODE_EA);
    if (active) {
        vr_status s = ensure_mask(vol);
        if (s != VR_OK) return s;
    }
    if (h_active) *h_active = active ? 1 : 0;
    if (h_build_ms) *h_build_ms = active ? vol->mask_build_ms : 0.f;
    if (h_mask_bytes) *h_mask_bytes = active ? (long long)(vol->mask_words * sizeof(unsigned long long)) : 0;
    if (h_occupied_fraction)
        *h_occupied_fraction = active ? (double)vol->mask_occupied / mask_cells(vol) : 1.0;
    return VR_OK;
}

vr_status vr_set_slab_staging(vr_volume* vol, int mode) {
    if (!vol) return fail(VR_ERR_INVALID_ARG, "vr_set_slab_staging: volume is NULL");
    if (mode < 0 || mode > 2) return fail(VR_ERR_INVALID_ARG, "vr_set_slab_staging: mode must be 0 (off), 1 (auto) or 2 (whenever it fits)");
    vol->slab_mode = mode;
    return VR_OK;
}

vr_status vr_get_slab_info(const vr_volume* vol, int h_info[6], float* h_linearize_ms, long long* h_linear_bytes) {
    if (!vol) return fail(VR_ERR_INVALID_ARG, "vr_get_slab_info: volume is NULL");
    if (h_info) for (int k = 0; k < 6; ++k) h_info[k] = vol->last_slab[k];
    if (h_linearize_ms) *h_linearize_ms = vol->linearize_ms + vol->transpose_ms;
    if (h_linear_bytes) {
        const vr::LinearDims L = vr::linear_dims(vol->dims[0], vol->dims[1], vol->dims[2]);
        const vr::LinearDims T = vr::linear_dims_t(vol->dims[0], vol->dims[1], vol->dims[2]);
        *h_linear_bytes = (vol->d_linear ? (long long)L.LX * L.LY * L.LZ * 4 : 0) + (vol->d_linear_t ? (long long)T.LX * T.LY * T.LZ * 4 : 0);
    }
    return VR_OK;
}

vr_status vr_volume_info(const vr_volume* vol, float* h_relayout_ms, long long* h_tiled_bytes) {
    if (!vol) return fail(VR_ERR_INVALID_ARG, "vr_volume_info: volume is NULL");
    if (h_relayout_ms) *h_relayout_ms = vol->relayout_ms;
    if (h_tiled_bytes) *h_tiled_bytes = (long long)(vol->tiled_elems * sizeof(float));
    return VR_OK;
}

vr_status vr_volume_range(const vr_volume* vol, float* h_min, float* h_max) {
    if (!vol) return fail(VR_ERR_INVALID_ARG, "vr_volume_range: volume is NULL");
    if (!vol->has_range) return fail(VR_ERR_STATE, "vr_volume_range: the cube holds no finite-ordered value (all NaN)");
    if (h_min) *h_min = vol->data_min;
    if (h_max) *h_max = vol->data_max;
    return VR_OK;
}

vr_status vr_volume_histogram(vr_volume* vol, int n_bins, float lo, float hi, long long* h_counts, long long* h_nan) {
    if (!vol || !h_counts) return fail(VR_ERR_INVALID_ARG, "vr_volume_histogram: NULL argument");
    if (n_bins < 1 || n_bins > vr::HIST_MAX_BINS) return fail(VR_ERR_INVALID_ARG, "vr_volume_histogram: n_bins must be in [1,4096]");
    if (!std::isfinite(lo) || !std::isfinite(hi) || !(hi > lo)) return fail(VR_ERR_INVALID_ARG, "vr_volume_histogram: need finite lo < hi");
    unsigned long long* d_bins = nullptr;
    VR_CUDA(cudaMalloc(&d_bins, (size_t)(n_bins + 1) * sizeof(unsigned long long)), "allocate histogram");
    cudaError_t e = cudaMemsetAsync(d_bins, 0, (size_t)(n_bins + 1) * sizeof(unsigned long long), vol->stream);
    std::vector<unsigned long long> h((size_t)n_bins + 1, 0ull);
    if (e == cudaSuccess) {
        const size_t n_tiles = (size_t)vol->TX * vol->TY * vol->TZ;
        const float scale = (float)n_bins / (hi - lo);
        // one CTA covers many tiles; sub-2^32 counts per CTA bin: at most n_tiles/grid * 512 voxels per CTA
        const int grid = (int)std::min<size_t>(n_tiles, 148 * 8);
        vr::histogram_kernel<<<grid, 256, (size_t)n_bins * sizeof(unsigned), vol->stream>>>(
            vol->d_tiled, n_tiles, vol->TX, vol->TY, vol->dims[0], vol->dims[1], vol->dims[2], lo, scale, n_bins, d_bins,
            d_bins + n_bins);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaMemcpyAsync(h.data(), d_bins, h.size() * sizeof(unsigned long long), cudaMemcpyDeviceToHost, vol->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(vol->stream);
    cudaFree(d_bins);
    if (e != cudaSuccess) return cuda_fail(e, "vr_volume_histogram");
    for (int i = 0; i < n_bins; ++i) h_counts[i] = (long long)h[i];
    if (h_nan) *h_nan = (long long)h[n_bins];
    return VR_OK;
}

vr_status vr_export_linear(vr_volume* vol, float* d_linear) {
    if (!vol || !d_linear) return fail(VR_ERR_INVALID_ARG, "vr_export_linear: NULL argument");
    vr::export_linear_kernel<<<1184, 256, 0, vol->stream>>>(vol->d_tiled, d_linear, vol->dims[0], vol->dims[1],
                                                             vol->dims[2], ty_stride_of(vol), slab_stride_of(vol));
    VR_CUDA(cudaGetLastError(), "export kernel launch");
    return VR_OK;
}

}  // extern "C"

// ------------------------------------------------------------------------------------------------
// vr_volume_histogram_noalloc — the histogram of vr_volume_histogram for callers that must not allocate.
//
// vr_volume_histogram gets its device-side bins from cudaMalloc and gives them back with cudaFree on every call.
// That is wrong for two kinds of user of this library:
//   * a viewer embedded in a process whose own allocator (PyTorch's caching allocator, an RMM pool ...) already
//     holds nearly all of the GPU's memory — normal once a 26.8 GB cube and its copies are resident.  A cudaMalloc
//     issued from inside this library bypasses that allocator and fails with "out of memory" although the host
//     application still has free blocks;
//   * an interaction loop that has frames in flight on other streams: cudaFree waits for the whole device, so a
//     histogram requested while the user drags the colour-map range would stall every frame being rendered.
// Here the bins live in the array below, which is part of the library image: every GPU that loads libvr_b200.so
// holds its (HIST_MAX_BINS + 1) x 8 bytes = 32 776 bytes from then until the process exits, used or not.
//
// hist_scratch is a DEVICE symbol.  In host code its name stands for a host-side shadow, not for device memory, so
// it is never handed to a kernel as it is: the address the kernels get comes from cudaGetSymbolAddress, asked once per
// device while that device is current (hist_scratch_address).
// ------------------------------------------------------------------------------------------------
static __device__ __align__(256) unsigned long long hist_scratch[vr::HIST_MAX_BINS + 1];   // bins, then the NaN count

namespace {

constexpr int NOALLOC_MAX_DEVICES = 64;

// Device address of hist_scratch on the CURRENT device, looked up on the first call per device and remembered.
vr_status hist_scratch_address(int device, unsigned long long** out) {
    static std::mutex mtx;
    static unsigned long long* known[NOALLOC_MAX_DEVICES] = {nullptr};
    std::lock_guard<std::mutex> lock(mtx);
    if (device >= 0 && device < NOALLOC_MAX_DEVICES && known[device]) { *out = known[device]; return VR_OK; }
    void* p = nullptr;
    VR_CUDA(cudaGetSymbolAddress(&p, hist_scratch), "cudaGetSymbolAddress(histogram scratch)");
    if (!p) return fail(VR_ERR_CUDA, "vr_volume_histogram_noalloc: the scratch array has no address on this device");
    if (device >= 0 && device < NOALLOC_MAX_DEVICES) known[device] = static_cast<unsigned long long*>(p);
    *out = static_cast<unsigned long long*>(p);
    return VR_OK;
}

}  // namespace

extern "C" vr_status vr_volume_histogram_noalloc(vr_volume* vol, int n_bins, float lo, float hi, long long* h_counts,
                                                 long long* h_nan) {
    if (!vol || !h_counts) return fail(VR_ERR_INVALID_ARG, "vr_volume_histogram_noalloc: NULL argument");
    if (n_bins < 1) return fail(VR_ERR_INVALID_ARG, "vr_volume_histogram_noalloc: n_bins must be at least 1");
    if (n_bins > vr::HIST_MAX_BINS)
        return fail(VR_ERR_INVALID_ARG, "vr_volume_histogram_noalloc: n_bins = " + std::to_string(n_bins) + " exceeds the " +
                                            std::to_string(vr::HIST_MAX_BINS) +
                                            " bins the built-in scratch array holds (it cannot grow: this call never allocates)");
    if (!std::isfinite(lo) || !std::isfinite(hi) || !(hi > lo))
        return fail(VR_ERR_INVALID_ARG, "vr_volume_histogram_noalloc: need finite lo < hi");
    // The scratch array exists once per GPU, and the address below is the current device's copy: the volume must live there.
    int device = -1;
    VR_CUDA(cudaGetDevice(&device), "cudaGetDevice");
    cudaPointerAttributes attr;
    VR_CUDA(cudaPointerGetAttributes(&attr, vol->d_tiled), "cudaPointerGetAttributes(volume)");
    if (attr.type != cudaMemoryTypeDevice || attr.device != device)
        return fail(VR_ERR_STATE, "vr_volume_histogram_noalloc: the volume lives on GPU " + std::to_string(attr.device) +
                                      " but GPU " + std::to_string(device) + " is current (cudaSetDevice to the volume's GPU first)");
    unsigned long long* d_bins = nullptr;
    vr_status s = hist_scratch_address(device, &d_bins);
    if (s != VR_OK) return s;
    // the array still holds the previous call's counts: bins and NaN counter start from zero
    VR_CUDA(cudaMemsetAsync(d_bins, 0, (size_t)(n_bins + 1) * sizeof(unsigned long long), vol->stream),
            "vr_volume_histogram_noalloc: clear scratch");
    const size_t n_tiles = (size_t)vol->TX * vol->TY * vol->TZ;
    const float scale = (float)n_bins / (hi - lo);
    const int grid = (int)std::min<size_t>(n_tiles, 148 * 8);
    vr::histogram_kernel<<<grid, 256, (size_t)n_bins * sizeof(unsigned), vol->stream>>>(
        vol->d_tiled, n_tiles, vol->TX, vol->TY, vol->dims[0], vol->dims[1], vol->dims[2], lo, scale, n_bins, d_bins,
        d_bins + n_bins);
    VR_CUDA(cudaGetLastError(), "histogram kernel launch");
    unsigned long long nan = 0;
    static_assert(sizeof(long long) == sizeof(unsigned long long), "counts are copied as they are");
    VR_CUDA(cudaMemcpyAsync(h_counts, d_bins, (size_t)n_bins * sizeof(unsigned long long), cudaMemcpyDeviceToHost, vol->stream),
            "vr_volume_histogram_noalloc: copy bins");
    VR_CUDA(cudaMemcpyAsync(&nan, d_bins + n_bins, sizeof(nan), cudaMemcpyDeviceToHost, vol->stream),
            "vr_volume_histogram_noalloc: copy NaN count");
    VR_CUDA(cudaStreamSynchronize(vol->stream), "vr_volume_histogram_noalloc");
    if (h_nan) *h_nan = (long long)nan;
    return VR_OK;
}
