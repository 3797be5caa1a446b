/* include/vr.h — C ABI of the B200 ray-casting volume renderer (libvr_b200.so).
 *
 * The hot path of Hassan, Fluke & Barnes, "Interactive Visualization of the Largest
 * Radioastronomy Cubes": ray casting of a float32 spectral cube that is
 * partitioned object-wise into bricks (section 2.3), one image per brick inside
 * its "rendering rectangle" (section 2.4), then depth-ordered sort-last
 * composition of the brick images into one frame (section 2.5).  The paper
 * states the problem as "cube of floats + colour map + transformation/projection matrices in,
 * W x H frame out" and gives no formulas; the formulas are the readings
 * O1-O11 / A1-A16 of DESIGN.md ("Readings of the paper").
 *
 * Pointer convention: names starting with d_ are DEVICE pointers owned by the caller (e.g.
 * torch-allocated); every other pointer is HOST memory.  No torch types cross this boundary.
 * All work is enqueued on the volume's stream (vr_set_stream; default = legacy stream 0) and the
 * calls return without synchronising unless stated.  Every call returns a vr_status; the message
 * for the last failure on the calling thread is vr_last_error().  Nothing throws or aborts.
 * There is NO CPU fallback: without a CUDA device every compute call returns VR_ERR_CUDA.
 * Environment: one variable, read at vr_create_volume.  VR_DEBUG=1 makes every frame call wait for each of its
 * kernels (caster, compositor) and return that kernel's failure, instead of letting an asynchronous fault surface at
 * a later call; for debugging only, it serialises the stream.  Nothing else is read from the environment.
 *
 * Geometry conventions (O1-O3, O11):
 *   cube       float32, dims (nx,ny,nz), x fastest: data[(z*ny + y)*nx + x]; voxel (i,j,k) is the
 *              unit cell [i,i+1)x[j,j+1)x[k,k+1) with its value at the cell centre; the volume
 *              box is [0,nx]x[0,ny]x[0,nz] in voxel units.
 *   image      float32 RGBA, row-major [py][px][4]; py = 0 is the BOTTOM row; rays go through
 *              pixel centres; emission-absorption colours are premultiplied by alpha; pixels
 *              whose ray misses the volume are (0,0,0,0).
 */
#ifndef VR_H
#define VR_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct vr_volume vr_volume; /* opaque: owns the tiled copy, the tables, the brick images */

typedef enum {
    VR_OK = 0,
    VR_ERR_INVALID_ARG = 1, /* NULL pointer, non-positive size, non-finite value, bad enum ...  */
    VR_ERR_STATE = 2,       /* e.g. render before a transfer function was set                   */
    VR_ERR_OOM = 3,         /* device allocation failed                                         */
    VR_ERR_CUDA = 4         /* CUDA runtime failure (no device, launch error ...)               */
} vr_status;

typedef enum { VR_MODE_EA = 0, VR_MODE_MIP = 1 } vr_mode;     /* PAPER.md:80 / PAPER.md:150    */
typedef enum { VR_PROJ_ORTHO = 0, VR_PROJ_PERSP = 1 } vr_proj;

/* The "transformation and projection matrices" the viewer sends per frame. */
typedef struct {
    float view[16];     /* row-major 4x4, voxel space -> eye space, rigid (rotation+translation);
                           the eye looks down -z_eye, +x_eye is right, +y_eye is up             */
    int   projection;   /* vr_proj                                                              */
    float fovy_deg;     /* PERSP: full vertical field of view, in (0,180)                       */
    float ortho_half_h; /* ORTHO: half height of the view window in voxels (half width = *W/H)  */
} vr_camera;

#define VR_MAX_BRICKS 512 /* bx*by*bz */
#define VR_MAX_CHANNEL_RUNS 16 /* runs of consecutive enabled channels a channel mask may have */

/* a0  Brick partitioner / tiled re-layout ("loads its portion").
 *     Copies the linear cube d_data[nz][ny][nx] into the library's own tiled layout (8x8x8-voxel
 *     tiles, edge-replicated padding) with one streaming kernel.
 *     d_data is read during the call only (the call synchronises the stream before returning, so
 *     the caller may free d_data afterwards).  Allocates ~1.01x the cube on the device.
 *     INVALID_ARG: NULL, dim <= 0, dim > 65528.  OOM / CUDA on failure.                         */
vr_status vr_create_volume(const int dims[3] /* nx,ny,nz */, const float* d_data, vr_volume** out);
void      vr_destroy_volume(vr_volume* vol);

/* Stream for all later work of this volume (a cudaStream_t passed as void*). */
vr_status vr_set_stream(vr_volume* vol, void* cuda_stream);

/* Colour map ("transfer function"; PAPER.md:138 colour map sent by the viewer).
 *     rgba: 256 entries (r,g,b,a) in [0,1], un-premultiplied, HOST; entry j sits at data value
 *     vmin + (vmax-vmin)*j/255; values between entries are linearly interpolated, values outside
 *     [vmin,vmax] clamp (O6).  Alpha is opacity per voxel of path length; each render
 *     corrects it per entry for its step: 1-(1-a)^step.  INVALID_ARG: NULL, vmax <= vmin,
 *     non-finite, entry outside [0,1].                                                          */
vr_status vr_set_transfer_function(vr_volume* vol, const float rgba[256 * 4], float vmin, float vmax);

/* Object-space partition into bx*by*bz bricks with faces at floor(m*n_a/b_a) (
 *     DESIGN.md O9/A10).  Default 1,1,1.  INVALID_ARG: b_a < 1, b_a > n_a, product > VR_MAX_BRICKS. */
vr_status vr_set_bricks(vr_volume* vol, int bx, int by, int bz);

/* Sub-cube / spectral-channel selection ("a manual sub-cube"; PAPER.md:138 channels enabled or
 *     disabled by the user): only samples inside [lo, hi) voxels are taken — e.g. lo = {0,0,z0}, hi = {nx,ny,z1}
 *     renders channels z0..z1-1.  The sample lattice and the sampling (which still reads neighbouring voxels
 *     across the sub-cube's faces) are unchanged: the sub-cube is one more box every brick is intersected with
 *     (S1).  NULL, NULL restores the whole cube.  INVALID_ARG unless 0 <= lo_a <= hi_a <= n_a.       */
vr_status vr_set_subcube(vr_volume* vol, const int lo[3], const int hi[3]);

/* Spectral-channel mask ("enabling/disabling spectral channel(s)"): enabled[z] != 0 keeps channel z,
 *     HOST array of nz bytes, copied; NULL enables every channel again.  The enabled channels form maximal runs
 *     [za, zb) of consecutive channels, and a sample of the ray lattice is taken iff it lies in the slab
 *     za <= z <= zb of some run — decided in double precision with the rule that assigns samples to bricks
 *     (S2, O9), so a mask with one run equals vr_set_subcube on that z range.  The lattice and the
 *     sampling (which reads neighbouring channels across a run's faces) are unchanged.  Combines with bricks, the
 *     sub-cube, both modes and early termination.  INVALID_ARG: more than VR_MAX_CHANNEL_RUNS runs.             */
vr_status vr_set_channel_mask(vr_volume* vol, const unsigned char* enabled);

/* NEXT-2  Empty-space skipping keyed to the transfer function ("keeping the size of these tasks
 *     balanced"; PAPER.md:205 the work "varies based on the dataset characteristics"; PAPER.md:294 transfer functions
 *     that suppress the noise).  The library keeps one bit per voxel cell (the unit cube between 8 neighbouring
 *     voxel centres) saying whether a sample inside it can contribute under the current table: the bit is clear
 *     when a corner is NaN (the sample is skipped, O5/A14) or when all 8 corners classify below the
 *     table's first entry with alpha > 0 (the sample's alpha is exactly 0, O6/O7).  Emission-absorption rays pass
 *     over such cells without reading the cube.  The frame is IDENTICAL to the one rendered without skipping —
 *     only exactly-zero contributions are dropped — so this is a switch for measurements, not a quality setting.
 *     The mask (1/32 of the cube) is rebuilt by one pass over the cube at the first emission-absorption render
 *     after vr_set_transfer_function changed vmin, vmax or the length of the table's leading run of alpha = 0
 *     (that render synchronises the stream); tables whose second entry already has alpha > 0, and MIP, do not
 *     use it.  Default: enabled.
 *     MIP frames use the same switch with a different structure: the largest voxel of every block of 4x4x4 cells
 *     (built once per volume at the first MIP frame, 1/64 of the cube); a sample is passed over when its block's
 *     maximum (stored with a margin of 2^-21 of the block's value range and magnitude, which covers what the rounding of
 *     the fp32 blend can add to its largest corner) is not above the maximum the ray has reached before the current
 *     64-sample segment, so the raw maxima are bit-identical with the switch on and off.
 * vr_get_skip_info: builds the mask if it is due, then reports whether skipping is active for the current table,
 *     the build time of the mask in ms, its size in bytes and the fraction of cells whose bit is set.            */
vr_status vr_set_empty_space_skipping(vr_volume* vol, int enabled);
vr_status vr_get_skip_info(vr_volume* vol, int* h_active, float* h_build_ms, long long* h_mask_bytes,
                           double* h_occupied_fraction);

/* Slab staging (north_star kernel (2): "brick slabs staged through shared memory via TMA where the view is near
 *     axis-aligned"; section 2.4: GPU memory and the per-ray sampling loop).  The library has a
 *     second caster: a CTA marches its 16x8-pixel tile through the brick slab by slab along the dominant axis of the
 *     view direction; the box of voxels the tile's rays can touch inside a slab is copied into shared memory by one
 *     bulk tensor copy (TMA) from a LINEAR padded copy of the cube (made by the library at the first such frame and
 *     kept: x fastest for views whose dominant axis is y or z, a second one with z fastest for views whose dominant
 *     axis is x; + 1 x the cube in device memory each, the frame that makes one synchronises the stream), and samples
 *     are interpolated from shared memory.  Same lattice, cells, fractions, classification and blending as the other caster (O4-O9):
 *     frames agree with it to fp32 rounding of the interpolation and both meet the same parity gates.  Frames with a
 *     channel mask, frames some of whose rays do not advance along the dominant axis (eye inside the cube, very wide
 *     field of view) and frames whose window does not fit shared memory always use the other caster.
 *     mode 0: never.  mode 1 (default): when the window stages at most ~80 bytes per sample (dense sampling: small pixel
 *     pitch x step), ~130 bytes x the occupied-cell fraction when empty-space skipping is active for the table;
 *     orthographic frames only (perspective windows must hold the far corner tiles; measured, they never paid).
 *     mode 2: whenever the window fits, perspective frames included.  If the
 *     linear copy cannot be allocated the library stays on the other caster.
 * vr_get_slab_info: h_info[6] = {last frame used the slab caster, dominant axis, slab thickness D in cell layers,
 *     (largest) window extent in voxels along x, y, z}; time spent making the linear copies in ms; their size in bytes
 *     (0: none made). */
vr_status vr_set_slab_staging(vr_volume* vol, int mode);
vr_status vr_get_slab_info(const vr_volume* vol, int h_info[6], float* h_linearize_ms, long long* h_linear_bytes);

/* Host-only planning step of the slab-staged caster, no device needed (what vr_set_slab_staging(vol, 2) would decide
 *     for this frame): h_plan[8] = {eligible, dominant axis, slab thickness D, window extent x, y, z, window sizes
 *     in use (1: orthographic), shared memory per CTA in bytes}; *h_bytes_per_sample = window bytes staged per sample.
 *     h_ray[18] = the affine ray description the kernel's window placement uses, in padded voxel coordinates
 *     (voxel + (8,1,1) - 1/2): the ray of pixel (px,py) passes through Q = q0 + px*dqx + py*dqy with direction
 *     V = v0 + px*dvx + py*dvy; order q0[3], dqx[3], dqy[3], v0[3], dvx[3], dvy[3].  Window rule (slab.cuh): for the
 *     slab of cells [s*D, s*D + D) along the dominant axis the window starts at floor(lo - 1e-3) on the two other
 *     axes, lo/hi = min/max over the tile's four corner rays and the slab's two faces of
 *     U_a(c) = Q_a + (c - Q_dom) V_a / V_dom, rounded down to a multiple of 4 on the source's fastest axis (x; z for
 *     x-dominant views), and must hold voxels up to floor(hi + 1e-3) + 1.                                          */
vr_status vr_plan_slab(const int dims[3], const int bricks[3], const vr_camera* cam, int W, int H, float step_voxels,
                       int h_plan[8], double* h_bytes_per_sample, double h_ray[18]);

/* a1-a7  One frame: per-brick ray casting inside each brick's rendering rectangle
 *     (PAPER.md:150), then depth-ordered composition into d_out_rgba.
 *     step_voxels: sampling distance along the ray in voxels, > 0.
 *     mode: VR_MODE_EA (front-to-back emission-absorption) or VR_MODE_MIP (maximum intensity,
 *           colour-mapped at the end, un-premultiplied).
 *     ert_alpha: early ray termination (Levoy 1990) when a brick's accumulated
 *           opacity reaches this value; <= 0 or >= 1 disables it.  Ignored for MIP.
 *     d_out_rgba: DEVICE, H*W*4 floats.  d_out_scalar: DEVICE, H*W floats or NULL; MIP only:
 *           the raw maximum per pixel ("2D floating point array of maximum recorded
 *           scalar value"), -inf where the ray takes no sample.
 *     INVALID_ARG: NULL, W/H <= 0 or > 32768, step <= 0 or non-finite, unknown mode/projection,
 *     view not rigid within 1e-4, fovy outside (0,180), ortho_half_h <= 0.  STATE: no transfer
 *     function yet.  Asynchronous on the stream (first use at a new image size allocates).      */
vr_status vr_render(vr_volume* vol, const vr_camera* cam, int W, int H, float step_voxels, int mode,
                    float ert_alpha, float* d_out_rgba, float* d_out_scalar);

/* Same frame delivered to HOST memory (the frame is returned to the viewer): vr_render into an
 *     internal device frame, then a device->host copy of it into h_out_rgba (H*W*4 floats; pinned memory makes the
 *     copy asynchronous), then a wait for that copy.  This is the end-to-end call bench.py times.
 * vr_render_to_host_async: the same without the wait.  Two internal device frames are used alternately and the
 *     copy runs on a stream of its own, so the copy of frame k overlaps the ray casting of frame k+1; the caller
 *     keeps h_out_rgba untouched until vr_wait_frames (which waits for every copy issued so far) and uses a
 *     different host buffer for the next frame.                                                                */
vr_status vr_render_to_host(vr_volume* vol, const vr_camera* cam, int W, int H, float step_voxels,
                            int mode, float ert_alpha, float* h_out_rgba);
vr_status vr_render_to_host_async(vr_volume* vol, const vr_camera* cam, int W, int H, float step_voxels,
                                  int mode, float ert_alpha, float* h_out_rgba);
vr_status vr_wait_frames(vr_volume* vol);

/* Inspection level (the paper's two stages taken apart):
 * vr_render_bricks: steps a1-a5 only.  d_brick_images: DEVICE, caller-owned, B*H*W*4 floats (EA:
 *     premultiplied C_b, A_b) or B*H*W floats (MIP: M_b, -inf = no sample), full frames, brick
 *     index b = (bk*by + bj)*bx + bi; pixels outside a brick's rectangle are 0 / -inf.
 * vr_composite: steps a6-a7 on such a stack of brick images.                                    */
vr_status vr_render_bricks(vr_volume* vol, const vr_camera* cam, int W, int H, float step_voxels,
                           int mode, float ert_alpha, float* d_brick_images);
vr_status vr_composite(vr_volume* vol, const vr_camera* cam, int W, int H, int mode,
                       const float* d_brick_images, float* d_out_rgba, float* d_out_scalar);

/* Host-only planning step (a2 rendering rectangles, a6 depth order), no device needed:
 *     out_rect[b] = {x0, y0, w, h} of brick b's rendering rectangle (w = 0: off-screen),
 *     out_order[k] = brick index of the k-th brick front to back (A11, A12).         */
vr_status vr_plan_bricks(const int dims[3], const int bricks[3], const vr_camera* cam, int W, int H,
                         int out_rect[][4], int out_order[]);

/* Minimum and maximum of the cube (NaN voxels ignored), computed by the re-layout pass of vr_create_volume at
 *     no extra memory traffic: the data range a transfer function is set over when the file metadata does not
 *     give one ("each GPU computes the minimum and maximum of its portion").
 *     STATE if every voxel is NaN.                                                               */
vr_status vr_volume_range(const vr_volume* vol, float* h_min, float* h_max);
/* Histogram of the cube's voxels (the data range — and with it the colour map and the threshold
 *     of a noise-suppressing table, PAPER.md:294 — is chosen from the data).  n_bins (1..4096) equal bins over
 *     [lo, hi): bin = floor((v - lo) * (n_bins / (hi - lo))) evaluated in float32, values outside the range are
 *     counted in the first / last bin, NaN voxels only in *h_nan (may be NULL).  h_counts: HOST, n_bins entries.
 *     One streaming pass over the tiled copy; synchronises.  INVALID_ARG: NULL, n_bins out of range, lo >= hi.     */
vr_status vr_volume_histogram(vr_volume* vol, int n_bins, float lo, float hi, long long* h_counts, long long* h_nan);
/* The same histogram for callers that must not allocate device memory: same arguments, same counts, bit for bit.
 *     Who needs it: (1) an application whose own allocator (PyTorch's caching allocator, an RMM pool) already owns
 *     nearly all of the GPU — usual once a cube of tens of GB is resident — where a cudaMalloc made behind its back by
 *     this library fails with "out of memory" although the application has free blocks; (2) a viewer with frames in
 *     flight on other streams: vr_volume_histogram frees its bins with cudaFree, which waits for the WHOLE device, so
 *     a histogram asked for while the user drags the data range would stall the frames.  This call makes no
 *     cudaMalloc / cudaFree and calls nothing that allocates: its bins are a fixed array inside the library image.
 *     Cost and limit: every GPU that loads libvr_b200.so holds that array — 4097 x 8 = 32 776 bytes — until the
 *     process ends, whether this call is used or not, and n_bins beyond 4096 is refused (INVALID_ARG, message names
 *     the limit); the array cannot grow.
 *     The volume's GPU must be the current device (STATE otherwise): the array exists once per GPU.  The first call
 *     on each GPU looks up the array's device address (cudaGetSymbolAddress) and remembers it; make that first call
 *     outside any stream capture.  All calls on one GPU share the array.  Each call clears the part it uses first, so
 *     what an earlier call left behind does not matter, but two calls that overlap on the GPU (two host threads, two
 *     volumes on different streams) count into the same bins and both results are garbage: the library takes no
 *     lock — serialise such calls yourself.  Like vr_volume_histogram it waits for the volume's stream before
 *     returning.  h_counts: HOST, n_bins entries; h_nan may be NULL.                                              */
vr_status vr_volume_histogram_noalloc(vr_volume* vol, int n_bins, float lo, float hi, long long* h_counts,
                                      long long* h_nan);
const char* vr_last_error(void); /* thread-local, never NULL */

#ifdef __cplusplus
}
#endif
#endif /* VR_H */
