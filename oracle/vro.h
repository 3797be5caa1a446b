/* oracle/vro.h — declarations of the CPU oracle (TEST INFRASTRUCTURE, not the product).
 *
 * A plain, slow, double-precision ray caster written from the paper
 * (/root/reference/PAPER.md, Hassan, Fluke & Barnes) and the readings O1-O11 /
 * A1-A16 recorded in DESIGN.md ("Readings of the paper").  It shares no code,
 * header, table or helper with the CUDA path under paper_1008_0135_b200/csrc:
 * this header re-declares its own camera struct on purpose.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may load this library.
 *
 * All pointers are HOST pointers.  The cube is float32, x fastest:
 * data[(z*ny + y)*nx + x]  ("regular, scalar 3D data lattice";
 * PAPER.md:40 4-byte floats).
 */
#ifndef VRO_H
#define VRO_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct {
    float view[16];     /* row-major 4x4, voxel space -> eye space, rigid; eye looks down -z_eye   */
    int   projection;   /* 0 = orthographic, 1 = perspective                                       */
    float fovy_deg;     /* perspective: full vertical field of view                                */
    float ortho_half_h; /* orthographic: half height of the window in voxels (half width = *W/H)   */
} vro_camera;

enum { VRO_MODE_EA = 0, VRO_MODE_MIP = 1 };

/* O1  camera -> right, up, fwd (unit, double), eye.  PAPER.md:138 "transformation and projection
 *     matrices".                                                                                 */
void vro_basis(const vro_camera* cam, double right[3], double up[3], double fwd[3], double eye[3]);

/* O2  ray through the centre of pixel (px,py) of a WxH image (py = 0 is the bottom row).
 *     PAPER.md:80 "a ray originating at this pixel".                                             */
void vro_ray(const vro_camera* cam, int W, int H, int px, int py, double o[3], double d[3]);

/* O3  slab clip of the ray against the box [lo,hi]; returns 1 and [t0,t1] (t0 NOT yet clamped to
 *     >= 0) when the slabs overlap, else 0.  PAPER.md:150 "tested against the bounding cube ...
 *     entry and exit points are calculated".                                                     */
int vro_slab(const double o[3], const double d[3], const double lo[3], const double hi[3],
             double* t0, double* t1);

/* O3+O4  global clip and sample count: returns n (0 on a miss) and t_near / t_far.               */
long long vro_ray_extent(const double o[3], const double d[3], const int dims[3], double step,
                         double* t_near, double* t_far);

/* O5  clamp-to-edge trilinear sample of the cube at voxel-space point p (cell-centred values).  */
double vro_sample(const float* data, const int dims[3], const double p[3]);

/* O6  classification: value -> (r,g,b,a) through the 256-entry table over [vmin,vmax];
 *     alpha is opacity-corrected per entry for `step` (step = 1: table used as given).          */
void vro_classify(const float rgba[1024], double vmin, double vmax, double step, double value,
                  double out[4]);

/* O9  brick boundaries P_a[m] = floor(m*n_a/b_a); for brick (i,j,k) and one ray the owned sample
 *     range [i_lo,i_hi) of the global lattice and t_in.  Returns 1 if the range is non-empty.   */
int vro_brick_span(const double o[3], const double d[3], const int dims[3], const int bricks[3],
                   int bi, int bj, int bk, double step, double t_near, double t_far,
                   double* t_in, long long* i_lo, long long* i_hi);

/* O1-O11  render a list of pixels.
 *   route 0: unbricked (O1-O8).  route 1: per brick (O9) then per-pixel t_in-sorted "over" (O10).
 *   ert_alpha <= 0 or >= 1 disables early termination (O7); in route 1 it is per brick.
 *   out_rgba   [n_pix][4]        final pixel (EA premultiplied; MIP colour-mapped, un-premultiplied)
 *   out_scalar [n_pix] or NULL   MIP: raw maximum (-inf = no sample); EA: untouched
 *   out_brick  NULL or [B][n_pix][4] (EA: C_b,A_b) / [B][n_pix] (MIP: M_b), route 1 only,
 *              brick index b = (bk*by + bj)*bx + bi
 *   out_samples NULL or one counter: samples evaluated over all listed pixels
 *   threads <= 0: all available (OpenMP).  Returns 0, or -1 on invalid arguments.               */
int vro_render_pixels(const float* data, const int dims[3], const float rgba[1024], float vmin,
                      float vmax, const int bricks[3], const vro_camera* cam, int W, int H,
                      float step, int mode, float ert_alpha, int route, long long n_pix,
                      const int* px, const int* py, float* out_rgba, float* out_scalar,
                      float* out_brick, long long* out_samples, int threads);

/* S1  Same with a sub-cube [sub_lo, sub_hi) in voxels (NULL, NULL = the whole cube): only lattice samples inside
 *     it are taken (PAPER.md:128 manual sub-cube; PAPER.md:138 spectral channels enabled/disabled = a z range);
 *     lattice (O4) and sampling (O5) are unchanged, every brick box is intersected with the sub-cube.            */
int vro_render_pixels_sub(const float* data, const int dims[3], const float rgba[1024], float vmin,
                          float vmax, const int bricks[3], const int sub_lo[3], const int sub_hi[3],
                          const vro_camera* cam, int W, int H, float step, int mode, float ert_alpha, int route,
                          long long n_pix, const int* px, const int* py, float* out_rgba, float* out_scalar,
                          float* out_brick, long long* out_samples, int threads);

/* S2  Same with a spectral-channel mask ("enabling/disabling spectral channel(s)"): chan_mask[z] != 0
 *     enables channel z (NULL = all enabled).  The enabled channels form maximal runs [za, zb); a lattice sample is
 *     taken iff O9's ownership rule gives it to the slab [za, zb] of some run (intersected with the sub-cube and,
 *     in route 1, the brick): each run is one more box, so a mask with a single run equals the sub-cube
 *     {0,0,za}..{nx,ny,zb} of S1.  Lattice (O4) and sampling (O5, whole cube, all channels) are unchanged;
 *     accumulation runs front to back through the runs' sample ranges, termination (O7) as before.            */
int vro_render_pixels_mask(const float* data, const int dims[3], const float rgba[1024], float vmin,
                           float vmax, const int bricks[3], const int sub_lo[3], const int sub_hi[3],
                           const unsigned char* chan_mask, const vro_camera* cam, int W, int H, float step, int mode,
                           float ert_alpha, int route, long long n_pix, const int* px, const int* py, float* out_rgba,
                           float* out_scalar, float* out_brick, long long* out_samples, int threads);

/* Full frame: every pixel, row-major [py][px].  out_brick then is [B][H][W][4] / [B][H][W].      */
int vro_render(const float* data, const int dims[3], const float rgba[1024], float vmin,
               float vmax, const int bricks[3], const vro_camera* cam, int W, int H, float step,
               int mode, float ert_alpha, int route, float* out_rgba, float* out_scalar,
               float* out_brick, long long* out_samples, int threads);

int vro_max_threads(void);

#ifdef __cplusplus
}
#endif
#endif
