/* oracle/vro.c — CPU oracle for the ray-casting volume renderer.  TEST INFRASTRUCTURE.
 *
 * Written from /root/reference/PAPER.md (Hassan, Fluke & Barnes, "Interactive Visualization of
 * the Largest Radioastronomy Cubes") and the readings O1-O11 listed in DESIGN.md.  The paper
 * gives the outline of the method (PAPER.md:80 ray casting with a transfer function and
 * accumulation of colour and opacity; PAPER.md:142 object-based partitioning
 * ray/box test, entry/exit points, sampling distance, early ray termination, MIP;
 * PAPER.md:156-161 image composition, associativity) and no formulas, so every formula below
 * is a DESIGN.md reading and is named by its rule number.
 *
 * Everything is double precision; cube and table values are read as stored float32.  No
 * blocking, no reordering, no shared code with the CUDA path.  Build: see oracle/build.py
 * (gcc -O2 -ffp-contract=off -fopenmp).
 *
 * Pins (tests/test_oracle_*.py, all -m "not gpu"): constant cube closed form, axis-aligned MIP
 * = max over an axis, axis-aligned EA = 1-D cumprod recurrence, continuous-limit integral of a
 * ramp, trilinear identities, brute force on tiny cubes, bricked = unbricked, symmetries; and, in
 * tests/test_oracle_branches.py, the three branches a mutant once survived: the t_near >= 0 clamp (eye
 * inside the box, box behind the eye), the d_a == 0 half-open containment rule (rays lying exactly on a
 * face or brick plane) and the termination point (exact sample count of a terminated ray).
 * General oblique / perspective views of noisy cubes: PARITY UNPINNED beyond those invariants
 * (the oracle is the definition there) — stated in DESIGN.md as well.
 */
#include "vro.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* ---------------------------------------------------------------- O1 basis ---------------- */
static void normalize3(double v[3]) {
    double l = sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
    v[0] /= l; v[1] /= l; v[2] /= l;
}

void vro_basis(const vro_camera* cam, double right[3], double up[3], double fwd[3], double eye[3]) {
    double R[3][3], tau[3];
    for (int r = 0; r < 3; ++r) {
        for (int c = 0; c < 3; ++c) R[r][c] = (double)cam->view[4 * r + c];
        tau[r] = (double)cam->view[4 * r + 3];
    }
    for (int c = 0; c < 3; ++c) {
        right[c] = R[0][c];
        up[c] = R[1][c];
        fwd[c] = -R[2][c];
    }
    normalize3(right); normalize3(up); normalize3(fwd);
    /* eye = -R^T tau : the point that the view matrix maps to the origin of eye space */
    for (int c = 0; c < 3; ++c) eye[c] = -(R[0][c] * tau[0] + R[1][c] * tau[1] + R[2][c] * tau[2]);
}

/* ---------------------------------------------------------------- O2 ray ------------------ */
void vro_ray(const vro_camera* cam, int W, int H, int px, int py, double o[3], double d[3]) {
    double right[3], up[3], fwd[3], eye[3];
    vro_basis(cam, right, up, fwd, eye);
    double u = 2.0 * ((double)px + 0.5) / (double)W - 1.0;
    double v = 2.0 * ((double)py + 0.5) / (double)H - 1.0;
    double asp = (double)W / (double)H;
    if (cam->projection == 0) {
        double h = (double)cam->ortho_half_h;
        for (int c = 0; c < 3; ++c) {
            o[c] = eye[c] + u * h * asp * right[c] + v * h * up[c];
            d[c] = fwd[c];
        }
    } else {
        double T = tan(0.5 * (double)cam->fovy_deg * (M_PI / 180.0));
        for (int c = 0; c < 3; ++c) {
            o[c] = eye[c];
            d[c] = fwd[c] + u * T * asp * right[c] + v * T * up[c];
        }
        normalize3(d);
    }
}

/* ---------------------------------------------------------------- O3 slab clip ------------ */
int vro_slab(const double o[3], const double d[3], const double lo[3], const double hi[3],
             double* t0_out, double* t1_out) {
    double tn = -INFINITY, tf = INFINITY;
    for (int a = 0; a < 3; ++a) {
        if (d[a] == 0.0) {
            if (!(lo[a] <= o[a] && o[a] < hi[a])) return 0;
        } else {
            double t0 = (lo[a] - o[a]) / d[a];
            double t1 = (hi[a] - o[a]) / d[a];
            double tmin = t0 < t1 ? t0 : t1;
            double tmax = t0 < t1 ? t1 : t0;
            if (tmin > tn) tn = tmin;
            if (tmax < tf) tf = tmax;
        }
    }
    *t0_out = tn;
    *t1_out = tf;
    return 1;
}

/* ---------------------------------------------------------------- O4 lattice -------------- */
/* I(t) = max(0, ceil((t - t_near)/step - 1/2)): index of the first lattice sample at or after t */
static long long lattice_index(double t, double t_near, double step) {
    double x = ceil((t - t_near) / step - 0.5);
    if (!(x > 0.0)) return 0;
    return (long long)x;
}

long long vro_ray_extent(const double o[3], const double d[3], const int dims[3], double step,
                         double* t_near, double* t_far) {
    double lo[3] = {0.0, 0.0, 0.0};
    double hi[3] = {(double)dims[0], (double)dims[1], (double)dims[2]};
    double tn, tf;
    *t_near = 0.0;
    *t_far = 0.0;
    if (!vro_slab(o, d, lo, hi, &tn, &tf)) return 0;
    if (tn < 0.0) tn = 0.0;
    if (!(tf > tn)) return 0;
    *t_near = tn;
    *t_far = tf;
    return lattice_index(tf, tn, step);
}

/* ---------------------------------------------------------------- O5 sample --------------- */
double vro_sample(const float* data, const int dims[3], const double p[3]) {
    long long i0[3], i1[3];
    double f[3];
    for (int a = 0; a < 3; ++a) {
        double q = p[a] - 0.5;
        double qmax = (double)(dims[a] - 1);
        if (q < 0.0) q = 0.0;
        if (q > qmax) q = qmax;
        double fl = floor(q);
        i0[a] = (long long)fl;
        i1[a] = i0[a] + 1 < dims[a] ? i0[a] + 1 : dims[a] - 1;
        f[a] = q - fl;
    }
    long long nx = dims[0], ny = dims[1];
    double acc = 0.0;
    for (int cz = 0; cz < 2; ++cz)
        for (int cy = 0; cy < 2; ++cy)
            for (int cx = 0; cx < 2; ++cx) {
                long long x = cx ? i1[0] : i0[0];
                long long y = cy ? i1[1] : i0[1];
                long long z = cz ? i1[2] : i0[2];
                double w = (cx ? f[0] : 1.0 - f[0]) * (cy ? f[1] : 1.0 - f[1]) *
                           (cz ? f[2] : 1.0 - f[2]);
                acc += w * (double)data[(z * ny + y) * nx + x];
            }
    return acc;
}

/* ---------------------------------------------------------------- O6 classify ------------- */
static void lookup(const double tab[256][4], double vmin, double vmax, double value,
                   double out[4]) {
    double s = (value - vmin) / (vmax - vmin);
    if (s < 0.0) s = 0.0;
    if (s > 1.0) s = 1.0;
    double x = 255.0 * s;
    double fl = floor(x);
    int m = (int)fl;
    if (m > 254) m = 254;
    double w = x - (double)m;
    for (int c = 0; c < 4; ++c) out[c] = (1.0 - w) * tab[m][c] + w * tab[m + 1][c];
}

/* table with alpha corrected per entry for the step: a -> 1 - (1-a)^step (step 1: unchanged) */
static void corrected_table(const float rgba[1024], double step, double tab[256][4]) {
    for (int j = 0; j < 256; ++j) {
        tab[j][0] = (double)rgba[4 * j + 0];
        tab[j][1] = (double)rgba[4 * j + 1];
        tab[j][2] = (double)rgba[4 * j + 2];
        double a = (double)rgba[4 * j + 3];
        tab[j][3] = (step == 1.0) ? a : 1.0 - pow(1.0 - a, step);
    }
}

void vro_classify(const float rgba[1024], double vmin, double vmax, double step, double value,
                  double out[4]) {
    double tab[256][4];
    corrected_table(rgba, step, tab);
    lookup(tab, vmin, vmax, value, out);
}

/* ---------------------------------------------------------------- O9 brick span ----------- */
static void brick_box(const int dims[3], const int bricks[3], const int idx[3], double lo[3],
                      double hi[3]) {
    for (int a = 0; a < 3; ++a) {
        long long n = dims[a], b = bricks[a];
        lo[a] = (double)(((long long)idx[a] * n) / b);
        hi[a] = (double)((((long long)idx[a] + 1) * n) / b);
    }
}

/* O9 for an explicit box [lo,hi] (voxel units): owned range of the global lattice. */
static int box_span(const double o[3], const double d[3], const double lo[3], const double hi[3], double step,
                    double t_near, double t_far, double* t_in, long long* i_lo, long long* i_hi) {
    double t0, t1;
    *t_in = 0.0; *i_lo = 0; *i_hi = 0;
    for (int a = 0; a < 3; ++a) if (!(hi[a] > lo[a])) return 0;
    if (!vro_slab(o, d, lo, hi, &t0, &t1)) return 0;
    if (t0 < t_near) t0 = t_near;
    if (t1 > t_far) t1 = t_far;
    if (!(t1 > t0)) return 0;
    *t_in = t0;
    *i_lo = lattice_index(t0, t_near, step);
    *i_hi = lattice_index(t1, t_near, step);
    return *i_hi > *i_lo;
}

/* O9 for brick (bi,bj,bk) of the regular grid: its box, then box_span — the same code the renderer runs
 * (route 1 below calls brick_box + box_span), so pins on this function pin the rendering path. */
int vro_brick_span(const double o[3], const double d[3], const int dims[3], const int bricks[3],
                   int bi, int bj, int bk, double step, double t_near, double t_far,
                   double* t_in, long long* i_lo, long long* i_hi) {
    int idx[3] = {bi, bj, bk};
    double lo[3], hi[3];
    brick_box(dims, bricks, idx, lo, hi);
    return box_span(o, d, lo, hi, step, t_near, t_far, t_in, i_lo, i_hi);
}

/* ---------------------------------------------------------------- O5-O8 sample loop ------- */
typedef struct {
    double C[3]; /* EA: accumulated premultiplied colour */
    double A;    /* EA: accumulated opacity              */
    double M;    /* MIP: running maximum, -inf initially */
} accum;

static void accum_reset(accum* acc) {
    acc->C[0] = acc->C[1] = acc->C[2] = 0.0;
    acc->A = 0.0;
    acc->M = -INFINITY;
}

/* samples i_lo <= i < i_hi of the global lattice t_i = t_near + (i + 1/2) step (O4), continuing the accumulation
 * in *acc; returns the number of samples taken and sets *terminated when O7 stopped the ray */
static long long march(const float* data, const int dims[3], const double tab[256][4], double vmin,
                       double vmax, const double o[3], const double d[3], double t_near,
                       double step, long long i_lo, long long i_hi, int mode, double ert,
                       accum* acc, int* terminated) {
    long long count = 0;
    int ert_on = (ert > 0.0 && ert < 1.0);
    for (long long i = i_lo; i < i_hi; ++i) {
        double t = t_near + ((double)i + 0.5) * step;
        double p[3] = {o[0] + t * d[0], o[1] + t * d[1], o[2] + t * d[2]};
        double value = vro_sample(data, dims, p);
        ++count;
        if (isnan(value)) continue; /* O5/A14: blanked voxels are skipped */
        if (mode == VRO_MODE_MIP) {
            if (value > acc->M) acc->M = value; /* O8 */
        } else {
            double e[4];
            lookup(tab, vmin, vmax, value, e); /* O6 */
            double wgt = (1.0 - acc->A) * e[3]; /* O7 front-to-back "over" */
            acc->C[0] += wgt * e[0];
            acc->C[1] += wgt * e[1];
            acc->C[2] += wgt * e[2];
            acc->A += wgt;
            if (ert_on && acc->A >= ert) { *terminated = 1; break; }
        }
    }
    return count;
}

/* S2 channel mask ("enabling/disabling spectral channel(s)"): the enabled channels form maximal runs
 * [za, zb) of consecutive channels; a lattice sample is taken iff it is owned, by O9's rule, by the slab
 * [za, zb] of some run (intersected with the box it is rendered in).  One run [0, nz) = no mask. */
typedef struct { int za, zb; } zrun;
typedef struct { double t_in; long long lo, hi; } span;
static int cmp_span(const void* x, const void* y) {
    const span* a = (const span*)x;
    const span* b = (const span*)y;
    return (a->lo > b->lo) - (a->lo < b->lo);
}

/* All samples of the lattice inside box [lo,hi] AND an enabled run, front to back, accumulated into *acc (reset
 * here).  Returns samples taken; *t_first = entry parameter of the first non-empty span (sort key of O10);
 * *any = 1 if at least one sample range was non-empty. */
static long long march_box(const float* data, const int dims[3], const double tab[256][4], double vmin, double vmax,
                           const double o[3], const double d[3], double t_near, double t_far, double step,
                           const double lo[3], const double hi[3], const zrun* runs, int n_runs, span* work,
                           int mode, double ert, accum* acc, double* t_first, int* any) {
    int ns = 0;
    for (int r = 0; r < n_runs; ++r) {
        double blo[3] = {lo[0], lo[1], lo[2]}, bhi[3] = {hi[0], hi[1], hi[2]};
        if (blo[2] < (double)runs[r].za) blo[2] = (double)runs[r].za;
        if (bhi[2] > (double)runs[r].zb) bhi[2] = (double)runs[r].zb;
        if (box_span(o, d, blo, bhi, step, t_near, t_far, &work[ns].t_in, &work[ns].lo, &work[ns].hi)) ++ns;
    }
    qsort(work, (size_t)ns, sizeof(span), cmp_span);
    accum_reset(acc);
    *any = ns > 0;
    *t_first = ns > 0 ? work[0].t_in : 0.0;
    long long count = 0;
    int terminated = 0;
    for (int k = 0; k < ns && !terminated; ++k)
        count += march(data, dims, tab, vmin, vmax, o, d, t_near, step, work[k].lo, work[k].hi, mode, ert, acc,
                       &terminated);
    return count;
}

typedef struct { double t_in; int b; } brick_key;
static int cmp_key(const void* x, const void* y) {
    const brick_key* a = (const brick_key*)x;
    const brick_key* b = (const brick_key*)y;
    if (a->t_in < b->t_in) return -1;
    if (a->t_in > b->t_in) return 1;
    return a->b - b->b;
}

/* ---------------------------------------------------------------- O1-O11 pixels ----------- */
int vro_render_pixels_mask(const float* data, const int dims[3], const float rgba[1024], float vmin_f,
                           float vmax_f, const int bricks_in[3], const int sub_lo[3], const int sub_hi[3],
                           const unsigned char* chan_mask, const vro_camera* cam, int W, int H, float step_f, int mode,
                           float ert_f, int route, long long n_pix, const int* px, const int* py, float* out_rgba,
                           float* out_scalar, float* out_brick, long long* out_samples, int threads) {
    if (!data || !dims || !rgba || !cam || !out_rgba || n_pix < 0) return -1;
    /* S1 sub-cube ("a manual sub-cube", PAPER.md:138 channel enable/disable): only samples of the
     * global lattice that lie in [sub_lo, sub_hi) are taken; the lattice itself (O4) and the sampling (O5, whole
     * cube) are unchanged, i.e. the sub-cube acts as one more box every brick is intersected with. */
    int slo[3] = {0, 0, 0}, shi[3] = {dims[0], dims[1], dims[2]};
    if (sub_lo && sub_hi)
        for (int a = 0; a < 3; ++a) {
            if (sub_lo[a] < 0 || sub_hi[a] > dims[a] || sub_hi[a] < sub_lo[a]) return -1;
            slo[a] = sub_lo[a]; shi[a] = sub_hi[a];
        }
    const int has_sub = (sub_lo && sub_hi);
    if (dims[0] <= 0 || dims[1] <= 0 || dims[2] <= 0 || W <= 0 || H <= 0) return -1;
    if (!(step_f > 0.0f) || !(vmax_f > vmin_f)) return -1;
    if (mode != VRO_MODE_EA && mode != VRO_MODE_MIP) return -1;
    if (route != 0 && route != 1) return -1;
    int bricks[3] = {1, 1, 1};
    if (bricks_in) { bricks[0] = bricks_in[0]; bricks[1] = bricks_in[1]; bricks[2] = bricks_in[2]; }
    for (int a = 0; a < 3; ++a) if (bricks[a] < 1 || bricks[a] > dims[a]) return -1;
    const int B = bricks[0] * bricks[1] * bricks[2];
    const double step = (double)step_f, vmin = (double)vmin_f, vmax = (double)vmax_f;
    const double ert = (double)ert_f;

    /* O6: per-step table for EA; O8: the uncorrected table colours the MIP result */
    double (*tabs)[4] = malloc(sizeof(double) * 256 * 4 * 2);
    if (!tabs) return -1;
    double (*tstep)[4] = tabs, (*traw)[4] = tabs + 256;
    corrected_table(rgba, step, tstep);
    corrected_table(rgba, 1.0, traw);

    /* S2: maximal runs of enabled channels (no mask: the single run [0, nz)) */
    zrun* runs = malloc(sizeof(zrun) * (size_t)(dims[2] / 2 + 2));
    if (!runs) { free(tabs); return -1; }
    int n_runs = 0;
    if (!chan_mask) {
        runs[0].za = 0; runs[0].zb = dims[2]; n_runs = 1;
    } else {
        for (int z = 0; z < dims[2];) {
            if (!chan_mask[z]) { ++z; continue; }
            int z1 = z;
            while (z1 < dims[2] && chan_mask[z1]) ++z1;
            runs[n_runs].za = z; runs[n_runs].zb = z1; ++n_runs;
            z = z1;
        }
    }
    const int plain = (!chan_mask && !has_sub);   /* route 0 then marches [0, n) directly, as O4 states it */

    long long total = 0;
#ifdef _OPENMP
    if (threads <= 0) threads = omp_get_max_threads();
#else
    threads = 1;
#endif
#pragma omp parallel for schedule(dynamic, 64) num_threads(threads) reduction(+ : total)
    for (long long k = 0; k < n_pix; ++k) {
        double o[3], d[3], t_near, t_far;
        vro_ray(cam, W, H, px[k], py[k], o, d);
        long long n = vro_ray_extent(o, d, dims, step, &t_near, &t_far);
        accum fin;
        fin.C[0] = fin.C[1] = fin.C[2] = 0.0; fin.A = 0.0; fin.M = -INFINITY;
        span work[n_runs > 0 ? n_runs : 1];
        if (route == 0) {
            if (plain) {
                int terminated = 0;
                if (n > 0)
                    total += march(data, dims, (const double(*)[4])tstep, vmin, vmax, o, d, t_near, step, 0, n, mode,
                                   ert, &fin, &terminated);
            } else if (n > 0) {                                /* S1 / S2: the sub-cube and the enabled runs */
                double blo[3] = {(double)slo[0], (double)slo[1], (double)slo[2]};
                double bhi[3] = {(double)shi[0], (double)shi[1], (double)shi[2]};
                double t_first; int any;
                total += march_box(data, dims, (const double(*)[4])tstep, vmin, vmax, o, d, t_near, t_far, step, blo,
                                   bhi, runs, n_runs, work, mode, ert, &fin, &t_first, &any);
            }
        } else {
            brick_key keys[B > 0 ? B : 1];
            accum parts[B > 0 ? B : 1];
            int nk = 0;
            for (int bk = 0; bk < bricks[2]; ++bk)
                for (int bj = 0; bj < bricks[1]; ++bj)
                    for (int bi = 0; bi < bricks[0]; ++bi) {
                        int b = (bk * bricks[1] + bj) * bricks[0] + bi;
                        accum* part = &parts[b];
                        accum_reset(part);
                        int idx3[3] = {bi, bj, bk};
                        double blo[3], bhi[3];
                        brick_box(dims, bricks, idx3, blo, bhi);
                        for (int a = 0; a < 3; ++a) {          /* S1: brick box intersected with the sub-cube */
                            if (blo[a] < (double)slo[a]) blo[a] = (double)slo[a];
                            if (bhi[a] > (double)shi[a]) bhi[a] = (double)shi[a];
                        }
                        if (n > 0) {
                            double t_first; int any;
                            total += march_box(data, dims, (const double(*)[4])tstep, vmin, vmax, o, d, t_near, t_far,
                                               step, blo, bhi, runs, n_runs, work, mode, ert, part, &t_first, &any);
                            if (any) { keys[nk].t_in = t_first; keys[nk].b = b; ++nk; }
                        }
                        if (out_brick) {
                            if (mode == VRO_MODE_MIP) {
                                out_brick[(long long)b * n_pix + k] = (float)part->M;
                            } else {
                                float* ob = out_brick + ((long long)b * n_pix + k) * 4;
                                ob[0] = (float)part->C[0]; ob[1] = (float)part->C[1];
                                ob[2] = (float)part->C[2]; ob[3] = (float)part->A;
                            }
                        }
                    }
            /* O10: per-pixel visibility order = ascending t_in; then "over" */
            qsort(keys, (size_t)nk, sizeof(brick_key), cmp_key);
            double T = 1.0; /* transparency of everything in front */
            for (int j = 0; j < nk; ++j) {
                const accum* part = &parts[keys[j].b];
                if (mode == VRO_MODE_MIP) {
                    if (part->M > fin.M) fin.M = part->M;
                } else {
                    fin.C[0] += T * part->C[0];
                    fin.C[1] += T * part->C[1];
                    fin.C[2] += T * part->C[2];
                    T *= (1.0 - part->A);
                }
            }
            if (mode == VRO_MODE_EA) fin.A = 1.0 - T;
        }
        /* O11 / O8 output */
        float* op = out_rgba + 4 * k;
        if (mode == VRO_MODE_MIP) {
            if (out_scalar) out_scalar[k] = (float)fin.M;
            if (fin.M == -INFINITY) {
                op[0] = op[1] = op[2] = op[3] = 0.0f;
            } else {
                double e[4];
                lookup((const double(*)[4])traw, vmin, vmax, fin.M, e);
                op[0] = (float)e[0]; op[1] = (float)e[1]; op[2] = (float)e[2]; op[3] = (float)e[3];
            }
        } else {
            op[0] = (float)fin.C[0]; op[1] = (float)fin.C[1]; op[2] = (float)fin.C[2];
            op[3] = (float)fin.A;
        }
    }
    free(tabs);
    free(runs);
    if (out_samples) *out_samples = total;
    return 0;
}

int vro_render_pixels_sub(const float* data, const int dims[3], const float rgba[1024], float vmin,
                          float vmax, const int bricks[3], const int sub_lo[3], const int sub_hi[3],
                          const vro_camera* cam, int W, int H, float step, int mode, float ert_alpha, int route,
                          long long n_pix, const int* px, const int* py, float* out_rgba, float* out_scalar,
                          float* out_brick, long long* out_samples, int threads) {
    return vro_render_pixels_mask(data, dims, rgba, vmin, vmax, bricks, sub_lo, sub_hi, NULL, cam, W, H, step, mode,
                                  ert_alpha, route, n_pix, px, py, out_rgba, out_scalar, out_brick, out_samples,
                                  threads);
}

int vro_render_pixels(const float* data, const int dims[3], const float rgba[1024], float vmin,
                      float vmax, const int bricks[3], const vro_camera* cam, int W, int H, float step, int mode,
                      float ert_alpha, int route, long long n_pix, const int* px, const int* py, float* out_rgba,
                      float* out_scalar, float* out_brick, long long* out_samples, int threads) {
    return vro_render_pixels_sub(data, dims, rgba, vmin, vmax, bricks, NULL, NULL, cam, W, H, step, mode, ert_alpha,
                                 route, n_pix, px, py, out_rgba, out_scalar, out_brick, out_samples, threads);
}

int vro_render(const float* data, const int dims[3], const float rgba[1024], float vmin,
               float vmax, const int bricks[3], const vro_camera* cam, int W, int H, float step,
               int mode, float ert_alpha, int route, float* out_rgba, float* out_scalar,
               float* out_brick, long long* out_samples, int threads) {
    if (W <= 0 || H <= 0) return -1;
    long long n_pix = (long long)W * H;
    int* px = malloc(sizeof(int) * (size_t)n_pix);
    int* py = malloc(sizeof(int) * (size_t)n_pix);
    if (!px || !py) { free(px); free(py); return -1; }
    for (int y = 0; y < H; ++y)
        for (int x = 0; x < W; ++x) {
            px[(long long)y * W + x] = x;
            py[(long long)y * W + x] = y;
        }
    int rc = vro_render_pixels(data, dims, rgba, vmin, vmax, bricks, cam, W, H, step, mode,
                               ert_alpha, route, n_pix, px, py, out_rgba, out_scalar, out_brick,
                               out_samples, threads);
    free(px); free(py);
    return rc;
}

int vro_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
