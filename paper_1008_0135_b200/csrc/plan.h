// plan.h — host-side per-frame planning of the CUDA path (double precision, no device code).
//
// Steps a1 (camera -> ray basis), a2 (rendering rectangle per brick), a6 (brick
// depth order, implied by PAPER.md:156-161) of DESIGN.md's hot-path table.  Formulas are the
// readings O1, O9, A10, A11, A12 of DESIGN.md.  Independent of oracle/ (no shared code).
#pragma once
#include <algorithm>
#include <cmath>
#include <vector>

#include "../../include/vr.h"

namespace vr {

struct Basis {            // O1: unit vectors and eye position in voxel space
    double right[3], up[3], fwd[3], eye[3];
};

struct BrickPlan {
    int lo[3], hi[3];     // brick box in voxels, faces at floor(m*n/b)  (O9/A10)
    int rx0, ry0, rw, rh; // rendering rectangle in pixels (A12); rw == 0 -> nothing to draw
    int key;              // depth key (A11): ascending = front to back
};

inline void normalize3(double v[3]) {
    double l = std::sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
    v[0] /= l; v[1] /= l; v[2] /= l;
}

// O1: right/up/fwd = rows 0, 1, -2 of the rotation part, re-normalised; eye = -R^T tau.
inline Basis make_basis(const vr_camera& cam) {
    Basis b;
    double R[3][3], tau[3];
    for (int r = 0; r < 3; ++r) {
        for (int c = 0; c < 3; ++c) R[r][c] = (double)cam.view[4 * r + c];
        tau[r] = (double)cam.view[4 * r + 3];
    }
    for (int c = 0; c < 3; ++c) {
        b.right[c] = R[0][c];
        b.up[c] = R[1][c];
        b.fwd[c] = -R[2][c];
        b.eye[c] = -(R[0][c] * tau[0] + R[1][c] * tau[1] + R[2][c] * tau[2]);
    }
    normalize3(b.right); normalize3(b.up); normalize3(b.fwd);
    return b;
}

// Returns nullptr if the camera is acceptable, else the reason.
inline const char* check_camera(const vr_camera& cam) {
    for (int i = 0; i < 16; ++i)
        if (!std::isfinite(cam.view[i])) return "camera: view has a non-finite entry";
    for (int r = 0; r < 3; ++r)
        for (int s = r; s < 3; ++s) {
            double dot = 0.0;
            for (int c = 0; c < 3; ++c) dot += (double)cam.view[4 * r + c] * (double)cam.view[4 * s + c];
            if (std::fabs(dot - (r == s ? 1.0 : 0.0)) > 1e-4)
                return "camera: upper-left 3x3 of view is not orthonormal within 1e-4";
        }
    if (cam.projection == VR_PROJ_PERSP) {
        if (!(cam.fovy_deg > 0.0f && cam.fovy_deg < 180.0f)) return "camera: fovy_deg must be in (0,180)";
    } else if (cam.projection == VR_PROJ_ORTHO) {
        if (!(cam.ortho_half_h > 0.0f) || !std::isfinite(cam.ortho_half_h))
            return "camera: ortho_half_h must be positive and finite";
    } else {
        return "camera: unknown projection";
    }
    return nullptr;
}

inline double tan_half_fov(const vr_camera& cam) {
    const double kPi = 3.14159265358979323846;
    return std::tan(0.5 * (double)cam.fovy_deg * (kPi / 180.0));
}

// A10: P_a[m] = floor(m*n_a/b_a)
inline int brick_face(int m, int n, int b) { return (int)(((long long)m * n) / b); }

// a2 + a6 for every brick; order[k] = k-th brick front to back.
// sub_lo/sub_hi (may be null): sub-cube every brick box is intersected with (S1).
inline void plan_bricks(const int dims[3], const int bricks[3], const vr_camera& cam, int W, int H,
                        std::vector<BrickPlan>& plan, std::vector<int>& order, const int* sub_lo = nullptr,
                        const int* sub_hi = nullptr) {
    const Basis bs = make_basis(cam);
    const bool persp = cam.projection == VR_PROJ_PERSP;
    const double asp = (double)W / (double)H;
    const double h = (double)cam.ortho_half_h;
    const double T = persp ? tan_half_fov(cam) : 0.0;
    const int B = bricks[0] * bricks[1] * bricks[2];
    plan.assign(B, BrickPlan());
    order.resize(B);

    // A11 (PERSP): index of the slab that holds the eye, -1 / b_a when outside the volume
    int eslab[3] = {0, 0, 0};
    for (int a = 0; a < 3; ++a) {
        if (bs.eye[a] < 0.0) eslab[a] = -1;
        else if (bs.eye[a] >= (double)dims[a]) eslab[a] = bricks[a];
        else {
            int m = 0;
            while (m + 1 < bricks[a] && (double)brick_face(m + 1, dims[a], bricks[a]) <= bs.eye[a]) ++m;
            eslab[a] = m;
        }
    }
    const double diag = std::sqrt((double)dims[0] * dims[0] + (double)dims[1] * dims[1] +
                                  (double)dims[2] * dims[2]);
    for (int bk = 0; bk < bricks[2]; ++bk)
        for (int bj = 0; bj < bricks[1]; ++bj)
            for (int bi = 0; bi < bricks[0]; ++bi) {
                const int idx[3] = {bi, bj, bk};
                BrickPlan& p = plan[(bk * bricks[1] + bj) * bricks[0] + bi];
                p.key = 0;
                for (int a = 0; a < 3; ++a) {
                    p.lo[a] = brick_face(idx[a], dims[a], bricks[a]);
                    p.hi[a] = brick_face(idx[a] + 1, dims[a], bricks[a]);
                    if (sub_lo && sub_hi) {            // S1: only the part of the brick inside the sub-cube
                        p.lo[a] = std::max(p.lo[a], sub_lo[a]);
                        p.hi[a] = std::min(p.hi[a], sub_hi[a]);
                    }
                    if (persp) p.key += std::abs(idx[a] - eslab[a]);
                    else p.key += (bs.fwd[a] >= 0.0) ? idx[a] : bricks[a] - 1 - idx[a];
                }
                // A12: bounding rectangle of the 8 projected corners (+1 pixel of slack), in
                // continuous pixel coordinates where pixel px covers [px, px+1).
                double xmin = 1e300, xmax = -1e300, ymin = 1e300, ymax = -1e300;
                bool full = false;
                if (p.hi[0] <= p.lo[0] || p.hi[1] <= p.lo[1] || p.hi[2] <= p.lo[2]) {   // empty after S1
                    p.rx0 = p.ry0 = p.rw = p.rh = 0;
                    continue;
                }
                for (int c = 0; c < 8 && !full; ++c) {
                    double rel[3];
                    for (int a = 0; a < 3; ++a)
                        rel[a] = (double)(((c >> a) & 1) ? p.hi[a] : p.lo[a]) - bs.eye[a];
                    double xe = rel[0] * bs.right[0] + rel[1] * bs.right[1] + rel[2] * bs.right[2];
                    double ye = rel[0] * bs.up[0] + rel[1] * bs.up[1] + rel[2] * bs.up[2];
                    double u, v;
                    if (persp) {
                        double depth = rel[0] * bs.fwd[0] + rel[1] * bs.fwd[1] + rel[2] * bs.fwd[2];
                        if (!(depth > 1e-6 * diag)) { full = true; break; }
                        u = xe / (depth * T * asp);
                        v = ye / (depth * T);
                    } else {
                        u = xe / (h * asp);
                        v = ye / h;
                    }
                    double fx = (u + 1.0) * 0.5 * (double)W, fy = (v + 1.0) * 0.5 * (double)H;
                    xmin = std::min(xmin, fx); xmax = std::max(xmax, fx);
                    ymin = std::min(ymin, fy); ymax = std::max(ymax, fy);
                }
                int x0 = 0, y0 = 0, x1 = W, y1 = H;
                if (!full) {
                    auto lo_px = [](double f, int n) {
                        double g = std::floor(f) - 1.0;
                        return (int)std::min(std::max(g, 0.0), (double)n);
                    };
                    auto hi_px = [](double f, int n) {
                        double g = std::ceil(f) + 1.0;
                        return (int)std::min(std::max(g, 0.0), (double)n);
                    };
                    x0 = lo_px(xmin, W); x1 = hi_px(xmax, W);
                    y0 = lo_px(ymin, H); y1 = hi_px(ymax, H);
                }
                if (x1 <= x0 || y1 <= y0) { p.rx0 = p.ry0 = p.rw = p.rh = 0; }
                else { p.rx0 = x0; p.ry0 = y0; p.rw = x1 - x0; p.rh = y1 - y0; }
            }
    for (int b = 0; b < B; ++b) order[b] = b;
    std::stable_sort(order.begin(), order.end(),
                     [&](int a, int b) { return plan[a].key < plan[b].key; });
}

}  // namespace vr
