"""Pins for three branches of the oracle that no other CPU test reaches (round-1 review: a mutant of each
passed the whole suite).  Each test names the line of oracle/vro.c it pins and the mutant it kills.

  O3  t_near = max(t_near, 0)          vro_ray_extent       eye inside the volume / box partly behind the eye
  O3  d_a == 0: hit iff lo <= o_a < hi  vro_slab             axis-parallel rays lying exactly on a face / brick plane
  O7  stop when A >= ert AFTER the update   march            exact sample count of a terminated ray

Expected values come from closed forms, hand-written recurrences over the listed voxels and the library route
of tests/helpers.py — never from the oracle itself.
"""
import math

import numpy as np
import pytest

from paper_1008_0135_b200 import workloads as wl
from tests.helpers import independent_pixel, oracle_camera

RAMP = wl.tf_ramp(0.1)


def noisy_cube(dims, seed):
    g = np.random.default_rng(seed)
    nx, ny, nz = dims
    return (g.normal(size=(nz, ny, nx)) * 1.5 + 2.0).astype(np.float32)


def camera_at(eye, target, projection, fovy=60.0, half_h=4.0):
    return wl.CameraSpec(wl.look_at(eye, target), projection, fovy, half_h)


# ------------------------------------------------------------------ O3: t_near = max(t_near, 0) ------
@pytest.mark.parametrize("name,eye,target,proj", [
    ("persp_eye_inside", (4.3, 3.1, 5.2), (9.0, 5.0, 0.5), wl.PROJ_PERSP),
    ("persp_box_behind_the_eye", (-1.5, 3.0, 4.0), (-5.0, 3.3, 3.6), wl.PROJ_PERSP),  # looks AWAY from the box
    ("ortho_box_behind_the_plane", (12.0, 3.0, 4.0), (15.0, 3.3, 3.6), wl.PROJ_ORTHO),
    ("ortho_plane_inside", (5.1, 3.4, 4.2), (0.3, 2.0, 7.7), wl.PROJ_ORTHO),
])
def test_eye_inside_or_box_behind_the_eye(oracle, name, eye, target, proj):
    """vro.c `if (tn < 0.0) tn = 0.0;` — samples start AT the eye, never behind it.  Without the clamp the
    lattice would be anchored at the (negative) entry parameter and the ray would integrate what lies behind
    the camera: with the eye inside the box (t_near < 0 < t_far) the picture changes, and a box that lies wholly
    behind the eye (t_near < t_far < 0) would be drawn, point-mirrored, instead of an empty frame.  Every pixel against the library route (inverse view matrix, face-by-face box hits,
    map_coordinates, interp, cumprod), which clamps with max(t, 0) in its own words."""
    dims = (10, 7, 9)
    cube = noisy_cube(dims, 21)
    cs = camera_at(eye, target, proj)
    W, H = 12, 9
    for step in (1.0, 0.5):
        r = oracle.render(cube, RAMP, -3.0, 8.0, (1, 1, 1), oracle_camera(oracle, cs), W, H, step, 0, 0.0, route=0)
        n_total, n_behind = 0, 0
        for py in range(H):
            for px in range(W):
                want, _, n = independent_pixel(cube, RAMP, -3.0, 8.0, cs, W, H, step, 0, px, py)
                assert np.abs(r["rgba"][py, px] - want).max() < 2e-6, (name, step, px, py)
                n_total += n
                o, d = oracle.ray(oracle_camera(oracle, cs), W, H, px, py)
                hit, t0, t1 = oracle.slab(o, d, (0, 0, 0), dims)
                n_behind += bool(hit and t0 < 0.0 and t1 > t0)      # entry behind the eye: the clamp decides
        assert r["samples"] == n_total
        assert n_behind > 0.2 * W * H, "the camera does not exercise the clamp"
        if "behind" in name:                              # the whole box lies behind every ray: an empty frame
            assert n_total == 0 and not r["rgba"].any()
    # the bricked route clips every brick against the same clamped [t_near, t_far]
    rb = oracle.render(cube, RAMP, -3.0, 8.0, (2, 2, 2), oracle_camera(oracle, cs), W, H, 0.5, 0, 0.0, route=1)
    assert np.abs(rb["rgba"] - r["rgba"]).max() < 1e-6 and rb["samples"] == r["samples"]


def test_eye_inside_mip_sees_only_what_is_in_front(oracle):
    """Same clamp through MIP: a bright voxel BEHIND an eye that sits inside the cube must not be seen."""
    dims = (9, 9, 9)
    cube = np.zeros((9, 9, 9), dtype=np.float32)
    cube[4, 4, 1] = 7.0                                   # voxel (x=1, y=4, z=4): behind the eye below
    cs = camera_at((4.5, 4.5, 4.5), (8.5, 4.5, 4.5), wl.PROJ_PERSP, fovy=40.0)   # looks along +x
    r = oracle.render(cube, RAMP, -3.0, 8.0, (1, 1, 1), oracle_camera(oracle, cs), 8, 8, 0.5, 1, 0.0, route=0)
    assert r["scalar"].max() == 0.0
    cs2 = camera_at((4.5, 4.5, 4.5), (0.5, 4.5, 4.5), wl.PROJ_PERSP, fovy=40.0)  # looks along -x: now in front
    r2 = oracle.render(cube, RAMP, -3.0, 8.0, (1, 1, 1), oracle_camera(oracle, cs2), 8, 8, 0.5, 1, 0.0, route=0)
    assert r2["scalar"].max() > 3.0


# ------------------------------------------------------------------ O3: d_a == 0 containment ---------
def on_plane_camera(n, sign):
    """Orthographic view exactly along sign*z of an n^3 cube, one pixel per voxel column plus one ring, shifted
    by half a voxel in x so that the rays of pixel column px run at x = px - 1 EXACTLY (dyadic numbers: the
    products and sums below are exact in double, so o_x == 0, == n/2 and == n hold bit for bit).
    W = H = 2n, ortho_half_h = n: pixel pitch 1 voxel, centre of the window at x = n/2 + 1/2."""
    f = np.array([0.0, 0.0, float(sign)])
    u = np.array([0.0, 1.0, 0.0])
    r = np.cross(f, u)                                   # sign=-1: r = (+1,0,0)
    assert r[0] == 1.0 or r[0] == -1.0
    c = np.array([0.5 * n + 0.5 * r[0], 0.5 * n, 0.5 * n])   # window centre half a voxel along +right
    eye = c - f * (0.5 * n + 3.0)
    R = np.stack([r, u, -f])
    M = np.eye(4)
    M[:3, :3] = R
    M[:3, 3] = -R @ eye
    return wl.CameraSpec(M.astype(np.float32), wl.PROJ_ORTHO, 45.0, float(n)), 2 * n, 2 * n, r[0]


def column_recurrence(values, table, vmin, vmax):
    """Front-to-back emission-absorption over voxel values listed in the order the ray meets them (step 1,
    samples on voxel centres): the O6 lookup and O7 blend written out with numpy.interp."""
    xp = vmin + (vmax - vmin) * np.arange(256) / 255.0
    tab = np.asarray(table, dtype=np.float64)
    C, A = np.zeros(3), 0.0
    for v in values:
        e = np.array([np.interp(float(v), xp, tab[:, c]) for c in range(4)])
        C += (1.0 - A) * e[3] * e[:3]
        A += (1.0 - A) * e[3]
    return np.array([C[0], C[1], C[2], A])


def test_axis_parallel_rays_on_faces_and_brick_planes(oracle):
    """vro.c `if (!(lo[a] <= o[a] && o[a] < hi[a])) return 0;` — with d_x == 0 a ray lying exactly on the lower
    face x = 0 is INSIDE (it samples voxel column x = 0 with weight 1: q = clamp(-1/2) = 0), a ray lying exactly
    on the upper face x = n is OUTSIDE (pixel exactly zero), and a ray on the plane x = n/2 shared by two
    bricks belongs to the brick whose LOWER face it is.  The mutant `lo < o <= hi` flips all three."""
    n = 4
    g = np.random.default_rng(3)
    cube = (g.uniform(0.0, 8.0, size=(n, n, n))).astype(np.float32)
    cs, W, H, rsign = on_plane_camera(n, -1)             # looking down -z; right = +x
    assert rsign == 1.0
    cam = oracle_camera(oracle, cs)
    xs = {}
    for px in range(W):
        o, d = oracle.ray(cam, W, H, px, 0)
        assert d[0] == 0.0 and d[1] == 0.0 and d[2] == -1.0
        xs[px] = o[0]
    assert xs[1] == 0.0 and xs[1 + n // 2] == n / 2 and xs[1 + n] == float(n)     # exactly on the planes
    r1 = oracle.render(cube, RAMP, -3.0, 8.0, (1, 1, 1), cam, W, H, 1.0, 0, 0.0, route=0)
    rb = oracle.render(cube, RAMP, -3.0, 8.0, (2, 1, 1), cam, W, H, 1.0, 0, 0.0, route=1, want_bricks=True)
    rm = oracle.render(cube, RAMP, -3.0, 8.0, (2, 1, 1), cam, W, H, 1.0, 1, 0.0, route=1, want_bricks=True)
    for py in range(H):
        y = py + 0.5 - (0.5 * H - 0.5 * n)               # o_y of this pixel row (window centred on n/2)
        inside_y = 0.0 < y < n
        for px in range(W):
            x = px - 1.0
            got = r1["rgba"][py, px]
            if not inside_y or not (0.0 <= x < n):        # the half-open rule, written out
                assert (got == 0).all(), (px, py)
                assert (rb["rgba"][py, px] == 0).all() and np.isneginf(rm["scalar"][py, px])
                continue
            # the sample sits at q = (x - 1/2, y - 1/2, k): x integer -> blend of columns x-1 and x with weight 1/2,
            # except on the face x = 0 where the clamp gives column 0 alone; y - 1/2 is an integer: one row
            iy = int(round(y - 0.5))
            if x == 0.0:
                col = cube[::-1, iy, 0].astype(np.float64)
            else:
                col = 0.5 * (cube[::-1, iy, int(x) - 1].astype(np.float64) + cube[::-1, iy, int(x)])
            want = column_recurrence(col, RAMP, -3.0, 8.0)
            assert np.abs(got - want).max() < 2e-7, (px, py, got, want)
            assert np.abs(rb["rgba"][py, px] - want).max() < 2e-7
            # ownership: brick 0 = [0, n/2), brick 1 = [n/2, n): a ray ON x = n/2 is brick 1's
            owner = 0 if x < n / 2 else 1
            assert rb["bricks"][owner, py, px, 3] > 0 and (rb["bricks"][1 - owner, py, px] == 0).all(), (px, py)
            assert rm["bricks"][owner, py, px] == np.float32(col.max()) and np.isneginf(rm["bricks"][1 - owner, py, px])
    assert r1["samples"] == n * n * n and rb["samples"] == n * n * n       # n columns x n rows x n samples


def test_brick_span_on_shared_plane_partitions_the_lattice(oracle):
    """O9 through the exported span function (now the same code the renderer runs): for an axis-parallel ray on
    a brick plane and for an oblique ray, the owned ranges are contiguous, disjoint and sum to n."""
    dims, bricks = (8, 8, 8), (2, 2, 2)
    for o, d in [((4.0, 4.0, -3.0), (0.0, 0.0, 1.0)),         # on two brick planes at once
                 ((0.0, 2.5, 9.0), (0.0, 0.0, -1.0)),         # on the volume face x = 0
                 ((-1.0, 0.7, 0.2), (0.8, 0.36, 0.48))]:
        n, tn, tf = oracle.ray_extent(o, d, dims, 0.5)
        assert n > 0
        spans = []
        for bk in range(2):
            for bj in range(2):
                for bi in range(2):
                    ok, t_in, lo, hi = oracle.brick_span(o, d, dims, bricks, (bi, bj, bk), 0.5, tn, tf)
                    if ok:
                        spans.append((lo, hi, (bi, bj, bk)))
        spans.sort()
        assert spans[0][0] == 0 and spans[-1][1] == n
        for a, b in zip(spans, spans[1:]):
            assert a[1] == b[0]
        if d[0] == 0.0 and o[0] == 4.0:
            assert all(s[2][0] == 1 and s[2][1] == 1 for s in spans)          # the lower-face owners


# ------------------------------------------------------------------ O7: termination point ------------
@pytest.mark.parametrize("a,ert", [(0.05, 0.9), (0.2, 0.995), (0.5, 0.75)])
def test_terminated_ray_takes_exactly_the_closed_form_count(oracle, a, ert):
    """vro.c `if (ert_on && acc->A >= ert) break;` AFTER the update.  Constant cube, constant table alpha a,
    step 1: A_k = 1 - (1-a)^k, so the ray stops after n* = ceil(log(1-ert)/log(1-a)) samples with
    A = 1 - (1-a)^n*.  Testing before the update (one sample late) gives n* + 1 and a larger A."""
    n_star = math.ceil(math.log(1.0 - ert) / math.log(1.0 - a))
    assert 1.0 - (1.0 - a) ** (n_star - 1) < ert - 1e-6 < ert + 1e-6 < 1.0 - (1.0 - a) ** n_star + 1e-3
    depth = n_star + 9
    cube = np.full((depth, 3, 3), 1.0, dtype=np.float32)
    tab = np.zeros((256, 4), dtype=np.float32)
    tab[:, 0], tab[:, 3] = 1.0, a
    a32 = float(np.float32(a))
    cs, W, H, *_ = wl.axis_camera((3, 3, depth), 2, -1)
    cam = oracle_camera(oracle, cs)
    r = oracle.render_pixels(cube, tab, 0.0, 2.0, (1, 1, 1), cam, W, H, 1.0, 0, ert, 0, [1], [1])
    assert r["samples"] == n_star
    assert abs(r["rgba"][0, 3] - (1.0 - (1.0 - a32) ** n_star)) < 1e-6
    off = oracle.render_pixels(cube, tab, 0.0, 2.0, (1, 1, 1), cam, W, H, 1.0, 0, 0.0, 0, [1], [1])
    assert off["samples"] == depth
    # per brick (route 1, 3 slabs along the ray): each brick restarts from A = 0 and stops on its own count
    rb = oracle.render_pixels(cube, tab, 0.0, 2.0, (1, 1, 3), cam, W, H, 1.0, 0, ert, 1, [1], [1])
    faces = [(m * depth) // 3 for m in range(4)]
    assert rb["samples"] == sum(min(n_star, faces[m + 1] - faces[m]) for m in range(3))


def test_termination_point_on_a_noisy_cube_against_the_library_route(oracle):
    """RGBA and SAMPLE COUNT under termination, pixel by pixel, against tests/helpers.independent_pixel
    (cumprod; stops after the first sample whose running opacity reaches ert)."""
    dims = (14, 11, 12)
    cube = noisy_cube(dims, 8) + 1.0
    tab = wl.tf_ramp(0.9)
    W, H = 10, 8
    checked = stopped = 0
    for proj, ert in ((wl.PROJ_ORTHO, 0.8), (wl.PROJ_PERSP, 0.95)):
        cs = wl.orbit_camera(dims, 35.0, 25.0, proj)
        cam = oracle_camera(oracle, cs)
        for py in range(H):
            for px in range(W):
                want, _, n = independent_pixel(cube, tab, -3.0, 8.0, cs, W, H, 0.5, 0, px, py, ert=ert)
                if n < 0:
                    continue
                full = independent_pixel(cube, tab, -3.0, 8.0, cs, W, H, 0.5, 0, px, py)[2]
                r = oracle.render_pixels(cube, tab, -3.0, 8.0, (1, 1, 1), cam, W, H, 0.5, 0, ert, 0, [px], [py])
                assert r["samples"] == n, (px, py, r["samples"], n)
                assert np.abs(r["rgba"][0] - want).max() < 2e-6
                checked += 1
                stopped += n < full
    assert checked > 100 and stopped > 40
