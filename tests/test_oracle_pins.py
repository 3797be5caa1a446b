"""Pins of the CPU oracle against things other than itself (all CPU, -m "not gpu").

Each test names the oracle rule (O1-O11) it would catch a mistake in.  Expected values
are closed forms, library routines (numpy.max, cumprod, scipy map_coordinates, numpy.interp),
invariants, or brute force on tiny inputs; golden numbers live in tests/golden/ with citations.
"""
import json
import math
import os

import numpy as np
import pytest

from paper_1008_0135_b200 import workloads as wl
from tests.helpers import independent_pixel, oracle_camera, pixel_ray_linalg

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "closed_forms.json")))
RAMP = wl.tf_ramp(0.1)


def rng_cube(dims, seed=0, scale=1.0):
    r = np.random.default_rng(seed)
    nx, ny, nz = dims
    return (scale * r.standard_normal((nz, ny, nx))).astype(np.float32)


# ---------------------------------------------------------------- O1/O2: rays -----------------
@pytest.mark.parametrize("proj", [0, 1])
def test_rays_match_inverse_view_matrix(oracle, proj):
    """O1/O2: a transposed R, a wrong sign of fwd, a wrong eye or pixel-centre offset fails."""
    cs = wl.orbit_camera((40, 30, 20), 37.0, -25.0, proj)
    cam = oracle_camera(oracle, cs)
    W, H = 13, 7
    for px, py in [(0, 0), (12, 6), (3, 5), (6, 3)]:
        o, d = oracle.ray(cam, W, H, px, py)
        o2, d2 = pixel_ray_linalg(cs, W, H, px, py)
        assert np.allclose(d, d2, atol=1e-6)
        # origins may differ along d for ORTHO (any point of the line is fine for the test)
        assert np.linalg.norm(np.cross(o - o2, d2)) < 1e-3 * np.linalg.norm(o2)
        # projecting back: the eye-space x,y of any point on the ray is the pixel centre
        V = cs.view.astype(np.float64)
        p = o + 17.0 * d
        e = V @ np.array([p[0], p[1], p[2], 1.0])
        u = 2 * (px + 0.5) / W - 1
        v = 2 * (py + 0.5) / H - 1
        if proj == 0:
            assert abs(e[0] - u * cs.ortho_half_h * W / H) < 1e-3
            assert abs(e[1] - v * cs.ortho_half_h) < 1e-3
        else:
            T = math.tan(math.radians(cs.fovy_deg / 2))
            assert abs(e[0] / -e[2] - u * T * W / H) < 1e-6
            assert abs(e[1] / -e[2] - v * T) < 1e-6


# ---------------------------------------------------------------- O2-O4 + O6/O7: constant cube
def test_constant_cube_closed_form_golden(oracle):
    """north_star closed form 1 with the worked numbers of SURVEY.md 8(c): 64^3 cube of 2.5,
    range [-3,8], ramp table, axis-aligned ray, n = 64/step."""
    cube = np.full((64, 64, 64), 2.5, dtype=np.float32)
    cs, W, H, *_ = wl.axis_camera((64, 64, 64), 2, +1)
    cam = oracle_camera(oracle, cs)
    for key, step in (("step1", 1.0), ("step0.5", 0.5), ("step0.25", 0.25)):
        r = oracle.render(cube, RAMP, -3.0, 8.0, (1, 1, 1), cam, W, H, step, 0)
        g = GOLD["constant_cube_64"][key]
        assert r["samples"] == int(64 / step) * W * H
        assert np.allclose(r["rgba"][..., 3], g["A"], atol=2e-7)
        assert np.allclose(r["rgba"][..., :3], g["C"], atol=2e-7)


@pytest.mark.parametrize("proj,az,el,step", [(0, 30.0, 20.0, 0.5), (1, 200.0, -35.0, 1.0),
                                             (0, 90.0, 0.0, 0.25), (1, 0.0, 89.0, 0.7)])
def test_constant_cube_oblique(oracle, proj, az, el, step):
    """O2-O4: A = 1 - (1 - a_step)^n with n from an independent per-face box intersection;
    pixels outside the silhouette are exactly zero."""
    dims = (20, 14, 9)
    cube = np.full((dims[2], dims[1], dims[0]), 4.0, dtype=np.float32)
    cs = wl.orbit_camera(dims, az, el, proj)
    cam = oracle_camera(oracle, cs)
    W, H = 24, 16
    r = oracle.render(cube, RAMP, -3.0, 8.0, (1, 1, 1), cam, W, H, step, 0)
    a1 = 0.1 * (4.0 + 3.0) / 11.0       # ramp alpha at the value, interpolated linearly
    for py in range(H):
        for px in range(W):
            exp, _, n = independent_pixel(cube, RAMP, -3.0, 8.0, cs, W, H, step, 0, px, py)
            got = r["rgba"][py, px]
            if n == 0:
                assert np.all(got == 0.0)
                continue
            s = (4.0 + 3.0) / 11.0
            # per-entry corrected alpha, interpolated between the two entries around 255*s
            x = 255 * s; m = int(x); w = x - m
            tab = RAMP.astype(np.float64)
            ad = (1 - w) * (1 - (1 - tab[m, 3]) ** step) + w * (1 - (1 - tab[m + 1, 3]) ** step)
            A = 1 - (1 - ad) ** n
            rgb = (1 - w) * tab[m, :3] + w * tab[m + 1, :3]
            assert abs(got[3] - A) < 1e-6, (px, py, n)
            assert np.allclose(got[:3], rgb * A, atol=1e-6)
            assert abs(a1 - ((1 - w) * tab[m, 3] + w * tab[m + 1, 3])) < 1e-7


# ---------------------------------------------------------------- O5: trilinear ---------------
def test_trilinear_identities(oracle):
    """O5: centre of a 2^3 cube = mean of 8; outer half voxel = nearest face value; a cube linear
    in (x,y,z) is reproduced exactly inside [1/2, n-1/2]."""
    r = np.random.default_rng(1)
    c2 = r.standard_normal((2, 2, 2)).astype(np.float32)
    assert abs(oracle.sample(c2, (1.0, 1.0, 1.0)) - float(c2.astype(np.float64).mean())) < 1e-15
    assert oracle.sample(c2, (0.2, 0.1, 0.4)) == float(c2[0, 0, 0])
    assert oracle.sample(c2, (1.9, 0.1, 1.7)) == float(c2[1, 0, 1])          # [z][y][x]
    nx, ny, nz = 7, 5, 6
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    lin = (0.5 * (x + 0.5) - 0.25 * (y + 0.5) + 2.0 * (z + 0.5) + 1.0).astype(np.float32)
    for p in r.uniform([0.5, 0.5, 0.5], [nx - 0.5, ny - 0.5, nz - 0.5], size=(50, 3)):
        assert abs(oracle.sample(lin, p) - (0.5 * p[0] - 0.25 * p[1] + 2.0 * p[2] + 1.0)) < 1e-12


def test_trilinear_matches_map_coordinates(oracle):
    """O5 against scipy.ndimage.map_coordinates(order=1, mode='nearest') incl. outside points."""
    from scipy import ndimage
    cube = rng_cube((9, 6, 5), 3)
    r = np.random.default_rng(4)
    P = r.uniform([-1, -1, -1], [10, 7, 6], size=(200, 3))
    ref = ndimage.map_coordinates(cube.astype(np.float64),
                                  np.stack([P[:, 2] - 0.5, P[:, 1] - 0.5, P[:, 0] - 0.5]),
                                  order=1, mode="nearest")
    got = np.array([oracle.sample(cube, p) for p in P])
    assert np.allclose(got, ref, atol=1e-12)


# ---------------------------------------------------------------- O6: lookup ------------------
def test_lookup_linear_table_is_identity_and_clamps(oracle):
    tab = RAMP
    for v in (-10.0, -3.0, 0.123, 2.5, 7.999, 8.0, 50.0):
        s = min(max((v + 3.0) / 11.0, 0.0), 1.0)
        e = oracle.classify(tab, -3.0, 8.0, 1.0, v)
        exp = (1 - s) * tab[0].astype(np.float64) + s * tab[255].astype(np.float64)
        assert np.allclose(e, exp, atol=1e-7)


def test_lookup_matches_numpy_interp(oracle):
    tab = wl.tf_piecewise(-3.0, 60.0, [(2.5, 0.0), (5.0, 0.02), (15.0, 0.2), (50.0, 0.6)])
    xp = -3.0 + 63.0 * np.arange(256) / 255.0
    for step in (1.0, 0.5, 0.3):
        ac = 1.0 - (1.0 - tab[:, 3].astype(np.float64)) ** step
        for v in np.linspace(-5, 65, 141):
            e = oracle.classify(tab, -3.0, 60.0, step, v)
            for c in range(3):
                assert abs(e[c] - np.interp(v, xp, tab[:, c].astype(np.float64))) < 1e-12
            assert abs(e[3] - np.interp(v, xp, ac)) < 1e-12


# ---------------------------------------------------------------- O5+O8: axis-aligned MIP -----
@pytest.mark.parametrize("axis", [0, 1, 2])
@pytest.mark.parametrize("sign", [+1, -1])
@pytest.mark.parametrize("step", [1.0, 1.0 / 3.0, 0.2])
def test_axis_aligned_mip_is_max_over_axis(oracle, axis, sign, step):
    """north_star closed form 2: samples sit on voxel centres, so MIP = numpy max over the axis."""
    dims = (22, 18, 14)
    cube = rng_cube(dims, 5, 3.0)
    cs, W, H, ra, rs, ua, us = wl.axis_camera(dims, axis, sign)
    cam = oracle_camera(oracle, cs)
    r = oracle.render(cube, RAMP, -3.0, 8.0, (1, 1, 1), cam, W, H, step, 1)
    mx = cube.astype(np.float64).max(axis=2 - axis)          # numpy axes are (z,y,x)
    for py in range(H):
        for px in range(W):
            col = [0, 0, 0]
            col[ra] = px if rs > 0 else dims[ra] - 1 - px
            col[ua] = py if us > 0 else dims[ua] - 1 - py
            rest = [col[a] for a in (2, 1, 0) if a != axis]   # index into mx in (z,y,x) order
            # step is a float32 argument: 1/3 and 0.2 are inexact, so samples drift off the
            # voxel centres by ~1e-6 voxel over the ray; at step 1 the match is to rounding
            tol = (1e-6 if step == 1.0 else 2e-5) * max(1, abs(mx[tuple(rest)]))
            assert abs(r["scalar"][py, px] - mx[tuple(rest)]) <= tol
    # colour = lookup of the max in the uncorrected table, un-premultiplied
    e = oracle.classify(RAMP, -3.0, 8.0, 1.0, float(r["scalar"][3, 4]))
    assert np.allclose(r["rgba"][3, 4], e, atol=1e-6)


# ---------------------------------------------------------------- O6+O7: 1-D recurrence -------
@pytest.mark.parametrize("axis,sign", [(2, +1), (2, -1), (0, +1), (1, -1)])
def test_axis_aligned_ea_is_cumprod_recurrence(oracle, axis, sign):
    """Step 1 along an axis on any cube = the 1-D front-to-back recurrence, written with cumprod."""
    dims = (11, 9, 13)
    cube = rng_cube(dims, 6, 3.0)
    tab = wl.tf_piecewise(-3.0, 8.0, [(0.0, 0.0), (3.0, 0.3), (8.0, 0.9)])
    cs, W, H, ra, rs, ua, us = wl.axis_camera(dims, axis, sign)
    cam = oracle_camera(oracle, cs)
    r = oracle.render(cube, tab, -3.0, 8.0, (1, 1, 1), cam, W, H, 1.0, 0)
    xp = -3.0 + 11.0 * np.arange(256) / 255.0
    c64 = cube.astype(np.float64)
    for py in range(H):
        for px in range(W):
            col = [slice(None)] * 3
            idx = {ra: px if rs > 0 else dims[ra] - 1 - px, ua: py if us > 0 else dims[ua] - 1 - py}
            sl = tuple(idx.get(a, slice(None)) for a in (2, 1, 0))
            v = c64[sl]
            if sign < 0:
                v = v[::-1]
            a = np.interp(v, xp, tab[:, 3].astype(np.float64))
            rgb = np.stack([np.interp(v, xp, tab[:, c].astype(np.float64)) for c in range(3)], 1)
            trans = np.concatenate([[1.0], np.cumprod(1 - a)[:-1]])
            C = (trans[:, None] * a[:, None] * rgb).sum(0)
            A = 1 - np.prod(1 - a)
            assert np.allclose(r["rgba"][py, px], [C[0], C[1], C[2], A], atol=2e-7)
            del col


def test_ramp_cube_worked_values_and_continuous_limit(oracle):
    """north_star closed form 3.  Ramp cube v[k] = -3 + 11k/63 along z, ramp table: worked values
    of SURVEY.md 8(c) at step 1 from both sides, and the analytic integral as step -> 0:
    ln(1-A) = 63 * I + (1/2) ln 0.9,  I = int_0^1 ln(1 - 0.1 s) ds = -(0.9 ln 0.9 + 0.1)/0.1."""
    k = np.arange(64, dtype=np.float64)
    cube = np.broadcast_to((-3.0 + 11.0 * k / 63.0)[:, None, None], (64, 4, 4)).astype(np.float32)
    g = GOLD["ramp_cube_64"]
    for sign, key in ((+1, "from_k0"), (-1, "from_k63")):
        cs, W, H, *_ = wl.axis_camera((4, 4, 64), 2, sign)
        r = oracle.render(cube, RAMP, -3.0, 8.0, (1, 1, 1), oracle_camera(oracle, cs), W, H, 1.0, 0)
        assert np.allclose(r["rgba"][1, 2, 3], g[key]["A"], atol=2e-7)
        assert np.allclose(r["rgba"][1, 2, :3], g[key]["C"], atol=2e-7)
    I = -(0.9 * math.log(0.9) + 0.1) / 0.1
    A_lim = 1.0 - math.exp(63.0 * I + 0.5 * math.log(0.9))
    assert abs(A_lim - g["continuous_limit_A"]) < 1e-10
    cs, W, H, *_ = wl.axis_camera((4, 4, 64), 2, +1)
    cam = oracle_camera(oracle, cs)
    errs = []
    for step in (1.0, 0.5, 0.25, 0.125):
        r = oracle.render(cube, RAMP, -3.0, 8.0, (1, 1, 1), cam, W, H, step, 0)
        errs.append(abs(float(r["rgba"][0, 0, 3]) - A_lim))
    assert errs[0] < 1e-6 and errs[1] < 2e-7 and errs[2] < 2e-7 and errs[3] < 2e-7
    assert errs[1] < errs[0] / 3          # second-order convergence until the f32 output floor
