"""Pins of the oracle's spectral-channel mask, rule S2 ("enabling/disabling spectral channel(s)"):
the enabled channels form maximal runs [za, zb); a lattice sample is taken iff O9's ownership rule gives it to the
slab of some run.  Pinned by: the closed form on a constant cube (n = number of enabled channels), the library
max over the enabled channels (axis-aligned MIP), the 1-D cumprod recurrence over the enabled, NON-contiguous
channels, mask of all ones = no mask, a single run = the sub-cube of S1, complementary masks (MIP: max of the two
= whole; sample counts add up), and an oblique view against the library route with the per-sample rule
"channel floor(p_z) is enabled" (equal to the run rule whenever no sample sits exactly on a channel plane)."""
import numpy as np
import pytest
from scipy import ndimage

from paper_1008_0135_b200 import workloads as wl
from tests.helpers import pixel_ray_linalg, box_hits_by_faces


def _cam(oracle, cs):
    return oracle.make_camera(cs.view, cs.projection, cs.fovy_deg, cs.ortho_half_h)


def _mask(nz, enabled):
    m = np.zeros(nz, dtype=np.uint8)
    for a, b in enabled:
        m[a:b] = 1
    return m


RUNS = [(2, 5), (9, 10), (14, 21)]          # three runs, 11 channels of 24


def test_all_ones_is_no_mask_and_single_run_is_the_subcube(oracle):
    dims = (20, 14, 24)
    cube = wl.cube_blobs(dims, 3, "cpu", n_blobs=3, amp=6.0, sigma=3.0).numpy()
    tab = wl.tf_ramp(0.2)
    for proj, route, bricks in ((0, 0, (1, 1, 1)), (1, 1, (2, 1, 3))):
        cs = wl.orbit_camera(dims, 40.0, 25.0, proj)
        a = oracle.render(cube, tab, -3, 8, bricks, _cam(oracle, cs), 30, 26, 0.5, 0, 0.0, route=route)
        b = oracle.render(cube, tab, -3, 8, bricks, _cam(oracle, cs), 30, 26, 0.5, 0, 0.0, route=route,
                          chan_mask=np.ones(24))
        assert np.array_equal(a["rgba"], b["rgba"]) and a["samples"] == b["samples"]
        c = oracle.render(cube, tab, -3, 8, bricks, _cam(oracle, cs), 30, 26, 0.5, 0, 0.9, route=route,
                          chan_mask=_mask(24, [(7, 18)]))
        d = oracle.render(cube, tab, -3, 8, bricks, _cam(oracle, cs), 30, 26, 0.5, 0, 0.9, route=route,
                          subcube=((0, 0, 7), (20, 14, 18)))
        assert np.array_equal(c["rgba"], d["rgba"]) and c["samples"] == d["samples"] and c["samples"] > 0
        z = oracle.render(cube, tab, -3, 8, bricks, _cam(oracle, cs), 30, 26, 0.5, 0, 0.0, route=route,
                          chan_mask=np.zeros(24))
        assert not z["rgba"].any() and z["samples"] == 0


@pytest.mark.parametrize("sign", [1, -1])
def test_constant_cube_closed_form_over_enabled_channels(oracle, sign):
    """Axis-aligned ray, step 1 and 1/2: n = enabled channels / step, A = 1 - (1 - a_step)^n (closed form 1)."""
    dims = (8, 8, 24)
    cube = np.full((24, 8, 8), 2.5, dtype=np.float32)
    tab = wl.tf_ramp(0.1)                                   # alpha(2.5) over [-3,8] = 0.05 per voxel of path
    cs, W, H, *_ = wl.axis_camera(dims, 2, sign)
    m = _mask(24, RUNS)
    for step in (1.0, 0.5):
        r = oracle.render(cube, tab, -3, 8, (1, 1, 2), _cam(oracle, cs), W, H, step, 0, 0.0, route=1, chan_mask=m)
        n = int(m.sum() / step)
        a = 1.0 - 0.95 ** step
        assert np.allclose(r["rgba"][..., 3], 1.0 - (1.0 - a) ** n, atol=3e-7)
        assert r["samples"] == W * H * n


def test_axis_mip_equals_library_max_over_enabled_channels(oracle):
    dims = (18, 14, 24)
    cube = wl.cube_blobs(dims, 4, "cpu", n_blobs=3, amp=6.0, sigma=3.0).numpy()
    cs, W, H, ra, rs, ua, us = wl.axis_camera(dims, 2, -1)
    m = _mask(24, RUNS)
    r = oracle.render(cube, wl.tf_ramp(0.1), -3, 8, (1, 2, 2), _cam(oracle, cs), W, H, 1.0, 1, 0.0, route=1, chan_mask=m)
    want = cube[m.astype(bool)].max(axis=0)
    if rs < 0:
        want = want[:, ::-1]
    assert np.abs(r["scalar"] - want).max() <= 1e-6


@pytest.mark.parametrize("sign", [1, -1])
def test_axis_ea_equals_cumprod_over_enabled_channels(oracle, sign):
    """View along +/-z, step 1: the frame is the 1-D recurrence over the enabled channels in the order the ray
    meets them (disabled channels simply do not appear in the product)."""
    dims = (10, 9, 24)
    cube = wl.cube_blobs(dims, 5, "cpu", n_blobs=2, amp=6.0, sigma=3.0).numpy()
    tab = wl.tf_ramp(0.3)
    cs, W, H, ra, rs, ua, us = wl.axis_camera(dims, 2, sign)
    m = _mask(24, RUNS).astype(bool)
    r = oracle.render(cube, tab, -3, 8, (1, 1, 1), _cam(oracle, cs), W, H, 1.0, 0, 0.0, route=0, chan_mask=m)["rgba"]
    col = cube[m]                                           # enabled channels, ascending z
    if sign < 0:
        col = col[::-1]
    xp = -3 + 11 * np.arange(256) / 255.0
    a = np.interp(col, xp, tab[:, 3].astype(np.float64))
    trans = np.concatenate([np.ones((1,) + a.shape[1:]), np.cumprod(1 - a, axis=0)[:-1]], axis=0)
    A = 1 - np.prod(1 - a, axis=0)
    C = [(trans * a * np.interp(col, xp, tab[:, c].astype(np.float64))).sum(axis=0) for c in range(3)]
    want = np.stack(C + [A], axis=-1)                       # [y][x]
    if rs < 0:
        want = want[:, ::-1]
    assert np.abs(r - want).max() < 3e-7


def test_complementary_masks(oracle):
    """Any view: every lattice sample belongs to exactly one of two complementary masks (counts add up), and the
    MIP of the whole cube is the larger of the two masked MIPs."""
    dims = (22, 17, 24)
    cube = wl.cube_blobs(dims, 6, "cpu", n_blobs=4, amp=6.0, sigma=3.0).numpy()
    tab = wl.tf_ramp(0.2)
    m = _mask(24, RUNS)
    for proj, bricks, route in ((wl.PROJ_PERSP, (2, 2, 2), 1), (wl.PROJ_ORTHO, (1, 1, 1), 0)):
        cs = wl.orbit_camera(dims, 55.0, 35.0, proj)
        W, H = 33, 27
        whole = oracle.render(cube, tab, -3, 8, bricks, _cam(oracle, cs), W, H, 0.5, 1, 0.0, route=route)
        a = oracle.render(cube, tab, -3, 8, bricks, _cam(oracle, cs), W, H, 0.5, 1, 0.0, route=route, chan_mask=m)
        b = oracle.render(cube, tab, -3, 8, bricks, _cam(oracle, cs), W, H, 0.5, 1, 0.0, route=route, chan_mask=1 - m)
        assert a["samples"] + b["samples"] == whole["samples"]
        assert np.array_equal(np.maximum(a["scalar"], b["scalar"]), whole["scalar"])
        # bricked = unbricked under a mask as well
        u = oracle.render(cube, tab, -3, 8, (1, 1, 1), _cam(oracle, cs), W, H, 0.5, 0, 0.0, route=0, chan_mask=m)
        k = oracle.render(cube, tab, -3, 8, (2, 3, 2), _cam(oracle, cs), W, H, 0.5, 0, 0.0, route=1, chan_mask=m)
        assert np.abs(u["rgba"] - k["rgba"]).max() < 1e-6 and u["samples"] == k["samples"]


def test_oblique_view_against_the_per_sample_rule(oracle):
    """Library route (tests/helpers.py pieces): samples listed one by one, a sample is kept iff channel
    floor(p_z) is enabled; map_coordinates, interp, cumprod.  Pixels with a sample within 1e-9 of a channel
    plane are left out (there the two statements of the rule may differ)."""
    dims = (13, 11, 24)
    g = np.random.default_rng(12)
    cube = (g.normal(size=(24, 11, 13)) * 1.5 + 2.0).astype(np.float32)
    tab = wl.tf_ramp(0.4)
    m = _mask(24, RUNS).astype(bool)
    W, H = 12, 10
    xp = -3 + 11 * np.arange(256) / 255.0
    checked = 0
    for proj in (wl.PROJ_ORTHO, wl.PROJ_PERSP):
        cs = wl.orbit_camera(dims, 35.0, 25.0, proj)
        r = oracle.render(cube, tab, -3, 8, (1, 1, 1), _cam(oracle, cs), W, H, 0.5, 0, 0.0, route=0, chan_mask=m)
        for py in range(H):
            for px in range(W):
                o, d = pixel_ray_linalg(cs, W, H, px, py)
                hit = box_hits_by_faces(o, d, np.zeros(3), np.array(dims, dtype=np.float64))
                if hit is None or not hit[1] > max(hit[0], 0.0):
                    assert not r["rgba"][py, px].any()
                    continue
                tn, tf = max(hit[0], 0.0), hit[1]
                ts = tn + (np.arange(int(np.ceil((tf - tn) / 0.5)) + 2) + 0.5) * 0.5
                ts = ts[ts < tf]
                if ts.size == 0:
                    assert not r["rgba"][py, px].any()
                    continue
                P = o[None, :] + ts[:, None] * d[None, :]
                if np.abs(P[:, 2] - np.round(P[:, 2])).min() < 1e-9:
                    continue
                keep = m[np.clip(np.floor(P[:, 2]).astype(int), 0, 23)]
                P = P[keep]
                if len(P) == 0:
                    assert not r["rgba"][py, px].any()
                    continue
                vals = ndimage.map_coordinates(cube.astype(np.float64), [P[:, 2] - .5, P[:, 1] - .5, P[:, 0] - .5],
                                               order=1, mode="nearest")
                a = np.interp(vals, xp, 1 - (1 - tab[:, 3].astype(np.float64)) ** 0.5)
                trans = np.concatenate([[1.0], np.cumprod(1 - a)[:-1]])
                want = [(trans * a * np.interp(vals, xp, tab[:, c].astype(np.float64))).sum() for c in range(3)]
                want.append(1 - np.prod(1 - a))
                assert np.abs(r["rgba"][py, px] - np.array(want)).max() < 2e-6, (proj, px, py)
                checked += 1
    assert checked > 50
