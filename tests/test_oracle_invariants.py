"""Oracle invariants and brute force (CPU, -m "not gpu"): bricks (O9/O10), termination (O7),
symmetries of the whole renderer, NaN voxels (A14), and a full independent render of small
cubes through library routines (tests/helpers.independent_pixel)."""
import numpy as np
import pytest

from paper_1008_0135_b200 import workloads as wl
from tests.helpers import independent_pixel, oracle_camera

RAMP = wl.tf_ramp(0.1)
PW = wl.tf_piecewise(-3.0, 8.0, [(0.5, 0.0), (3.0, 0.25), (8.0, 0.8)])


def blob_cube(dims, seed):
    r = np.random.default_rng(seed)
    nx, ny, nz = dims
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    c = r.standard_normal((nz, ny, nx))
    c += 6.0 * np.exp(-((x - nx * 0.4) ** 2 + (y - ny * 0.6) ** 2 + (z - nz * 0.5) ** 2) / 18.0)
    return c.astype(np.float32)


# ---------------------------------------------------------------- brute force, general views --
@pytest.mark.parametrize("proj,az,el,step,mode", [
    (0, 30.0, 20.0, 0.5, 0), (1, 30.0, 20.0, 0.5, 0), (1, 215.0, -40.0, 1.0, 0),
    (0, 100.0, 65.0, 0.25, 0), (0, 30.0, 20.0, 1.0, 1), (1, 300.0, 10.0, 0.5, 1)])
def test_general_view_matches_independent_library_render(oracle, proj, az, el, step, mode):
    """Every pixel of an oblique / perspective frame of a small noisy cube against the
    library-routine renderer: pins O1-O8 together on general views (small inputs)."""
    dims = (10, 7, 6)
    cube = blob_cube(dims, 11)
    cs = wl.orbit_camera(dims, az, el, proj)
    cam = oracle_camera(oracle, cs)
    W, H = 14, 10
    r = oracle.render(cube, PW, -3.0, 8.0, (1, 1, 1), cam, W, H, step, mode)
    total = 0
    for py in range(H):
        for px in range(W):
            rgba, M, n = independent_pixel(cube, PW, -3.0, 8.0, cs, W, H, step, mode, px, py)
            total += n
            assert np.allclose(r["rgba"][py, px], rgba, atol=3e-7), (px, py)
            if mode == 1 and n > 0:
                assert abs(r["scalar"][py, px] - M) < 1e-6
    assert r["samples"] == total


def test_tiny_cube_hand_rolled(oracle):
    """4^3 cube, 8x8 image, axis-tilted ortho view: every sample listed by plain loops."""
    dims = (4, 4, 4)
    cube = blob_cube(dims, 2)
    cs = wl.orbit_camera(dims, 45.0, 0.0, 0)
    cam = oracle_camera(oracle, cs)
    r = oracle.render(cube, RAMP, -3.0, 8.0, (1, 1, 1), cam, 8, 8, 1.0, 0)
    for py in range(8):
        for px in range(8):
            rgba, _, _ = independent_pixel(cube, RAMP, -3.0, 8.0, cs, 8, 8, 1.0, 0, px, py)
            assert np.allclose(r["rgba"][py, px], rgba, atol=3e-7)


# ---------------------------------------------------------------- O9/O10 bricks ---------------
@pytest.mark.parametrize("bricks", [(1, 1, 1), (2, 2, 1), (2, 2, 2), (4, 4, 4), (3, 1, 2)])
@pytest.mark.parametrize("proj", [0, 1])
@pytest.mark.parametrize("mode", [0, 1])
def test_bricked_composite_equals_unbricked(oracle, bricks, proj, mode):
    """north_star closed form 4; also every lattice sample is owned by exactly one brick."""
    dims = (22, 18, 14)
    cube = blob_cube(dims, 7)
    cs = wl.orbit_camera(dims, 30.0, 20.0, proj)
    cam = oracle_camera(oracle, cs)
    W, H = 24, 24
    a = oracle.render(cube, PW, -3.0, 8.0, (1, 1, 1), cam, W, H, 0.5, mode, 0.0, 0)
    b = oracle.render(cube, PW, -3.0, 8.0, bricks, cam, W, H, 0.5, mode, 0.0, 1, want_bricks=True)
    assert a["samples"] == b["samples"]
    assert np.abs(a["rgba"] - b["rgba"]).max() <= 1.2e-7        # f32 outputs of ~1e-16 doubles
    if mode == 1:
        assert np.array_equal(a["scalar"], b["scalar"])
    for py in (0, 5, 11, 17, 23):
        for px in (0, 6, 12, 13, 23):
            o, d = oracle.ray(cam, W, H, px, py)
            n, tn, tf = oracle.ray_extent(o, d, dims, 0.5)
            owned = []
            for bk in range(bricks[2]):
                for bj in range(bricks[1]):
                    for bi in range(bricks[0]):
                        ok, t_in, lo, hi = oracle.brick_span(o, d, dims, bricks, (bi, bj, bk), 0.5,
                                                             tn, tf)
                        if ok:
                            owned.append((lo, hi))
            owned.sort()
            assert sum(h - l for l, h in owned) == n
            for (l0, h0), (l1, h1) in zip(owned, owned[1:]):
                assert h0 == l1                                  # contiguous, no overlap


def test_brick_boundaries_are_floor_splits(oracle):
    """A10: P_a[m] = floor(m n_a / b_a), e.g. 1721 -> 860 + 861 (only the slab test sees them)."""
    o = np.array([-5.0, 0.5, 0.5]); d = np.array([1.0, 0.0, 0.0])
    n, tn, tf = oracle.ray_extent(o, d, (1721, 1, 1), 1.0)
    assert n == 1721
    ok, t_in, lo, hi = oracle.brick_span(o, d, (1721, 1, 1), (2, 1, 1), (0, 0, 0), 1.0, tn, tf)
    assert (lo, hi) == (0, 860)
    ok, t_in, lo, hi = oracle.brick_span(o, d, (1721, 1, 1), (2, 1, 1), (1, 0, 0), 1.0, tn, tf)
    assert (lo, hi) == (860, 1721)


def test_over_is_associative_through_brick_groupings(oracle):
    """any grouping of depth-ordered partial images gives the same frame: splitting
    along the view axis into 2, 3 or 6 slabs composites to the same pixel values."""
    dims = (8, 8, 24)
    cube = blob_cube(dims, 9)
    cs, W, H, *_ = wl.axis_camera(dims, 2, -1)
    cam = oracle_camera(oracle, cs)
    ref = oracle.render(cube, PW, -3.0, 8.0, (1, 1, 1), cam, W, H, 1.0, 0)["rgba"]
    for bz in (2, 3, 6):
        r = oracle.render(cube, PW, -3.0, 8.0, (1, 1, bz), cam, W, H, 1.0, 0, 0.0, 1,
                          want_bricks=True)
        assert np.abs(r["rgba"] - ref).max() <= 1.2e-7
        # explicit "over" of the per-brick images, back to front grouping (right-associated)
        imgs = r["bricks"].astype(np.float64)                    # view along -z: far slab first
        order = list(range(bz))[::-1]
        C = np.zeros((H, W, 3)); A = np.zeros((H, W))
        for b in order[::-1]:                                    # fold from the back
            C = imgs[b, ..., :3] + (1 - imgs[b, ..., 3:4]) * C
            A = imgs[b, ..., 3] + (1 - imgs[b, ..., 3]) * A
        assert np.abs(C - ref[..., :3]).max() < 3e-7 and np.abs(A - ref[..., 3]).max() < 3e-7


# ---------------------------------------------------------------- O7 termination --------------
@pytest.mark.parametrize("route,bricks", [(0, (1, 1, 1)), (1, (2, 2, 2))])
def test_early_termination_bound(oracle, route, bricks):
    """A7: |ERT-on - ERT-off| <= 1 - ert_alpha per channel; fewer samples; with one brick a
    terminated ray has A >= ert_alpha."""
    dims = (24, 24, 24)
    cube = blob_cube(dims, 3) + 2.0
    tab = wl.tf_ramp(0.5)
    cs = wl.orbit_camera(dims, 30.0, 20.0, 1)
    cam = oracle_camera(oracle, cs)
    off = oracle.render(cube, tab, -3.0, 8.0, bricks, cam, 32, 32, 0.5, 0, 0.0, route)
    on = oracle.render(cube, tab, -3.0, 8.0, bricks, cam, 32, 32, 0.5, 0, 0.9, route)
    assert on["samples"] < off["samples"]
    assert np.abs(on["rgba"] - off["rgba"]).max() <= 0.1 + 1e-6
    changed = np.abs(on["rgba"] - off["rgba"]).max(axis=2) > 1e-7
    assert changed.any()
    if route == 0:
        assert (on["rgba"][..., 3][changed] >= 0.9 - 1e-6).all()


# ---------------------------------------------------------------- symmetries ------------------
def test_mirror_symmetry(oracle):
    """Cube flipped in x and the camera mirrored in x gives the x-mirrored image."""
    dims = (12, 10, 8)
    cube = blob_cube(dims, 5)
    cs = wl.orbit_camera(dims, 25.0, 15.0, 0)
    W, H = 20, 16
    a = oracle.render(cube, PW, -3.0, 8.0, (2, 1, 2), oracle_camera(oracle, cs), W, H, 0.5, 0, 0, 1)
    cs2 = wl.orbit_camera(dims, -25.0, 15.0, 0)
    b = oracle.render(cube[:, :, ::-1].copy(), PW, -3.0, 8.0, (2, 1, 2), oracle_camera(oracle, cs2),
                      W, H, 0.5, 0, 0, 1)
    assert np.abs(a["rgba"] - b["rgba"][:, ::-1]).max() < 2e-6


def test_quarter_turn_of_cube_and_camera(oracle):
    """Rotating cube and camera together by 90 deg about y leaves the image unchanged."""
    n = 10
    cube = blob_cube((n, n, n), 8)
    W = H = 16
    cs = wl.orbit_camera((n, n, n), 20.0, 30.0, 1)
    a = oracle.render(cube, PW, -3.0, 8.0, (1, 1, 1), oracle_camera(oracle, cs), W, H, 0.5, 0)
    # new cube: (x', z') = (z, n-1-x)  <=>  rotate the content by +90 deg about y
    rot = np.ascontiguousarray(np.transpose(cube, (2, 1, 0))[::-1, :, :])
    cs2 = wl.orbit_camera((n, n, n), 20.0 + 90.0, 30.0, 1)
    b = oracle.render(rot, PW, -3.0, 8.0, (1, 1, 1), oracle_camera(oracle, cs2), W, H, 0.5, 0)
    assert np.abs(a["rgba"] - b["rgba"]).max() < 2e-6


def test_step_halving_converges(oracle):
    dims = (16, 16, 16)
    z, y, x = np.meshgrid(*[np.arange(16)] * 3, indexing="ij")
    cube = (4.0 * np.exp(-((x - 8) ** 2 + (y - 7) ** 2 + (z - 9) ** 2) / 30.0)).astype(np.float32)
    cs = wl.orbit_camera(dims, 30.0, 20.0, 0)
    cam = oracle_camera(oracle, cs)
    imgs = [oracle.render(cube, RAMP, -3.0, 8.0, (1, 1, 1), cam, 16, 16, s, 0)["rgba"]
            for s in (1.0, 0.5, 0.25, 0.125)]
    e = [np.abs(imgs[i] - imgs[i + 1]).max() for i in range(3)]
    # first order at grazing rays (the last partial step), second order elsewhere
    assert e[1] < 0.6 * e[0] and e[2] < 0.6 * e[1]


# ---------------------------------------------------------------- A14 NaN ---------------------
def test_nan_voxels_are_skipped(oracle):
    dims = (6, 6, 12)
    cube = blob_cube(dims, 4)
    cs, W, H, *_ = wl.axis_camera(dims, 2, +1)
    cam = oracle_camera(oracle, cs)
    holed = cube.copy()
    holed[4:8] = np.nan                       # 4 blank channels
    a = oracle.render(holed, PW, -3.0, 8.0, (1, 1, 1), cam, W, H, 1.0, 0)
    # O5: "if the blend is NaN the sample is skipped" - IEEE 0*NaN = NaN, so a sample is lost as
    # soon as ANY voxel of its 2x2x2 footprint is NaN, also at weight 0: the sample on the centre
    # of channel 3 has channel 4 as its (zero-weight) upper neighbour and is skipped as well.
    kept = np.concatenate([cube[:3], cube[8:]], axis=0)
    cs2, *_ = wl.axis_camera((6, 6, 7), 2, +1)
    b = oracle.render(kept, PW, -3.0, 8.0, (1, 1, 1), oracle_camera(oracle, cs2), W, H, 1.0, 0)
    assert np.abs(a["rgba"] - b["rgba"]).max() < 2e-7
    m = oracle.render(holed, PW, -3.0, 8.0, (1, 1, 1), cam, W, H, 1.0, 1)
    assert np.array_equal(m["scalar"], kept.max(axis=0)[:, ::-1])    # looking along +z: right = -x
    allnan = np.full((4, 4, 4), np.nan, dtype=np.float32)
    cs3, W3, H3, *_ = wl.axis_camera((4, 4, 4), 0, +1)
    z = oracle.render(allnan, PW, -3.0, 8.0, (1, 1, 1), oracle_camera(oracle, cs3), W3, H3, 1.0, 1)
    assert np.all(z["rgba"] == 0) and np.all(np.isneginf(z["scalar"]))
