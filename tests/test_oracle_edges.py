"""Pins for two edge rules of the oracle that survived mutation in the round-2 review.

  O4/O9  I(t) = max(0, ceil((t - t_near)/step - 1/2))   lattice_index   a sample that lands EXACTLY on the exit face is
         outside (t_i < t_far is strict), and one that lands exactly on a brick plane belongs to the brick behind
         the plane (every brick box is half-open, [lo, hi)).  The mutant floor(x + 1/2) differs only on such ties.
  O6     m = min(floor x, 254)                          lookup          the LAST table interval [254, 255]
         interpolates between entries 254 and 255.  The mutant min(floor x, 253) extrapolates from entries 253 and 254,
         which is the same thing on every table that is linear over its last two intervals.

Geometry is dyadic (positions, steps and plane distances are exact binary fractions) so the ties are ties in floating
point too.  Expected values are hand-written sample lists, the strict `while t < t_far` loop of tests/helpers.py,
numpy.interp and closed forms (O4, O6, O9; PAPER.md:150 entry and exit points, PAPER.md:80 transfer function)
— never the oracle itself.
"""
import numpy as np
import pytest
from scipy import ndimage

from paper_1008_0135_b200 import workloads as wl
from tests.helpers import independent_pixel, oracle_camera


def hand_samples(o_z, step, nz):
    """z of the samples of a +z ray that starts INSIDE the cube at height o_z: t_i = (i + 1/2) step, kept while the
    position is strictly below the exit face z = nz."""
    zs, i = [], 0
    while o_z + (i + 0.5) * step < nz:
        zs.append(o_z + (i + 0.5) * step)
        i += 1
    return zs


def blend_of(cube, table, vmin, vmax, step, x, y, zs):
    """Front-to-back blend (premultiplied C, A) of the listed sample positions, from library routines."""
    if not zs:
        return np.zeros(4)
    coords = np.array([[z - 0.5 for z in zs], [y - 0.5] * len(zs), [x - 0.5] * len(zs)])
    vals = ndimage.map_coordinates(cube.astype(np.float64), coords, order=1, mode="nearest")
    xp = vmin + (vmax - vmin) * np.arange(256) / 255.0
    tab = np.asarray(table, dtype=np.float64)
    rgb = np.stack([np.interp(vals, xp, tab[:, c]) for c in range(3)], axis=1)
    a = np.interp(vals, xp, 1.0 - (1.0 - tab[:, 3]) ** step)
    trans = np.concatenate([[1.0], np.cumprod(1.0 - a)[:-1]])
    C = (trans[:, None] * a[:, None] * rgb).sum(axis=0)
    return np.array([C[0], C[1], C[2], 1.0 - np.prod(1.0 - a)])


# ------------------------------------------------------------------ O4: a sample exactly on the exit face ------
@pytest.mark.parametrize("o_z,step,nz,want", [
    (1.5, 1.0, 4, 2),      # samples at z = 2, 3; the next one is z = 4 = the exit face
    (1.25, 0.5, 4, 5),     # z = 1.5 ... 3.5; the sixth would be 4.0
    (1.0, 2.0, 8, 3),      # z = 2, 4, 6; then 8.0
    (0.5, 1.0, 4, 3),      # no tie: z = 1, 2, 3 and 4.0 again excluded
    (1.5, 1.0, 5, 3),      # one more layer: z = 4 is now inside
    (0.0, 0.25, 1, 4),     # from the entry face itself: z = 1/8, 3/8, 5/8, 7/8
])
def test_a_sample_exactly_on_the_exit_face_is_not_taken(oracle, o_z, step, nz, want):
    """vro.c lattice_index: ceil((t_far - t_near)/step - 1/2).  When (t_far - t_near)/step = k + 1/2 the (k+1)-th
    sample sits exactly on the exit face: t_i < t_far is false, n = k.  floor(x + 1/2) would count it."""
    assert len(hand_samples(o_z, step, nz)) == want                    # the hand list is what the table says
    n, t_near, t_far = oracle.ray_extent((0.5, 0.5, o_z), (0.0, 0.0, 1.0), (1, 1, nz), step)
    assert (t_near, t_far) == (0.0, nz - o_z)
    assert n == want
    # the same ray from the far side (entering through a face, t_near > 0), marching towards -z
    n, t_near, t_far = oracle.ray_extent((0.5, 0.5, nz + 3.0), (0.0, 0.0, -1.0), (1, 1, nz), step)
    assert (t_near, t_far) == (3.0, 3.0 + nz)
    k, i = 0, 0
    while 3.0 + (i + 0.5) * step < 3.0 + nz:
        k, i = k + 1, i + 1
    assert n == k


def inside_plane_camera(dims, z0):
    """Orthographic camera looking along +z whose image plane lies INSIDE the cube at height z0, one ray per voxel
    column (rays start at (px + 1/2, py + 1/2, z0): t_near = 0 by O3's clamp)."""
    nx, ny, _ = dims
    cs = wl.CameraSpec(wl.look_at((nx / 2.0, ny / 2.0, z0), (nx / 2.0, ny / 2.0, z0 + 4.0)), wl.PROJ_ORTHO, 45.0, ny / 2.0)
    return cs, nx, ny


def test_frame_with_samples_on_the_exit_face_and_on_a_brick_plane(oracle):
    """dims (4,4,8), image plane at z = 1, step 2: every ray's samples are z = 2, 4, 6 — z = 8 falls on the exit face
    (not taken) and z = 4 falls on the plane between the two bricks of a (1,1,2) partition.  Brick boxes are half-open
    (O9, A10): the sample at z = 4 belongs to brick 1 = [4, 8).  Checked: the sample count, the frame against the
    library route (whose loop is `while t < t_far`), and BOTH brick images against blends of hand-written owner lists."""
    dims = (4, 4, 8)
    g = np.random.default_rng(5)
    cube = (g.normal(size=(8, 4, 4)) * 1.5 + 2.0).astype(np.float32)
    table = wl.tf_ramp(0.3)
    vmin, vmax, step = -3.0, 8.0, 2.0
    cs, W, H = inside_plane_camera(dims, 1.0)
    cam = oracle_camera(oracle, cs)
    o, d = oracle.ray(cam, W, H, 1, 2)
    assert np.array_equal(d, [0.0, 0.0, 1.0]) and o[2] == 1.0          # the geometry is exact
    zs = hand_samples(1.0, step, 8)
    assert zs == [2.0, 4.0, 6.0]
    owners = {0: [2.0], 1: [4.0, 6.0]}                                 # hand-written: [0,4) and [4,8)
    r0 = oracle.render(cube, table, vmin, vmax, (1, 1, 1), cam, W, H, step, 0, 0.0, route=0)
    r1 = oracle.render(cube, table, vmin, vmax, (1, 1, 2), cam, W, H, step, 0, 0.0, route=1, want_bricks=True)
    assert r0["samples"] == r1["samples"] == W * H * 3
    for py in range(H):
        for px in range(W):
            o, _ = oracle.ray(cam, W, H, px, py)
            want, _, n = independent_pixel(cube, table, vmin, vmax, cs, W, H, step, 0, px, py)
            assert n == 3
            assert np.abs(r0["rgba"][py, px] - want).max() < 2e-6
            assert np.abs(r1["rgba"][py, px] - want).max() < 2e-6
            for b in (0, 1):
                wb = blend_of(cube, table, vmin, vmax, step, o[0], o[1], owners[b])
                assert np.abs(r1["bricks"][b, py, px] - wb).max() < 2e-6, (b, px, py)
    # the spans themselves: brick 0 owns lattice index 0 only, brick 1 owns 1 and 2
    o, d = oracle.ray(cam, W, H, 0, 0)
    n, t_near, t_far = oracle.ray_extent(o, d, dims, step)
    assert (n, t_near, t_far) == (3, 0.0, 7.0)
    ok0, t_in0, lo0, hi0 = oracle.brick_span(o, d, dims, (1, 1, 2), (0, 0, 0), step, t_near, t_far)
    ok1, t_in1, lo1, hi1 = oracle.brick_span(o, d, dims, (1, 1, 2), (0, 0, 1), step, t_near, t_far)
    assert ok0 and ok1 and (t_in0, lo0, hi0) == (0.0, 0, 1) and (t_in1, lo1, hi1) == (3.0, 1, 3)


def test_mip_ignores_the_sample_on_the_exit_face(oracle):
    """Same geometry, MIP: a cube whose last layer's far side would win if z = 8 were sampled.  Samples z = 2, 4, 6
    read voxel layers (1,2), (3,4), (5,6); layer 7 holds the largest values and must not be seen."""
    cube = np.zeros((8, 4, 4), dtype=np.float32)
    for k in range(8):
        cube[k] = float(k)
    cube[7] = 100.0
    cs, W, H = inside_plane_camera((4, 4, 8), 1.0)
    r = oracle.render(cube, wl.tf_ramp(0.1), 0.0, 100.0, (1, 1, 1), oracle_camera(oracle, cs), W, H, 2.0, 1, 0.0, route=0)
    assert np.array_equal(r["scalar"], np.full((H, W), 5.5, dtype=np.float32))      # z = 6: half of layers 5 and 6


# ------------------------------------------------------------------ O6: the top interval of the table ------
def curved_top_table():
    t = wl.tf_ramp(0.05).astype(np.float64)
    t[253] = (0.9, 0.1, 0.2, 0.1)
    t[254] = (0.2, 0.8, 0.3, 0.2)
    t[255] = (0.1, 0.3, 0.7, 0.9)          # not on the line through entries 253 and 254
    return t.astype(np.float32)


@pytest.mark.parametrize("x", [252.5, 253.0, 253.5, 254.0, 254.25, 254.5, 254.999, 255.0, 300.0])
def test_top_interval_of_the_table_interpolates_between_entries_254_and_255(oracle, x):
    """vro.c lookup: m = min(floor x, 254).  With vmin = 0, vmax = 255 a value IS its table position."""
    tab = curved_top_table()
    got = oracle.classify(tab, 0.0, 255.0, 1.0, x)
    want = np.array([np.interp(min(x, 255.0), np.arange(256.0), tab[:, c].astype(np.float64)) for c in range(4)])
    assert np.abs(got - want).max() < 1e-12, (x, got, want)
    if x == 254.5:                          # spelled out: half way between entries 254 and 255
        assert abs(got[3] - 0.55) < 1e-7 and abs(got[1] - 0.55) < 1e-7


def test_constant_cube_in_the_top_interval_has_the_closed_form_opacity(oracle):
    """The same rule through the renderer: a cube of 254.5 everywhere, 4 samples per ray at step 1 ->
    A = 1 - (1 - 0.55)^4 and C = A * colour(254.5)  (north_star closed form 1, at the top of the table)."""
    tab = curved_top_table()
    cube = np.full((4, 4, 4), 254.5, dtype=np.float32)
    cs, W, H, *_ = wl.axis_camera((4, 4, 4), 2, 1)
    r = oracle.render(cube, tab, 0.0, 255.0, (1, 1, 1), oracle_camera(oracle, cs), W, H, 1.0, 0, 0.0, route=0)
    t64 = tab.astype(np.float64)
    a = 0.5 * (t64[254, 3] + t64[255, 3])
    A = 1.0 - (1.0 - a) ** 4
    col = 0.5 * (t64[254, :3] + t64[255, :3])
    assert r["samples"] == 4 * W * H
    assert np.abs(r["rgba"][..., 3] - A).max() < 1e-6
    assert np.abs(r["rgba"][..., :3] - A * col).max() < 1e-6
