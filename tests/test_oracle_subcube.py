"""Pins of the oracle's sub-cube / channel-range rule S1 (PAPER.md:128 manual sub-cube, PAPER.md:138 channels
enabled or disabled): closed form on a constant cube, library max over the enabled channels for an axis-aligned
MIP, the 1-D cumprod recurrence over the enabled channels, complementary sub-cubes composited = whole cube,
whole-cube sub-cube = no sub-cube."""
import numpy as np

from paper_1008_0135_b200 import workloads as wl


def _cam(oracle, cs):
    return oracle.make_camera(cs.view, cs.projection, cs.fovy_deg, cs.ortho_half_h)


def test_whole_cube_subcube_is_identity(oracle):
    dims = (20, 14, 12)
    cube = wl.cube_blobs(dims, 3, "cpu", n_blobs=3, amp=6.0, sigma=3.0).numpy()
    tab = wl.tf_ramp(0.2)
    for proj, route, bricks in ((0, 0, (1, 1, 1)), (1, 1, (2, 1, 2))):
        cs = wl.orbit_camera(dims, 40.0, 25.0, proj)
        a = oracle.render(cube, tab, -3, 8, bricks, _cam(oracle, cs), 30, 26, 0.5, 0, 0.0, route=route)
        b = oracle.render(cube, tab, -3, 8, bricks, _cam(oracle, cs), 30, 26, 0.5, 0, 0.0, route=route,
                          subcube=((0, 0, 0), dims))
        assert np.array_equal(a["rgba"], b["rgba"]) and a["samples"] == b["samples"]


def test_constant_cube_channel_range_closed_form(oracle):
    """Axis-aligned ray, step 1: n = number of enabled channels, A = 1 - (1-a)^n (north_star closed form 1)."""
    dims = (16, 16, 64)
    cube = np.full((64, 16, 16), 2.5, dtype=np.float32)
    tab = wl.tf_ramp(0.1)                                   # alpha(2.5) over [-3,8] = 0.05
    cs, W, H, *_ = wl.axis_camera(dims, 2, 1)
    for z0, z1 in ((0, 64), (10, 30), (63, 64), (17, 17)):
        r = oracle.render(cube, tab, -3, 8, (1, 1, 1), _cam(oracle, cs), W, H, 1.0, 0, 0.0, route=0,
                          subcube=((0, 0, z0), (16, 16, z1)))
        A = 1.0 - 0.95 ** (z1 - z0)
        assert np.allclose(r["rgba"][..., 3], A, atol=2e-7)
        assert r["samples"] == W * H * (z1 - z0)


def test_axis_mip_over_enabled_channels_equals_library_max(oracle):
    dims = (18, 14, 22)
    cube = wl.cube_blobs(dims, 4, "cpu", n_blobs=3, amp=6.0, sigma=3.0).numpy()
    cs, W, H, ra, rs, ua, us = wl.axis_camera(dims, 2, -1)
    z0, z1 = 5, 16
    r = oracle.render(cube, wl.tf_ramp(0.1), -3, 8, (1, 2, 2), _cam(oracle, cs), W, H, 1.0, 1, 0.0, route=1,
                      subcube=((0, 0, z0), (dims[0], dims[1], z1)))
    m = cube[z0:z1].max(axis=0)                             # [y][x]
    if rs < 0:
        m = m[:, ::-1]
    assert np.abs(r["scalar"] - m).max() <= 1e-6


def test_axis_ea_over_enabled_channels_equals_cumprod(oracle):
    dims = (10, 9, 24)
    cube = wl.cube_blobs(dims, 5, "cpu", n_blobs=2, amp=6.0, sigma=3.0).numpy()
    tab = wl.tf_ramp(0.3)
    cs, W, H, ra, rs, ua, us = wl.axis_camera(dims, 2, 1)   # looking towards +z: front = small z
    z0, z1 = 4, 19
    r = oracle.render(cube, tab, -3, 8, (1, 1, 1), _cam(oracle, cs), W, H, 1.0, 0, 0.0, route=0,
                      subcube=((0, 0, z0), (dims[0], dims[1], z1)))["rgba"]
    xp = -3 + 11 * np.arange(256) / 255.0
    v = cube[z0:z1].astype(np.float64)                      # [k][y][x]
    a = np.interp(v, xp, tab[:, 3].astype(np.float64))
    trans = np.cumprod(np.concatenate([np.ones((1,) + a.shape[1:]), 1 - a[:-1]]), axis=0)
    A = 1 - np.prod(1 - a, axis=0)
    Cr = (trans * a * np.interp(v, xp, tab[:, 0].astype(np.float64))).sum(axis=0)
    if rs < 0:
        A, Cr = A[:, ::-1], Cr[:, ::-1]
    assert np.abs(r[..., 3] - A).max() <= 1e-6 and np.abs(r[..., 0] - Cr).max() <= 1e-6


def test_complementary_subcubes_composite_to_the_whole(oracle):
    """Every lattice sample lies in exactly one of two complementary sub-cubes; "over" of the two = the frame."""
    dims = (22, 18, 14)
    cube = wl.cube_blobs(dims, 6, "cpu", n_blobs=3, amp=6.0, sigma=3.0).numpy()
    tab = wl.tf_ramp(0.25)
    for proj in (0, 1):
        cs = wl.orbit_camera(dims, 30.0, 20.0, proj)       # eye at +x,+y,+z looking at the centre: large x in front
        cam = _cam(oracle, cs)
        full = oracle.render(cube, tab, -3, 8, (2, 2, 1), cam, 28, 24, 0.5, 0, 0.0, route=1)
        front = oracle.render(cube, tab, -3, 8, (2, 2, 1), cam, 28, 24, 0.5, 0, 0.0, route=1,
                              subcube=((9, 0, 0), dims))
        back = oracle.render(cube, tab, -3, 8, (2, 2, 1), cam, 28, 24, 0.5, 0, 0.0, route=1,
                             subcube=((0, 0, 0), (9, dims[1], dims[2])))
        assert front["samples"] + back["samples"] == full["samples"]
        f, b = front["rgba"].astype(np.float64), back["rgba"].astype(np.float64)
        comp = f.copy()
        comp[..., :3] += (1 - f[..., 3:4]) * b[..., :3]
        comp[..., 3] = 1 - (1 - f[..., 3]) * (1 - b[..., 3])
        assert np.abs(comp - full["rgba"]).max() <= 3e-7
