"""GPU parity of the slab-staged caster (slab.cuh: shared-memory windows filled by bulk tensor copies) against the
CPU oracle, and against the row-cache caster, through the C ABI.  Same gates as tests/test_gpu_parity.py."""
import numpy as np
import pytest

from paper_1008_0135_b200 import workloads as wl

pytestmark = pytest.mark.gpu

TOL_EA = 1e-4
TOL_ERT = 5e-3


@pytest.fixture(scope="module")
def vr():
    import torch
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    from paper_1008_0135_b200 import vr as binding
    binding.lib()
    return binding


def ocam(oracle, cs):
    return oracle.make_camera(cs.view, cs.projection, cs.fovy_deg, cs.ortho_half_h)


def noisy_cube(dims, seed):
    import torch
    g = torch.Generator(device="cuda").manual_seed(seed)
    cube = torch.randn((dims[2], dims[1], dims[0]), generator=g, device="cuda", dtype=torch.float32)
    zz, yy, xx = torch.meshgrid(torch.arange(dims[2], device="cuda"), torch.arange(dims[1], device="cuda"),
                                torch.arange(dims[0], device="cuda"), indexing="ij")
    c = [d / 2.0 for d in dims]
    cube += 6.0 * torch.exp(-((xx - c[0]) ** 2 + (yy - c[1]) ** 2 + (zz - c[2]) ** 2) / (2.0 * (min(dims) / 5.0) ** 2))
    return cube.contiguous()


def render(vr, vol, cs, W, H, step, mode, ert, slab_mode, want_scalar=False):
    import torch
    vol.vr_set_slab_staging(slab_mode)
    sc = torch.empty((H, W), dtype=torch.float32, device="cuda") if want_scalar else None
    out = vol.vr_render(vr.camera_from_spec(cs), W, H, step, mode, ert, out_scalar=sc)
    torch.cuda.synchronize()
    info = vol.vr_get_slab_info()
    return out.cpu().numpy(), (sc.cpu().numpy() if want_scalar else None), info


# az/el chosen so that each axis is the dominant one, in both directions
VIEWS = [(30.0, 20.0, 2), (210.0, -15.0, 2), (100.0, 10.0, 0), (280.0, 25.0, 0), (20.0, 70.0, 1), (140.0, -65.0, 1),
         (0.0, 0.0, 2), (90.0, 0.0, 0)]


@pytest.mark.parametrize("az,el,dom", VIEWS)
def test_slab_caster_matches_oracle_every_dominant_axis(vr, oracle, az, el, dom):
    dims = (61, 35, 47)
    cube = noisy_cube(dims, 11)
    table = wl.tf_ramp(0.08)
    vmin, vmax = -3.0, 9.0
    vol = vr.Volume(cube)
    vol.vr_set_transfer_function(table, vmin, vmax)
    cs = wl.orbit_camera(dims, az, el, wl.PROJ_ORTHO)
    W, H = 150, 131
    for bricks in [(1, 1, 1), (2, 2, 2), (3, 1, 2)]:
        vol.vr_set_bricks(*bricks)
        for step in (0.5, 0.25):
            got, _, info = render(vr, vol, cs, W, H, step, 0, 0.0, 2)
            assert info["used"] and info["dominant_axis"] == dom, info
            ref = oracle.render(cube.cpu().numpy(), table, vmin, vmax, bricks, ocam(oracle, cs), W, H, step, 0, 0.0,
                                route=0)["rgba"]
            err = np.abs(got - ref).max(axis=(0, 1))
            assert (err <= TOL_EA).all(), (bricks, step, err)
            assert ref[..., 3].max() > 0.3
            assert (got[ref[..., 3] == 0] == 0).all()
            other, _, info0 = render(vr, vol, cs, W, H, step, 0, 0.0, 0)
            assert not info0["used"]
            assert np.abs(got - other).max() <= 2e-5
    vol.close()


def test_slab_caster_mip_and_termination(vr, oracle):
    dims = (70, 44, 52)
    cube = noisy_cube(dims, 12)
    table = wl.tf_ramp(0.2)
    vmin, vmax = -3.0, 9.0
    vol = vr.Volume(cube)
    vol.vr_set_transfer_function(table, vmin, vmax)
    vol.vr_set_bricks(2, 1, 2)
    W, H = 160, 120
    for az, el in [(30.0, 20.0), (100.0, 10.0), (20.0, 70.0)]:
        cs = wl.orbit_camera(dims, az, el, wl.PROJ_ORTHO)
        got, sc, info = render(vr, vol, cs, W, H, 0.5, 1, 0.0, 2, want_scalar=True)
        assert info["used"]
        ref = oracle.render(cube.cpu().numpy(), table, vmin, vmax, (2, 1, 2), ocam(oracle, cs), W, H, 0.5, 1, 0.0, route=0)
        m = ref["scalar"]
        hit = np.isfinite(m)
        assert (np.isfinite(sc) == hit).all()
        assert (np.abs(sc[hit] - m[hit]) <= 1e-4 * np.maximum(1.0, np.abs(m[hit]))).all()
        assert np.abs(got - ref["rgba"]).max() <= 1e-4
        # termination: against the ERT-off and the ERT-on oracle (A7's bound)
        got_t, _, info = render(vr, vol, cs, W, H, 0.5, 0, 0.9, 2)
        assert info["used"]
        ref_off = oracle.render(cube.cpu().numpy(), table, vmin, vmax, (2, 1, 2), ocam(oracle, cs), W, H, 0.5, 0, 0.0, route=1)["rgba"]
        ref_on = oracle.render(cube.cpu().numpy(), table, vmin, vmax, (2, 1, 2), ocam(oracle, cs), W, H, 0.5, 0, 0.9, route=1)["rgba"]
        assert np.abs(got_t - ref_on).max() <= TOL_ERT
        assert np.abs(got_t - ref_off).max() <= 1.0 - 0.9 + 1e-6
    vol.close()


def test_slab_caster_config0_and_nan_block(vr, oracle):
    w = wl.config(0)
    cube = w.cube("cuda").clone()
    vol = vr.Volume(cube)
    vol.vr_set_transfer_function(w.table, w.vmin, w.vmax)
    cs = w.camera()
    got, _, info = render(vr, vol, cs, w.W, w.H, w.step, 0, 0.0, 1)      # auto picks the slab caster for config 0
    assert info["used"], info
    ref = oracle.render(cube.cpu().numpy(), w.table, w.vmin, w.vmax, (1, 1, 1), ocam(oracle, cs), w.W, w.H, w.step, 0, 0.0,
                        route=0)["rgba"]
    assert np.abs(got - ref).max() <= TOL_EA
    vol.close()
    cube[20:30, 10:25, 30:40] = float("nan")                              # blanked voxels (A14)
    vol = vr.Volume(cube)
    vol.vr_set_transfer_function(w.table, w.vmin, w.vmax)
    vol.vr_set_bricks(2, 2, 1)
    got, _, info = render(vr, vol, cs, w.W, w.H, w.step, 0, 0.0, 2)
    assert info["used"]
    ref = oracle.render(cube.cpu().numpy(), w.table, w.vmin, w.vmax, (2, 2, 1), ocam(oracle, cs), w.W, w.H, w.step, 0, 0.0,
                        route=0)["rgba"]
    assert np.isfinite(got).all()
    assert np.abs(got - ref).max() <= TOL_EA
    vol.close()


def test_slab_caster_not_used_where_it_does_not_apply(vr):
    w = wl.config(0)
    cube = w.cube("cuda")
    vol = vr.Volume(cube)
    vol.vr_set_transfer_function(w.table, w.vmin, w.vmax)
    cs = w.camera()
    mask = np.ones(w.dims[2], dtype=np.uint8)
    mask[10:20] = 0
    vol.vr_set_channel_mask(mask)
    _, _, info = render(vr, vol, cs, 64, 64, 0.5, 0, 0.0, 2)
    assert not info["used"]                                               # channel masks: row-cache caster
    vol.vr_set_channel_mask(None)
    _, _, info = render(vr, vol, cs, 64, 64, 0.5, 0, 0.0, 0)
    assert not info["used"]
    vol.close()


PVIEWS = [(30.0, 20.0), (215.0, -10.0), (95.0, 15.0), (10.0, 75.0), (0.0, 0.0)]


@pytest.mark.parametrize("az,el", PVIEWS)
def test_slab_caster_perspective_matches_oracle(vr, oracle, az, el):
    """Perspective frames: the window of a slab follows the diverging rays (several window sizes per frame)."""
    dims = (72, 50, 41)
    cube = noisy_cube(dims, 13)
    table = wl.tf_ramp(0.06)
    vmin, vmax = -3.0, 9.0
    vol = vr.Volume(cube)
    vol.vr_set_transfer_function(table, vmin, vmax)
    cs = wl.orbit_camera(dims, az, el, wl.PROJ_PERSP)
    W, H = 200, 170
    for bricks, step, ert in [((1, 1, 1), 0.5, 0.0), ((2, 2, 1), 0.25, 0.0), ((2, 3, 2), 0.5, 0.995)]:
        vol.vr_set_bricks(*bricks)
        got, _, info = render(vr, vol, cs, W, H, step, 0, ert, 2)
        assert info["used"], info
        ref = oracle.render(cube.cpu().numpy(), table, vmin, vmax, bricks, ocam(oracle, cs), W, H, step, 0, ert, route=1)["rgba"]
        err = np.abs(got - ref).max()
        assert err <= (TOL_ERT if ert > 0 else TOL_EA), (bricks, step, ert, err)
        assert ref[..., 3].max() > 0.3
        other, _, info0 = render(vr, vol, cs, W, H, step, 0, ert, 0)
        assert not info0["used"]
        if ert == 0:
            assert np.abs(got - other).max() <= 2e-5
    got, sc, info = render(vr, vol, cs, W, H, 0.5, 1, 0.0, 2, want_scalar=True)
    assert info["used"]
    ref = oracle.render(cube.cpu().numpy(), table, vmin, vmax, (2, 3, 2), ocam(oracle, cs), W, H, 0.5, 1, 0.0, route=0)
    m = ref["scalar"]
    hit = np.isfinite(m)
    assert (np.isfinite(sc) == hit).all()
    assert (np.abs(sc[hit] - m[hit]) <= 1e-4 * np.maximum(1.0, np.abs(m[hit]))).all()
    vol.close()


def test_slab_caster_perspective_eye_inside_or_wide(vr, oracle):
    """An eye inside the cube and a very wide field of view: rays that do not advance along the dominant axis make the
    frame ineligible (row-cache caster); either way the frame matches the oracle."""
    import dataclasses
    dims = (48, 40, 36)
    cube = noisy_cube(dims, 14)
    table = wl.tf_ramp(0.1)
    vol = vr.Volume(cube)
    vol.vr_set_transfer_function(table, -3.0, 9.0)
    vol.vr_set_bricks(2, 2, 2)
    eye = (20.0, 18.0, 15.0)
    view = wl.look_at(eye, (40.0, 30.0, 30.0))
    for fov in (45.0, 150.0):
        cs = wl.CameraSpec(view=view, projection=wl.PROJ_PERSP, fovy_deg=fov, ortho_half_h=1.0)
        got, _, info = render(vr, vol, cs, 96, 80, 0.5, 0, 0.0, 2)
        ref = oracle.render(cube.cpu().numpy(), table, -3.0, 9.0, (2, 2, 2), ocam(oracle, cs), 96, 80, 0.5, 0, 0.0, route=0)["rgba"]
        assert np.abs(got - ref).max() <= TOL_EA, (fov, info)
    vol.close()


def test_slab_caster_coarse_steps_and_tiny_images(vr, oracle):
    """Steps longer than a slab is thick (a ray then has slabs without a sample of its own) and images smaller than one
    CTA tile."""
    dims = (90, 64, 77)
    cube = noisy_cube(dims, 15)
    table = wl.tf_ramp(0.15)
    vol = vr.Volume(cube)
    vol.vr_set_transfer_function(table, -3.0, 9.0)
    vol.vr_set_bricks(2, 1, 3)
    for (az, el), (W, H), step in [((30.0, 20.0), (300, 260), 2.5), ((100.0, 10.0), (300, 260), 9.3), ((20.0, 70.0), (11, 5), 0.5),
                                   ((200.0, -30.0), (1, 1), 0.25)]:
        cs = wl.orbit_camera(dims, az, el, wl.PROJ_ORTHO)
        got, _, info = render(vr, vol, cs, W, H, step, 0, 0.0, 2)
        assert info["used"] == (W > 16), info                 # a few pixels across the cube: the window cannot fit
        ref = oracle.render(cube.cpu().numpy(), table, -3.0, 9.0, (2, 1, 3), ocam(oracle, cs), W, H, step, 0, 0.0, route=0)["rgba"]
        assert np.abs(got - ref).max() <= TOL_EA, (az, el, W, H, step, np.abs(got - ref).max())
    vol.close()


def test_slab_caster_image_smaller_than_a_tile(vr, oracle):
    dims = (9, 7, 8)
    cube = noisy_cube(dims, 16)
    table = wl.tf_ramp(0.3)
    vol = vr.Volume(cube)
    vol.vr_set_transfer_function(table, -3.0, 9.0)
    for (W, H) in [(11, 5), (3, 2), (1, 1)]:
        cs = wl.orbit_camera(dims, 40.0, 25.0, wl.PROJ_ORTHO)
        got, _, info = render(vr, vol, cs, W, H, 0.25, 0, 0.0, 2)
        assert info["used"] == (W == 11), info                # windows are sized for a whole 16x8-pixel tile
        ref = oracle.render(cube.cpu().numpy(), table, -3.0, 9.0, (1, 1, 1), ocam(oracle, cs), W, H, 0.25, 0, 0.0, route=0)["rgba"]
        assert np.abs(got - ref).max() <= TOL_EA
    vol.close()
