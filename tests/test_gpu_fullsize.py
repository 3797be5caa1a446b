"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (config 3:
2048x2048x1600 f32, 2x2x2 bricks, 1024^2, perspective, step 1), on sampled outputs the oracle can
compute one by one (a lattice of every 8th pixel in x and y = 16384 rays), plus properties that
hold at any size (library max for the axis-aligned MIP, sample-count law for orthographic views).
Needs ~55 GB of HBM and ~30 GB of host RAM; skipped (loudly) when the box has less."""
import numpy as np
import pytest

from paper_1008_0135_b200 import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def vr():
    import torch
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    from paper_1008_0135_b200 import vr as binding
    binding.lib()
    return binding


def _enough_memory(n_bytes):
    import torch
    free, _ = torch.cuda.mem_get_info()
    try:
        import psutil
        host = psutil.virtual_memory().available
    except Exception:
        host = 1 << 62
    return free > 2.2 * n_bytes and host > 1.3 * n_bytes


@pytest.fixture(scope="module")
def gass(vr):
    """Config 3's cube on the device, its host copy, and a volume handle with table and bricks set."""
    import torch
    w = wl.config(3)
    n_bytes = 4 * w.dims[0] * w.dims[1] * w.dims[2]
    if not _enough_memory(n_bytes):
        pytest.skip("not enough device/host memory for the 26.8 GB cube on this box")
    cube = w.cube("cuda")
    torch.cuda.synchronize()
    host = cube.cpu().numpy()
    vol = vr.Volume(cube)
    vol.vr_set_transfer_function(w.table, w.vmin, w.vmax)
    vol.vr_set_bricks(*w.bricks)
    yield w, cube, host, vol
    vol.close()


def report(tag, got, ref, gate):
    """Print the measured per-channel margin (pytest -s / the captured log keeps it on record)."""
    err = np.abs(np.asarray(got, dtype=np.float64) - ref).reshape(-1, ref.shape[-1] if ref.ndim > 1 else 1).max(axis=0)
    print(f"[margin] {tag}: max abs err per channel {np.array2string(err, precision=3)} gate {gate:g} "
          f"({err.max() / gate:.2f} of the gate)")


def lattice(W, H, stride=8, offset=3):
    xs = np.arange(offset, W, stride, dtype=np.int32)
    ys = np.arange(offset, H, stride, dtype=np.int32)
    yy, xx = np.meshgrid(ys, xs, indexing="ij")
    return xx.reshape(-1), yy.reshape(-1)


@pytest.mark.parametrize("az", [30.0, 90.0, 200.0])
def test_config3_full_size_sampled_pixels(vr, oracle, gass, az):
    import torch
    w, cube, host, vol = gass
    cs = w.camera(az_deg=az)
    cam = vr.camera_from_spec(cs)
    oc = oracle.make_camera(cs.view, cs.projection, cs.fovy_deg, cs.ortho_half_h)
    px, py = lattice(w.W, w.H)
    ref_off = oracle.render_pixels(host, w.table, w.vmin, w.vmax, w.bricks, oc, w.W, w.H, w.step, w.mode, 0.0, 0,
                                   px, py)["rgba"]
    ref_on = oracle.render_pixels(host, w.table, w.vmin, w.vmax, w.bricks, oc, w.W, w.H, w.step, w.mode,
                                  w.ert_alpha, 1, px, py)["rgba"]
    got_off = vol.vr_render(cam, w.W, w.H, w.step, w.mode, 0.0).cpu().numpy()[py, px]
    got_on = vol.vr_render(cam, w.W, w.H, w.step, w.mode, w.ert_alpha).cpu().numpy()[py, px]
    assert ref_off[:, 3].max() > 0.5 and (ref_off[:, 3] > 0).mean() > 0.3       # a real picture
    report(f"cfg3 az {az:g} ERT off", got_off, ref_off, 1e-4)
    report(f"cfg3 az {az:g} ERT on vs oracle ERT on", got_on, ref_on, 5e-3)
    assert np.abs(got_off - ref_off).max() <= 1e-4, np.abs(got_off - ref_off).max(axis=0)
    assert np.abs(got_on - ref_off).max() <= 5e-3
    assert np.abs(got_on - ref_on).max() <= 5e-3


def test_config3_full_size_bricks_1_8_64_agree(vr, oracle, gass):
    """north_star closed form 4 at full size: 1, 8 and 64 bricks give the unbricked oracle frame (each within
    1e-4 on the pixel lattice) and therefore agree with one another within 2e-4 everywhere."""
    w, cube, host, vol = gass
    cs = w.camera(az_deg=40.0)
    cam = vr.camera_from_spec(cs)
    oc = oracle.make_camera(cs.view, cs.projection, cs.fovy_deg, cs.ortho_half_h)
    px, py = lattice(w.W, w.H)
    ref = oracle.render_pixels(host, w.table, w.vmin, w.vmax, (1, 1, 1), oc, w.W, w.H, w.step, w.mode, 0.0, 0,
                               px, py)["rgba"]
    frames = []
    for b in ((1, 1, 1), (2, 2, 2), (4, 4, 4)):
        vol.vr_set_bricks(*b)
        f = vol.vr_render(cam, w.W, w.H, w.step, w.mode, 0.0).cpu().numpy()
        report(f"cfg3 az 40 bricks {b}", f[py, px], ref, 1e-4)
        assert np.abs(f[py, px] - ref).max() <= 1e-4, (b, np.abs(f[py, px] - ref).max(axis=0))
        frames.append(f)
    vol.vr_set_bricks(*w.bricks)
    assert np.abs(frames[1] - frames[0]).max() <= 2e-4
    assert np.abs(frames[2] - frames[0]).max() <= 2e-4


def test_full_size_axis_mip_equals_library_max(vr, gass):
    """north_star closed form 2 at the full 26.8 GB: axis-aligned orthographic MIP = torch.amax."""
    import torch
    w, cube, host, vol = gass
    cs, W, H, ra, rs, ua, us = wl.axis_camera(w.dims, 2, -1)        # looking down -z at the sky plane
    sc = torch.empty((H, W), dtype=torch.float32, device="cuda")
    vol.vr_render(vr.camera_from_spec(cs), W, H, 1.0, 1, 0.0, out_scalar=sc)
    m = torch.amax(cube, dim=0)                                     # [y][x]
    if rs < 0:
        m = torch.flip(m, dims=[1])
    torch.cuda.synchronize()
    assert (ra, ua) == (0, 1)
    err = (sc - m).abs().max().item()
    assert err <= 1e-4 * max(1.0, m.abs().max().item()), err


def test_full_size_ortho_sample_count_law(vr, gass):
    """Any size: for an orthographic view S = V / (p^2 * step) within 1 % (p = voxels per pixel)."""
    w, cube, host, vol = gass
    cs = wl.orbit_camera(w.dims, 30.0, 20.0, wl.PROJ_ORTHO)
    samples, sectors = vol.vr_measure(vr.camera_from_spec(cs), 1024, 1024, 1.0, 0, 0.0)
    V = float(w.dims[0]) * w.dims[1] * w.dims[2]
    p = 2.0 * cs.ortho_half_h / 1024.0
    assert abs(samples / (V / (p * p)) - 1.0) < 0.01
    total_sectors = (-(-(w.dims[0] + 9) // 8)) * (-(-(w.dims[1] + 2) // 8)) * (-(-(w.dims[2] + 2) // 8)) * 64
    assert 0.5 * total_sectors < sectors <= total_sectors


# ---- BASELINE.json configs[4]: the sweep's corners at full size (config 3's cube, ORTHO az 30 el 20, ERT off) ----
@pytest.mark.parametrize("size,step,bricks", [(1024, 0.5, (2, 2, 2)), (1024, 0.25, (2, 2, 2)), (2048, 1.0, (2, 2, 2)),
                                              (1024, 0.5, (4, 4, 4)), (512, 0.25, (1, 1, 1)), (2048, 0.25, (2, 2, 2))])
def test_config4_sweep_points_full_size(vr, oracle, gass, size, step, bricks):
    """Step < 1 exercises what step 1 does not: the per-step opacity correction of the table (O6), the hi+lo
    split of the fp32 step vector, several samples per voxel in the row cache (PAPER.md:185 sampling distance;
    PAPER.md:207 output sizes).  16384-pixel lattice, gate 1e-4 per channel, margins printed."""
    w, cube, host, vol = gass
    cs = wl.orbit_camera(w.dims, 30.0, 20.0, wl.PROJ_ORTHO)
    oc = oracle.make_camera(cs.view, cs.projection, cs.fovy_deg, cs.ortho_half_h)
    px, py = lattice(size, size, stride=size // 128)
    ref = oracle.render_pixels(host, w.table, w.vmin, w.vmax, bricks, oc, size, size, step, 0, 0.0, 0, px, py)["rgba"]
    vol.vr_set_bricks(*bricks)
    assert ref[:, 3].max() > 0.5
    # both casters at full size: the row-cache caster (slab staging off) and the slab-staged one wherever its window fits
    used = []
    for slab_mode in (0, 2, 1):
        vol.vr_set_slab_staging(slab_mode)
        got = vol.vr_render(vr.camera_from_spec(cs), size, size, step, 0, 0.0).cpu().numpy()[py, px]
        info = vol.vr_get_slab_info()
        used.append(info["used"])
        if slab_mode == 2 and not info["used"]:
            continue                                          # window does not fit: same frame as mode 0
        name = "slab-staged" if info["used"] else "row-cache"
        report(f"cfg4 EA {size}^2 step {step} bricks {bricks} [{name} caster, staging mode {slab_mode}]", got, ref, 1e-4)
        assert np.abs(got - ref).max() <= 1e-4, (slab_mode, np.abs(got - ref).max(axis=0))
    vol.vr_set_bricks(*w.bricks)
    assert not used[0]
    if size == 2048:
        assert used[1] and used[2]                            # the dense points run on the slab caster by default


def test_slab_caster_x_dominant_view_full_size(vr, oracle, gass):
    """A view whose dominant axis is x (az 100, el 10) at 2048^2, step 1/2: the slab caster reads its z-fastest second
    copy of the 26.8 GB cube (`transpose_kernel`).  Same lattice and gate as the other config-4 points."""
    w, cube, host, vol = gass
    size, step, bricks = 2048, 0.5, (2, 2, 2)
    cs = wl.orbit_camera(w.dims, 100.0, 10.0, wl.PROJ_ORTHO)
    oc = oracle.make_camera(cs.view, cs.projection, cs.fovy_deg, cs.ortho_half_h)
    px, py = lattice(size, size, stride=size // 128)
    ref = oracle.render_pixels(host, w.table, w.vmin, w.vmax, bricks, oc, size, size, step, 0, 0.0, 0, px, py)["rgba"]
    assert ref[:, 3].max() > 0.5
    vol.vr_set_bricks(*bricks)
    for slab_mode in (0, 2):
        vol.vr_set_slab_staging(slab_mode)
        got = vol.vr_render(vr.camera_from_spec(cs), size, size, step, 0, 0.0).cpu().numpy()[py, px]
        info = vol.vr_get_slab_info()
        assert info["used"] == (slab_mode == 2) and (slab_mode == 0 or info["dominant_axis"] == 0), info
        report(f"x-dominant view {size}^2 step {step} [{'slab-staged' if info['used'] else 'row-cache'} caster]", got, ref, 1e-4)
        assert np.abs(got - ref).max() <= 1e-4
    print(f"[info] linear copies: {info['linear_bytes'] / 1e9:.2f} GB, made in {info['linearize_ms']:.1f} ms")
    vol.vr_set_slab_staging(1)
    vol.vr_set_bricks(*w.bricks)


def test_config4_mip_point_oblique_full_size(vr, oracle, gass):
    """The sweep's MIP point (8 bricks, 1024^2, step 1) on the oblique az 30 / el 20 view: raw maxima within
    1e-4 * max(1, |M|) of the oracle's, colours within 1e-4."""
    import torch
    w, cube, host, vol = gass
    cs = wl.orbit_camera(w.dims, 30.0, 20.0, wl.PROJ_ORTHO)
    oc = oracle.make_camera(cs.view, cs.projection, cs.fovy_deg, cs.ortho_half_h)
    px, py = lattice(1024, 1024)
    ref = oracle.render_pixels(host, w.table, w.vmin, w.vmax, w.bricks, oc, 1024, 1024, 1.0, 1, 0.0, 1, px, py)
    sc = torch.empty((1024, 1024), dtype=torch.float32, device="cuda")
    got = vol.vr_render(vr.camera_from_spec(cs), 1024, 1024, 1.0, 1, 0.0, out_scalar=sc).cpu().numpy()[py, px]
    sc = sc.cpu().numpy()[py, px]
    hit = np.isfinite(ref["scalar"])
    assert hit.mean() > 0.3 and (np.isfinite(sc) == hit).all()
    scale = np.maximum(1.0, np.abs(ref["scalar"][hit]))
    rel = np.abs(sc[hit] - ref["scalar"][hit]) / scale
    print(f"[margin] cfg4 MIP oblique: max |M - M_oracle| / max(1,|M|) = {rel.max():.3e} gate 1e-4; colours "
          f"{np.abs(got - ref['rgba']).max():.3e}")
    assert rel.max() <= 1e-4
    assert np.abs(got - ref["rgba"]).max() <= 1e-4


def test_config2_full_size_sampled_pixels(vr, oracle):
    """Config 2 (HIPASS-shaped 1721x1721x1024, 12.1 GB, orthographic, ERT off, piecewise table)."""
    import torch
    w = wl.config(2)
    if not _enough_memory(4 * w.dims[0] * w.dims[1] * w.dims[2]):
        pytest.skip("not enough memory for the 12.1 GB cube on this box")
    cube = w.cube("cuda")
    host = cube.cpu().numpy()
    vol = vr.Volume(cube)
    vol.vr_set_transfer_function(w.table, w.vmin, w.vmax)
    vol.vr_set_bricks(*w.bricks)
    cs = w.camera()
    oc = oracle.make_camera(cs.view, cs.projection, cs.fovy_deg, cs.ortho_half_h)
    px, py = lattice(w.W, w.H)
    ref = oracle.render_pixels(host, w.table, w.vmin, w.vmax, w.bricks, oc, w.W, w.H, w.step, w.mode, 0.0, 0, px, py)["rgba"]
    got = vol.vr_render(vr.camera_from_spec(cs), w.W, w.H, w.step, w.mode, 0.0).cpu().numpy()[py, px]
    vol.close()
    assert ref[:, 3].max() > 0.3
    report("cfg2 full size", got, ref, 1e-4)
    assert np.abs(got - ref).max() <= 1e-4, np.abs(got - ref).max(axis=0)
