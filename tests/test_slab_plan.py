"""Host logic of the slab-staged caster (no GPU): the window the host sizes and the placement rule the kernel applies
(include/vr.h, vr_plan_slab) must hold the 2x2x2 footprint of every sample a CTA tile can take inside a slab.  The rays
are re-derived here from the camera with DESIGN.md O1/O2, independently of the library's affine description."""
import numpy as np
import pytest

from paper_1008_0135_b200 import workloads as wl

PAD = np.array([8.0, 1.0, 1.0])
CTA_W, CTA_H = 16, 8


@pytest.fixture(scope="module")
def vr():
    from paper_1008_0135_b200 import vr as binding
    binding.lib()
    return binding


def rays_of(cs, W, H, px, py):
    """O1/O2 in numpy: origins and directions of the pixels (px, py), in voxel coordinates."""
    M = np.asarray(cs.view, dtype=np.float64).reshape(4, 4)
    R, tau = M[:3, :3], M[:3, 3]
    right, up, fwd = R[0] / np.linalg.norm(R[0]), R[1] / np.linalg.norm(R[1]), -R[2] / np.linalg.norm(R[2])
    eye = -R.T @ tau
    u = 2.0 * (px + 0.5) / W - 1.0
    v = 2.0 * (py + 0.5) / H - 1.0
    asp = W / H
    if cs.projection == wl.PROJ_ORTHO:
        h = float(np.float32(cs.ortho_half_h))           # the camera struct carries float32 (include/vr.h)
        o = eye[None, :] + (u * h * asp)[:, None] * right[None, :] + (v * h)[:, None] * up[None, :]
        d = np.repeat(fwd[None, :], len(px), axis=0)
    else:
        T = np.tan(np.radians(0.5 * float(np.float32(cs.fovy_deg))))
        o = np.repeat(eye[None, :], len(px), axis=0)
        d = fwd[None, :] + (u * T * asp)[:, None] * right[None, :] + (v * T)[:, None] * up[None, :]
        d /= np.linalg.norm(d, axis=1)[:, None]
    return o, d


def position_at(o, d, dom, c):
    """Padded position of each ray where its padded dominant coordinate equals c."""
    q = o + PAD[None, :] - 0.5
    t = (c - q[:, dom]) / d[:, dom]
    return q + t[:, None] * d


CASES = [
    # dims, bricks, az, el, projection, image, step
    ((2048, 2048, 1600), (2, 2, 2), 30.0, 20.0, wl.PROJ_ORTHO, 2048, 0.25),
    ((1024, 1024, 1024), (2, 2, 2), 90.0, 0.0, wl.PROJ_ORTHO, 1024, 1.0),
    ((1024, 1024, 1024), (1, 1, 1), 130.0, 0.0, wl.PROJ_ORTHO, 1024, 1.0),
    ((300, 200, 260), (3, 1, 2), 20.0, 70.0, wl.PROJ_ORTHO, 400, 0.5),
    ((300, 200, 260), (2, 2, 2), 215.0, -10.0, wl.PROJ_PERSP, 700, 0.5),
    ((512, 512, 256), (2, 2, 1), 30.0, 20.0, wl.PROJ_PERSP, 512, 0.5),
    ((72, 50, 41), (2, 3, 2), 95.0, 15.0, wl.PROJ_PERSP, 200, 0.25),
]


@pytest.mark.parametrize("dims,bricks,az,el,proj,size,step", CASES)
def test_window_holds_every_footprint_of_its_tile(vr, dims, bricks, az, el, proj, size, step):
    cs = wl.orbit_camera(dims, az, el, proj)
    cam = vr.camera_from_spec(cs)
    W = H = size
    plan = vr.vr_plan_slab(dims, bricks, cam, W, H, step)
    assert plan["eligible"], plan
    dom, D, w = plan["dominant_axis"], plan["slab_layers"], np.array(plan["window"])
    fast = 2 if dom == 0 else 0
    assert w[dom] == D + 1 and w[fast] % 4 == 0 and plan["smem_bytes"] <= 113 * 1024
    others = [a for a in range(3) if a != dom]
    rects, _ = vr.vr_plan_bricks(dims, bricks, cam, W, H)
    nb = np.array(bricks)
    rng = np.random.default_rng(7)
    checked = 0
    for b, (rx0, ry0, rw, rh) in enumerate(rects):
        if rw <= 0 or rh <= 0:
            continue
        bi = np.array([b % nb[0], (b // nb[0]) % nb[1], b // (nb[0] * nb[1])])
        lo_b = (bi * np.array(dims)) // nb
        hi_b = ((bi + 1) * np.array(dims)) // nb
        tiles_x, tiles_y = -(-rw // CTA_W), -(-rh // CTA_H)
        picks = {(0, 0), (tiles_x - 1, 0), (0, tiles_y - 1), (tiles_x - 1, tiles_y - 1), (tiles_x // 2, tiles_y // 2)}
        picks |= {(int(rng.integers(tiles_x)), int(rng.integers(tiles_y))) for _ in range(3)}
        for tx, ty in picks:
            px0, py0 = rx0 + tx * CTA_W, ry0 + ty * CTA_H
            gx, gy = np.meshgrid(np.arange(CTA_W), np.arange(CTA_H))
            px, py = (px0 + gx).reshape(-1).astype(np.float64), (py0 + gy).reshape(-1).astype(np.float64)
            o, d = rays_of(cs, W, H, px, py)
            assert (np.sign(d[:, dom]) == np.sign(d[0, dom])).all() and (d[:, dom] != 0).all()
            corners = np.array([0, CTA_W - 1, (CTA_H - 1) * CTA_W, CTA_H * CTA_W - 1])
            # the library's affine description reproduces the corner rays (positions where the dominant coordinate is c)
            c_probe = float(lo_b[dom] + PAD[dom] + 3.0)
            for k in corners:
                Q = plan["q0"] + px[k] * plan["dqx"] + py[k] * plan["dqy"]
                V = plan["v0"] + px[k] * plan["dvx"] + py[k] * plan["dvy"]
                U = Q + (c_probe - Q[dom]) * V / V[dom]
                ref = position_at(o[k:k + 1], d[k:k + 1], dom, c_probe)[0]
                assert np.abs(U - ref).max() <= 1e-6 * max(1.0, np.abs(ref).max())
            # slabs over the brick's depth range (padded cells lo - 1 + PAD .. hi + PAD)
            s_lo = int(lo_b[dom] + PAD[dom] - 1) // D
            s_hi = int(hi_b[dom] + PAD[dom]) // D
            for s in {s_lo, s_hi, (s_lo + s_hi) // 2, int(rng.integers(s_lo, s_hi + 1))}:
                c0, c1 = float(s * D), float(s * D + D)
                ends = np.concatenate([position_at(o[corners], d[corners], dom, c0), position_at(o[corners], d[corners], dom, c1)])
                org = np.zeros(3, dtype=np.int64)
                need_hi = np.zeros(3, dtype=np.int64)
                org[dom], need_hi[dom] = s * D, s * D + D
                for a in others:
                    org[a] = int(np.floor(ends[:, a].min() - 1e-3))
                    need_hi[a] = int(np.floor(ends[:, a].max() + 1e-3)) + 1
                org[fast] &= ~3
                assert (need_hi - org + 1 <= w).all(), (b, tx, ty, s, org, need_hi, w)
                # every pixel of the tile, anywhere inside the slab: footprint cells floor(U), floor(U) + 1 lie in the window
                cs_rand = rng.uniform(c0, c1, size=len(px))
                U = position_at(o, d, dom, cs_rand)
                for a in others:
                    cells = np.floor(U[:, a]).astype(np.int64)
                    assert (cells >= org[a]).all() and (cells + 1 < org[a] + w[a]).all(), (b, tx, ty, s, a)
                checked += len(px)
    assert checked > 1000


def test_frames_the_slab_caster_cannot_take(vr):
    dims = (128, 128, 128)
    # an eye inside the cube: some rays do not advance along the dominant axis in the direction of fwd
    eye = (60.0, 60.0, 60.0)
    cs = wl.CameraSpec(view=wl.look_at(eye, (128.0, 100.0, 90.0)), projection=wl.PROJ_PERSP, fovy_deg=170.0, ortho_half_h=1.0)
    plan = vr.vr_plan_slab(dims, (1, 1, 1), vr.camera_from_spec(cs), 256, 256, 0.5)
    assert not plan["eligible"]
    # a coarse image of a large cube: the window of a 16x8-pixel tile does not fit shared memory
    cs = wl.orbit_camera((2048, 2048, 1600), 30.0, 20.0, wl.PROJ_ORTHO)
    plan = vr.vr_plan_slab((2048, 2048, 1600), (2, 2, 2), vr.camera_from_spec(cs), 256, 256, 1.0)
    assert not plan["eligible"]
