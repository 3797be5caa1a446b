"""Host-side planning of the CUDA path (a2 rendering rectangles, a6 depth order; A11/A12)
checked against the oracle's per-ray brick spans: every pixel whose ray takes a sample in a brick
lies inside that brick's rectangle, and the brick order never contradicts the per-pixel t_in order."""
import numpy as np
import pytest

from paper_1008_0135_b200 import build as vr_build
from paper_1008_0135_b200 import workloads as wl


@pytest.fixture(scope="module")
def vr():
    vr_build.build()
    from paper_1008_0135_b200 import vr as binding
    binding.lib()
    return binding


CASES = [
    ((22, 18, 14), (2, 2, 2), wl.PROJ_ORTHO, 30.0, 20.0, 40, 32),
    ((22, 18, 14), (3, 1, 2), wl.PROJ_PERSP, 200.0, -35.0, 36, 36),
    ((22, 18, 14), (4, 4, 4), wl.PROJ_PERSP, 75.0, 60.0, 33, 29),
    ((16, 16, 16), (2, 2, 1), wl.PROJ_ORTHO, 0.0, 0.0, 24, 24),
    ((16, 16, 16), (2, 2, 2), wl.PROJ_ORTHO, 90.0, 0.0, 24, 24),
    ((31, 17, 9), (5, 2, 3), wl.PROJ_ORTHO, 310.0, 5.0, 48, 20),
]


@pytest.mark.parametrize("dims,bricks,proj,az,el,W,H", CASES)
def test_rectangles_and_order_agree_with_oracle_spans(vr, oracle, dims, bricks, proj, az, el, W, H):
    cs = wl.orbit_camera(dims, az, el, proj)
    rect, order = vr.vr_plan_bricks(dims, bricks, vr.camera_from_spec(cs), W, H)
    rank = np.empty(len(order), dtype=np.int64)
    rank[order] = np.arange(len(order))
    ocam = oracle.make_camera(cs.view, cs.projection, cs.fovy_deg, cs.ortho_half_h)
    step = 0.5
    covered = 0
    for py in range(H):
        for px in range(W):
            o, d = oracle.ray(ocam, W, H, px, py)
            n, tn, tf = oracle.ray_extent(o, d, dims, step)
            if n == 0:
                continue
            spans = []
            for bk in range(bricks[2]):
                for bj in range(bricks[1]):
                    for bi in range(bricks[0]):
                        ok, t_in, lo, hi = oracle.brick_span(o, d, dims, bricks, (bi, bj, bk), step, tn, tf)
                        if ok:
                            b = (bk * bricks[1] + bj) * bricks[0] + bi
                            x0, y0, w, h = rect[b]
                            assert x0 <= px < x0 + w and y0 <= py < y0 + h, (b, px, py, rect[b])
                            spans.append((t_in, b))
                            covered += 1
            spans.sort()
            ranks = [rank[b] for _, b in spans]
            assert ranks == sorted(ranks), (px, py, spans, ranks)
    assert covered > 0


def test_rectangle_is_not_trivially_the_whole_image(vr):
    dims, bricks = (64, 64, 64), (4, 4, 4)
    cs = wl.orbit_camera(dims, 30, 20, wl.PROJ_ORTHO)
    rect, _ = vr.vr_plan_bricks(dims, bricks, vr.camera_from_spec(cs), 256, 256)
    area = (rect[:, 2] * rect[:, 3]).astype(np.int64)
    assert area.max() < 0.25 * 256 * 256
    assert (area > 0).all()


def test_eye_inside_volume_gives_full_rectangles(vr):
    dims, bricks = (32, 32, 32), (2, 2, 2)
    view = wl.look_at((16.2, 15.7, 16.4), (40.0, 20.0, 18.0))
    cam = vr.make_camera(view, wl.PROJ_PERSP, 60.0, 1.0)
    rect, order = vr.vr_plan_bricks(dims, bricks, cam, 40, 30)
    assert sorted(order.tolist()) == list(range(8))
    assert any((r == np.array([0, 0, 40, 30])).all() for r in rect)
