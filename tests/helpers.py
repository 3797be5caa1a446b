"""Test-side helpers.  `independent_render` is a second, structurally different route to a frame
built from LIBRARY routines (numpy.linalg for the camera, per-face plane intersection for the
clip, scipy.ndimage.map_coordinates(order=1, mode='nearest') for the clamp-to-edge trilinear
sample, numpy.interp for the 256-entry table, cumprod for the front-to-back blend).  It is used
to pin the oracle by brute force on small cubes; it calls nothing under oracle/ or the CUDA path.
"""
import numpy as np
from scipy import ndimage


def oracle_camera(vro, cs):
    return vro.make_camera(cs.view, cs.projection, cs.fovy_deg, cs.ortho_half_h)


def pixel_ray_linalg(cs, W, H, px, py):
    """Ray through a pixel centre from the inverse view matrix (eye-space construction)."""
    V = np.asarray(cs.view, dtype=np.float64).reshape(4, 4)
    Vi = np.linalg.inv(V)
    u = 2.0 * (px + 0.5) / W - 1.0
    v = 2.0 * (py + 0.5) / H - 1.0
    asp = W / H
    if cs.projection == 0:
        h = float(np.float32(cs.ortho_half_h))
        a = Vi @ np.array([u * h * asp, v * h, 0.0, 1.0])
        b = Vi @ np.array([u * h * asp, v * h, -1.0, 1.0])
    else:
        T = np.tan(np.radians(float(np.float32(cs.fovy_deg))) / 2.0)
        a = Vi @ np.array([0.0, 0.0, 0.0, 1.0])
        b = Vi @ np.array([u * T * asp, v * T, -1.0, 1.0])
    o = a[:3]
    d = b[:3] - a[:3]
    return o, d / np.linalg.norm(d)


def box_hits_by_faces(o, d, lo, hi, eps=1e-9):
    """Entry/exit parameters of a line through a box, found face by face (not the slab method)."""
    ts = []
    for a in range(3):
        if abs(d[a]) < 1e-300:
            continue
        for plane in (lo[a], hi[a]):
            t = (plane - o[a]) / d[a]
            p = o + t * d
            ok = all(lo[b] - eps <= p[b] <= hi[b] + eps for b in range(3) if b != a)
            if ok:
                ts.append(t)
    if len(ts) < 2:
        return None
    return min(ts), max(ts)


def independent_pixel(cube, table, vmin, vmax, cs, W, H, step, mode, px, py, ert=0.0):
    """(rgba, scalar, n_samples) of one pixel, no bricks.  ert in (0,1): the ray stops after the FIRST sample
    whose accumulated opacity 1 - prod(1 - a) reaches ert (O7) and n_samples counts the samples up to and
    including that one; n_samples is -1 when some partial opacity lies within 1e-9 of ert (the crossing sample
    is then not decidable independently of the rounding order)."""
    nz, ny, nx = cube.shape
    o, d = pixel_ray_linalg(cs, W, H, px, py)
    hit = box_hits_by_faces(o, d, np.zeros(3), np.array([nx, ny, nz], dtype=np.float64))
    if hit is None:
        return np.zeros(4), -np.inf, 0
    t_near, t_far = max(hit[0], 0.0), hit[1]
    if not t_far > t_near:
        return np.zeros(4), -np.inf, 0
    ts = []
    i = 0
    while t_near + (i + 0.5) * step < t_far:
        ts.append(t_near + (i + 0.5) * step)
        i += 1
    if not ts:
        return np.zeros(4), -np.inf, 0
    ts = np.array(ts)
    P = o[None, :] + ts[:, None] * d[None, :]
    coords = np.stack([P[:, 2] - 0.5, P[:, 1] - 0.5, P[:, 0] - 0.5])        # (z, y, x) index space
    vals = ndimage.map_coordinates(cube.astype(np.float64), coords, order=1, mode="nearest")
    xp = vmin + (vmax - vmin) * np.arange(256) / 255.0
    tab = np.asarray(table, dtype=np.float64)
    if mode == 1:
        M = vals.max()
        rgba = np.array([np.interp(M, xp, tab[:, c]) for c in range(4)])
        return rgba, M, len(ts)
    rgb = np.stack([np.interp(vals, xp, tab[:, c]) for c in range(3)], axis=1)
    a = np.interp(vals, xp, 1.0 - (1.0 - tab[:, 3]) ** step)
    n_taken = len(ts)
    if 0.0 < ert < 1.0:
        A_run = 1.0 - np.cumprod(1.0 - a)
        if np.any(np.abs(A_run - ert) < 1e-9):
            n_taken = -1
        else:
            hit = np.nonzero(A_run >= ert)[0]
            if hit.size:
                n_taken = int(hit[0]) + 1
                a, rgb = a[:n_taken], rgb[:n_taken]
    trans = np.concatenate([[1.0], np.cumprod(1.0 - a)[:-1]])
    C = (trans[:, None] * a[:, None] * rgb).sum(axis=0)
    A = 1.0 - np.prod(1.0 - a)
    return np.array([C[0], C[1], C[2], A]), None, n_taken
