"""ctypes binding of the CPU oracle (oracle/vro.c).  TEST INFRASTRUCTURE, not the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs import
this.  Argument marshalling only: every formula lives in vro.c (rules O1-O11 of DESIGN.md).
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

MODE_EA, MODE_MIP = 0, 1
PROJ_ORTHO, PROJ_PERSP = 0, 1


class Camera(C.Structure):
    _fields_ = [("view", C.c_float * 16), ("projection", C.c_int), ("fovy_deg", C.c_float),
                ("ortho_half_h", C.c_float)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        d3 = C.POINTER(C.c_double)
        i3 = C.POINTER(C.c_int)
        fp = C.POINTER(C.c_float)
        _lib.vro_basis.argtypes = [C.POINTER(Camera), d3, d3, d3, d3]
        _lib.vro_basis.restype = None
        _lib.vro_ray.argtypes = [C.POINTER(Camera), C.c_int, C.c_int, C.c_int, C.c_int, d3, d3]
        _lib.vro_ray.restype = None
        _lib.vro_slab.argtypes = [d3, d3, d3, d3, d3, d3]
        _lib.vro_slab.restype = C.c_int
        _lib.vro_ray_extent.argtypes = [d3, d3, i3, C.c_double, d3, d3]
        _lib.vro_ray_extent.restype = C.c_longlong
        _lib.vro_sample.argtypes = [fp, i3, d3]
        _lib.vro_sample.restype = C.c_double
        _lib.vro_classify.argtypes = [fp, C.c_double, C.c_double, C.c_double, C.c_double, d3]
        _lib.vro_classify.restype = None
        _lib.vro_brick_span.argtypes = [d3, d3, i3, i3, C.c_int, C.c_int, C.c_int, C.c_double,
                                        C.c_double, C.c_double, d3, C.POINTER(C.c_longlong),
                                        C.POINTER(C.c_longlong)]
        _lib.vro_brick_span.restype = C.c_int
        _lib.vro_render_pixels.argtypes = [fp, i3, fp, C.c_float, C.c_float, i3, C.POINTER(Camera),
                                           C.c_int, C.c_int, C.c_float, C.c_int, C.c_float, C.c_int,
                                           C.c_longlong, i3, i3, fp, fp, fp,
                                           C.POINTER(C.c_longlong), C.c_int]
        _lib.vro_render_pixels.restype = C.c_int
        _lib.vro_render_pixels_sub.argtypes = [fp, i3, fp, C.c_float, C.c_float, i3, i3, i3, C.POINTER(Camera),
                                               C.c_int, C.c_int, C.c_float, C.c_int, C.c_float, C.c_int,
                                               C.c_longlong, i3, i3, fp, fp, fp,
                                               C.POINTER(C.c_longlong), C.c_int]
        _lib.vro_render_pixels_sub.restype = C.c_int
        _lib.vro_render_pixels_mask.argtypes = [fp, i3, fp, C.c_float, C.c_float, i3, i3, i3, C.POINTER(C.c_ubyte),
                                                C.POINTER(Camera), C.c_int, C.c_int, C.c_float, C.c_int, C.c_float,
                                                C.c_int, C.c_longlong, i3, i3, fp, fp, fp,
                                                C.POINTER(C.c_longlong), C.c_int]
        _lib.vro_render_pixels_mask.restype = C.c_int
        _lib.vro_max_threads.argtypes = []
        _lib.vro_max_threads.restype = C.c_int
    return _lib


def make_camera(view, projection, fovy_deg=45.0, ortho_half_h=1.0):
    cam = Camera()
    v = np.asarray(view, dtype=np.float32).reshape(16)
    for i in range(16):
        cam.view[i] = float(v[i])
    cam.projection = int(projection)
    cam.fovy_deg = float(fovy_deg)
    cam.ortho_half_h = float(ortho_half_h)
    return cam


def _d3(a):
    return (C.c_double * 3)(*[float(x) for x in a])


def _i3(a):
    return (C.c_int * 3)(*[int(x) for x in a])


def _fp(a):
    return a.ctypes.data_as(C.POINTER(C.c_float))


def basis(cam):
    r, u, f, e = _d3([0] * 3), _d3([0] * 3), _d3([0] * 3), _d3([0] * 3)
    lib().vro_basis(C.byref(cam), r, u, f, e)
    return np.array(r), np.array(u), np.array(f), np.array(e)


def ray(cam, W, H, px, py):
    o, d = _d3([0] * 3), _d3([0] * 3)
    lib().vro_ray(C.byref(cam), W, H, px, py, o, d)
    return np.array(o), np.array(d)


def slab(o, d, lo, hi):
    t0, t1 = C.c_double(0), C.c_double(0)
    hit = lib().vro_slab(_d3(o), _d3(d), _d3(lo), _d3(hi), C.byref(t0), C.byref(t1))
    return bool(hit), t0.value, t1.value


def ray_extent(o, d, dims, step):
    tn, tf = C.c_double(0), C.c_double(0)
    n = lib().vro_ray_extent(_d3(o), _d3(d), _i3(dims), float(step), C.byref(tn), C.byref(tf))
    return int(n), tn.value, tf.value


def _cube(data):
    """data: numpy float32 array of shape (nz, ny, nx), C-contiguous (x fastest)."""
    a = np.ascontiguousarray(data, dtype=np.float32)
    assert a.ndim == 3
    dims = (a.shape[2], a.shape[1], a.shape[0])
    return a, dims


def sample(data, p):
    a, dims = _cube(data)
    return float(lib().vro_sample(_fp(a), _i3(dims), _d3(p)))


def classify(rgba, vmin, vmax, step, value):
    t = np.ascontiguousarray(rgba, dtype=np.float32).reshape(1024)
    out = (C.c_double * 4)()
    lib().vro_classify(_fp(t), float(vmin), float(vmax), float(step), float(value), out)
    return np.array(out)


def brick_span(o, d, dims, bricks, ijk, step, t_near, t_far):
    t_in = C.c_double(0)
    lo, hi = C.c_longlong(0), C.c_longlong(0)
    ok = lib().vro_brick_span(_d3(o), _d3(d), _i3(dims), _i3(bricks), ijk[0], ijk[1], ijk[2],
                              float(step), float(t_near), float(t_far), C.byref(t_in),
                              C.byref(lo), C.byref(hi))
    return bool(ok), t_in.value, lo.value, hi.value


def render_pixels(data, rgba, vmin, vmax, bricks, cam, W, H, step, mode, ert_alpha, route, px, py,
                  want_bricks=False, threads=0, subcube=None, chan_mask=None):
    """Render the listed pixels.  Returns dict(rgba [n,4], scalar [n] (MIP), bricks, samples).
    chan_mask: None or nz values, non-zero = channel enabled (rule S2)."""
    a, dims = _cube(data)
    t = np.ascontiguousarray(rgba, dtype=np.float32).reshape(1024)
    px = np.ascontiguousarray(px, dtype=np.int32).reshape(-1)
    py = np.ascontiguousarray(py, dtype=np.int32).reshape(-1)
    n = px.size
    assert py.size == n
    out = np.zeros((n, 4), dtype=np.float32)
    scalar = np.zeros(n, dtype=np.float32) if mode == MODE_MIP else None
    B = int(bricks[0]) * int(bricks[1]) * int(bricks[2])
    ob = None
    if want_bricks:
        assert route == 1
        ob = np.zeros((B, n, 4) if mode == MODE_EA else (B, n), dtype=np.float32)
    samples = C.c_longlong(0)
    ip = C.POINTER(C.c_int)
    sub_lo = _i3(subcube[0]) if subcube is not None else None
    sub_hi = _i3(subcube[1]) if subcube is not None else None
    cm = None
    if chan_mask is not None:
        cm_arr = np.ascontiguousarray(np.asarray(chan_mask) != 0, dtype=np.uint8)
        assert cm_arr.size == dims[2]
        cm = cm_arr.ctypes.data_as(C.POINTER(C.c_ubyte))
    rc = lib().vro_render_pixels_mask(
        _fp(a), _i3(dims), _fp(t), float(vmin), float(vmax), _i3(bricks), sub_lo, sub_hi, cm, C.byref(cam), int(W),
        int(H), float(step), int(mode), float(ert_alpha), int(route), n,
        px.ctypes.data_as(ip), py.ctypes.data_as(ip), _fp(out),
        _fp(scalar) if scalar is not None else None, _fp(ob) if ob is not None else None,
        C.byref(samples), int(threads))
    if rc != 0:
        raise ValueError("vro_render_pixels: invalid arguments")
    return {"rgba": out, "scalar": scalar, "bricks": ob, "samples": samples.value}


def render(data, rgba, vmin, vmax, bricks, cam, W, H, step, mode, ert_alpha=0.0, route=0,
           want_bricks=False, threads=0, subcube=None, chan_mask=None):
    """Full frame; arrays come back shaped [H, W, ...] (py = 0 is the bottom row)."""
    yy, xx = np.meshgrid(np.arange(H, dtype=np.int32), np.arange(W, dtype=np.int32), indexing="ij")
    r = render_pixels(data, rgba, vmin, vmax, bricks, cam, W, H, step, mode, ert_alpha, route,
                      xx.reshape(-1), yy.reshape(-1), want_bricks, threads, subcube, chan_mask)
    r["rgba"] = r["rgba"].reshape(H, W, 4)
    if r["scalar"] is not None:
        r["scalar"] = r["scalar"].reshape(H, W)
    if r["bricks"] is not None:
        B = r["bricks"].shape[0]
        r["bricks"] = r["bricks"].reshape((B, H, W, 4) if mode == MODE_EA else (B, H, W))
    return r


def max_threads():
    return int(lib().vro_max_threads())
