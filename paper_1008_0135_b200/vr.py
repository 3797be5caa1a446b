"""Thin ctypes binding of include/vr.h (libvr_b200.so).  Argument marshalling only.

Same names as the C ABI.  Device buffers are torch CUDA tensors (torch supplies memory and the
stream; nothing is computed in torch).  Loading fails loudly when the library is missing: there is
no CPU fallback and nothing here imports oracle/.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

HERE = os.path.dirname(os.path.abspath(__file__))
# libvr_b200.so; an experiment variant's own file only while VR_DEFINES names that variant (build.py)
LIB_PATH = _build.lib_path()

VR_OK, VR_ERR_INVALID_ARG, VR_ERR_STATE, VR_ERR_OOM, VR_ERR_CUDA = 0, 1, 2, 3, 4
VR_MODE_EA, VR_MODE_MIP = 0, 1
VR_PROJ_ORTHO, VR_PROJ_PERSP = 0, 1
VR_MAX_BRICKS = 512
VR_MAX_CHANNEL_RUNS = 16

SYMBOLS = ["vr_create_volume", "vr_destroy_volume", "vr_set_stream", "vr_set_transfer_function",
           "vr_set_bricks", "vr_set_subcube", "vr_set_channel_mask", "vr_render", "vr_render_to_host", "vr_render_to_host_async", "vr_wait_frames", "vr_render_bricks", "vr_composite",
           "vr_plan_bricks", "vr_measure", "vr_measure_units", "vr_set_empty_space_skipping", "vr_get_skip_info",
           "vr_set_slab_staging", "vr_get_slab_info", "vr_plan_slab",
           "vr_get_stage_ms", "vr_volume_info", "vr_volume_range", "vr_volume_histogram", "vr_volume_histogram_noalloc", "vr_export_linear", "vr_last_error"]


class vr_camera(C.Structure):
    _fields_ = [("view", C.c_float * 16), ("projection", C.c_int), ("fovy_deg", C.c_float),
                ("ortho_half_h", C.c_float)]


class VrError(RuntimeError):
    def __init__(self, status, message):
        super().__init__(f"vr status {status}: {message}")
        self.status = status


_lib = None


def lib():
    """Load libvr_b200.so (built by paper_1008_0135_b200/build.py); raises if it is not there."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_1008_0135_b200.build` "
                              "(or __graft_entry__.build()); there is no CPU fallback")
        L = C.CDLL(LIB_PATH)
        vp, ip, fp = C.c_void_p, C.POINTER(C.c_int), C.POINTER(C.c_float)
        cam = C.POINTER(vr_camera)
        L.vr_create_volume.argtypes = [ip, vp, C.POINTER(vp)]
        L.vr_destroy_volume.argtypes = [vp]
        L.vr_destroy_volume.restype = None
        L.vr_set_stream.argtypes = [vp, vp]
        L.vr_set_transfer_function.argtypes = [vp, fp, C.c_float, C.c_float]
        L.vr_set_bricks.argtypes = [vp, C.c_int, C.c_int, C.c_int]
        L.vr_set_subcube.argtypes = [vp, ip, ip]
        L.vr_set_channel_mask.argtypes = [vp, C.POINTER(C.c_ubyte)]
        L.vr_render.argtypes = [vp, cam, C.c_int, C.c_int, C.c_float, C.c_int, C.c_float, vp, vp]
        L.vr_render_to_host.argtypes = [vp, cam, C.c_int, C.c_int, C.c_float, C.c_int, C.c_float, vp]
        L.vr_render_to_host_async.argtypes = [vp, cam, C.c_int, C.c_int, C.c_float, C.c_int, C.c_float, vp]
        L.vr_wait_frames.argtypes = [vp]
        L.vr_render_bricks.argtypes = [vp, cam, C.c_int, C.c_int, C.c_float, C.c_int, C.c_float, vp]
        L.vr_composite.argtypes = [vp, cam, C.c_int, C.c_int, C.c_int, vp, vp, vp]
        L.vr_plan_bricks.argtypes = [ip, ip, cam, C.c_int, C.c_int, vp, ip]
        L.vr_measure.argtypes = [vp, cam, C.c_int, C.c_int, C.c_float, C.c_int, C.c_float,
                                 C.POINTER(C.c_longlong), C.POINTER(C.c_longlong)]
        L.vr_measure_units.argtypes = [vp, cam, C.c_int, C.c_int, C.c_float, C.c_int, C.c_float,
                                       C.POINTER(C.c_longlong), C.POINTER(C.c_longlong)]
        L.vr_set_empty_space_skipping.argtypes = [vp, C.c_int]
        L.vr_get_skip_info.argtypes = [vp, ip, fp, C.POINTER(C.c_longlong), C.POINTER(C.c_double)]
        L.vr_set_slab_staging.argtypes = [vp, C.c_int]
        L.vr_get_slab_info.argtypes = [vp, ip, fp, C.POINTER(C.c_longlong)]
        L.vr_plan_slab.argtypes = [ip, ip, cam, C.c_int, C.c_int, C.c_float, ip, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.vr_get_stage_ms.argtypes = [vp, fp, fp]
        L.vr_volume_info.argtypes = [vp, fp, C.POINTER(C.c_longlong)]
        L.vr_volume_range.argtypes = [vp, fp, fp]
        L.vr_volume_histogram.argtypes = [vp, C.c_int, C.c_float, C.c_float, C.POINTER(C.c_longlong), C.POINTER(C.c_longlong)]
        L.vr_volume_histogram_noalloc.argtypes = L.vr_volume_histogram.argtypes
        L.vr_export_linear.argtypes = [vp, vp]
        L.vr_last_error.argtypes = []
        L.vr_last_error.restype = C.c_char_p
        for name in SYMBOLS:
            if name not in ("vr_destroy_volume", "vr_last_error"):
                getattr(L, name).restype = C.c_int
        _lib = L
    return _lib


def vr_last_error():
    return lib().vr_last_error().decode()


def _check(status):
    if status != VR_OK:
        raise VrError(status, vr_last_error())


def make_camera(view, projection, fovy_deg=45.0, ortho_half_h=1.0):
    cam = vr_camera()
    v = np.asarray(view, dtype=np.float32).reshape(16)
    for i in range(16):
        cam.view[i] = float(v[i])
    cam.projection = int(projection)
    cam.fovy_deg = float(fovy_deg)
    cam.ortho_half_h = float(ortho_half_h)
    return cam


def camera_from_spec(cs):
    """cs: workloads.CameraSpec (or anything with view/projection/fovy_deg/ortho_half_h)."""
    return make_camera(cs.view, cs.projection, cs.fovy_deg, cs.ortho_half_h)


def _i3(a):
    return (C.c_int * 3)(*[int(x) for x in a])


def _dptr(t, dtype_name="float32"):
    """Device pointer of a contiguous torch CUDA tensor (None -> NULL)."""
    if t is None:
        return None
    import torch
    assert isinstance(t, torch.Tensor) and t.is_cuda and t.is_contiguous(), "need a contiguous CUDA tensor"
    assert str(t.dtype) == "torch." + dtype_name, f"need {dtype_name}"
    return C.c_void_p(t.data_ptr())


def vr_plan_bricks(dims, bricks, cam, W, H):
    """Host-only: (rects [B,4] = x0,y0,w,h ; order [B] front to back)."""
    B = int(bricks[0]) * int(bricks[1]) * int(bricks[2])
    rect = np.zeros((max(B, 1), 4), dtype=np.int32)
    order = np.zeros(max(B, 1), dtype=np.int32)
    _check(lib().vr_plan_bricks(_i3(dims), _i3(bricks), C.byref(cam), int(W), int(H),
                                rect.ctypes.data_as(C.c_void_p), order.ctypes.data_as(C.POINTER(C.c_int))))
    return rect[:B], order[:B]


def vr_plan_slab(dims, bricks, cam, W, H, step):
    """Host-only: what the slab-staged caster would plan for this frame (include/vr.h)."""
    plan = (C.c_int * 8)()
    bps = C.c_double(0.0)
    ray = (C.c_double * 18)()
    _check(lib().vr_plan_slab(_i3(dims), _i3(bricks), C.byref(cam), int(W), int(H), float(step), plan, C.byref(bps), ray))
    r = np.array(list(ray), dtype=np.float64).reshape(6, 3)
    return {"eligible": bool(plan[0]), "dominant_axis": plan[1], "slab_layers": plan[2], "window": (plan[3], plan[4], plan[5]),
            "n_maps": plan[6], "smem_bytes": plan[7], "bytes_per_sample": bps.value,
            "q0": r[0], "dqx": r[1], "dqy": r[2], "v0": r[3], "dvx": r[4], "dvy": r[5]}


class Volume:
    """Owner of one vr_volume handle.  `cube` is a torch float32 CUDA tensor of shape (nz,ny,nx)."""

    def __init__(self, cube, stream=None):
        import torch
        assert cube.dim() == 3
        self.dims = (int(cube.shape[2]), int(cube.shape[1]), int(cube.shape[0]))
        self.device = cube.device
        self.bricks = (1, 1, 1)
        self._h = C.c_void_p()
        with torch.cuda.device(self.device):
            torch.cuda.current_stream().synchronize()      # the cube must be complete: a0 runs on stream 0
            _check(lib().vr_create_volume(_i3(self.dims), _dptr(cube), C.byref(self._h)))
            self.vr_set_stream(torch.cuda.current_stream() if stream is None else stream)

    def close(self):
        if self._h:
            lib().vr_destroy_volume(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- same names as the C ABI ------------------------------------------------------------------
    def vr_set_stream(self, stream):
        _check(lib().vr_set_stream(self._h, C.c_void_p(stream.cuda_stream)))

    def vr_set_transfer_function(self, rgba, vmin, vmax):
        t = np.ascontiguousarray(rgba, dtype=np.float32).reshape(1024)
        _check(lib().vr_set_transfer_function(self._h, t.ctypes.data_as(C.POINTER(C.c_float)),
                                              float(vmin), float(vmax)))

    def vr_set_bricks(self, bx, by, bz):
        _check(lib().vr_set_bricks(self._h, int(bx), int(by), int(bz)))
        self.bricks = (int(bx), int(by), int(bz))

    def vr_set_subcube(self, lo=None, hi=None):
        if lo is None and hi is None:
            _check(lib().vr_set_subcube(self._h, None, None))
        else:
            _check(lib().vr_set_subcube(self._h, _i3(lo), _i3(hi)))

    def vr_set_channel_mask(self, enabled=None):
        """enabled: None (all channels) or nz values, non-zero = channel enabled."""
        if enabled is None:
            _check(lib().vr_set_channel_mask(self._h, None))
            return
        m = np.ascontiguousarray(np.asarray(enabled) != 0, dtype=np.uint8)
        assert m.size == self.dims[2], "one value per spectral channel"
        _check(lib().vr_set_channel_mask(self._h, m.ctypes.data_as(C.POINTER(C.c_ubyte))))

    def vr_render(self, cam, W, H, step, mode, ert_alpha=0.0, out=None, out_scalar=None):
        import torch
        if out is None:
            out = torch.empty((H, W, 4), dtype=torch.float32, device=self.device)
        _check(lib().vr_render(self._h, C.byref(cam), int(W), int(H), float(step), int(mode),
                               float(ert_alpha), _dptr(out), _dptr(out_scalar)))
        return out

    def vr_render_to_host(self, cam, W, H, step, mode, ert_alpha, host_out):
        """host_out: torch CPU float32 tensor [H,W,4] (pinned for an asynchronous copy)."""
        assert not host_out.is_cuda and host_out.is_contiguous() and host_out.numel() == H * W * 4
        _check(lib().vr_render_to_host(self._h, C.byref(cam), int(W), int(H), float(step), int(mode),
                                       float(ert_alpha), C.c_void_p(host_out.data_ptr())))
        return host_out

    def vr_render_to_host_async(self, cam, W, H, step, mode, ert_alpha, host_out):
        """As vr_render_to_host without the wait; host_out must stay untouched until vr_wait_frames()."""
        assert not host_out.is_cuda and host_out.is_contiguous() and host_out.numel() == H * W * 4
        _check(lib().vr_render_to_host_async(self._h, C.byref(cam), int(W), int(H), float(step), int(mode),
                                             float(ert_alpha), C.c_void_p(host_out.data_ptr())))
        return host_out

    def vr_wait_frames(self):
        _check(lib().vr_wait_frames(self._h))

    def vr_render_bricks(self, cam, W, H, step, mode, ert_alpha=0.0):
        import torch
        B = self.bricks[0] * self.bricks[1] * self.bricks[2]
        shape = (B, H, W, 4) if mode == VR_MODE_EA else (B, H, W)
        imgs = torch.empty(shape, dtype=torch.float32, device=self.device)
        _check(lib().vr_render_bricks(self._h, C.byref(cam), int(W), int(H), float(step), int(mode),
                                      float(ert_alpha), _dptr(imgs)))
        return imgs

    def vr_composite(self, cam, W, H, mode, brick_images, out=None, out_scalar=None):
        import torch
        if out is None:
            out = torch.empty((H, W, 4), dtype=torch.float32, device=self.device)
        _check(lib().vr_composite(self._h, C.byref(cam), int(W), int(H), int(mode), _dptr(brick_images),
                                  _dptr(out), _dptr(out_scalar)))
        return out

    def vr_measure(self, cam, W, H, step, mode, ert_alpha=0.0):
        """(lattice samples visited, distinct 32-byte sectors of the cube touched) from the instrumented caster."""
        s, k = C.c_longlong(0), C.c_longlong(0)
        _check(lib().vr_measure(self._h, C.byref(cam), int(W), int(H), float(step), int(mode),
                                float(ert_alpha), C.byref(s), C.byref(k)))
        return s.value, k.value

    def vr_measure_units(self, cam, W, H, step, mode, ert_alpha=0.0):
        """([lattice samples visited, samples evaluated], [distinct 32-byte sectors, 64-byte pairs, 128-byte lines of
        the cube touched, 32-byte sectors of the occupancy mask read])."""
        s, u = (C.c_longlong * 2)(0, 0), (C.c_longlong * 4)(0, 0, 0, 0)
        _check(lib().vr_measure_units(self._h, C.byref(cam), int(W), int(H), float(step), int(mode),
                                      float(ert_alpha), s, u))
        return [int(s[0]), int(s[1])], [int(u[k]) for k in range(4)]

    def vr_set_empty_space_skipping(self, enabled):
        _check(lib().vr_set_empty_space_skipping(self._h, 1 if enabled else 0))

    def vr_set_slab_staging(self, mode):
        _check(lib().vr_set_slab_staging(self._h, int(mode)))

    def vr_get_slab_info(self):
        info = (C.c_int * 6)()
        ms = C.c_float(0.0)
        nb = C.c_longlong(0)
        _check(lib().vr_get_slab_info(self._h, info, C.byref(ms), C.byref(nb)))
        return {"used": bool(info[0]), "dominant_axis": info[1], "slab_layers": info[2],
                "window": (info[3], info[4], info[5]), "linearize_ms": ms.value, "linear_bytes": nb.value}

    def vr_get_skip_info(self):
        """dict(active, build_ms, mask_bytes, occupied_fraction); builds the mask if it is due."""
        a, ms, nb, fr = C.c_int(0), C.c_float(0), C.c_longlong(0), C.c_double(0)
        _check(lib().vr_get_skip_info(self._h, C.byref(a), C.byref(ms), C.byref(nb), C.byref(fr)))
        return {"active": bool(a.value), "build_ms": ms.value, "mask_bytes": nb.value, "occupied_fraction": fr.value}

    def vr_get_stage_ms(self):
        """(cast ms, composite ms) of the most recent vr_render; waits for it."""
        a, b = C.c_float(0), C.c_float(0)
        _check(lib().vr_get_stage_ms(self._h, C.byref(a), C.byref(b)))
        return a.value, b.value

    def vr_volume_info(self):
        ms, nb = C.c_float(0), C.c_longlong(0)
        _check(lib().vr_volume_info(self._h, C.byref(ms), C.byref(nb)))
        return ms.value, nb.value

    def vr_volume_range(self):
        """(min, max) of the cube, NaN ignored, from the re-layout pass."""
        a, b = C.c_float(0), C.c_float(0)
        _check(lib().vr_volume_range(self._h, C.byref(a), C.byref(b)))
        return a.value, b.value

    def vr_volume_histogram(self, n_bins, lo, hi):
        """(counts [n_bins] int64, number of NaN voxels); outliers fall into the end bins."""
        counts = np.zeros(int(n_bins), dtype=np.int64)
        nan = C.c_longlong(0)
        _check(lib().vr_volume_histogram(self._h, int(n_bins), float(lo), float(hi),
                                         counts.ctypes.data_as(C.POINTER(C.c_longlong)), C.byref(nan)))
        return counts, nan.value

    def vr_volume_histogram_noalloc(self, n_bins, lo, hi):
        """vr_volume_histogram for callers that must not allocate device memory (a host allocator owns the GPU, or
        frames are in flight and cudaFree would stall them): same result, bins in a fixed 4096-bin array inside the
        library.  Calls that overlap on one GPU race; see include/vr.h."""
        counts = np.zeros(max(int(n_bins), 0), dtype=np.int64)
        nan = C.c_longlong(0)
        _check(lib().vr_volume_histogram_noalloc(self._h, int(n_bins), float(lo), float(hi),
                                                 counts.ctypes.data_as(C.POINTER(C.c_longlong)), C.byref(nan)))
        return counts, nan.value

    def vr_export_linear(self):
        import torch
        out = torch.empty((self.dims[2], self.dims[1], self.dims[0]), dtype=torch.float32, device=self.device)
        _check(lib().vr_export_linear(self._h, _dptr(out)))
        return out
