"""Seeded synthetic inputs: cubes, cameras, transfer functions and the BASELINE.json configs.

This module serves BOTH the CUDA path's tests/bench and the oracle's tests.  It holds none of
the method's arithmetic (no ray, sample, classification or blend code): it only makes inputs.
It imports neither the C-ABI binding nor oracle/.

The paper measures on the HIPASS, GASS and an N-body cube (Table 3); none is
available, so the cubes below take their shapes and statistics and STAND IN for them (low-SNR
noise, compact sources elongated along the spectral axis, a bright band across the sky, extended
emission confined in velocity: Fig 5).  Recipe: DESIGN.md "Inputs".

Cube tensors are torch float32 of shape (nz, ny, nx), x fastest (FITS order; z = spectral axis).
"""
import math
from dataclasses import dataclass, field

import numpy as np
import torch

PROJ_ORTHO, PROJ_PERSP = 0, 1
MODE_EA, MODE_MIP = 0, 1


# ------------------------------------------------------------------ cameras -------------------
@dataclass
class CameraSpec:
    view: np.ndarray            # (4,4) float32 row-major, voxel -> eye
    projection: int
    fovy_deg: float = 45.0
    ortho_half_h: float = 1.0


def look_at(eye, centre, up=(0.0, 1.0, 0.0)):
    """Rigid view matrix (OpenGL convention: eye looks down -z_eye, +x right, +y up)."""
    eye = np.asarray(eye, dtype=np.float64)
    centre = np.asarray(centre, dtype=np.float64)
    f = centre - eye
    f /= np.linalg.norm(f)
    upv = np.asarray(up, dtype=np.float64)
    r = np.cross(f, upv)
    if np.linalg.norm(r) < 1e-9:            # looking along `up`: pick another up
        upv = np.array([0.0, 0.0, 1.0]) if abs(f[2]) < 0.9 else np.array([1.0, 0.0, 0.0])
        r = np.cross(f, upv)
    r /= np.linalg.norm(r)
    u = np.cross(r, f)
    R = np.stack([r, u, -f])
    M = np.eye(4)
    M[:3, :3] = R
    M[:3, 3] = -R @ eye
    return M.astype(np.float32)


def orbit_camera(dims, az_deg, el_deg, projection, fovy_deg=45.0):
    """Camera on a sphere around the cube centre; az = rotation about the y axis (the paper's
    theta), az = el = 0 looks down the spectral (z) axis at the sky plane."""
    dims = np.asarray(dims, dtype=np.float64)
    c = 0.5 * dims
    R = 0.5 * float(np.linalg.norm(dims))
    az, el = math.radians(az_deg), math.radians(el_deg)
    direction = np.array([math.cos(el) * math.sin(az), math.sin(el), math.cos(el) * math.cos(az)])
    if projection == PROJ_PERSP:
        D = R / math.sin(math.radians(0.5 * fovy_deg))
    else:
        D = 2.0 * R
    eye = c + D * direction
    return CameraSpec(look_at(eye, c), projection, fovy_deg, R)


def axis_camera(dims, axis, sign):
    """Orthographic view exactly along +/- one cube axis, one pixel per voxel column.
    Returns (CameraSpec, W, H, right_axis, right_sign, up_axis, up_sign)."""
    dims = [int(v) for v in dims]
    up_axis = 1 if axis != 1 else 2
    f = np.zeros(3); f[axis] = float(sign)
    u = np.zeros(3); u[up_axis] = 1.0
    r = np.cross(f, u)
    right_axis = int(np.argmax(np.abs(r)))
    right_sign = int(np.sign(r[right_axis]))
    c = 0.5 * np.asarray(dims, dtype=np.float64)
    eye = c - f * (dims[axis] * 0.5 + 10.0)
    R = np.stack([r, u, -f])
    M = np.eye(4)
    M[:3, :3] = R
    M[:3, 3] = -R @ eye
    W, H = dims[right_axis], dims[up_axis]
    cam = CameraSpec(M.astype(np.float32), PROJ_ORTHO, 45.0, 0.5 * H)
    return cam, W, H, right_axis, right_sign, up_axis, 1


# ------------------------------------------------------------------ transfer functions --------
def tf_ramp(alpha_max=0.1):
    """T[j] = (u, u/2, 1-u, alpha_max*u), u = j/255."""
    u = np.arange(256, dtype=np.float64) / 255.0
    return np.stack([u, 0.5 * u, 1.0 - u, alpha_max * u], axis=1).astype(np.float32)


def tf_piecewise(vmin, vmax, knots):
    """Piecewise-linear alpha through `knots` [(value, alpha), ...] (flat outside), colour
    blue -> green -> red over the range.  A noise-suppressing table."""
    v = vmin + (vmax - vmin) * np.arange(256, dtype=np.float64) / 255.0
    kv = np.array([k[0] for k in knots], dtype=np.float64)
    ka = np.array([k[1] for k in knots], dtype=np.float64)
    a = np.interp(v, kv, ka)
    u = np.arange(256, dtype=np.float64) / 255.0
    r = np.clip(2.0 * u - 1.0, 0.0, 1.0)
    b = np.clip(1.0 - 2.0 * u, 0.0, 1.0)
    g = 1.0 - r - b
    return np.stack([r, g, b, a], axis=1).astype(np.float32)


# ------------------------------------------------------------------ cubes ---------------------
def _add_sources(cube, gen, n, amp_lo, amp_hi, sxy_lo, sxy_hi, sz_lo, sz_hi, log_amp=True):
    """Add n separable Gaussian sources (truncated at 4 sigma) at uniform random centres."""
    nz, ny, nx = cube.shape
    dev = cube.device
    r = torch.rand((n, 7), generator=gen, device=dev, dtype=torch.float64).cpu().numpy()
    for k in range(n):
        cx, cy, cz = r[k, 0] * nx, r[k, 1] * ny, r[k, 2] * nz
        if log_amp:
            amp = amp_lo * (amp_hi / amp_lo) ** r[k, 3]
        else:
            amp = amp_lo + (amp_hi - amp_lo) * r[k, 3]
        sxy = sxy_lo + (sxy_hi - sxy_lo) * r[k, 4]
        sz = sz_lo + (sz_hi - sz_lo) * r[k, 5]
        prof = []
        sl = []
        for c, s, nn in ((cz, sz, nz), (cy, sxy, ny), (cx, sxy, nx)):
            lo = max(0, int(math.floor(c - 4.0 * s)))
            hi = min(nn, int(math.ceil(c + 4.0 * s)) + 1)
            x = torch.arange(lo, hi, device=dev, dtype=torch.float32) + 0.5
            prof.append(torch.exp(-0.5 * ((x - float(c)) / float(s)) ** 2))
            sl.append(slice(lo, hi))
        cube[sl[0], sl[1], sl[2]] += float(amp) * (prof[0][:, None, None] * prof[1][None, :, None]
                                                   * prof[2][None, None, :])


def _noise(dims, gen, device):
    nx, ny, nz = dims
    cube = torch.empty((nz, ny, nx), dtype=torch.float32, device=device)
    chunk = max(1, (1 << 28) // (nx * ny))        # ~1 GiB of floats per call
    for z0 in range(0, nz, chunk):
        z1 = min(nz, z0 + chunk)
        cube[z0:z1].normal_(0.0, 1.0, generator=gen)
    return cube


def _gen(seed, device):
    g = torch.Generator(device=device)
    g.manual_seed(int(seed))
    return g


def cube_blobs(dims, seed, device="cpu", n_blobs=4, amp=5.0, sigma=4.0):
    """Config 0: N(0,1) noise + isotropic Gaussian blobs."""
    g = _gen(seed, device)
    cube = _noise(dims, g, device)
    _add_sources(cube, g, n_blobs, amp, amp, sigma, sigma, sigma, sigma, log_amp=False)
    return cube


def cube_blobs_band(dims, seed, device="cpu", n_blobs=200, band_amp=10.0, band_w=32.0):
    """Config 1: noise + Gaussians (amplitude log-uniform 2-20, sigma 2-8, isotropic) + a smooth
    band of amplitude 10 across the y sky axis, all channels."""
    nx, ny, nz = dims
    g = _gen(seed, device)
    cube = _noise(dims, g, device)
    r = torch.rand((n_blobs,), generator=g, device=device, dtype=torch.float64).cpu().numpy()
    for k in range(n_blobs):
        s = 2.0 + 6.0 * r[k]
        _add_sources(cube, g, 1, 2.0, 20.0, s, s, s, s, log_amp=True)
    y = torch.arange(ny, device=device, dtype=torch.float32) + 0.5
    cube += (band_amp * torch.exp(-0.5 * ((y - 0.5 * ny) / band_w) ** 2))[None, :, None]
    return cube


def cube_hipass_like(dims, seed, device="cpu", n_sources=5000, band_amp=50.0, band_sigma=40.0,
                     band_half_channels=30):
    """Config 2: low-SNR noise + compact sources elongated along the spectral axis + a
    galactic-plane band across y spanning 60 spectral channels."""
    nx, ny, nz = dims
    g = _gen(seed, device)
    cube = _noise(dims, g, device)
    _add_sources(cube, g, n_sources, 3.0, 30.0, 1.0, 3.0, 2.0, 20.0, log_amp=True)
    y = torch.arange(ny, device=device, dtype=torch.float32) + 0.5
    band = band_amp * torch.exp(-0.5 * ((y - 0.5 * ny) / band_sigma) ** 2)
    z0 = max(0, nz // 2 - band_half_channels)
    z1 = min(nz, nz // 2 + band_half_channels)
    cube[z0:z1] += band[None, :, None]
    return cube


def cube_gass_like(dims, seed, device="cpu", n_sources=10000, field_amp=20.0, chan_frac=(0.375, 0.625),
                   taper=20):
    """Config 3/4: noise + extended emission (20/3)*max(g,0), g a unit-rms Gaussian random field
    with P(k) ~ k^-3 made at 1/4 resolution by FFT and trilinearly upsampled, confined to the
    middle quarter of the spectral axis (channels 600-1000 of 1600) with a cosine taper
    + compact sources (Fig 5)."""
    nx, ny, nz = dims
    g = _gen(seed, device)
    cube = _noise(dims, g, device)
    za, zb = int(round(chan_frac[0] * nz)), int(round(chan_frac[1] * nz))
    nzf = zb - za
    q = 4
    cz, cy, cx = max(2, -(-nzf // q)), max(2, -(-ny // q)), max(2, -(-nx // q))
    white = torch.randn((cz, cy, cx), generator=g, device=device, dtype=torch.float32)
    kz = torch.fft.fftfreq(cz, device=device)[:, None, None]
    ky = torch.fft.fftfreq(cy, device=device)[None, :, None]
    kx = torch.fft.rfftfreq(cx, device=device)[None, None, :]
    k = torch.sqrt(kz * kz + ky * ky + kx * kx)
    k[0, 0, 0] = 1.0
    amp = k ** (-1.5)
    amp[0, 0, 0] = 0.0
    coarse = torch.fft.irfftn(torch.fft.rfftn(white) * amp, s=(cz, cy, cx))
    coarse = coarse / coarse.std()
    coarse = (field_amp / 3.0) * torch.clamp(coarse, min=0.0)
    zi = torch.arange(nzf, device=device, dtype=torch.float32)
    tp = min(taper, max(1, nzf // 4))
    w = torch.ones(nzf, device=device)
    ramp = 0.5 - 0.5 * torch.cos(math.pi * (torch.arange(tp, device=device) + 0.5) / tp)
    w[:tp] = ramp
    w[nzf - tp:] = torch.flip(ramp, dims=[0])
    del zi
    chunk = max(1, (1 << 27) // (nx * ny))
    for s0 in range(0, nzf, chunk):
        s1 = min(nzf, s0 + chunk)
        # trilinear upsample of the coarse field to output channels [s0,s1) (align_corners=False)
        zc = (torch.arange(s0, s1, device=device, dtype=torch.float32) + 0.5) / q - 0.5
        zc = zc.clamp(0, cz - 1)
        i0 = zc.floor().long()
        i1 = (i0 + 1).clamp(max=cz - 1)
        fz = (zc - i0.float())[:, None, None]
        slab = coarse[i0] * (1 - fz) + coarse[i1] * fz            # (s1-s0, cy, cx)
        up = torch.nn.functional.interpolate(slab[None], size=(ny, nx), mode="bilinear",
                                             align_corners=False)[0]
        cube[za + s0:za + s1] += up * w[s0:s1, None, None]
        del slab, up
    _add_sources(cube, g, n_sources, 3.0, 30.0, 1.0, 3.0, 2.0, 20.0, log_amp=True)
    return cube


def cube_nbody_like(dims, seed, device="cpu", sigma=1.6, coarse=2):
    """Second workload (the paper's third dataset, an N-body density cube of 1024^3,
    Table 3): a log-normal density field rho = exp(sigma*g - sigma^2/2), g a unit-rms Gaussian random
    field with P(k) ~ k^-2 generated at 1/coarse resolution by FFT and trilinearly upsampled (smooth at the voxel
    scale, like a CIC-binned simulation), plus 2 % multiplicative white noise.  Positive, mean ~1, filaments and
    knots reaching ~50."""
    nx, ny, nz = dims
    g = _gen(seed, device)
    q = int(coarse)
    cz, cy, cx = max(2, -(-nz // q)), max(2, -(-ny // q)), max(2, -(-nx // q))
    white = torch.randn((cz, cy, cx), generator=g, device=device, dtype=torch.float32)
    kz = torch.fft.fftfreq(cz, device=device)[:, None, None]
    ky = torch.fft.fftfreq(cy, device=device)[None, :, None]
    kx = torch.fft.rfftfreq(cx, device=device)[None, None, :]
    k = torch.sqrt(kz * kz + ky * ky + kx * kx)
    k[0, 0, 0] = 1.0
    amp = k ** (-1.0)
    amp[0, 0, 0] = 0.0
    field = torch.fft.irfftn(torch.fft.rfftn(white) * amp, s=(cz, cy, cx))
    del white, k, amp
    field = field / field.std()
    cube = torch.empty((nz, ny, nx), dtype=torch.float32, device=device)
    chunk = max(1, (1 << 27) // (nx * ny))
    for s0 in range(0, nz, chunk):
        s1 = min(nz, s0 + chunk)
        zc = ((torch.arange(s0, s1, device=device, dtype=torch.float32) + 0.5) / q - 0.5).clamp(0, cz - 1)
        i0 = zc.floor().long()
        i1 = (i0 + 1).clamp(max=cz - 1)
        fz = (zc - i0.float())[:, None, None]
        slab = field[i0] * (1 - fz) + field[i1] * fz
        up = torch.nn.functional.interpolate(slab[None], size=(ny, nx), mode="bilinear", align_corners=False)[0]
        noise = torch.empty_like(up).normal_(0.0, 0.02, generator=g)
        cube[s0:s1] = torch.exp(sigma * up - 0.5 * sigma * sigma) * (1.0 + noise)
        del slab, up, noise
    return cube


# ------------------------------------------------------------------ configs -------------------
@dataclass
class Workload:
    name: str
    dims: tuple                 # (nx, ny, nz)
    seed: int
    cube_fn: str                # name of the generator above
    bricks: tuple
    W: int
    H: int
    projection: int
    az_deg: float
    el_deg: float
    step: float
    mode: int
    ert_alpha: float            # 0 = off
    table: np.ndarray = field(repr=False, default=None)
    vmin: float = -3.0
    vmax: float = 8.0
    cube_kwargs: dict = field(default_factory=dict)

    def cube(self, device="cpu"):
        return globals()[self.cube_fn](self.dims, self.seed, device=device, **self.cube_kwargs)

    def camera(self, az_deg=None, el_deg=None):
        return orbit_camera(self.dims, self.az_deg if az_deg is None else az_deg,
                            self.el_deg if el_deg is None else el_deg, self.projection)

    def scaled(self, factor, W=None, H=None):
        """Same recipe on a cube `factor` times smaller per axis (for oracle-speed parity cases).
        Source counts scale with the volume; sizes in voxels stay."""
        dims = tuple(max(8, int(round(d * factor))) for d in self.dims)
        kw = dict(self.cube_kwargs)
        vol = (dims[0] * dims[1] * dims[2]) / (self.dims[0] * self.dims[1] * self.dims[2])
        key, base = {"cube_blobs": ("n_blobs", 4), "cube_blobs_band": ("n_blobs", 200),
                     "cube_hipass_like": ("n_sources", 5000), "cube_gass_like": ("n_sources", 10000),
                     "cube_nbody_like": (None, 0)}[self.cube_fn]
        if key is not None and self.cube_fn != "cube_blobs":
            kw[key] = max(1, int(round(kw.get(key, base) * vol)))
        return Workload(self.name + f"_x{factor:g}", dims, self.seed, self.cube_fn, self.bricks,
                        W or self.W, H or self.H, self.projection, self.az_deg, self.el_deg,
                        self.step, self.mode, self.ert_alpha, self.table, self.vmin, self.vmax, kw)


def config(i):
    """BASELINE.json `configs[i]` (i = 0..3; config 4 is a sweep over config 3's cube, see
    sweep_points(); 5 is the extra N-body-like workload).  Items BASELINE.json leaves open are fixed as DESIGN.md "Inputs" says."""
    if i == 0:
        return Workload("cfg0_64cube", (64, 64, 64), 0, "cube_blobs", (1, 1, 1), 256, 256,
                        PROJ_ORTHO, 30.0, 20.0, 0.5, MODE_EA, 0.0, tf_ramp(0.1), -3.0, 8.0)
    if i == 1:
        return Workload("cfg1_512x512x256", (512, 512, 256), 1, "cube_blobs_band", (2, 2, 1), 512,
                        512, PROJ_PERSP, 30.0, 20.0, 0.5, MODE_EA, 0.995, tf_ramp(0.05), -3.0, 20.0)
    if i == 2:
        tab = tf_piecewise(-3.0, 60.0, [(2.5, 0.0), (5.0, 0.02), (15.0, 0.2), (50.0, 0.6)])
        return Workload("cfg2_hipass_1721x1721x1024", (1721, 1721, 1024), 2, "cube_hipass_like",
                        (2, 2, 2), 1024, 1024, PROJ_ORTHO, 30.0, 20.0, 1.0, MODE_EA, 0.0, tab,
                        -3.0, 60.0)
    if i == 3:
        tab = tf_piecewise(-3.0, 30.0, [(2.0, 0.0), (20.0, 0.3)])
        return Workload("cfg3_gass_2048x2048x1600", (2048, 2048, 1600), 3, "cube_gass_like",
                        (2, 2, 2), 1024, 1024, PROJ_PERSP, 30.0, 20.0, 1.0, MODE_EA, 0.995, tab,
                        -3.0, 30.0)
    if i == 5:
        # not a BASELINE.json config: the paper's N-body cube (Table 3) with the rotation-about-y protocol of
        # Figs 7 and 12: el = 0, orthographic, early termination off
        tab = tf_piecewise(0.0, 20.0, [(1.0, 0.0), (4.0, 0.05), (20.0, 0.4)])
        return Workload("cfg5_nbody_1024cube", (1024, 1024, 1024), 5, "cube_nbody_like", (2, 2, 2), 1024, 1024,
                        PROJ_ORTHO, 30.0, 0.0, 1.0, MODE_EA, 0.0, tab, 0.0, 20.0)
    raise ValueError("config index must be 0..3 or 5")


def orbit_azimuths():
    """Config 3: 36-view orbit about the y axis, el = 20 deg."""
    return [10.0 * k for k in range(36)]


def sweep_points():
    """Config 4: MIP point + EA sweep (bricks x step x image), ORTHO az 30 el 20, ERT off."""
    pts = [dict(mode=MODE_MIP, bricks=(2, 2, 2), step=1.0, size=1024)]
    for b in ((1, 1, 1), (2, 2, 2), (4, 4, 4)):
        for step in (0.25, 0.5, 1.0):
            for size in (512, 1024, 2048):
                pts.append(dict(mode=MODE_EA, bricks=b, step=step, size=size))
    return pts
