"""Seeded synthetic inputs for the RTM-with-probing hot path.

This module serves BOTH the CPU oracle (``oracle/``) and the CUDA path
(``paper_2201_06914_b200/``).  It holds none of the method's arithmetic: no
stencil, no damping profile, no coefficient (K1/K2) formula, no interpolation
weight, no estimator.  It only produces *inputs*: earth models (vp, epsilon,
delta, theta), acquisition geometry (positions in metres), source wavelets,
time step / step count, and the random probing matrices Z.

The models STAND IN for the paper's SEAM slice (Sec. 4.1) and the
BP 2007 TTI model (Sec. 4.2), which are not available; only the
shapes and value ranges of BASELINE.json:configs are used.  Every array is drawn
from ``numpy.random.default_rng(20220106 + c)`` (c = config number).

All returned arrays are C-contiguous; z is the contiguous (last) axis.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np
from scipy.ndimage import gaussian_filter

SEED0 = 20220106

# sum_j |w_j| of the order-8 second-derivative weights (|w0| + 2*sum_{j>=1}|w_j|); used only to
# pick a stable time step (an input), SURVEY.md 8(c) O7.
_S_ABS = 205.0 / 72.0 + 2.0 * (8.0 / 5.0 + 1.0 / 5.0 + 8.0 / 315.0 + 1.0 / 560.0)


def cfl_dt_acoustic(h: float, vmax: float, ndim: int) -> float:
    """von-Neumann limit of the 2nd-order-time / 8th-order-space scheme."""
    return 2.0 * h / (vmax * math.sqrt(ndim * _S_ABS))


def cfl_dt_tti(h: float, vmax: float, eps_max: float) -> float:
    """Frozen-coefficient bound for the rotated first-derivative TTI operator."""
    return 0.8172 * h / (vmax * math.sqrt(1.0 + 2.0 * eps_max))


def ricker(nt: int, dt: float, f0: float) -> np.ndarray:
    """Ricker wavelet (1-2a)exp(-a), a=(pi f0 (t-1/f0))^2, sampled at t=n*dt, made exactly
    zero-sum, returned as fp32 [nt]."""
    t = np.arange(nt, dtype=np.float64) * dt
    a = (np.pi * f0 * (t - 1.0 / f0)) ** 2
    w = (1.0 - 2.0 * a) * np.exp(-a)
    w -= w.mean()
    w32 = w.astype(np.float32)
    # make the fp32 samples sum to zero as closely as fp32 allows
    w32[-1] = np.float32(w32[-1] - np.float32(w32.astype(np.float64).sum()))
    return w32


def gaussian_probes(nt: int, r: int, seed: int) -> np.ndarray:
    """Z[nt][r] i.i.d. N(0,1) (BASELINE.json configs; E[zz^T]=I reading C1), fp32."""
    return np.random.default_rng(seed).standard_normal((nt, r)).astype(np.float32)


def rademacher_probes(nt: int, r: int, seed: int) -> np.ndarray:
    """Z[nt][r] i.i.d. +-1."""
    return (np.random.default_rng(seed).integers(0, 2, size=(nt, r)) * 2 - 1).astype(np.float32)


def identity_probes(nt: int) -> np.ndarray:
    """Z = sqrt(nt) * I (r = nt), so (1/r) Z Z^T = I exactly (reading C1)."""
    return (math.sqrt(nt) * np.eye(nt)).astype(np.float32)


@dataclass
class Problem:
    """One shot of one configuration.  Positions are metres from the physical origin."""
    name: str
    ndim: int
    n: tuple                      # physical points (x,(y),z)
    h: float
    nb: int
    physics: int                  # 0 acoustic, 1 TTI
    nt: int
    dt: float
    r: int
    f0: float
    vp_true: np.ndarray           # fp32 [n]
    vp: np.ndarray                # fp32 [n] migration (smoothed) model
    eps: np.ndarray | None = None
    delta: np.ndarray | None = None
    theta: np.ndarray | None = None   # radians: tilt of the symmetry axis from the z axis
    phi: np.ndarray | None = None     # radians: its azimuth from the x axis (3D TTI only)
    src_xyz: np.ndarray = field(default=None)   # fp32 [nsrc][ndim]
    rec_xyz: np.ndarray = field(default=None)   # fp32 [nrec][ndim]
    wav: np.ndarray = field(default=None)       # fp32 [nt][nsrc]
    Z: np.ndarray = field(default=None)         # fp32 [nt][r]
    offsets: np.ndarray | None = None           # int32 [nh]  (grid points along x)

    @property
    def N(self) -> int:
        return int(np.prod(self.n))

    @property
    def P(self) -> tuple:
        return tuple(int(a) + 2 * self.nb for a in self.n)

    @property
    def Np(self) -> int:
        return int(np.prod(self.P))


def _smooth_noise(rng, shape, sigma):
    f = gaussian_filter(rng.standard_normal(shape), sigma, mode="reflect")
    f -= f.min()
    m = f.max()
    return f / m if m > 0 else f


def _star_body(shape, h, centre, rad_x, rad_z, rng, nvert=10):
    """Mask of a random star-shaped body: radius interpolated linearly in angle between nvert
    random vertices; elliptical scaling (rad_x, rad_z are (lo, hi) ranges in metres)."""
    nx, nz = shape
    ang = np.sort(rng.uniform(0, 2 * np.pi, nvert))
    fx = rng.uniform(rad_x[0], rad_x[1], nvert)
    fz = rng.uniform(rad_z[0], rad_z[1], nvert)
    X = (np.arange(nx) * h - centre[0])[:, None]
    Zc = (np.arange(nz) * h - centre[1])[None, :]
    th = np.mod(np.arctan2(Zc, X), 2 * np.pi)
    angp = np.concatenate([ang, [ang[0] + 2 * np.pi]])
    fxp = np.concatenate([fx, [fx[0]]])
    fzp = np.concatenate([fz, [fz[0]]])
    th2 = np.where(th < ang[0], th + 2 * np.pi, th)
    ax = np.interp(th2, angp, fxp)
    az = np.interp(th2, angp, fzp)
    return (X / ax) ** 2 + (Zc / az) ** 2 <= 1.0


def _smooth_slowness(vp, sigma):
    return (1.0 / gaussian_filter(1.0 / vp.astype(np.float64), sigma, mode="nearest")).astype(np.float32)


def make_c0(nt: int = 500, r: int = 8, n=(101, 101), nb: int = 20) -> Problem:
    """configs[0]: 2D acoustic 101x101 @10 m, 3 layers 1500/2500/3500, interfaces z=150,300 m (C15)."""
    c = 0
    h = 10.0
    nx, nz = n
    z = np.arange(nz) * h
    col = np.where(z < 150.0, 1500.0, np.where(z < 300.0, 2500.0, 3500.0))
    vp = np.broadcast_to(col[None, :], (nx, nz)).astype(np.float32).copy()
    dt = 0.4 * cfl_dt_acoustic(h, float(vp.max()), 2)
    f0 = 15.0
    src = np.array([[(nx - 1) * h / 2.0, 0.0]], np.float32)
    rec = np.stack([np.arange(nx) * h, np.zeros(nx)], 1).astype(np.float32)
    wav = ricker(nt, dt, f0)[:, None].copy()
    Z = gaussian_probes(nt, r, SEED0 + c)
    return Problem("c0", 2, (nx, nz), h, nb, 0, nt, dt, r, f0, vp, _smooth_slowness(vp, 3.0),
                   src_xyz=src, rec_xyz=rec, wav=wav, Z=Z)


def make_c1(n=(1751, 751), nt: int = 6000, r: int = 32, nb: int = 80, node: int = 1,
            h: float = 20.0, record_s: float | None = 10.0) -> Problem:
    """configs[1]: 2D acoustic long-offset subsalt, water layer, gradient, star-shaped salt.
    ``n`` may be cropped (same recipe, geometry scaled to the cropped extent).  ``node`` picks one
    of three timed OBN positions (x = 1/14, 1/2, 13/14 of the line), used as a reciprocal source."""
    c = 1
    rng = np.random.default_rng(SEED0 + c)
    nx, nz = n
    Lx, Lz = (nx - 1) * h, (nz - 1) * h
    zwater = 0.1 * Lz                      # 1500 m of 15 km
    z = np.arange(nz) * h
    grad = 1500.0 + 3000.0 * np.clip((z - zwater) / max(Lz - zwater, h), 0.0, 1.0)
    sig = 25.0 * min(1.0, nx / 1751.0) + 1.0
    noise = gaussian_filter(rng.standard_normal((nx, nz)), sig, mode="reflect")
    noise *= 0.03 / max(np.abs(noise).max(), 1e-30)
    vp = grad[None, :] * (1.0 + noise)
    salt = _star_body((nx, nz), h, (0.5 * Lx, 7.0 / 15.0 * Lz),
                      (2.0 / 35.0 * Lx, 5.0 / 35.0 * Lx), (1.0 / 15.0 * Lz, 2.5 / 15.0 * Lz), rng)
    vp = np.where(salt, 4500.0, vp)
    vp = np.clip(vp, 1500.0, 4500.0)
    vp[:, z < zwater] = 1500.0
    vp = vp.astype(np.float32)
    vmax = 4500.0
    dtmax = cfl_dt_acoustic(h, vmax, 2)
    if record_s is not None and nt == 6000:
        dt = record_s / nt                 # 1.6667 ms = 0.676 dt_max (C15)
    else:
        dt = 0.676 * dtmax
    assert dt < dtmax
    f0 = 15.0
    xs = (1.0 / 14.0, 0.5, 13.0 / 14.0)[node] * Lx
    zs = math.floor(zwater / h) * h        # node on the sea floor
    src = np.array([[xs, zs]], np.float32)
    rec = np.stack([np.arange(nx) * h, np.zeros(nx)], 1).astype(np.float32)
    wav = ricker(nt, dt, f0)[:, None].copy()
    Z = gaussian_probes(nt, r, SEED0 + c)
    sm = 10.0 * min(1.0, nx / 1751.0) + 1.0
    return Problem("c1", 2, (nx, nz), h, nb, 0, nt, dt, r, f0, vp, _smooth_slowness(vp, sm),
                   src_xyz=src, rec_xyz=rec, wav=wav, Z=Z)


def make_c2(n=(2000, 800), nt: int = 8000, r: int = 64, nb: int = 40, h: float = 12.5,
            nrec: int | None = None) -> Problem:
    """configs[2]: 2D pseudo-acoustic TTI; smooth eps in [0,.25], delta in [0,.1] (<= eps),
    theta in [-45,45] deg; isotropic in the top 5 cells; off-grid receivers (C10, C15)."""
    c = 2
    rng = np.random.default_rng(SEED0 + c)
    nx, nz = n
    Lx, Lz = (nx - 1) * h, (nz - 1) * h
    z = np.arange(nz) * h
    grad = 1500.0 + 3300.0 * (z / max(Lz, h))
    vp = np.broadcast_to(grad[None, :], (nx, nz)).copy()
    salt = _star_body((nx, nz), h, (0.55 * Lx, 0.5 * Lz), (0.08 * Lx, 0.2 * Lx), (0.1 * Lz, 0.25 * Lz), rng)
    vp = np.where(salt, 4800.0, vp).astype(np.float32)
    sig = 30.0 * min(1.0, nx / 2000.0) + 1.0
    eps = 0.25 * _smooth_noise(rng, (nx, nz), sig)
    delta = 0.10 * _smooth_noise(rng, (nx, nz), sig)
    theta = (np.pi / 4.0) * (2.0 * _smooth_noise(rng, (nx, nz), sig) - 1.0)
    delta = np.minimum(delta, eps)
    eps[:, :5] = 0.0
    delta[:, :5] = 0.0
    theta[:, :5] = 0.0
    dt = 1.0e-3 if n == (2000, 800) else 0.576 * cfl_dt_tti(h, 4800.0, 0.25)
    assert dt < cfl_dt_tti(h, 4800.0, 0.25)
    f0 = 20.0
    # cell-centred source (x = (nx/2 + 1/2) h, z = 1.5 h): the centred rotated operator has the grid
    # Nyquist modes in its null space (C10); a cell-centred bilinear source does not excite them
    src = np.array([[(nx // 2 + 0.5) * h, 1.5 * h]], np.float32)
    if nrec is None:
        nrec = 800 if nx >= 800 else max(8, nx // 3)
    xr = (np.arange(nrec) + 0.37) * (Lx / nrec)                  # off-grid => exercises interpolation
    rec = np.stack([xr, np.full(nrec, 1.5 * h)], 1).astype(np.float32)
    wav = ricker(nt, dt, f0)[:, None].copy()
    Z = gaussian_probes(nt, r, SEED0 + c)
    sm = 10.0 * min(1.0, nx / 2000.0) + 1.0
    return Problem("c2", 2, (nx, nz), h, nb, 1, nt, dt, r, f0, vp, _smooth_slowness(vp, sm),
                   eps=eps.astype(np.float32), delta=delta.astype(np.float32),
                   theta=theta.astype(np.float32), src_xyz=src, rec_xyz=rec, wav=wav, Z=Z)


def make_c3(**kw) -> Problem:
    """configs[3]: offset gather on c1's model and centre shot, nh=41 offsets h in [-20,20]."""
    p = make_c1(**kw)
    p.name = "c3"
    hmax = min(20, (p.n[0] - 1) // 2)
    p.offsets = np.arange(-hmax, hmax + 1, dtype=np.int32)
    return p


def make_c4(n=(512, 512, 256), nt: int = 3000, r: int = 16, nb: int = 40, h: float = 12.5,
            rec_stride: int = 2) -> Problem:
    """configs[4]: 3D acoustic, 6 undulating layers 1500..4000 with a salt ellipsoid at 4000."""
    c = 4
    rng = np.random.default_rng(SEED0 + c)
    nx, ny, nz = n
    Lx, Ly, Lz = (nx - 1) * h, (ny - 1) * h, (nz - 1) * h
    vels = np.linspace(1500.0, 4000.0, 6)
    # low-resolution undulation of each interface (+-50 m), bilinear up-sampling by index
    vp = np.full((nx, ny, nz), vels[0], np.float32)
    zz = (np.arange(nz) * h)[None, None, :]
    gx = np.linspace(0, 1, nx)[:, None]
    gy = np.linspace(0, 1, ny)[None, :]
    for k in range(1, 6):
        a = rng.uniform(-50.0, 50.0, 4)
        und = a[0] * (1 - gx) * (1 - gy) + a[1] * gx * (1 - gy) + a[2] * (1 - gx) * gy + a[3] * gx * gy
        und = und + 25.0 * np.sin(2 * np.pi * (gx * rng.uniform(0.5, 2) + gy * rng.uniform(0.5, 2)))
        zi = k * Lz / 6.0 + np.clip(und, -50.0, 50.0)
        vp[zz[0, 0][None, None, :] >= zi[:, :, None]] = vels[k]
    X = (np.arange(nx) * h - 0.5 * Lx)[:, None, None]
    Y = (np.arange(ny) * h - 0.5 * Ly)[None, :, None]
    Zc = (np.arange(nz) * h - 0.55 * Lz)[None, None, :]
    ax, ay, az = 0.25 * Lx, 0.1875 * Ly, 0.1875 * Lz       # 1.6 x 1.2 x 0.6 km at full size
    vp[(X / ax) ** 2 + (Y / ay) ** 2 + (Zc / az) ** 2 <= 1.0] = 4000.0
    dt = 0.6 * cfl_dt_acoustic(h, 4000.0, 3)
    f0 = 10.0
    src = np.array([[0.5 * Lx, 0.5 * Ly, h]], np.float32)
    rx = np.arange(0, nx, rec_stride) * h
    ry = np.arange(0, ny, rec_stride) * h
    RX, RY = np.meshgrid(rx, ry, indexing="ij")
    rec = np.stack([RX.ravel(), RY.ravel(), np.full(RX.size, h)], 1).astype(np.float32)
    wav = ricker(nt, dt, f0)[:, None].copy()
    Z = gaussian_probes(nt, r, SEED0 + c)
    sm = 4.0 * min(1.0, nx / 512.0) + 1.0
    return Problem("c4", 3, (nx, ny, nz), h, nb, 0, nt, dt, r, f0, vp, _smooth_slowness(vp, sm),
                   src_xyz=src, rec_xyz=rec, wav=wav, Z=Z)


def homogeneous(ndim: int, n, h: float, c: float, f0: float, nt: int, cfl_frac: float,
                nb: int, src, recs, r: int = 1, seed: int = 7) -> Problem:
    """Homogeneous medium for the analytic Green's-function pin."""
    vp = np.full(tuple(n), c, np.float32)
    dt = cfl_frac * cfl_dt_acoustic(h, c, ndim)
    t = np.arange(nt, dtype=np.float64) * dt
    a = (np.pi * f0 * (t - 1.0 / f0)) ** 2
    wav = ((1.0 - 2.0 * a) * np.exp(-a)).astype(np.float32)[:, None].copy()   # NOT mean-subtracted
    return Problem("homog", ndim, tuple(n), h, nb, 0, nt, dt, r, f0, vp, vp.copy(),
                   src_xyz=np.asarray(src, np.float32).reshape(-1, ndim),
                   rec_xyz=np.asarray(recs, np.float32).reshape(-1, ndim),
                   wav=wav, Z=gaussian_probes(nt, r, seed))


def random_tti(n=(40, 36), nb: int = 8, nt: int = 60, r: int = 4, seed: int = 11, h: float = 10.0,
               nsrc: int = 2, nrec: int = 5) -> Problem:
    """Small random TTI problem with off-grid positions (dot tests, parity edge cases)."""
    rng = np.random.default_rng(seed)
    nx, nz = n
    vp = (1500.0 + 2000.0 * _smooth_noise(rng, n, 4.0)).astype(np.float32)
    eps = 0.25 * _smooth_noise(rng, n, 4.0)
    delta = np.minimum(0.1 * _smooth_noise(rng, n, 4.0), eps)
    theta = (np.pi / 4) * (2 * _smooth_noise(rng, n, 4.0) - 1)
    dt = 0.55 * cfl_dt_tti(h, float(vp.max()), 0.25)
    Lx, Lz = (nx - 1) * h, (nz - 1) * h
    src = np.stack([rng.uniform(0, Lx, nsrc), rng.uniform(0, Lz, nsrc)], 1).astype(np.float32)
    rec = np.stack([rng.uniform(0, Lx, nrec), rng.uniform(0, Lz, nrec)], 1).astype(np.float32)
    wav = rng.standard_normal((nt, nsrc)).astype(np.float32)
    return Problem("rtti", 2, n, h, nb, 1, nt, dt, r, 15.0, vp, vp.copy(), eps=eps.astype(np.float32),
                   delta=delta.astype(np.float32), theta=theta.astype(np.float32),
                   src_xyz=src, rec_xyz=rec, wav=wav, Z=gaussian_probes(nt, r, seed))


def random_tti3d(n=(20, 18, 22), nb: int = 6, nt: int = 40, r: int = 4, seed: int = 21, h: float = 10.0,
                 nsrc: int = 2, nrec: int = 5) -> Problem:
    """Small random 3D TTI problem (tilt and azimuth fields) with off-grid positions."""
    rng = np.random.default_rng(seed)
    vp = (1500.0 + 2000.0 * _smooth_noise(rng, n, 3.0)).astype(np.float32)
    eps = 0.25 * _smooth_noise(rng, n, 3.0)
    delta = np.minimum(0.1 * _smooth_noise(rng, n, 3.0), eps)
    theta = (np.pi / 4) * (2 * _smooth_noise(rng, n, 3.0) - 1)
    phi = np.pi * (2 * _smooth_noise(rng, n, 3.0) - 1)
    dt = 0.5 * cfl_dt_tti(h, float(vp.max()), 0.25) * math.sqrt(2.0 / 3.0)      # three axes instead of two
    L = [(a - 1) * h for a in n]
    src = np.stack([rng.uniform(0, l, nsrc) for l in L], 1).astype(np.float32)
    rec = np.stack([rng.uniform(0, l, nrec) for l in L], 1).astype(np.float32)
    wav = rng.standard_normal((nt, nsrc)).astype(np.float32)
    return Problem("rtti3", 3, tuple(n), h, nb, 1, nt, dt, r, 15.0, vp, vp.copy(), eps=eps.astype(np.float32),
                   delta=delta.astype(np.float32), theta=theta.astype(np.float32), phi=phi.astype(np.float32),
                   src_xyz=src, rec_xyz=rec, wav=wav, Z=gaussian_probes(nt, r, seed))


def make_c4_tti(n=(512, 512, 256), nt: int = 3000, r: int = 16, nb: int = 40, h: float = 12.5,
                rec_stride: int = 2) -> Problem:
    """configs[4]'s grid, layered model and acquisition with the anisotropy of configs[2] added (SURVEY 8(f) item 4:
    3D TTI): seeded smooth epsilon in [0, 0.25], delta in [0, 0.1] (<= epsilon), tilt in [-45, 45] deg and azimuth in
    [-180, 180] deg; isotropic in the top 5 cells; cell-centred source and receivers (C10)."""
    p = make_c4(n=n, nt=nt, r=r, nb=nb, h=h, rec_stride=rec_stride)
    rng = np.random.default_rng(SEED0 + 14)
    nx, ny, nz = n
    sig = 30.0 * min(1.0, nx / 512.0) + 1.0

    def smooth():       # low-resolution noise, up-sampled by index (a 512 x 512 x 256 Gaussian filter is too slow)
        c = [max(4, a // 16) for a in n]
        f = gaussian_filter(rng.standard_normal(c), sig / 16.0 + 0.5, mode="reflect")
        f -= f.min()
        f /= max(f.max(), 1e-30)
        ix = np.minimum(np.arange(nx) * c[0] // nx, c[0] - 1)
        iy = np.minimum(np.arange(ny) * c[1] // ny, c[1] - 1)
        iz = np.minimum(np.arange(nz) * c[2] // nz, c[2] - 1)
        return f[np.ix_(ix, iy, iz)]

    eps = 0.25 * smooth()
    delta = np.minimum(0.10 * smooth(), eps)
    theta = (np.pi / 4.0) * (2.0 * smooth() - 1.0)
    phi = np.pi * (2.0 * smooth() - 1.0)
    for a in (eps, delta, theta, phi):
        a[:, :, :5] = 0.0
    p.name, p.physics = "c4tti", 1
    p.eps, p.delta, p.theta, p.phi = (a.astype(np.float32) for a in (eps, delta, theta, phi))
    p.dt = 0.5 * cfl_dt_tti(h, 4000.0, 0.25) * math.sqrt(2.0 / 3.0)
    p.wav = ricker(nt, p.dt, p.f0)[:, None].copy()
    Lx, Ly = (nx - 1) * h, (ny - 1) * h
    p.src_xyz = np.array([[(nx // 2 + 0.5) * h, (ny // 2 + 0.5) * h, 1.5 * h]], np.float32)
    rx = (np.arange(0, nx - 1, rec_stride) + 0.5) * h
    ry = (np.arange(0, ny - 1, rec_stride) + 0.5) * h
    RX, RY = np.meshgrid(rx, ry, indexing="ij")
    p.rec_xyz = np.stack([RX.ravel(), RY.ravel(), np.full(RX.size, 1.5 * h)], 1).astype(np.float32)
    return p


def random_acoustic(ndim: int = 2, n=(40, 36), nb: int = 8, nt: int = 60, r: int = 4, seed: int = 5,
                    h: float = 10.0, nsrc: int = 2, nrec: int = 5) -> Problem:
    """Small random acoustic problem with off-grid positions (dot tests, parity edge cases)."""
    rng = np.random.default_rng(seed)
    vp = (1500.0 + 2500.0 * _smooth_noise(rng, tuple(n), 3.0)).astype(np.float32)
    dt = 0.6 * cfl_dt_acoustic(h, float(vp.max()), ndim)
    L = [(a - 1) * h for a in n]
    src = np.stack([rng.uniform(0, l, nsrc) for l in L], 1).astype(np.float32)
    rec = np.stack([rng.uniform(0, l, nrec) for l in L], 1).astype(np.float32)
    wav = rng.standard_normal((nt, nsrc)).astype(np.float32)
    return Problem("racou", ndim, tuple(n), h, nb, 0, nt, dt, r, 15.0, vp, vp.copy(),
                   src_xyz=src, rec_xyz=rec, wav=wav, Z=gaussian_probes(nt, r, seed))
