"""ctypes binding of include/rtm.h -- argument marshalling only; every step runs in the CUDA kernels.

PyTorch is used for device memory and streams (tensor.data_ptr(), torch.cuda.current_stream())."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIBPATH = os.path.join(_HERE, "csrc", "librtm.so")
_lib = None

EXPORTS = ["rtm_workspace_bytes", "rtm_create", "rtm_destroy", "rtm_coeffs_host", "rtm_coeffs_host3", "rtm_set_model", "rtm_set_model3",
           "rtm_set_probes", "rtm_probes_dtt_host", "rtm_probes_qr_host", "rtm_forward_probe", "rtm_adjoint_image", "rtm_image", "rtm_offset_gather",
           "rtm_offset_gather_xy", "rtm_offset_gather_static",
           "rtm_shot_staging_bytes", "rtm_shot_host", "rtm_export_probes", "rtm_set_snapshots",
           "rtm_export_coeff", "rtm_last_pass_ms", "rtm_pass_ms_mean", "rtm_launch_count", "rtm_set_option", "rtm_strerror", "rtm_last_cuda_error"]


class RTMError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(msg)
        self.code = code


class RtmConfig(C.Structure):
    _fields_ = [("ndim", C.c_int), ("n", C.c_int * 3), ("h", C.c_float), ("nb", C.c_int),
                ("physics", C.c_int), ("nt", C.c_int), ("dt", C.c_double), ("r", C.c_int),
                ("max_pts", C.c_int), ("probe_block", C.c_int), ("probe_fields", C.c_int)]


def lib_path() -> str:
    return _LIBPATH


def load_library():
    """Load csrc/librtm.so; raises (no fallback) if it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIBPATH):
        raise ImportError("CUDA library %s is missing: run `python -c 'import __graft_entry__ as g; g.build()'` "
                          "(there is no CPU fallback)" % _LIBPATH)
    lib = C.CDLL(_LIBPATH)
    vp, ip, fp = C.c_void_p, C.c_int, C.c_float
    cfgp = C.POINTER(RtmConfig)
    lib.rtm_workspace_bytes.restype = C.c_size_t
    lib.rtm_workspace_bytes.argtypes = [cfgp]
    lib.rtm_create.argtypes = [cfgp, vp, C.c_size_t, C.POINTER(vp)]
    lib.rtm_destroy.argtypes = [vp]
    lib.rtm_destroy.restype = None
    lib.rtm_coeffs_host.argtypes = [cfgp] + [vp] * 10
    lib.rtm_set_model.argtypes = [vp] * 8
    lib.rtm_coeffs_host3.argtypes = [cfgp] + [vp] * 13
    lib.rtm_set_model3.argtypes = [vp] * 10
    lib.rtm_set_probes.argtypes = [vp] * 4
    lib.rtm_probes_dtt_host.argtypes = [ip, ip, C.c_double, vp, vp]
    lib.rtm_probes_qr_host.argtypes = [ip, ip, ip, vp, vp, vp]
    lib.rtm_forward_probe.argtypes = [vp, ip, vp, vp, ip, vp, vp, vp]
    lib.rtm_adjoint_image.argtypes = [vp, ip, vp, vp, ip, vp, vp, fp, ip, vp, vp]
    lib.rtm_image.argtypes = [vp, fp, ip, vp, vp]
    lib.rtm_offset_gather.argtypes = [vp, ip, vp, fp, vp, vp]
    lib.rtm_offset_gather_xy.argtypes = [vp, ip, vp, fp, vp, vp]
    lib.rtm_offset_gather_static.argtypes = [ip, ip, ip, vp, vp, ip, vp, fp, vp, vp]
    lib.rtm_shot_staging_bytes.restype = C.c_size_t
    lib.rtm_shot_staging_bytes.argtypes = [cfgp, ip, ip, ip]
    lib.rtm_shot_host.argtypes = [vp, ip, vp, vp, ip, vp, vp, vp, fp, vp, ip, vp, vp, vp, C.c_size_t, vp]
    lib.rtm_export_probes.argtypes = [vp, ip, vp, vp]
    lib.rtm_set_snapshots.argtypes = [vp, ip, vp, vp]
    lib.rtm_export_coeff.argtypes = [vp, ip, vp, vp]
    if hasattr(lib, "rtm_debug_stamps"):          # -DRTM_DEBUG builds only
        lib.rtm_debug_stamps.argtypes = [vp, vp, ip]
    lib.rtm_launch_count.restype = C.c_longlong
    lib.rtm_launch_count.argtypes = [vp]
    lib.rtm_last_pass_ms.restype = C.c_float
    lib.rtm_last_pass_ms.argtypes = [vp, ip]
    lib.rtm_pass_ms_mean.restype = C.c_float
    lib.rtm_pass_ms_mean.argtypes = [vp, ip, ip]
    lib.rtm_set_option.argtypes = [vp, C.c_char_p, ip]
    lib.rtm_strerror.restype = C.c_char_p
    lib.rtm_strerror.argtypes = [ip]
    lib.rtm_last_cuda_error.restype = C.c_char_p
    _lib = lib
    return lib


def _check(rc):
    if rc != 0:
        lib = load_library()
        msg = lib.rtm_strerror(rc).decode()
        if rc == -3:
            msg += ": " + lib.rtm_last_cuda_error().decode()
        raise RTMError(rc, "rtm error %d: %s" % (rc, msg))


def make_config(ndim, n, h, nb, physics, nt, dt, r, max_pts, probe_block=0, probe_fields=0) -> RtmConfig:
    c = RtmConfig()
    c.ndim = int(ndim)
    for i, v in enumerate(n):
        c.n[i] = int(v)
    c.h = float(h)
    c.nb = int(nb)
    c.physics = int(physics)
    c.nt = int(nt)
    c.dt = float(dt)
    c.r = int(r)
    c.max_pts = int(max_pts)
    c.probe_block = int(probe_block)
    c.probe_fields = int(probe_fields)
    return c


def workspace_bytes(cfg: RtmConfig) -> int:
    return int(load_library().rtm_workspace_bytes(C.byref(cfg)))


def _hp(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def coeffs_host(cfg: RtmConfig, vp, eps=None, delta=None, theta=None):
    """rtm_coeffs_host: (K2, epsh, delh, cos, sin, damp1d) as numpy fp32 arrays (canonical [Np])."""
    lib = load_library()
    nd = cfg.ndim
    n = [cfg.n[i] for i in range(nd)]
    P = [a + 2 * cfg.nb for a in n]
    Np = int(np.prod(P))
    f32 = lambda a: None if a is None else np.ascontiguousarray(a, np.float32)
    vp, eps, delta, theta = f32(vp), f32(eps), f32(delta), f32(theta)
    K2 = np.empty(Np, np.float32)
    damp = np.empty(sum(P), np.float32)
    tti = cfg.physics == 1
    outs = [np.empty(Np, np.float32) if tti else None for _ in range(4)]
    _check(lib.rtm_coeffs_host(C.byref(cfg), _hp(vp), _hp(eps), _hp(delta), _hp(theta), _hp(K2),
                               _hp(outs[0]), _hp(outs[1]), _hp(outs[2]), _hp(outs[3]), _hp(damp)))
    return K2, outs[0], outs[1], outs[2], outs[3], damp


def coeffs_host3(cfg: RtmConfig, vp, eps, delta, theta, phi):
    """rtm_coeffs_host3 (3D TTI): (K2, epsh, delh, cos th, sin th, cos ph, sin ph, damp1d) as numpy fp32 arrays."""
    lib = load_library()
    n = [cfg.n[i] for i in range(3)]
    P = [a + 2 * cfg.nb for a in n]
    Np = int(np.prod(P))
    f32 = lambda a: np.ascontiguousarray(a, np.float32)
    vp, eps, delta, theta, phi = (f32(a) for a in (vp, eps, delta, theta, phi))
    outs = [np.empty(Np, np.float32) for _ in range(7)]
    damp = np.empty(sum(P), np.float32)
    _check(lib.rtm_coeffs_host3(C.byref(cfg), _hp(vp), _hp(eps), _hp(delta), _hp(theta), _hp(phi),
                                *[_hp(o) for o in outs], _hp(damp)))
    return tuple(outs) + (damp,)


def probes_qr_host(D, Z):
    """rtm_probes_qr_host: Q [nt][r], orthonormal basis of range(D D^T Z); use with scale = 1."""
    D = np.ascontiguousarray(D, np.float32)
    Z = np.ascontiguousarray(Z, np.float32)
    assert D.ndim == 2 and Z.ndim == 2 and D.shape[0] == Z.shape[0]
    out = np.empty_like(Z)
    _check(load_library().rtm_probes_qr_host(D.shape[0], D.shape[1], Z.shape[1], _hp(D), _hp(Z), _hp(out)))
    return out


def probes_dtt_host(Z, dt):
    """rtm_probes_dtt_host: Zdd [nt][r] such that probing with Zdd accumulates Z^T u_tt (Eq. 2-3)."""
    Z = np.ascontiguousarray(Z, np.float32)
    out = np.empty_like(Z)
    _check(load_library().rtm_probes_dtt_host(Z.shape[0], Z.shape[1], float(dt), _hp(Z), _hp(out)))
    return out


STATIC_SCRATCH_BYTES = 16 << 20     # rtm.h: RTM_STATIC_SCRATCH_BYTES
STATIC_MAX_OFFSETS = 64             # rtm.h: RTM_STATIC_MAX_OFFSETS


def offset_gather_static(U, V, offsets, scale, out, stream=None):
    """rtm_offset_gather_static: the entry point that allocates nothing.  U, V: CUDA fp32 tensors [r][nx][nz] on the
    current device; out: caller-allocated CUDA fp32 tensor [nh][nx][nz] (this wrapper allocates nothing on the device
    either); offsets: host ints.  Calls share one static device array: keep them ordered on the GPU."""
    import torch
    offs = np.ascontiguousarray(offsets, np.int32)
    r, nx, nz = (int(x) for x in U.shape)
    for x in (U, V, out):
        if not (x.is_cuda and x.dtype == torch.float32 and x.is_contiguous()):
            raise ValueError("offset_gather_static takes contiguous fp32 CUDA tensors")
    if tuple(V.shape) != (r, nx, nz) or tuple(out.shape) != (len(offs), nx, nz):
        raise ValueError("offset_gather_static: V must be [r][nx][nz], out [nh][nx][nz]")
    st = torch.cuda.current_stream().cuda_stream if stream is None else stream
    _check(load_library().rtm_offset_gather_static(nx, nz, r, C.c_void_p(U.data_ptr()), C.c_void_p(V.data_ptr()), len(offs),
                                                   _hp(offs), float(scale), C.c_void_p(out.data_ptr()), C.c_void_p(st)))
    return out


class Rtm:
    """One context = one (model, acquisition size) on one GPU.  Same calls as include/rtm.h."""

    def __init__(self, ndim, n, h, nb, physics, nt, dt, r, max_pts, device="cuda:0", probe_block=0, guard_bytes=0,
                 probe_fields=0):
        import torch
        self.torch = torch
        self.lib = load_library()
        self.cfg = make_config(ndim, n, h, nb, physics, nt, dt, r, max_pts, probe_block, probe_fields)
        self.probe_block = int(probe_block)
        self.probe_planes = (2 if int(probe_fields) == 2 else 1) * int(r)
        self.device = torch.device(device)
        nbytes = workspace_bytes(self.cfg)
        if nbytes == 0:
            raise RTMError(-1, "rtm error -1: invalid config")
        # Optional guard bands around the caller-owned workspace (tests only): filled with a byte pattern that
        # check_guards() verifies after a run -- an out-of-bounds WRITE of any kernel next to the workspace shows up.
        self._guard = int(guard_bytes) // 256 * 256
        self._alloc = torch.empty(nbytes + 2 * self._guard, dtype=torch.uint8, device=self.device)
        if self._guard:
            self._alloc[:self._guard] = 0xAB
            self._alloc[self._guard + nbytes:] = 0xAB
        self.workspace = self._alloc[self._guard:self._guard + nbytes]
        h_ = C.c_void_p()
        _check(self.lib.rtm_create(C.byref(self.cfg), self.workspace.data_ptr(), nbytes, C.byref(h_)))
        self.ctx = h_
        self.n = tuple(int(v) for v in n)
        self.N = int(np.prod(self.n))
        self.P = tuple(v + 2 * nb for v in self.n)
        self.Np = int(np.prod(self.P))
        self.nt, self.r, self.ndim, self.physics = int(nt), int(r), int(ndim), int(physics)
        self._keep = []

    @classmethod
    def from_problem(cls, p, device="cuda:0", nt=None, r=None, max_pts=None, probe_block=0, guard_bytes=0,
                     probe_fields=0):
        mp = max(len(p.src_xyz), len(p.rec_xyz)) if max_pts is None else max_pts
        return cls(p.ndim, p.n, p.h, p.nb, p.physics, p.nt if nt is None else nt, p.dt,
                   p.r if r is None else r, mp, device=device, probe_block=probe_block, guard_bytes=guard_bytes,
                   probe_fields=probe_fields)

    def check_guards(self) -> bool:
        """True if the guard bands around the workspace still hold their pattern (see __init__)."""
        if not self._guard:
            return True
        self.torch.cuda.synchronize(self.device)
        lo, hi = self._alloc[:self._guard], self._alloc[self._guard + self.workspace.numel():]
        return bool((lo == 0xAB).all().item()) and bool((hi == 0xAB).all().item())

    def close(self):
        if getattr(self, "ctx", None):
            self.torch.cuda.synchronize(self.device)
            self.lib.rtm_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- helpers -------------------------------------------------------------------------------------
    def _stream(self):
        return C.c_void_p(self.torch.cuda.current_stream(self.device).cuda_stream)

    def _dev(self, a):
        t = self.torch
        if a is None:
            return None
        if isinstance(a, t.Tensor):
            assert a.is_cuda and a.dtype == t.float32 and a.is_contiguous()
            return a
        return t.from_numpy(np.ascontiguousarray(a, np.float32)).to(self.device)

    @staticmethod
    def _ptr(tens):
        return None if tens is None else C.c_void_p(tens.data_ptr())

    # -- API ------------------------------------------------------------------------------------------
    def set_model_from_earth(self, vp, eps=None, delta=None, theta=None, phi=None):
        if self.physics == 1 and self.ndim == 3:            # 3D TTI: tilt and azimuth (reading C30)
            K2, eh, dh, cs, sn, cp, sp, damp = coeffs_host3(self.cfg, vp, eps, delta, theta, phi)
            d = [self._dev(a) for a in (K2, eh, dh, cs, sn, cp, sp)]
            damp = np.ascontiguousarray(damp, np.float32)
            _check(self.lib.rtm_set_model3(self.ctx, *[self._ptr(x) for x in d], _hp(damp), self._stream()))
            self._keep = [d, damp]
            return K2, eh, dh, cs, sn, damp, cp, sp
        K2, eh, dh, cs, sn, damp = coeffs_host(self.cfg, vp, eps, delta, theta)
        self.set_model(K2, eh, dh, cs, sn, damp)
        return K2, eh, dh, cs, sn, damp

    def set_model(self, K2, epsh, delh, cosT, sinT, damp1d):
        d = [self._dev(a) for a in (K2, epsh, delh, cosT, sinT)]
        damp = np.ascontiguousarray(damp1d, np.float32)
        _check(self.lib.rtm_set_model(self.ctx, *[self._ptr(x) for x in d], _hp(damp), self._stream()))
        self._keep = [d, damp]

    def set_probes(self, Zf, Za=None):
        zf = self._dev(Zf)
        za = zf if Za is None else self._dev(Za)
        assert tuple(zf.shape) == (self.nt, self.r) and tuple(za.shape) == (self.nt, self.r)
        _check(self.lib.rtm_set_probes(self.ctx, self._ptr(zf), self._ptr(za), self._stream()))
        self._keep_z = (zf, za)

    def forward_probe(self, src_xyz, wav, rec_xyz, data_out=True):
        t = self.torch
        src = np.ascontiguousarray(src_xyz, np.float32).reshape(-1, self.ndim)
        rec = np.ascontiguousarray(rec_xyz, np.float32).reshape(-1, self.ndim)
        w = self._dev(wav)
        assert w.numel() == self.nt * len(src)
        out = None
        if data_out is True:
            out = t.empty((self.nt, len(rec)), dtype=t.float32, device=self.device)
        elif data_out is not None and data_out is not False:
            out = data_out
        _check(self.lib.rtm_forward_probe(self.ctx, len(src), _hp(src), self._ptr(w), len(rec), _hp(rec),
                                          self._ptr(out), self._stream()))
        return out

    def adjoint_image(self, rec_xyz, data_in, src_xyz, scale=None, qadj_out=False, image=True, accumulate=False):
        t = self.torch
        src = np.ascontiguousarray(src_xyz, np.float32).reshape(-1, self.ndim)
        rec = np.ascontiguousarray(rec_xyz, np.float32).reshape(-1, self.ndim)
        din = self._dev(data_in)
        assert din.numel() == self.nt * len(rec)
        q = t.empty((self.nt, len(src)), dtype=t.float32, device=self.device) if qadj_out else None
        img = None
        if image is True:
            img = t.zeros(self.n, dtype=t.float32, device=self.device)
        elif image is not None and image is not False:
            img = image
        sc = 1.0 / self.r if scale is None else float(scale)
        _check(self.lib.rtm_adjoint_image(self.ctx, len(rec), _hp(rec), self._ptr(din), len(src), _hp(src),
                                          self._ptr(q), sc, 1 if accumulate else 0, self._ptr(img), self._stream()))
        return img, q

    def image(self, scale=None, out=None, accumulate=False):
        """rtm_image: Eq. 3 from the Uz / Vz of the last forward and adjoint passes."""
        t = self.torch
        if out is None:
            out = t.zeros(self.n, dtype=t.float32, device=self.device)
        sc = 1.0 / self.r if scale is None else float(scale)
        _check(self.lib.rtm_image(self.ctx, sc, 1 if accumulate else 0, self._ptr(out), self._stream()))
        return out

    def offset_gather(self, offsets, scale=None, out=None):
        t = self.torch
        offs = np.ascontiguousarray(offsets, np.int32)
        if out is None:
            out = t.empty((len(offs),) + self.n, dtype=t.float32, device=self.device)
        sc = 1.0 / self.r if scale is None else float(scale)
        _check(self.lib.rtm_offset_gather(self.ctx, len(offs), _hp(offs), sc, self._ptr(out), self._stream()))
        return out

    def offset_gather_xy(self, offsets_xy, scale=None, out=None):
        """rtm_offset_gather_xy: offsets_xy [nh][2] = (hx, hy) grid points, 3D grids only."""
        t = self.torch
        offs = np.ascontiguousarray(offsets_xy, np.int32).reshape(-1, 2)
        if out is None:
            out = t.empty((len(offs),) + self.n, dtype=t.float32, device=self.device)
        sc = 1.0 / self.r if scale is None else float(scale)
        _check(self.lib.rtm_offset_gather_xy(self.ctx, len(offs), _hp(offs), sc, self._ptr(out), self._stream()))
        return out

    def shot_host(self, src_xyz, h_wav, rec_xyz, h_data_in, h_data_out=None, h_image=None, offsets=None,
                  h_gather=None, scale=None, staging=None):
        """rtm_shot_host: h_* are pinned CPU torch tensors (or None)."""
        t = self.torch
        src = np.ascontiguousarray(src_xyz, np.float32).reshape(-1, self.ndim)
        rec = np.ascontiguousarray(rec_xyz, np.float32).reshape(-1, self.ndim)
        nh = 0 if offsets is None else len(offsets)
        offs = None if offsets is None else np.ascontiguousarray(offsets, np.int32)
        need = int(self.lib.rtm_shot_staging_bytes(C.byref(self.cfg), len(src), len(rec), nh))
        if staging is None or staging.numel() < need:
            staging = t.empty(need, dtype=t.uint8, device=self.device)
        self._staging = staging
        sc = 1.0 / self.r if scale is None else float(scale)
        hp = lambda x: None if x is None else C.c_void_p(x.data_ptr())
        _check(self.lib.rtm_shot_host(self.ctx, len(src), _hp(src), hp(h_wav), len(rec), _hp(rec), hp(h_data_in),
                                      hp(h_data_out), sc, hp(h_image), nh, _hp(offs), hp(h_gather),
                                      C.c_void_p(staging.data_ptr()), staging.numel(), self._stream()))
        return staging

    def export_probes(self, which):
        t = self.torch
        out = t.empty((self.probe_planes, self.N), dtype=t.float32, device=self.device)
        _check(self.lib.rtm_export_probes(self.ctx, int(which), self._ptr(out), self._stream()))
        return out

    def set_snapshots(self, steps):
        t = self.torch
        steps = np.ascontiguousarray(steps, np.int32)
        nf = 2 if self.physics == 1 else 1
        out = t.zeros((len(steps), nf, self.Np), dtype=t.float32, device=self.device)
        _check(self.lib.rtm_set_snapshots(self.ctx, len(steps), _hp(steps), self._ptr(out)))
        return out

    def export_coeff(self, which):
        t = self.torch
        out = t.empty(self.Np, dtype=t.float32, device=self.device)
        _check(self.lib.rtm_export_coeff(self.ctx, int(which), self._ptr(out), self._stream()))
        return out

    def debug_stamps(self, nblocks=1024):
        if not hasattr(self.lib, "rtm_debug_stamps"):
            raise RTMError(-1, "rtm_debug_stamps exists only in a library built with RTM_DEBUG=1")
        out = np.zeros((nblocks, 8), np.uint64)
        _check(self.lib.rtm_debug_stamps(self.ctx, _hp(out), int(nblocks)))
        return out

    def launch_count(self) -> int:
        return int(self.lib.rtm_launch_count(self.ctx))

    def last_pass_ms(self, which: int) -> float:
        return float(self.lib.rtm_last_pass_ms(self.ctx, int(which)))

    def pass_ms_mean(self, which: int, count: int) -> float:
        return float(self.lib.rtm_pass_ms_mean(self.ctx, int(which), int(count)))

    def set_option(self, name: str, value: int):
        _check(self.lib.rtm_set_option(self.ctx, name.encode(), int(value)))
