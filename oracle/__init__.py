"""CPU oracle -- TEST INFRASTRUCTURE ONLY (see rtm_oracle.c header).

Thin ctypes wrapper around ``oracle/rtm_oracle.c`` (plain C, fp64, OpenMP over the outer spatial
loop).  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline /
``--impl reference`` legs may import this package.  It imports nothing from the CUDA package.

Beside the C routines it holds two plain numpy functions for Eq. 2-3's gradient-type imaging condition
(``probes_dtt``, ``exact_gradient_image``; pins in tests/test_oracle_estimator.py).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "rtm_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, no fast-math, OpenMP)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-std=gnu11", "-fopenmp", "-shared", "-fPIC", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


class _Cfg(C.Structure):
    _fields_ = [("ndim", C.c_int), ("n", C.c_int * 3), ("nb", C.c_int), ("physics", C.c_int),
                ("nt", C.c_int), ("r", C.c_int), ("h", C.c_double), ("dt", C.c_double)]


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(_LIB)
        _lib.orc_num_threads.restype = C.c_int
    return _lib


def _cfg(p, nt=None, r=None) -> _Cfg:
    c = _Cfg()
    c.ndim = p.ndim
    for i, v in enumerate(p.n):
        c.n[i] = int(v)
    c.nb = p.nb
    c.physics = p.physics
    c.nt = int(p.nt if nt is None else nt)
    c.r = int(p.r if r is None else r)
    c.h = float(np.float32(p.h))
    c.dt = float(p.dt)
    return c


def _fp(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _f32(a):
    return None if a is None else np.ascontiguousarray(a, np.float32)


def num_threads() -> int:
    return int(_load().orc_num_threads())


class Coeffs:
    """fp32 coefficient arrays of O1 (canonical padded order)."""

    def __init__(self, K2, damp, epsh=None, delh=None, cosT=None, sinT=None, cosP=None, sinP=None):
        self.K2, self.damp, self.epsh, self.delh, self.cosT, self.sinT = K2, damp, epsh, delh, cosT, sinT
        self.cosP, self.sinP = cosP, sinP          # 3D TTI: azimuth of the symmetry axis (reading C30)


def coeffs(p, vp=None) -> Coeffs:
    """O1: coefficients from (vp, eps, delta, theta, dt, h, nb)."""
    lib = _load()
    c = _cfg(p)
    vp = _f32(p.vp if vp is None else vp)
    Np = p.Np
    K2 = np.zeros(Np, np.float32)
    damp = np.zeros(sum(p.P), np.float32)
    tti = p.physics == 1
    eh = np.zeros(Np, np.float32) if tti else None
    dh = np.zeros(Np, np.float32) if tti else None
    ct = np.zeros(Np, np.float32) if tti else None
    st = np.zeros(Np, np.float32) if tti else None
    if tti and p.ndim == 3:
        cp, sp = np.zeros(Np, np.float32), np.zeros(Np, np.float32)
        rc = lib.orc_coeffs3(C.byref(c), _fp(vp), _fp(_f32(p.eps)), _fp(_f32(p.delta)), _fp(_f32(p.theta)),
                             _fp(_f32(p.phi)), _fp(K2), _fp(damp), _fp(eh), _fp(dh), _fp(ct), _fp(st), _fp(cp), _fp(sp))
        assert rc == 0
        return Coeffs(K2, damp, eh, dh, ct, st, cp, sp)
    rc = lib.orc_coeffs(C.byref(c), _fp(vp), _fp(_f32(p.eps)), _fp(_f32(p.delta)), _fp(_f32(p.theta)),
                        _fp(K2), _fp(damp), _fp(eh), _fp(dh), _fp(ct), _fp(st))
    assert rc == 0
    return Coeffs(K2, damp, eh, dh, ct, st)


def propagate(p, co: Coeffs, adjoint: bool, inj_xyz, inj_val, smp_xyz=None, Z=None, want_hist=False,
              snap_steps=(), nt=None, want_samples=True, fields=1):
    """O2/O3/O5/O6.  Returns dict(samples [nt][nsmp], PZ [r][N], hist [nt][N], snaps [ns][nf][Np]).
    fields=2 (TTI, reading C29): p and r probed apart, PZ [2r][N] (p planes, then r planes), hist [nt][2][N]."""
    lib = _load()
    nt = int(p.nt if nt is None else nt)
    r = 0 if Z is None else int(Z.shape[1])
    c = _cfg(p, nt=nt, r=r)
    inj_xyz = _f32(inj_xyz).reshape(-1, p.ndim)
    inj_val = _f32(inj_val).reshape(nt, -1)
    ninj = inj_xyz.shape[0]
    assert inj_val.shape[1] == ninj
    if smp_xyz is None:
        smp_xyz = np.zeros((0, p.ndim), np.float32)
    smp_xyz = _f32(smp_xyz).reshape(-1, p.ndim)
    nsmp = smp_xyz.shape[0]
    N, Np = p.N, p.Np
    nf = 2 if p.physics == 1 else 1
    out = np.zeros((nt, nsmp), np.float64) if (want_samples and nsmp > 0) else None
    Zc = _f32(Z)
    assert fields in (1, 2)
    PZ = np.zeros((fields * r, N), np.float64) if r > 0 else None
    hist = np.zeros((nt, N) if fields == 1 else (nt, 2, N), np.float64) if want_hist else None
    ss = np.asarray(list(snap_steps), np.int32)
    snaps = np.zeros((len(ss), nf, Np), np.float64) if len(ss) else None
    if p.physics == 1 and p.ndim == 3:
        assert co.cosP is not None
        fn3 = lib.orc_propagate3 if fields == 1 else lib.orc_propagate3_pr      # readings C30 / C29 + C30
        rc = fn3(C.byref(c), C.c_int(1 if adjoint else 0), _fp(co.K2), _fp(co.damp), _fp(co.epsh),
                                _fp(co.delh), _fp(co.cosT), _fp(co.sinT), _fp(co.cosP), _fp(co.sinP), C.c_int(ninj),
                                _fp(inj_xyz), _fp(inj_val), C.c_int(nsmp), _fp(smp_xyz), _fp(out), _fp(Zc), _fp(PZ),
                                _fp(hist), C.c_int(len(ss)), _fp(ss), _fp(snaps))
    else:
        fn = lib.orc_propagate if fields == 1 else lib.orc_propagate_pr
        rc = fn(C.byref(c), C.c_int(1 if adjoint else 0), _fp(co.K2), _fp(co.damp), _fp(co.epsh),
                _fp(co.delh), _fp(co.cosT), _fp(co.sinT), C.c_int(ninj), _fp(inj_xyz), _fp(inj_val),
                C.c_int(nsmp), _fp(smp_xyz), _fp(out), _fp(Zc), _fp(PZ), _fp(hist),
                C.c_int(len(ss)), _fp(ss), _fp(snaps))
    if rc != 0:
        raise ValueError("orc_propagate failed rc=%d" % rc)
    return {"samples": out, "PZ": PZ, "hist": hist, "snaps": snaps}


def forward(p, co, Z=None, **kw):
    """O2/O5: source -> data, Uz."""
    return propagate(p, co, False, p.src_xyz, p.wav, p.rec_xyz, Z=Z, **kw)


def adjoint(p, co, din, Z=None, **kw):
    """O3/O6: data -> qadj, Vz."""
    return propagate(p, co, True, p.rec_xyz, din, p.src_xyz, Z=Z, **kw)


def image(Uz, Vz, scale):
    """Eq. 3."""
    lib = _load()
    r, N = Uz.shape
    Uz = np.ascontiguousarray(Uz, np.float64)
    Vz = np.ascontiguousarray(Vz, np.float64)
    I = np.zeros(N, np.float64)
    lib.orc_image(C.c_int(r), C.c_long(N), _fp(Uz), _fp(Vz), C.c_double(scale), _fp(I))
    return I


def exact_image(uh, vh):
    """Eq. 2 (u.v form) from stored histories [nt][N]."""
    lib = _load()
    nt, N = uh.shape
    uh = np.ascontiguousarray(uh, np.float64)
    vh = np.ascontiguousarray(vh, np.float64)
    I = np.zeros(N, np.float64)
    lib.orc_exact_image(C.c_int(nt), C.c_long(N), _fp(uh), _fp(vh), _fp(I))
    return I


def probes_dtt(Z, dt):
    """Reading C4 (Eq. 2-3 probe u_tt): Zdd[n] = (Z[n] - 2 Z[n+1] + Z[n+2]) / dt^2 with
    Z[nt] = Z[nt+1] = 0, so that  sum_n Z[n] (w[n] - 2 w[n-1] + w[n-2]) / dt^2 = sum_n Zdd[n] w[n]  for the fields
    w[n] computed by step n (w[-1] = w[-2] = 0).  fp64, one rounding to the fp32 the GPU receives (C18)."""
    Z = np.asarray(Z, np.float32).astype(np.float64)
    nt = Z.shape[0]
    Zp = np.vstack([Z, np.zeros((2, Z.shape[1]))])
    return (((Zp[:nt] - 2.0 * Zp[1:nt + 1]) + Zp[2:nt + 2]) * (1.0 / (float(dt) * float(dt)))).astype(np.float32)


def probes_qr(D, Z):
    """PAPER.md:L33 "[Q, ~] = qr(A Z) where Z is a Rademacher random matrix": range-finder probes (refs [21, 26, 27]).
    Reading C3: A = D D^T, the nt x nt temporal covariance of the shot record D [nt][nrec] that the
    adjoint pass back-propagates (never formed: Y = D (D^T Z)); Q [nt][r] = the orthonormal factor of the thin QR of
    Y with diag(R) > 0.  Q^T Q = I_r, so the estimator sum_k (Q^T u)_k (Q^T v)_k = u^T Q Q^T v is a projection and
    its scale is 1, not 1/r.  fp64 (numpy.linalg.qr as the library step), one rounding to the fp32 the GPU receives."""
    D = np.asarray(D, np.float32).astype(np.float64)
    Z = np.asarray(Z, np.float32).astype(np.float64)
    Y = D @ (D.T @ Z)
    Q, R = np.linalg.qr(Y)
    Q = Q * np.where(np.diag(R) < 0, -1.0, 1.0)[None, :]
    return Q.astype(np.float32)


def exact_gradient_image(uh, vh, dt):
    """Eq. 2 as printed: sum_t u_tt(t) v(t) from stored histories [nt][N], with the second time
    difference of the update itself, u_tt[n] = (w[n] - 2 w[n-1] + w[n-2]) / dt^2 (zero initial fields)."""
    uh = np.asarray(uh, np.float64)
    vh = np.asarray(vh, np.float64)
    nt = uh.shape[0]
    I = np.zeros(uh.shape[1], np.float64)
    for n in range(nt):
        w1 = uh[n - 1] if n >= 1 else 0.0
        w2 = uh[n - 2] if n >= 2 else 0.0
        I += ((uh[n] - 2.0 * w1) + w2) / (float(dt) * float(dt)) * vh[n]
    return I


def offset_gather(n, Uz, Vz, offsets, scale):
    """Eq. 4: [nh][N]; offsets in grid points along x."""
    lib = _load()
    r, N = Uz.shape
    nx = int(n[0])
    nrest = N // nx
    Uz = np.ascontiguousarray(Uz, np.float64)
    Vz = np.ascontiguousarray(Vz, np.float64)
    offs = np.ascontiguousarray(offsets, np.int32)
    G = np.zeros((len(offs), N), np.float64)
    lib.orc_offset_gather(C.c_int(nx), C.c_long(nrest), C.c_int(r), _fp(Uz), _fp(Vz), C.c_int(len(offs)),
                          _fp(offs), C.c_double(scale), _fp(G))
    return G


def offset_gather_xy(n, Uz, Vz, offsets_xy, scale):
    """Eq. 4 with vector offsets h = (hx, hy) on a 3D grid n = (nx, ny, nz): [nh][N] (reading C28)."""
    lib = _load()
    r, N = Uz.shape
    nx, ny, nz = (int(v) for v in n)
    assert N == nx * ny * nz
    Uz = np.ascontiguousarray(Uz, np.float64)
    Vz = np.ascontiguousarray(Vz, np.float64)
    offs = np.ascontiguousarray(offsets_xy, np.int32).reshape(-1, 2)
    G = np.zeros((len(offs), N), np.float64)
    lib.orc_offset_gather_xy(C.c_int(nx), C.c_int(ny), C.c_int(nz), C.c_int(r), _fp(Uz), _fp(Vz),
                             C.c_int(len(offs)), _fp(offs), C.c_double(scale), _fp(G))
    return G


def tti_H(p, co, which, f):
    """Test hook: H_perp (which=0) / H_par (which=1) applied to a padded-grid function [Np]."""
    lib = _load()
    c = _cfg(p)
    f = np.ascontiguousarray(f, np.float64).ravel()
    out = np.zeros_like(f)
    if p.ndim == 3:
        rc = lib.orc_tti_H3(C.byref(c), _fp(co.cosT), _fp(co.sinT), _fp(co.cosP), _fp(co.sinP), C.c_int(which), _fp(f), _fp(out))
    else:
        rc = lib.orc_tti_H(C.byref(c), _fp(co.cosT), _fp(co.sinT), C.c_int(which), _fp(f), _fp(out))
    assert rc == 0
    return out
