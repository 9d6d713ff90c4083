"""Pins for the oracle's 3D TTI operator (reading C30: PAPER.md:L77 says only "TTI", L81 "generalize to 3D").

  * adjointness <F q, d> = <q, F^T d> to 1e-12 with random tilt / azimuth fields and off-grid positions
  * H_perp, H_par symmetric and negative semi-definite
  * constant angles: H_perp + H_par = Dx Dx + Dy Dy + Dz Dz (the three directions are orthonormal; a wrong sign or a
    swapped component in n, e1 or e2 breaks it), and for th = 0 H_par = Dz Dz alone
  * eps = delta = 0: p == r bit for bit whatever the angles, and the data agree with the 3D acoustic scheme
  * kinematics in a homogeneous medium tilted by th = 30 deg at azimuth ph = 40 deg: the pulse travels at c along the
    axis n and at c sqrt(1 + 2 eps) along e1 and e2; the mirror images of e1 (th -> -th) and e2 (ph -> -ph) are slower
    (kills: a sign flip of sin th or sin ph, eps-hat on the wrong field, H_perp / H_par swapped)
"""
import math

import numpy as np

import oracle as orc
import rtm_inputs as ri


def test_dot_product_3d_tti():
    p = ri.random_tti3d(n=(15, 13, 14), nb=5, nt=40, seed=2)
    co = orc.coeffs(p)
    rng = np.random.default_rng(17)
    f = orc.forward(p, co)
    d = rng.standard_normal(f["samples"].shape).astype(np.float32)
    a = orc.adjoint(p, co, d)
    lhs = float((f["samples"] * d.astype(np.float64)).sum())
    rhs = float((p.wav.astype(np.float64) * a["samples"]).sum())
    assert abs(lhs) > 0 and abs(lhs - rhs) <= 1e-12 * abs(lhs)


def test_H3_symmetric_negative_semidefinite():
    p = ri.random_tti3d(n=(14, 12, 13), nb=4, nt=4)
    co = orc.coeffs(p)
    rng = np.random.default_rng(0)
    f, g = rng.standard_normal(p.Np), rng.standard_normal(p.Np)
    for which in (0, 1):
        Hf, Hg = orc.tti_H(p, co, which, f), orc.tti_H(p, co, which, g)
        a, b = float(f @ Hg), float(g @ Hf)
        assert abs(a - b) <= 1e-12 * max(abs(a), abs(b))
        assert float(f @ Hf) < 0.0 and float(g @ Hg) < 0.0


_C1 = [float(np.float32(x)) for x in (4.0 / 5.0, -1.0 / 5.0, 4.0 / 105.0, -1.0 / 280.0)]


def _d(f, axis):
    """undivided centred order-8 first derivative with zeros outside the array (numpy slicing)"""
    e = np.zeros(tuple(s + 8 for s in f.shape))
    e[4:-4, 4:-4, 4:-4] = f
    out = np.zeros_like(f)
    c = [slice(4, -4)] * 3
    for j, w in enumerate(_C1, 1):
        hi, lo = list(c), list(c)
        hi[axis] = slice(4 + j, e.shape[axis] - 4 + j)
        lo[axis] = slice(4 - j, e.shape[axis] - 4 - j)
        out += w * (e[tuple(hi)] - e[tuple(lo)])
    return out


def test_constant_angles_sum_to_the_laplacian():
    p = ri.random_tti3d(n=(18, 17, 16), nb=3, nt=4)
    rng = np.random.default_rng(1)
    f = rng.standard_normal(p.P)
    lap = sum(_d(_d(f, ax), ax) for ax in range(3))          # Dx Dx + Dy Dy + Dz Dz, zeros outside P
    s = slice(9, -9)                                           # away from the edge (g is cut off outside P)
    for th, ph in ((0.5, 0.7), (-0.6, 2.5), (0.0, 1.0)):
        p.theta[:], p.phi[:] = th, ph
        co = orc.coeffs(p)
        Hp = orc.tti_H(p, co, 0, f.ravel()).reshape(p.P)
        Hl = orc.tti_H(p, co, 1, f.ravel()).reshape(p.P)
        # 1e-6: cos / sin are the fp32-rounded inputs (C18), so the basis is orthonormal to 1e-7 only
        assert np.abs((Hp + Hl - lap)[s, s, s]).max() <= 1e-6 * np.abs(lap[s, s, s]).max(), (th, ph)
        if th == 0.0:
            dzz = _d(_d(f, 2), 2)
            assert np.abs((Hl - dzz)[s, s, s]).max() <= 1e-12 * np.abs(dzz).max()


def test_isotropic_limit_3d():
    args = (3, (41, 39, 40), 10.0, 2000.0, 10.0, 110, 0.3, 8, [195.0, 185.0, 195.0],
            [[195.0, 185.0, 295.0], [265.0, 185.0, 195.0], [195.0, 245.0, 235.0]])
    pa = ri.homogeneous(*args)
    pt = ri.homogeneous(*args)
    pt.physics = 1
    rng = np.random.default_rng(5)
    pt.eps = np.zeros(pt.n, np.float32)
    pt.delta = np.zeros(pt.n, np.float32)
    pt.theta = rng.uniform(-0.7, 0.7, pt.n).astype(np.float32)      # any angles: the medium is isotropic
    pt.phi = rng.uniform(-3.0, 3.0, pt.n).astype(np.float32)
    ca, ct = orc.coeffs(pa), orc.coeffs(pt)
    assert np.array_equal(ca.K2, ct.K2)
    ft = orc.forward(pt, ct, snap_steps=[60])
    assert np.array_equal(ft["snaps"][0, 0], ft["snaps"][0, 1]) and np.abs(ft["snaps"]).max() > 0     # p == r
    pt.theta[:], pt.phi[:] = 0.0, 0.0                                # constant angles: compare with the acoustic scheme
    f0 = orc.forward(pt, orc.coeffs(pt))["samples"]
    da = orc.forward(pa, ca)["samples"]
    assert 0 < np.linalg.norm(da - f0) <= 5e-2 * np.linalg.norm(da)   # different 2nd-derivative stencils: loose


def test_tilted_3d_kinematics():
    # elliptic anisotropy (delta = eps): no pseudo-acoustic shear artefact, which along the axis is stronger than the qP
    # pulse at these short distances and would fool the peak picker; orientation and eps-hat placement are pinned all the same
    c, h, f0, n, nb, eps, delta = 2000.0, 10.0, 20.0, (65, 65, 65), 10, 0.2, 0.2
    th, ph = math.radians(30.0), math.radians(40.0)
    st, ct, sp, cp = math.sin(th), math.cos(th), math.sin(ph), math.cos(ph)
    dirs = {"axis": (st * cp, st * sp, ct), "e1": (ct * cp, ct * sp, -st), "e2": (-sp, cp, 0.0),
            "e1_mirror": (ct * cp, ct * sp, st), "e2_mirror": (sp, cp, 0.0)}
    src = np.array([[325.0, 325.0, 325.0]])
    recs = []
    for d in dirs.values():
        for rho in (100.0, 250.0):
            q = src[0] + rho * np.array(d)
            recs.append((np.floor(q / h) + 0.5) * h)
    recs = np.array(recs)
    dt = 0.5 * ri.cfl_dt_tti(h, c, eps) * math.sqrt(2.0 / 3.0)
    nt = int(0.21 / dt)
    p = ri.homogeneous(3, n, h, c, f0, nt, 0.3, nb, src, recs)
    p.dt, p.physics = dt, 1
    t = np.arange(nt) * dt
    a = (np.pi * f0 * (t - 1.0 / f0)) ** 2
    p.wav = ((1.0 - 2.0 * a) * np.exp(-a)).astype(np.float32)[:, None].copy()
    p.eps, p.delta, p.theta, p.phi = (np.full(n, v, np.float32) for v in (eps, delta, th, ph))
    d = orc.forward(p, orc.coeffs(p))["samples"]

    def peak_time(tr):
        e = np.abs(tr)
        i = int(np.argmax(e >= 0.5 * e.max()))
        while i + 1 < len(e) and e[i + 1] >= e[i]:
            i += 1
        return (i + 0.5 * (e[i - 1] - e[i + 1]) / (e[i - 1] - 2.0 * e[i] + e[i + 1])) * dt

    v = {}
    for k, name in enumerate(dirs):
        r0, r1 = recs[2 * k], recs[2 * k + 1]
        v[name] = (np.linalg.norm(r1 - src[0]) - np.linalg.norm(r0 - src[0])) / (peak_time(d[:, 2 * k + 1]) - peak_time(d[:, 2 * k])) / c
    fast = math.sqrt(1.0 + 2.0 * eps)
    assert abs(v["axis"] - 1.0) <= 1e-2, v
    assert abs(v["e1"] / fast - 1.0) <= 1e-2 and abs(v["e2"] / fast - 1.0) <= 1e-2, v
    assert v["e1_mirror"] < 1.08 and v["e2_mirror"] < 1.16, v       # 30 deg / 60 deg off the axis: clearly slower than e1, e2


def test_two_probed_fields_3d():
    """Readings C29 + C30 (four compressed arrays of the TTI gradient, in 3D): with fields = 2 the pass probes p and r
    apart.  Pinned against things the one-field pass and numpy already fix: (i) plane k of p plus plane k of r, halved,
    is the one-field plane of 1/2 (p + r); (ii) PZ = hist^T Z by a numpy matmul, field by field; (iii) field 0 of the
    history is the physical part of the p snapshot and field 1 of the r snapshot (kills a swap of the two)."""
    p = ri.random_tti3d(n=(13, 11, 12), nb=4, nt=30, r=3, seed=5)
    co = orc.coeffs(p)
    one = orc.forward(p, co, Z=p.Z)
    steps = [7, 29]
    two = orc.forward(p, co, Z=p.Z, fields=2, want_hist=True, snap_steps=steps)
    P, R = two["PZ"][:p.r], two["PZ"][p.r:]
    assert np.abs(one["PZ"]).max() > 0 and np.abs(P - R).max() > 1e-3 * np.abs(P).max()      # p and r do differ
    assert np.abs(0.5 * (P + R) - one["PZ"]).max() <= 1e-12 * np.abs(one["PZ"]).max()
    assert np.array_equal(two["samples"], one["samples"])
    Z = p.Z.astype(np.float64)
    for f in range(2):
        ref = Z.T @ two["hist"][:, f, :]
        assert np.abs(ref - two["PZ"][f * p.r:(f + 1) * p.r]).max() <= 1e-12 * np.abs(ref).max()
    nb = p.nb
    for q, n in enumerate(steps):
        for f in range(2):
            full = two["snaps"][q, f].reshape(p.P)
            phys = full[nb:nb + p.n[0], nb:nb + p.n[1], nb:nb + p.n[2]].ravel()
            assert np.array_equal(phys, two["hist"][n, f])
    # the adjoint pass takes the same path
    d = one["samples"].astype(np.float32)
    a1 = orc.adjoint(p, co, d, Z=p.Z)
    a2 = orc.adjoint(p, co, d, Z=p.Z, fields=2)
    assert np.abs(0.5 * (a2["PZ"][:p.r] + a2["PZ"][p.r:]) - a1["PZ"]).max() <= 1e-12 * np.abs(a1["PZ"]).max()
