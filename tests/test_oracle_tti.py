"""Pins for the oracle's TTI operator (O5/O6; PAPER.md:L77 says only "TTI", equations per DESIGN.md C10).

  * H_perp, H_par are symmetric and negative semi-definite (they are -G^T G with D^T = -D, zeros outside P)
  * eps = delta = theta = 0  =>  p == r exactly, and the field agrees with the acoustic scheme to
    discretisation error (different 2nd-derivative stencils: loose 1e-2)
  * theta -> theta + pi leaves every result unchanged (the symmetry axis is a line, not a vector)
  * theta = 0, eps = delta = 0: H_perp + H_par = Dx Dx + Dz Dz applied to a polynomial gives its Laplacian
"""
import numpy as np

import oracle as orc
import rtm_inputs as ri


def test_H_symmetric_negative_semidefinite():
    p = ri.random_tti(n=(22, 19), nb=5, nt=4)
    co = orc.coeffs(p)
    rng = np.random.default_rng(0)
    f = rng.standard_normal(p.Np)
    g = rng.standard_normal(p.Np)
    for which in (0, 1):
        Hf = orc.tti_H(p, co, which, f)
        Hg = orc.tti_H(p, co, which, g)
        a, b = float(f @ Hg), float(g @ Hf)
        assert abs(a - b) <= 1e-12 * max(abs(a), abs(b))
        assert float(f @ Hf) < 0.0 and float(g @ Hg) < 0.0
    # constants away from the edge are annihilated
    one = np.ones(p.Np)
    H1 = orc.tti_H(p, co, 0, one).reshape(p.P)
    assert np.abs(H1[9:-9, 9:-9]).max() <= 1e-13


def test_untilted_H_is_second_derivative_of_polynomial():
    p = ri.random_tti(n=(30, 28), nb=4, nt=4)
    p.theta[:] = 0.0
    co = orc.coeffs(p)
    Px, Pz = p.P
    X, Zc = np.meshgrid(np.arange(Px, dtype=float), np.arange(Pz, dtype=float), indexing="ij")
    f = 0.5 * X ** 2 + 0.25 * Zc ** 3 + X * Zc                     # f_xx = 1, f_zz = 1.5 z  (undivided, h = 1)
    Hx = orc.tti_H(p, co, 0, f.ravel()).reshape(Px, Pz)            # theta = 0: H_perp = Dx Dx
    Hz = orc.tti_H(p, co, 1, f.ravel()).reshape(Px, Pz)            #            H_par  = Dz Dz
    s = slice(9, -9)
    # 2e-7: the FD weights are the fp32-rounded ones (reading C18), so sum_j 2 j c_j = 1 + O(1e-8)
    assert np.allclose(Hx[s, s], 1.0, rtol=2e-7, atol=0)
    assert np.allclose(Hz[s, s], 1.5 * Zc[s, s], rtol=2e-7, atol=0)


def test_isotropic_limit_p_equals_r_and_matches_acoustic():
    # Cell-centred source and receivers: the centred-first-derivative operator -G^T G has the grid
    # Nyquist modes in its null space (C10); bilinear weights (1/4 on 4 corners) neither
    # excite nor record them, so the comparison sees the physical branch only.
    args = (2, (61, 61), 10.0, 2000.0, 12.0, 260, 0.35, 10, [295.0, 295.0], [[295.0, 415.0], [385.0, 355.0]])
    pa = ri.homogeneous(*args)
    pt = ri.homogeneous(*args)
    pt.physics = 1
    pt.eps = np.zeros(pt.n, np.float32)
    pt.delta = np.zeros(pt.n, np.float32)
    pt.theta = np.zeros(pt.n, np.float32)
    ca, ct = orc.coeffs(pa), orc.coeffs(pt)
    assert np.array_equal(ca.K2, ct.K2)                              # reading C22: same K2 for both physics
    fa = orc.forward(pa, ca, snap_steps=[120])
    ft = orc.forward(pt, ct, snap_steps=[120])
    sp, sr = ft["snaps"][0, 0], ft["snaps"][0, 1]
    assert np.array_equal(sp, sr)
    da, dtt = fa["samples"], ft["samples"]
    assert np.linalg.norm(da - dtt) <= 1e-2 * np.linalg.norm(da)
    assert np.linalg.norm(da - dtt) > 0


def test_theta_plus_pi_invariance():
    p = ri.random_tti(n=(24, 22), nb=6, nt=50)
    co = orc.coeffs(p)
    f1 = orc.forward(p, co, Z=p.Z)
    p2 = ri.random_tti(n=(24, 22), nb=6, nt=50)
    p2.theta = (p2.theta.astype(np.float64) + np.pi).astype(np.float32)
    co2 = orc.coeffs(p2)
    f2 = orc.forward(p2, co2, Z=p2.Z)
    # cos, sin flip sign up to the fp32 rounding of theta + pi: loose but far below any real change
    assert np.linalg.norm(f1["samples"] - f2["samples"]) <= 1e-5 * np.linalg.norm(f1["samples"])
    assert np.linalg.norm(f1["PZ"] - f2["PZ"]) <= 1e-5 * np.linalg.norm(f1["PZ"])


def test_delta_is_clamped_to_epsilon():
    p = ri.random_tti(n=(12, 12), nb=4, nt=3)
    p.eps[:] = 0.05
    p.delta[:] = 0.09
    co = orc.coeffs(p)
    assert np.allclose(co.delh, np.sqrt(1.1), rtol=1e-7)
    assert np.allclose(co.epsh, 1.1, rtol=1e-7)


# ---- four compressed arrays for the TTI gradient (reading C29) -------------------------------
def _second_difference(H):
    """D[n] = H[n] - 2 H[n-1] + H[n-2] with zero fields before step 0; H [nt][...]."""
    Hp = np.concatenate([np.zeros((2,) + H.shape[1:]), H])
    return (Hp[2:] - 2.0 * Hp[1:-1]) + Hp[:-2]


def test_two_field_gradient_is_the_derivative_of_the_misfit():
    """What fixes the four-array condition is calculus, not the oracle: for J = 1/2 |F(K2) q - d_obs|^2 and
    K2 -> K2 (1 + eta) on the physical grid, dJ/d eta(x) = sum_n (D p[n] w_p[n] + D r[n] w_r[n])(x) / (K2(x) h^2),
    D the undivided second time difference of the stored forward fields and (w_p, w_r) the adjoint fields of the
    residual.  Central differences of J (the forward pass only) against that sum from the two-field histories: a
    dropped r term, a swapped field, a wrong time shift or scale all fail.  The one-field image of 1/2 (p + r)
    (reading C10) is not this gradient and misses by far more than the tolerance."""
    p = ri.random_tti(n=(34, 30), nb=8, nt=90, r=4, seed=5)
    co = orc.coeffs(p)
    rng = np.random.default_rng(3)
    d0 = orc.forward(p, co)["samples"]
    dobs = 0.7 * d0 + 0.01 * np.abs(d0).max() * rng.standard_normal(d0.shape)

    def J(K2):
        d = orc.forward(p, orc.Coeffs(K2, co.damp, co.epsh, co.delh, co.cosT, co.sinT))["samples"]
        return 0.5 * ((d - dobs) ** 2).sum()

    f = orc.forward(p, co, want_hist=True, fields=2)
    assert np.array_equal(f["samples"], d0)                       # probing does not touch the propagation
    a = orc.adjoint(p, co, f["samples"] - dobs, want_hist=True, fields=2)
    S = (_second_difference(f["hist"]) * a["hist"]).sum(axis=(0, 1))
    P = (p.n[0] + 2 * p.nb, p.n[1] + 2 * p.nb)
    K2 = np.asarray(co.K2, np.float64).reshape(P)
    K2phys = K2[p.nb:-p.nb, p.nb:-p.nb].ravel()
    g = S / (K2phys * float(np.float32(p.h)) ** 2)
    eta = rng.standard_normal(p.N)
    errs = []
    for t in (1e-2, 3e-3):
        def pert(sgn):
            K = K2.copy()
            K[p.nb:-p.nb, p.nb:-p.nb] *= 1.0 + sgn * t * eta.reshape(p.n)
            return K.ravel().astype(np.float32)
        fd = (J(pert(+1)) - J(pert(-1))) / (2 * t)
        errs.append(abs(fd / (g @ eta) - 1.0))
    assert errs[1] <= 2e-3, errs
    assert errs[1] < 0.2 * errs[0], errs                          # O(t^2): it converges to the sum, not near it
    f1 = orc.forward(p, co, want_hist=True)
    a1 = orc.adjoint(p, co, f["samples"] - dobs, want_hist=True)
    S1 = (_second_difference(f1["hist"]) * a1["hist"]).sum(axis=0)
    g1 = 2.0 * S1 / (K2phys * float(np.float32(p.h)) ** 2)
    assert abs((g1 @ eta) / (g @ eta) - 1.0) > 0.2


def test_two_field_probes_are_history_times_Z_and_split_the_one_field_probe():
    p = ri.random_tti(n=(30, 26), nb=8, nt=50, r=6, seed=8)
    co = orc.coeffs(p)
    f2 = orc.forward(p, co, Z=p.Z, want_hist=True, fields=2)
    f1 = orc.forward(p, co, Z=p.Z, want_hist=True)
    Z = p.Z.astype(np.float64)
    for fld in range(2):                                          # plane block fld == Z^T history of field fld
        ref = Z.T @ f2["hist"][:, fld, :]
        assert np.abs(f2["PZ"][fld * p.r:(fld + 1) * p.r] - ref).max() <= 1e-12 * np.abs(ref).max()
    assert np.abs(f2["hist"][:, 0] - f2["hist"][:, 1]).max() > 0  # anisotropic: p != r
    assert np.abs(0.5 * (f2["hist"][:, 0] + f2["hist"][:, 1]) - f1["hist"]).max() <= 1e-15 * np.abs(f1["hist"]).max()
    half = 0.5 * (f2["PZ"][:p.r] + f2["PZ"][p.r:])
    assert np.abs(half - f1["PZ"]).max() <= 1e-12 * np.abs(f1["PZ"]).max()


def test_two_field_identity_probes_give_the_exact_sum_and_the_isotropic_limit():
    """r = nt, Z = sqrt(nt) I: Eq. 3 over the 2r planes == sum_n (p w_p + r w_r) from the stored histories.
    eps = delta = 0: p == r and w_p == w_r, so the four-array image is twice the one-field image."""
    p = ri.random_tti(n=(28, 24), nb=8, nt=40, r=40, seed=9)
    co = orc.coeffs(p)
    Z = ri.identity_probes(p.nt)
    f = orc.forward(p, co, Z=Z, want_hist=True, fields=2)
    a = orc.adjoint(p, co, f["samples"], Z=Z, want_hist=True, fields=2)
    I = orc.image(f["PZ"], a["PZ"], 1.0 / p.nt)
    Iex = (f["hist"] * a["hist"]).sum(axis=(0, 1)) * (float(Z[0, 0]) ** 2 / p.nt)
    assert np.abs(I - Iex).max() <= 1e-12 * np.abs(Iex).max()
    p.eps[:] = 0
    p.delta[:] = 0
    p.theta[:] = 0
    p.Z = ri.gaussian_probes(p.nt, 5, 1)
    p.r = 5
    co = orc.coeffs(p)
    f2 = orc.forward(p, co, Z=p.Z, fields=2)
    a2 = orc.adjoint(p, co, f2["samples"], Z=p.Z, fields=2)
    f1 = orc.forward(p, co, Z=p.Z)
    a1 = orc.adjoint(p, co, f2["samples"], Z=p.Z)
    I2, I1 = orc.image(f2["PZ"], a2["PZ"], 0.2), orc.image(f1["PZ"], a1["PZ"], 0.2)
    assert np.abs(I1).max() > 0 and np.abs(I2 - 2.0 * I1).max() <= 1e-12 * np.abs(I1).max()


# ---- kinematics: which field carries eps-hat, and the sign of the tilt (reading C10) --------------------------------
def _axis_velocities(theta_deg, eps=0.2, delta=0.1):
    """Homogeneous TTI medium; velocity of the qP pulse along three directions from the peak-time difference of two
    receivers 200 m apart on each ray: 'perp' = (cos th, -sin th) (perpendicular to the symmetry axis),
    'axis' = (sin th, cos th) (along it), 'mirror' = (cos th, +sin th) (the perp direction of the medium tilted the
    other way).  Cell-centred source and receivers (they neither excite nor record the Nyquist null space, C10)."""
    import math
    c, h, f0, n, nb = 2000.0, 10.0, 15.0, (121, 121), 20
    th = math.radians(theta_deg)
    src = np.array([[605.0, 605.0]])
    dirs = {"perp": (math.cos(th), -math.sin(th)), "axis": (math.sin(th), math.cos(th)),
            "mirror": (math.cos(th), math.sin(th))}
    recs = []
    for d in dirs.values():
        for rho in (200.0, 400.0):
            q = src[0] + rho * np.array(d)
            recs.append((np.floor(q / h) + 0.5) * h)
    recs = np.array(recs)
    dt = 0.5 * ri.cfl_dt_tti(h, c, eps)
    nt = int(0.45 / dt)
    p = ri.homogeneous(2, n, h, c, f0, nt, 0.3, nb, src, recs)
    p.dt, p.physics = dt, 1
    t = np.arange(nt) * dt
    a = (np.pi * f0 * (t - 1.0 / f0)) ** 2
    p.wav = ((1.0 - 2.0 * a) * np.exp(-a)).astype(np.float32)[:, None].copy()
    p.eps, p.delta, p.theta = (np.full(n, v, np.float32) for v in (eps, delta, th))
    d = orc.forward(p, orc.coeffs(p))["samples"]

    def peak_time(tr):
        e = np.abs(tr)
        i = int(np.argmax(e >= 0.5 * e.max()))                   # first arrival (the qP pulse), then its local peak
        while i + 1 < len(e) and e[i + 1] >= e[i]:
            i += 1
        return (i + 0.5 * (e[i - 1] - e[i + 1]) / (e[i - 1] - 2.0 * e[i] + e[i + 1])) * dt

    out = {}
    for k, name in enumerate(dirs):
        r0, r1 = recs[2 * k], recs[2 * k + 1]
        out[name] = (np.linalg.norm(r1 - src[0]) - np.linalg.norm(r0 - src[0])) / (
            peak_time(d[:, 2 * k + 1]) - peak_time(d[:, 2 * k])) / c
    return out


def test_vti_is_faster_along_x_by_sqrt_1_plus_2eps():
    """theta = 0, eps = 0.2, delta = 0.1: the pulse travels at c sqrt(1 + 2 eps) along x and at c along z (the
    symmetry axis).  Mutant it kills: H_perp / H_par swapped between the two fields (eps-hat moved from p to r),
    which makes z the fast axis."""
    v = _axis_velocities(0.0)
    assert abs(v["perp"] / np.sqrt(1.4) - 1.0) <= 5e-3, v          # along x
    assert abs(v["axis"] - 1.0) <= 5e-3, v                         # along z
    assert abs(v["perp"] / v["axis"] / np.sqrt(1.4) - 1.0) <= 5e-3, v


def test_tilt_sign_fast_direction_is_perpendicular_to_the_axis():
    """theta = +30 deg tilts the symmetry axis n = (sin th, cos th) toward +x (reading C10): the fast direction is
    (cos th, -sin th), perpendicular to n -- not its mirror image (cos th, +sin th), which is 60 deg away from it and
    much slower.  Mutant it kills: sin(theta) taken with the opposite sign in tti_H (theta -> theta + pi cannot see it)."""
    v = _axis_velocities(30.0)
    assert abs(v["perp"] / np.sqrt(1.4) - 1.0) <= 5e-3, v
    assert abs(v["axis"] - 1.0) <= 5e-3, v
    assert v["mirror"] < 1.06 < v["perp"], v
