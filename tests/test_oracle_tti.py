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
