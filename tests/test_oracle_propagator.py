"""Pins for the oracle's propagators (not gpu).

  * adjointness   : <F q, d> = <q, F^T d> to 1e-12 (acoustic 2D/3D, TTI), random q, d, off-grid positions
                    (north_star check 3)
  * correctness   : homogeneous medium vs the analytic Green's functions
                      3D  u = s(t - rho/c) / (4 pi rho)
                      2D  u = (1/2pi) int_0^{acosh(t/a)} s(t - a cosh y) dy,  a = rho/c
                    within the stated dispersion error, and 2nd-order convergence in dt (north_star check 4)
  * coefficients  : closed forms of O1 (interior K1 = 1, K2 = c^2 dt^2/h^2; integral of the profile)
"""
import math

import numpy as np
import pytest

import oracle as orc
import rtm_inputs as ri


@pytest.mark.parametrize("make", [
    lambda: ri.random_acoustic(2, n=(30, 26), nb=7, nt=70, seed=1),
    lambda: ri.random_acoustic(3, n=(13, 11, 12), nb=5, nt=40, seed=2),
    lambda: ri.random_tti(n=(28, 30), nb=7, nt=70, seed=3),
])
def test_dot_product(make):
    p = make()
    co = orc.coeffs(p)
    rng = np.random.default_rng(17)
    f = orc.forward(p, co)
    d = rng.standard_normal(f["samples"].shape).astype(np.float32)
    a = orc.adjoint(p, co, d)
    lhs = float((f["samples"] * d.astype(np.float64)).sum())
    rhs = float((p.wav.astype(np.float64) * a["samples"]).sum())
    assert abs(lhs) > 0
    assert abs(lhs - rhs) <= 1e-12 * abs(lhs)


def _ricker(t, f0):
    a = (np.pi * f0 * (t - 1.0 / f0)) ** 2
    return (1.0 - 2.0 * a) * np.exp(-a)


def _green3d(t, rho, c, f0):
    return _ricker(t - rho / c, f0) / (4.0 * np.pi * rho)


def _green2d(t, rho, c, f0, ny=4001):
    a = rho / c
    out = np.zeros_like(t)
    for i, ti in enumerate(t):
        if ti <= a:
            continue
        ymax = math.acosh(ti / a)
        y = np.linspace(0.0, ymax, ny)
        v = _ricker(ti - a * np.cosh(y), f0)
        hh = y[1] - y[0]
        out[i] = hh / 3.0 * (v[0] + v[-1] + 4.0 * v[1:-1:2].sum() + 2.0 * v[2:-1:2].sum()) / (2.0 * np.pi)
    return out


def _homog_error(ndim, cfl_frac):
    c, h, f0 = 2000.0, 10.0, 10.0
    if ndim == 3:
        # the damping layer starts >= 250 m (x) / 350 m (y,z) from the source line: nothing reflected
        # from it can reach a receiver inside its comparison window
        n, src = (91, 71, 71), [250.0, 350.0, 350.0]
        recs = [[450.0, 350.0, 350.0], [650.0, 350.0, 350.0]]
    else:
        # large enough that no boundary reflection reaches a receiver inside the record (2D has tails)
        n, src = (171, 151), [650.0, 750.0]
        recs = [[850.0, 750.0], [1050.0, 750.0]]
    dt = cfl_frac * ri.cfl_dt_acoustic(h, c, ndim)
    nt = int(0.4 / dt)
    p = ri.homogeneous(ndim, n, h, c, f0, nt, cfl_frac, 30 if ndim == 2 else 20, src, recs)
    co = orc.coeffs(p)
    d = orc.forward(p, co)["samples"]                 # d[n] is the field at t = (n+1) dt  (reading C6)
    t = (np.arange(nt) + 1.0) * p.dt
    errs = []
    for j, rho in enumerate((200.0, 400.0)):
        ref = _green3d(t, rho, c, f0) if ndim == 3 else _green2d(t, rho, c, f0)
        # 3D: the pulse has passed by rho/c + 0.2 s; later samples could only hold boundary reflections
        m = t <= (rho / c + 0.2 if ndim == 3 else 1e9)
        errs.append(np.linalg.norm(d[m, j] - ref[m]) / np.linalg.norm(ref[m]))
    return errs


@pytest.mark.parametrize("ndim", [2, 3])
def test_green_function_and_time_order(ndim):
    e1 = _homog_error(ndim, 0.4)
    assert e1[0] <= 5e-3, e1          # stated dispersion error at rho = 200 m
    assert e1[1] <= 1e-2, e1          # ... at rho = 400 m
    e2 = _homog_error(ndim, 0.2)
    for a, b in zip(e1, e2):
        assert 3.3 <= a / b <= 4.7, (e1, e2)   # 2nd order in time


def test_coefficient_closed_forms():
    p = ri.make_c0()
    co = orc.coeffs(p)
    Px, Pz = p.P
    nb, h, dt = p.nb, float(np.float32(p.h)), p.dt
    K2 = co.K2.reshape(Px, Pz)
    # interior: no damping -> K2 = c^2 dt^2 / h^2 rounded once to fp32
    ref = (p.vp.astype(np.float64) ** 2 * dt * dt / (h * h)).astype(np.float32)
    assert np.array_equal(K2[nb:-nb, nb:-nb], ref)
    # tables: zero inside, monotone in the layer, symmetric, end value sigma_max*dt
    dx = co.damp[:Px].astype(np.float64)
    dz = co.damp[Px:].astype(np.float64)
    assert len(dz) == Pz
    assert np.all(dx[nb:Px - nb] == 0) and np.all(dz[nb:Pz - nb] == 0)
    assert np.all(np.diff(dx[:nb + 1]) < 0) and np.all(np.diff(dx[Px - nb - 1:]) > 0)
    assert np.allclose(dx, dx[::-1], rtol=1e-6)
    smax_dt = float(p.vp.max()) * math.log(1000.0) / (nb * h) * dt
    assert abs(dx[0] - smax_dt) <= 1e-6 * smax_dt          # phi(1) = 1
    # integral of sigma over one layer = sigma_max nb h / 2  (int_0^1 phi = 1/2): the round trip at v_max
    # attenuates by exp(-ln 1000) = 1e-3; trapezoid in s = d/nb is exact to O(1/nb^2) here
    integ = (dx[:nb + 1].sum() - 0.5 * dx[0]) / nb
    assert abs(integ - 0.5 * smax_dt) <= 2e-3 * smax_dt
    # layer K2 uses the edge-replicated velocity and 1/(1 + sigma dt)
    c_edge = float(p.vp[0, 0])
    k2 = c_edge ** 2 * dt * dt / (h * h * (1.0 + 2.0 * smax_dt))
    assert abs(K2[0, 0] - k2) <= 2e-7 * k2


def test_positions_outside_grid_are_rejected():
    p = ri.random_acoustic(2, n=(12, 10), nb=4, nt=5)
    co = orc.coeffs(p)
    p.src_xyz = np.array([[-1.0, 5.0], [10.0, 10.0]], np.float32)
    with pytest.raises(ValueError):
        orc.forward(p, co)


def test_on_grid_source_receiver_roundtrip():
    """A receiver placed on the source's node records exactly the injected value at step 0."""
    p = ri.random_acoustic(2, n=(12, 10), nb=4, nt=3, nsrc=1, nrec=1)
    p.src_xyz = np.array([[50.0, 40.0]], np.float32)
    p.rec_xyz = p.src_xyz.copy()
    co = orc.coeffs(p)
    d = orc.forward(p, co)["samples"]
    K2 = co.K2.reshape(p.P)[5 + p.nb, 4 + p.nb]
    assert d[0, 0] == pytest.approx(float(K2) * float(p.wav[0, 0]), rel=1e-14)   # h^(2-d) = 1 in 2D
