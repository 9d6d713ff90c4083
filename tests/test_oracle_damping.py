"""Pins for the oracle's damped update (reading C7/C23; not gpu).

The scheme is (1/c^2)(u_tt + 2 sigma u_t) - Lap u = q with centred differences in time; solving it for the new
time level fixes the update, K1 included -- it is mathematics, not a free choice:

    (u+ - 2u + u-)/dt^2 + sigma (u+ - u-)/dt = c^2 (Lap u + q)
    u+ = (2u - (1 - sigma dt) u- + c^2 dt^2 (Lap u + q)) / (1 + sigma dt)

  * test_damped_update_is_the_centred_scheme: a tiny 2D grid stepped in numpy with exactly that formula (sigma dt
    from the per-axis tables) against the oracle's snapshots on the whole padded grid, layer included, to 1e-12.
    Mutant it kills: K1_at returning 1/(1 + s) instead of (1 - s)/(1 + s) (survived every round-1 test).
  * test_layer_attenuation_is_exp_minus_integral_sigma_over_c: physics of the same term.  A pulse that has travelled a
    distance x into the layer at normal incidence is attenuated by exp(-int_0^x sigma/c) against the same pulse in a
    grid without a layer there; with sigma = sigma_max phi(x / (nb h)), sigma_max = c ln(1000) / (nb h) and
    phi(s) = s - sin(2 pi s)/(2 pi) that is 1000^-(s^2/2 + (cos(2 pi s) - 1)/(4 pi^2)).  Pins the strength and the
    profile of reading C7 as well as K1 (the 1/(1+s) mutant damps half as much: 0.81 / 0.46 instead of 0.65 / 0.20).
"""
import math

import numpy as np

import oracle as orc
import rtm_inputs as ri

# order-8 second-derivative side weights, rounded to fp32 (reading C18); centre = -2 sum (reading C21)
_W = [float(np.float32(x)) for x in (8.0 / 5.0, -1.0 / 5.0, 8.0 / 315.0, -1.0 / 560.0)]


def _lap(u):
    """Undivided order-8 Laplacian of a padded-grid field with zeros outside (reading C8)."""
    Px, Pz = u.shape
    e = np.zeros((Px + 8, Pz + 8))
    e[4:-4, 4:-4] = u
    L = np.zeros_like(u)
    for j, w in enumerate(_W, 1):
        L += w * (e[4 + j:Px + 4 + j, 4:-4] + e[4 - j:Px + 4 - j, 4:-4]
                  + e[4:-4, 4 + j:Pz + 4 + j] + e[4:-4, 4 - j:Pz + 4 - j] - 4.0 * u)
    return L


def test_damped_update_is_the_centred_scheme():
    p = ri.random_acoustic(2, n=(20, 17), nb=6, nt=60, nsrc=1, nrec=1, seed=3)
    p.src_xyz = np.array([[90.0, 70.0]], np.float32)            # node (9, 7): weight 1, h^(2-d) = 1
    co = orc.coeffs(p)
    Px, Pz = p.P
    s = co.damp[:Px].astype(np.float64)[:, None] + co.damp[Px:].astype(np.float64)[None, :]   # sigma dt
    assert s.max() > 0.05 and np.all(s[p.nb:-p.nb, p.nb:-p.nb] == 0)
    c2 = co.K2.astype(np.float64).reshape(Px, Pz) * (1.0 + s)    # c^2 dt^2 / h^2 (O1: K2 = that / (1 + sigma dt))
    steps = [0, 1, 5, 20, 59]
    snaps = orc.forward(p, co, snap_steps=steps)["snaps"]
    u, um, ref = np.zeros((Px, Pz)), np.zeros((Px, Pz)), {}
    for n in range(p.nt):
        q = np.zeros((Px, Pz))
        q[9 + p.nb, 7 + p.nb] = float(p.wav[n, 0])
        un = (2.0 * u - (1.0 - s) * um + c2 * (_lap(u) + q)) / (1.0 + s)
        um, u = u, un
        if n in steps:
            ref[n] = u.copy()
    mx = max(np.abs(v).max() for v in ref.values())
    assert np.abs(ref[59][:p.nb]).max() > 0.05 * mx              # the field is inside the layer by then
    for i, n in enumerate(steps):
        assert np.abs(snaps[i, 0].reshape(Px, Pz) - ref[n]).max() <= 1e-12 * mx, n


def test_layer_attenuation_is_exp_minus_integral_sigma_over_c():
    c, h, f0, nb = 2000.0, 10.0, 25.0, 40

    def line(nx, tsnap):
        dt = 0.4 * ri.cfl_dt_acoustic(h, c, 2)
        nt = int(tsnap / dt) + 1
        p = ri.homogeneous(2, (nx, 121), h, c, f0, nt, 0.4, nb, [600.0, 600.0], [[600.0, 600.0]])
        f = orc.forward(p, orc.coeffs(p), snap_steps=[nt - 1])
        return f["snaps"][0, 0].reshape(p.P)[:, 60 + nb]         # the line z = z_source, padded x index

    j0 = nb + 120                                                # padded index of the physical edge x = 1200 m
    for d, lo, hi in ((200.0, 0.55, 0.75), (300.0, 0.15, 0.25)):
        ts = 1.0 / f0 + (600.0 + d) / c                          # the pulse peak is d metres into the layer
        la, lb = line(121, ts), line(241, ts)                    # with the layer there / physical grid continues
        seg = slice(j0 + int(d / h) - 6, j0 + int(d / h) + 7)
        ia = seg.start + int(np.argmax(np.abs(la[seg])))
        ib = seg.start + int(np.argmax(np.abs(lb[seg])))
        assert abs(ia - ib) <= 1
        sdepth = (ia - j0) / nb
        expo = sdepth ** 2 / 2.0 + (math.cos(2.0 * math.pi * sdepth) - 1.0) / (4.0 * math.pi ** 2)
        want = 1000.0 ** (-expo)
        got = abs(la[ia]) / abs(lb[ib])
        assert lo < want < hi                                    # the test is where it is meant to be
        assert abs(got / want - 1.0) <= 0.03, (d, got, want)
