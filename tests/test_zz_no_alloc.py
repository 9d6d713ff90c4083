"""-m gpu: rtm_offset_gather_static, the one entry point that allocates nothing (include/rtm.h), against the existing
rtm_offset_gather on the same compressed wavefields, on calls in a row that share the static scratch array.

Collected last on purpose (the suite runs with `pytest -x`): a failure here hides no other test."""
import numpy as np
import pytest

import rtm_inputs as ri
from gpu_util import K_ELEM, TOL_IMAGE, elem

pytestmark = pytest.mark.gpu


def _existing(p, offsets):
    """Uz, Vz [r][nx][nz] (device) and the gather of the existing context path for `offsets`."""
    import torch
    from paper_2201_06914_b200 import Rtm
    m = Rtm.from_problem(p)
    m.set_model_from_earth(p.vp, p.eps, p.delta, p.theta, p.phi)
    m.set_probes(p.Z)
    data = m.forward_probe(p.src_xyz, p.wav, p.rec_xyz)
    m.adjoint_image(p.rec_xyz, data, p.src_xyz, qadj_out=False)
    U = m.export_probes(0).reshape(p.r, *p.n).clone()
    V = m.export_probes(1).reshape(p.r, *p.n).clone()
    G = [m.offset_gather(np.asarray(o, np.int32)).reshape(len(o), *p.n).clone() for o in offsets]
    torch.cuda.synchronize()
    m.close()
    return U, V, G


def _same(got, ref, exact, what):
    g, o = got.cpu().numpy(), ref.cpu().numpy()
    assert np.isfinite(g).all(), (what, "an element was not written")
    assert np.abs(o).max() > 0, what
    e = elem(g, o)
    assert e <= K_ELEM * TOL_IMAGE, (what, e)
    if exact:     # same gather_kernel, same products in the same order: the same bits
        assert np.array_equal(g, o), (what, e)


def test_static_gather_matches_the_context_path_on_calls_in_a_row():
    import torch
    from paper_2201_06914_b200 import offset_gather_static
    # nz = 61 and 50 are not multiples of 4: the re-pitched rows in the scratch have pad columns
    pa = ri.random_acoustic(2, n=(70, 61), nb=8, nt=70, r=6, seed=41, nsrc=2, nrec=6)
    pb = ri.random_acoustic(2, n=(45, 50), nb=4, nt=60, r=3, seed=42, nsrc=1, nrec=5)
    scattered = [-7, 0, 3, 12]                   # -> gather_kernel in the context path too
    run9 = list(range(-4, 5))                    # a run of consecutive offsets -> the register-tiled kernel there
    Ua, Va, (Ga_s, Ga_r) = _existing(pa, [scattered, run9])
    Ub, Vb, (Gb_s,) = _existing(pb, [[2, -1, 0]])
    nan = float("nan")
    new = lambda ref: torch.full_like(ref, nan)
    # several calls in a row on one stream; the smaller problem in the middle leaves the tail of the first call's
    # planes in the scratch, and the last call runs on what the middle one left behind
    o1 = offset_gather_static(Ua, Va, scattered, 1.0 / pa.r, new(Ga_s))
    o2 = offset_gather_static(Ub, Vb, [2, -1, 0], 1.0 / pb.r, new(Gb_s))
    o3 = offset_gather_static(Ua, Va, run9, 1.0 / pa.r, new(Ga_r))
    o4 = offset_gather_static(Ua, Va, scattered, 1.0 / pa.r, new(Ga_s))
    torch.cuda.synchronize()
    _same(o1, Ga_s, True, "first call")
    _same(o2, Gb_s, True, "second call (smaller grid)")
    _same(o3, Ga_r, False, "third call (against the tiled kernel)")
    _same(o4, Ga_s, True, "fourth call")
    # h = 0 is Eq. 3's image
    img = (Ua.double() * Va.double()).sum(0) / pa.r
    assert elem(o1[1].cpu().numpy(), img.cpu().numpy()) <= K_ELEM * TOL_IMAGE


def test_static_gather_rejects_sizes_beyond_the_static_array():
    import torch
    from paper_2201_06914_b200 import RTMError, offset_gather_static
    from paper_2201_06914_b200.binding import STATIC_MAX_OFFSETS, STATIC_SCRATCH_BYTES
    dev = torch.device("cuda:0")
    U = torch.zeros((2, 16, 12), device=dev)
    out = torch.zeros((STATIC_MAX_OFFSETS + 1, 16, 12), device=dev)
    with pytest.raises(RTMError) as ei:
        offset_gather_static(U, U, [0] * (STATIC_MAX_OFFSETS + 1), 1.0, out)
    assert ei.value.code == -5 and "static scratch" in str(ei.value)
    # largest nx that fits for r = 2, nz = 1024, and the first one that does not
    r, nz = 2, 1024
    nx_max = (STATIC_SCRATCH_BYTES - 256) // (2 * r * nz * 4)
    big = torch.zeros((r, nx_max + 1, nz), device=dev)
    out = torch.zeros((1, nx_max + 1, nz), device=dev)
    with pytest.raises(RTMError) as ei:
        offset_gather_static(big, big, [0], 1.0, out)
    assert ei.value.code == -5
    fit = big[:, :nx_max].contiguous()
    fit[:, -1, -1] = 3.0
    o = offset_gather_static(fit, fit, [0], 0.5, out[:, :nx_max].contiguous())
    torch.cuda.synchronize()
    assert float(o[0, -1, -1]) == 0.5 * r * 9.0 and float(o.sum()) == 0.5 * r * 9.0
    with pytest.raises(RTMError) as ei:       # |h| >= nx
        offset_gather_static(U, U, [16], 1.0, torch.zeros((1, 16, 12), device=dev))
    assert ei.value.code == -1
