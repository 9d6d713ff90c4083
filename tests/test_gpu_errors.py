"""-m gpu: error behaviour of the C ABI (include/rtm.h) on a device."""
import ctypes as C

import numpy as np
import pytest

import rtm_inputs as ri

pytestmark = pytest.mark.gpu


def _mk(p, **kw):
    from paper_2201_06914_b200 import Rtm
    m = Rtm.from_problem(p, **kw)
    return m


def test_state_and_argument_errors():
    import torch
    from paper_2201_06914_b200 import RTMError
    p = ri.random_acoustic(2, n=(30, 28), nb=4, nt=10, r=2)
    m = _mk(p)
    with pytest.raises(RTMError) as e:          # no model / probes yet
        m.forward_probe(p.src_xyz, p.wav, p.rec_xyz)
    assert e.value.code == -4
    m.set_model_from_earth(p.vp)
    m.set_probes(p.Z)
    with pytest.raises(RTMError) as e:          # adjoint image before forward
        m.adjoint_image(p.rec_xyz, np.zeros((p.nt, len(p.rec_xyz)), np.float32), p.src_xyz)
    assert e.value.code == -4
    bad = p.src_xyz.copy()
    bad[0, 0] = -5.0
    with pytest.raises(RTMError) as e:          # position outside the physical grid
        m.forward_probe(bad, p.wav, p.rec_xyz)
    assert e.value.code == -1
    bad[0, 0] = (p.n[0] - 1) * p.h + 0.5
    with pytest.raises(RTMError) as e:
        m.forward_probe(bad, p.wav, p.rec_xyz)
    assert e.value.code == -1
    d = m.forward_probe(p.src_xyz, p.wav, p.rec_xyz)
    with pytest.raises(RTMError) as e:          # gather before adjoint
        m.offset_gather(np.array([0], np.int32))
    assert e.value.code == -4
    m.adjoint_image(p.rec_xyz, d, p.src_xyz)
    with pytest.raises(RTMError) as e:          # |h| >= nx
        m.offset_gather(np.array([p.n[0]], np.int32))
    assert e.value.code == -1
    with pytest.raises(RTMError) as e:          # vector offsets are for 3D grids
        m.offset_gather_xy(np.array([[0, 0]], np.int32))
    assert e.value.code == -1
    many = np.tile(p.rec_xyz, (4, 1))           # more points than max_pts
    with pytest.raises(RTMError) as e:
        m.forward_probe(p.src_xyz, p.wav, many)
    assert e.value.code == -1
    torch.cuda.synchronize()
    m.close()


def test_create_errors():
    import torch
    from paper_2201_06914_b200 import binding as B
    lib = B.load_library()
    cfg = B.make_config(2, (20, 20), 10.0, 4, 0, 5, 1e-3, 2, 4)
    need = B.workspace_bytes(cfg)
    assert need > 0
    ws = torch.empty(need, dtype=torch.uint8, device="cuda")
    h = C.c_void_p()
    assert lib.rtm_create(C.byref(cfg), ws.data_ptr(), need - 1, C.byref(h)) == -2          # ENOMEM
    assert lib.rtm_create(C.byref(cfg), ws.data_ptr() + 4, need, C.byref(h)) == -1          # misaligned
    assert lib.rtm_create(C.byref(cfg), None, need, C.byref(h)) == -1
    host = np.zeros(need + 256, np.uint8)
    hp = (host.ctypes.data + 255) // 256 * 256
    assert lib.rtm_create(C.byref(cfg), hp, need, C.byref(h)) == -1                          # host pointer
    for bad in (dict(nb=-1), dict(nb=1025), dict(ndim=4), dict(r=0), dict(nt=0)):
        c2 = B.make_config(bad.get("ndim", 2), (20, 20, 20), 10.0, bad.get("nb", 4), bad.get("physics", 0),
                           bad.get("nt", 5), 1e-3, bad.get("r", 2), 4)
        assert B.workspace_bytes(c2) == 0
    assert lib.rtm_create(C.byref(cfg), ws.data_ptr(), need, C.byref(h)) == 0
    lib.rtm_destroy(h)


def test_no_receivers_and_no_image():
    """Degenerate calls: nrec = 0 forward (probing only), adjoint without image output."""
    import torch
    p = ri.random_acoustic(2, n=(30, 28), nb=4, nt=12, r=3)
    m = _mk(p)
    m.set_model_from_earth(p.vp)
    m.set_probes(p.Z)
    out = m.forward_probe(p.src_xyz, p.wav, np.zeros((0, 2), np.float32), data_out=None)
    assert out is None
    uz = m.export_probes(0).cpu().numpy()
    assert np.abs(uz).max() > 0
    din = np.ones((p.nt, len(p.rec_xyz)), np.float32)
    img, q = m.adjoint_image(p.rec_xyz, din, p.src_xyz, image=None)
    assert img is None
    torch.cuda.synchronize()
    m.close()


@pytest.mark.parametrize("T", [0, 8, 16])
def test_no_kernel_writes_outside_the_workspace_or_its_outputs(T):
    """compute-sanitizer is closed on this pool: guard bands around the caller-owned workspace and around every
    output buffer must keep their pattern after a whole shot (all step kernels, flush roles, image, both gather
    kernels), on grids with ragged tiles in every direction."""
    import numpy as np
    import torch
    import rtm_inputs as ri
    from paper_2201_06914_b200 import Rtm
    cases = [ri.random_acoustic(2, n=(70, 61), nb=8, nt=40, r=6, seed=31, nsrc=2, nrec=5),
             ri.random_acoustic(3, n=(21, 18, 37), nb=8, nt=36, r=5, seed=32),
             ri.random_tti(n=(75, 67), nb=12, nt=40, r=9, seed=33)]
    G = 1 << 16

    def guarded(shape):
        n = int(np.prod(shape))
        buf = torch.full((n + 2 * G,), float("nan"), dtype=torch.float32, device="cuda")
        return buf, buf[G:G + n].view(*shape)

    for p in cases:
        m = Rtm.from_problem(p, probe_block=T, guard_bytes=1 << 20)
        m.set_model_from_earth(p.vp, p.eps, p.delta, p.theta)
        m.set_probes(p.Z)
        bd, data = guarded((p.nt, len(p.rec_xyz)))
        bi, img = guarded(p.n)
        offs = np.arange(-4, 5, dtype=np.int32)
        bg, gat = guarded((len(offs),) + tuple(p.n))
        bg2, gat2 = guarded((3,) + tuple(p.n))
        m.forward_probe(p.src_xyz, p.wav, p.rec_xyz, data_out=data)
        m.adjoint_image(p.rec_xyz, data, p.src_xyz, image=img)
        m.offset_gather(offs, out=gat)                               # tiled kernel
        m.offset_gather(np.array([-2, 0, 3], np.int32), out=gat2)    # generic kernel
        assert m.check_guards()
        for buf, view in ((bd, data), (bi, img), (bg, gat), (bg2, gat2)):
            assert torch.isnan(buf[:G]).all() and torch.isnan(buf[-G:]).all()
            assert torch.isfinite(view).all()
        m.close()


def test_contexts_of_different_sizes_coexist():
    """The large-shared-memory opt-in belongs to a kernel function on a device, not to a context: a second, smaller
    context (2D resident kernel with a small slab, 3D streaming kernel) must not break the launches of a larger one that
    is still alive, whatever the order in which they are created and used."""
    import torch
    from paper_2201_06914_b200 import Rtm
    big = ri.random_acoustic(2, n=(300, 520), nb=20, nt=60, r=4, seed=3, nrec=40)       # resident: slabs of ~21 rows x 560 points
    small = ri.random_acoustic(2, n=(40, 36), nb=8, nt=60, r=4, seed=4)
    vol = ri.random_acoustic(3, n=(24, 20, 28), nb=4, nt=40, r=4, seed=5)
    ms = []
    for p in (big, small, vol):
        m = Rtm.from_problem(p, probe_block=8)
        m.set_model_from_earth(p.vp)
        m.set_probes(p.Z)
        ms.append((m, p))
    outs = {}
    for rnd in range(2):
        for i in (0, 1, 2, 1, 0):
            m, p = ms[i]
            d = m.forward_probe(p.src_xyz, p.wav, p.rec_xyz).cpu().numpy()
            assert np.isfinite(d).all() and np.abs(d).max() > 0
            if i in outs:
                assert np.array_equal(outs[i], d)
            outs[i] = d
    torch.cuda.synchronize()
    for m, _ in ms:
        m.close()


def test_option_values_are_validated():
    """rx = 32 used to be stored unchecked and left half of the rows un-updated; only the kernel's
    instances are accepted now, and unknown options / values return RTM_EINVAL."""
    from paper_2201_06914_b200 import RTMError
    p = ri.random_acoustic(2, n=(30, 28), nb=4, nt=10, r=2)
    m = _mk(p, probe_block=8)
    for name, bad in (("rx", 32), ("rx", 3), ("rx", -1), ("resident", 4), ("resident", -1), ("no_such_option", 1), ("dbg", 1)):
        with pytest.raises(RTMError) as e:
            m.set_option(name, bad)
        assert e.value.code == -1, (name, bad)
    for name, ok in (("rx", 16), ("rx", 0), ("resident", 0), ("resident", 3), ("pdl", 0), ("time_steps", 1)):
        m.set_option(name, ok)
    m.close()
    m3 = _mk(ri.random_acoustic(3, n=(14, 12, 10), nb=4, nt=5, r=2), probe_block=8)
    with pytest.raises(RTMError):
        m3.set_option("rx", 4)                      # the 2D streaming kernel's knob
    with pytest.raises(RTMError):
        m3.set_option("tti_tile", 16)               # the 2D TTI kernel's knob
    m3.close()
    q = ri.random_tti(n=(40, 36), nb=8, nt=10, r=3, seed=2)
    mt = _mk(q, probe_block=16)
    for bad in (0, 8, 24, 64):
        with pytest.raises(RTMError):
            mt.set_option("tti_tile", bad)
    mt.set_option("tti_tile", 16)
    mt.set_option("tti_tile", 32)
    mt.close()
    mt = _mk(q, probe_block=8)                      # the 32-row instance exists for time blocks of 9 .. 16 steps
    with pytest.raises(RTMError):
        mt.set_option("tti_tile", 32)
    mt.close()
