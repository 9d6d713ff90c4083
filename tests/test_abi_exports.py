"""Not gpu: the C-ABI library loads and exports every symbol include/rtm.h declares; the host-only
coefficient helper matches the oracle bit for bit (no device needed)."""
import os
import re

import numpy as np
import pytest

import oracle as orc
import rtm_inputs as ri

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _build():
    import __graft_entry__ as g
    g.build()


def test_library_exports_every_declared_symbol():
    _build()
    from paper_2201_06914_b200 import binding as B
    lib = B.load_library()
    hdr = open(os.path.join(ROOT, "include", "rtm.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    hdr = re.sub(r"#ifdef RTM_DEBUG.*?#endif", "", hdr, flags=re.S)      # timing experiments: -DRTM_DEBUG builds only
    assert not hasattr(lib, "rtm_debug_stamps")                          # the product library has no debug switches
    declared = sorted(set(re.findall(r"\b(rtm_[a-z0-9_]+)\s*\(", hdr)))
    assert len(declared) >= 15
    for name in declared:
        assert hasattr(lib, name), name
    assert sorted(B.EXPORTS) == declared


def test_workspace_bytes_model():
    """Probe storage is 2 r N floats (Table 1: O(N r) instead of O(N nt))."""
    _build()
    from paper_2201_06914_b200 import binding as B
    base = dict(ndim=2, n=(1751, 751), h=20.0, nb=80, physics=0, nt=6000, dt=1e-3, max_pts=1751)
    w32 = B.workspace_bytes(B.make_config(r=32, **base))
    w64 = B.workspace_bytes(B.make_config(r=64, **base))
    N = 1751 * 751
    # doubling r adds 2 * 32 probe planes (pitch-padded: 768/751) + the wider Z
    extra = w64 - w32
    assert 2 * 32 * N * 4 <= extra <= 2 * 32 * N * 4 * 1.03 + 2 * 6000 * 32 * 4 + 4096
    full_history = N * 6000 * 4
    assert full_history / (2 * 32 * N * 4) == 6000 / 64          # nt / (2 r): two arrays kept (reading C14)
    assert w32 < 0.5e9


def test_c4_workspace_fits_hbm_where_full_history_does_not():
    """north_star: a 3D case whose full wavefield history would not fit in HBM runs entirely in device memory.
    configs[4]: 512x512x256, nt = 3000, r = 16; with the T = 16 history ring the workspace is still O(N r)."""
    _build()
    from paper_2201_06914_b200 import binding as B
    base = dict(ndim=3, n=(512, 512, 256), h=12.5, nb=40, physics=0, nt=3000, dt=8.5e-4, r=16, max_pts=65536)
    N = 512 * 512 * 256
    full_history = N * 3000 * 4
    hbm = 180e9
    assert full_history > 4 * hbm                                   # 805 GB
    for T, extra in ((0, 0), (16, 2 * 16 * N * 4)):
        w = B.workspace_bytes(B.make_config(probe_block=T, **base))
        assert 2 * 16 * N * 4 + extra <= w <= 2 * 16 * N * 4 + extra + 3.0e9      # + 3 fields, K2, tables
        assert w < 0.15 * hbm and w < full_history / 40
    assert B.workspace_bytes(B.make_config(probe_block=33, **base)) == 0            # invalid config -> 0
    base2 = dict(base, ndim=2, n=(512, 256, 0), physics=1)
    assert B.workspace_bytes(B.make_config(probe_block=17, **base2)) == 0           # TTI: time blocks of <= 16 steps


def test_table1_memory_ratios_golden():
    """tests/golden/table1.txt holds the paper's Table 1; gain = standard / trace estimation."""
    rows = {}
    for line in open(os.path.join(ROOT, "tests", "golden", "table1.txt")):
        if line.startswith("#") or not line.strip():
            continue
        name, std_full, std_sub, te64, te32, g_hi, g_lo = line.split()
        rows[name] = tuple(map(float, (std_full, std_sub, te64, te32, g_hi, g_lo)))
    for name, (sf, ss, t64, t32, ghi, glo) in rows.items():
        assert abs(sf / t64 - ghi) <= 0.01 * ghi + 1        # printed gains are rounded
        assert abs(ss / t32 - glo) <= 0.01 * glo + 1
        assert abs(t64 / t32 - 2.0) < 1e-9                   # storage is linear in r  (O(N r), L47)


def test_host_coefficients_match_oracle_bitwise():
    _build()
    from paper_2201_06914_b200 import binding as B
    for p in (ri.make_c0(), ri.random_tti(), ri.random_acoustic(3, n=(14, 12, 10), nb=4, nt=30),
              ri.random_acoustic(2, n=(20, 17), nb=0, nt=5)):
        cfg = B.make_config(p.ndim, p.n, p.h, p.nb, p.physics, p.nt, p.dt, p.r, 8)
        K2, eh, dh, cs, sn, damp = B.coeffs_host(cfg, p.vp, p.eps, p.delta, p.theta)
        co = orc.coeffs(p)
        assert np.array_equal(K2, co.K2) and np.array_equal(damp, co.damp)
        if p.physics == 1:
            for a, b in ((eh, co.epsh), (dh, co.delh), (cs, co.cosT), (sn, co.sinT)):
                assert np.array_equal(a, b)


def test_host_coefficients_3d_tti_match_oracle_bitwise():
    _build()
    from paper_2201_06914_b200 import binding as B
    p = ri.random_tti3d(n=(11, 9, 10), nb=3, nt=5)
    cfg = B.make_config(p.ndim, p.n, p.h, p.nb, p.physics, p.nt, p.dt, p.r, 8)
    K2, eh, dh, cs, sn, cp, sp, damp = B.coeffs_host3(cfg, p.vp, p.eps, p.delta, p.theta, p.phi)
    co = orc.coeffs(p)
    for a, b in ((K2, co.K2), (damp, co.damp), (eh, co.epsh), (dh, co.delh), (cs, co.cosT), (sn, co.sinT), (cp, co.cosP), (sp, co.sinP)):
        assert np.array_equal(a, b)
    one = B.workspace_bytes(B.make_config(3, p.n, p.h, p.nb, 1, p.nt, p.dt, p.r, 8))
    two = B.workspace_bytes(B.make_config(3, p.n, p.h, p.nb, 1, p.nt, p.dt, p.r, 8, probe_fields=2))
    assert two > one > 0                                                     # four-array mode: TTI in 2D and 3D, twice the planes
    assert B.workspace_bytes(B.make_config(3, p.n, p.h, p.nb, 0, p.nt, p.dt, p.r, 8, probe_fields=2)) == 0    # not for acoustic physics


def test_coeffs_host_rejects_bad_time_step_and_spacing():
    """dt <= 0 or non-finite would give K2 = 0 / NaN tables with RTM_OK: rejected instead."""
    _build()
    from paper_2201_06914_b200 import RTMError
    from paper_2201_06914_b200 import binding as B
    p = ri.random_acoustic(2, n=(12, 10), nb=4, nt=5)
    for dt in (0.0, -1e-3, float("nan"), float("inf")):
        with pytest.raises(RTMError) as e:
            B.coeffs_host(B.make_config(p.ndim, p.n, p.h, p.nb, 0, p.nt, dt, p.r, 8), p.vp)
        assert e.value.code == -1
    for h in (float("inf"), float("nan"), 0.0):
        assert B.workspace_bytes(B.make_config(p.ndim, p.n, h, p.nb, 0, p.nt, p.dt, p.r, 8)) == 0
    for nb in (0, 3, 5, 6, 7):                                  # any layer thickness is a valid config (no nb % 4 rule)
        assert B.workspace_bytes(B.make_config(p.ndim, p.n, p.h, nb, 0, p.nt, p.dt, p.r, 8)) > 0


def test_qr_probes_host_match_oracle():
    """rtm_probes_qr_host (Gram-Schmidt with re-orthogonalisation, host fp64; no GPU needed) against the oracle's
    numpy.linalg.qr: the thin QR with diag(R) > 0 is unique, so Q itself is compared (reading C3), plus the projector
    and the error paths."""
    import oracle as orc
    import rtm_inputs as ri
    from paper_2201_06914_b200 import RTMError, probes_qr_host
    rng = np.random.default_rng(3)
    for nt, nrec, r in ((96, 40, 8), (61, 7, 5), (33, 50, 33)):
        D = rng.standard_normal((nt, nrec)).astype(np.float32) * np.linspace(1.0, 0.05, nrec, dtype=np.float32)
        Z = ri.rademacher_probes(nt, r, seed=nt)
        Q = probes_qr_host(D, Z)
        ref = orc.probes_qr(D, Z)
        assert np.abs(Q.astype(np.float64) - ref).max() <= 2e-6, (nt, nrec, r, np.abs(Q - ref).max())
        Q64 = Q.astype(np.float64)
        assert np.abs(Q64.T @ Q64 - np.eye(r)).max() <= 1e-6
    with pytest.raises(RTMError) as e:                       # r > rank D: D (D^T Z) is rank-deficient
        probes_qr_host(rng.standard_normal((20, 3)).astype(np.float32), ri.rademacher_probes(20, 5, seed=1))
    assert e.value.code == -1
    with pytest.raises(RTMError) as e:                       # r > nt
        probes_qr_host(rng.standard_normal((4, 9)).astype(np.float32), np.ones((4, 6), np.float32))
    assert e.value.code == -1


def test_static_gather_argument_checks_need_no_device():
    """rtm_offset_gather_static validates sizes against the static scratch (rtm.h: RTM_STATIC_SCRATCH_BYTES,
    RTM_STATIC_MAX_OFFSETS) before it touches CUDA, so the checks run here: no launch happens on any of these paths."""
    import ctypes as C
    _build()
    from paper_2201_06914_b200 import binding as B
    lib = B.load_library()
    fake = C.c_void_p(256)            # never dereferenced: every call below returns before any CUDA call
    offs = (C.c_int * 80)(*([0] * 80))
    call = lambda nx, nz, r, nh, U=fake, V=fake, G=fake, o=offs: lib.rtm_offset_gather_static(
        nx, nz, r, U, V, nh, C.cast(o, C.c_void_p), C.c_float(1.0), G, None)
    assert call(16, 12, 2, 65) == -5                                  # more than RTM_STATIC_MAX_OFFSETS
    r, nz = 2, 1024
    nx_max = (B.STATIC_SCRATCH_BYTES - 256) // (2 * r * nz * 4)
    assert call(nx_max + 1, nz, r, 1) == -5                           # one row beyond the static array
    assert call(1 << 30, 1 << 30, 1 << 30, 1) == -5                   # no overflow in the size check
    assert call(0, 12, 2, 1) == -1 and call(16, 12, 0, 1) == -1 and call(16, 12, 2, 0) == -1
    assert call(16, 12, 2, 1, U=None) == -1 and call(16, 12, 2, 1, G=None) == -1
    bad = (C.c_int * 80)(*([16] + [0] * 79))
    assert call(16, 12, 2, 1, o=bad) == -1                            # |h| >= nx
    assert b"static scratch" in lib.rtm_strerror(-5)
