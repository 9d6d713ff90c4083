"""Shared helpers for the -m gpu parity tests: run the CUDA path (through the C ABI binding) and the
oracle on the same seeded inputs."""
import numpy as np


def rel(a, b):
    a = np.asarray(a, np.float64).ravel()
    b = np.asarray(b, np.float64).ravel()
    nb = np.linalg.norm(b)
    return float(np.linalg.norm(a - b) / nb) if nb > 0 else float(np.linalg.norm(a))


K_ELEM = 4.0   # element-wise bound: max|g - o| <= K_ELEM * tol * max|o| (see elem_ok)


def elem(a, b):
    """Worst element: max|a - b| / max|b|."""
    a = np.asarray(a, np.float64).ravel()
    b = np.asarray(b, np.float64).ravel()
    mb = np.abs(b).max()
    return float(np.abs(a - b).max() / mb) if mb > 0 else float(np.abs(a).max())


def elem_ok(g, o, tol, what=""):
    """Element-by-element check beside the relative-L2 one (which is north_star's metric but cannot see a single
    wrong point in a quiet region):
      (i)  max|g - o| <= K_ELEM * tol * max|o|   -- rounding errors of the fp32 path are spread evenly, so the worst
           element, normalised by the largest one, stays below a small multiple of the tolerance (check_all
           prints the ratio worst element / relative L2 of every output: at most 2.4 over the whole suite on B200);
      (ii) wherever the oracle is EXACTLY zero (points no signal has reached yet, outputs outside the offset
           range: the fp64 oracle and the fp32 path have the same dependency cone) the CUDA path must be exactly
           zero too -- a stray write into a quiet corner fails this whatever its size."""
    g = np.asarray(g, np.float64).ravel()
    o = np.asarray(o, np.float64).ravel()
    e = elem(g, o)
    assert e <= K_ELEM * tol, (what, "worst element", e, K_ELEM * tol)
    z = o == 0.0
    assert not np.any(g[z] != 0.0), (what, "non-zero where the oracle is exactly zero", int(np.count_nonzero(g[z])))
    return e


def snap_rel(gs, rs):
    """reading C17: per-snapshot L2 error normalised by the largest snapshot norm."""
    gs = np.asarray(gs, np.float64)
    rs = np.asarray(rs, np.float64)
    den = max(np.linalg.norm(rs[i]) for i in range(len(rs)))
    return max(np.linalg.norm(gs[i] - rs[i]) for i in range(len(rs))) / den


def run_gpu(p, snap_steps=(), din=None, offsets=None, want_qadj=True, probe_block=0, options=None, offsets_xy=None):
    import torch
    from paper_2201_06914_b200 import Rtm
    m = Rtm.from_problem(p, probe_block=probe_block)
    for k, v in (options or {}).items():
        m.set_option(k, v)
    coef = m.set_model_from_earth(p.vp, p.eps, p.delta, p.theta, p.phi)
    m.set_probes(p.Z)
    out = {"coef": coef}
    sn = m.set_snapshots(list(snap_steps)) if len(snap_steps) else None
    data = m.forward_probe(p.src_xyz, p.wav, p.rec_xyz)
    out["data"] = data.cpu().numpy()
    if sn is not None:
        out["fsnaps"] = sn.cpu().numpy()
    out["Uz"] = m.export_probes(0).cpu().numpy()
    if din is None:
        din = out["data"]
    out["din"] = np.ascontiguousarray(din, np.float32)
    sn = m.set_snapshots(list(snap_steps)) if len(snap_steps) else None
    img, q = m.adjoint_image(p.rec_xyz, out["din"], p.src_xyz, qadj_out=want_qadj)
    out["image"] = img.cpu().numpy().ravel()
    out["qadj"] = None if q is None else q.cpu().numpy()
    if sn is not None:
        out["asnaps"] = sn.cpu().numpy()
    out["Vz"] = m.export_probes(1).cpu().numpy()
    if offsets is not None:
        out["gather"] = m.offset_gather(offsets).cpu().numpy().reshape(len(offsets), -1)
    if offsets_xy is not None:
        out["gather_xy"] = m.offset_gather_xy(offsets_xy).cpu().numpy().reshape(len(offsets_xy), -1)
    out["launches"] = m.launch_count()
    torch.cuda.synchronize()
    m.close()
    return out


def run_oracle(p, din, snap_steps=(), offsets=None):
    import oracle as orc
    co = orc.coeffs(p)
    f = orc.forward(p, co, Z=p.Z, snap_steps=snap_steps)
    a = orc.adjoint(p, co, din, Z=p.Z, snap_steps=snap_steps)
    out = {"co": co, "data": f["samples"], "Uz": f["PZ"], "fsnaps": f["snaps"], "qadj": a["samples"],
           "Vz": a["PZ"], "asnaps": a["snaps"]}
    out["image"] = orc.image(f["PZ"], a["PZ"], 1.0 / p.r)
    if offsets is not None:
        out["gather"] = orc.offset_gather(p.n, f["PZ"], a["PZ"], offsets, 1.0 / p.r)
    return out


TOL_FIELD = 1e-5   # north_star: wavefields and receiver data
TOL_IMAGE = 1e-4   # north_star: images, offset gathers (and the compressed wavefields they are made of)


def check_all(p, snap_steps=(), offsets=None, din=None, tol_field=TOL_FIELD, tol_image=TOL_IMAGE, probe_block=0,
              options=None):
    g = run_gpu(p, snap_steps=snap_steps, din=din, offsets=offsets, probe_block=probe_block, options=options)
    o = run_oracle(p, g["din"], snap_steps=snap_steps, offsets=offsets)
    errs = {}
    errs["data"] = rel(g["data"], o["data"])
    errs["qadj"] = rel(g["qadj"], o["qadj"])
    errs["Uz"] = rel(g["Uz"], o["Uz"])
    errs["Vz"] = rel(g["Vz"], o["Vz"])
    errs["image"] = rel(g["image"], o["image"])
    if len(snap_steps):
        errs["fsnaps"] = snap_rel(g["fsnaps"], o["fsnaps"])
        errs["asnaps"] = snap_rel(g["asnaps"], o["asnaps"])
    if offsets is not None:
        errs["gather"] = rel(g["gather"], o["gather"])
    print(p.name, p.n, "nt", p.nt, "r", p.r, {k: "%.2e" % v for k, v in errs.items()},
          "worst element / rel L2:", {k: "%.1f" % (elem(g[k], o[k]) / max(errs[k], 1e-30)) for k in errs})
    assert np.abs(o["data"]).max() > 0 and np.abs(o["image"]).max() > 0
    for k in ("data", "qadj", "fsnaps", "asnaps"):
        if k in errs:
            assert errs[k] <= tol_field, (k, errs)
            elem_ok(g[k], o[k], tol_field, k)
    for k in ("Uz", "Vz", "image", "gather"):
        if k in errs:
            assert errs[k] <= tol_image, (k, errs)
            elem_ok(g[k], o[k], tol_image, k)
    return g, o, errs
