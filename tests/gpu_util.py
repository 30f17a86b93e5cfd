"""Helpers shared by the -m gpu parity tests: run the CUDA path (through the C ABI binding) and the
oracle on the same seeded workload and return both sides' results."""
import numpy as np

from oracle.reference import OracleMetaD
from paper_2510_06873_b200.inputs import hill_walk, hill_walk_periodic, seeded_heights

TOL_CV = 1e-6       # BASELINE.json north_star: "CV, V and dV/ds within 1e-6 relative"
TOL_F = 1e-5        # "per-atom bias forces within 1e-5 * max|F| absolute"
TINY = 1e-300       # reading S


def rel(a, b):
    a, b = np.atleast_1d(a).astype(float), np.atleast_1d(b).astype(float)
    return float(np.max(np.abs(a - b) / np.maximum(np.abs(b), TINY)))


def positions_for(w, precision):
    """fp32 mode: the inputs ARE the fp32-rounded coordinates (both sides see the same numbers)."""
    if precision == 32:
        return np.ascontiguousarray(w.pos.astype(np.float32))
    return np.ascontiguousarray(w.pos)


def sorted_rows(cnt, lst):
    out = np.full_like(lst, np.iinfo(np.int32).max)
    for i in range(len(cnt)):
        out[i, :cnt[i]] = np.sort(lst[i, :cnt[i]])
    return out


def sorted_rows_fast(cnt, lst):
    big = np.iinfo(np.int32).max
    a = np.where(np.arange(lst.shape[1])[None, :] < cnt[:, None], lst, big)
    return np.sort(a, axis=1)


def make_hills(w, s_ref, seed=5):
    if w.hill_centers is not None:
        return np.asarray(w.hill_centers, float), np.asarray(w.hill_heights, float)
    if getattr(w, "period", None):
        c = hill_walk_periodic(seed, s_ref, w.sigma, w.n_hills, w.period, w.extra["period_lo"])
    else:
        c = hill_walk(seed, s_ref, w.sigma, w.n_hills)
    return c, seeded_heights(seed, w.n_hills, w.w0)


def stagewise(w, precision=None, threads=None, want_virial=False):
    """Runs both sides stage by stage (reading S): the oracle's s feeds the GPU bias, the oracle's
    dV/ds feeds the GPU forces.  Returns a dict of reference / measured arrays."""
    import torch
    from paper_2510_06873_b200.metad import MetaD
    precision = w.precision if precision is None else precision
    pos = positions_for(w, precision)
    o = OracleMetaD(w)
    o.build_neighbors(pos.astype(np.float64))
    s_ref = o.eval_cv()
    centers, heights = make_hills(w, s_ref)
    o.set_hills(centers, heights)
    V_ref, dV_ref = o.bias(s_ref, use_grid=False)
    F_ref = o.forces(dV_ref)

    md = MetaD(w, precision=precision, max_hills=len(heights) + 16, want_virial=want_virial)
    tdt = torch.float32 if precision == 32 else torch.float64
    with torch.cuda.stream(md.stream):
        dpos = torch.tensor(pos, device="cuda", dtype=tdt)
        F = torch.zeros((w.natoms, 3), device="cuda", dtype=tdt)
        s_in = torch.tensor(s_ref, device="cuda", dtype=torch.float64)
        dV_in = torch.tensor(dV_ref, device="cuda", dtype=torch.float64)
    md.synchronize()
    md.set_hills(centers, heights)
    md.build_neighbors(dpos)
    cnt, lst = md.neighbors()
    md.eval_cv()
    md.synchronize()
    s_gpu = md.cv.cpu().numpy()
    V, dV = md.bias(cv=s_in)
    md.synchronize()
    V_gpu, dV_gpu = float(V.cpu()[0]), dV.cpu().numpy()
    md.apply_forces(F, dVds=dV_in)
    md.synchronize()
    F_gpu = F.cpu().numpy().astype(np.float64)
    out = dict(o=o, md=md, pos=pos, cnt_ref=o.count, lst_ref=o.list, cnt=cnt, lst=lst, s_ref=s_ref, s=s_gpu,
               V_ref=V_ref, V=V_gpu, dV_ref=dV_ref, dV=dV_gpu, F_ref=F_ref, F=F_gpu, status=md.status(),
               centers=centers, heights=heights, dpos=dpos)
    if any(cv.kind in (1, 2) for cv in w.cvs):
        out["q6_ref"] = o.q6
        out["q6"] = md.q6()
    return out


def assert_stagewise(r, tol_cv=TOL_CV, tol_f=TOL_F):
    assert r["status"] == 0, f"sticky bits {r['status']}"
    assert np.array_equal(r["cnt"], np.minimum(r["cnt_ref"], r["lst_ref"].shape[1]))
    assert np.array_equal(sorted_rows_fast(r["cnt"], r["lst"]), sorted_rows_fast(r["cnt_ref"], r["lst_ref"])), \
        "neighbour sets differ"
    assert rel(r["s"], r["s_ref"]) <= tol_cv, (r["s"], r["s_ref"])
    assert rel(r["V"], r["V_ref"]) <= tol_cv, (r["V"], r["V_ref"])
    assert rel(r["dV"], r["dV_ref"]) <= tol_cv, (r["dV"], r["dV_ref"])
    fmax = np.abs(r["F_ref"]).max()
    assert np.abs(r["F"] - r["F_ref"]).max() <= tol_f * fmax, (np.abs(r["F"] - r["F_ref"]).max(), fmax)
