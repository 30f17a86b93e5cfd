"""Helpers shared by the -m gpu parity tests: run the CUDA path (through the C ABI binding) and the
oracle on the same seeded workload and return both sides' results."""
import numpy as np

from oracle.reference import OracleMetaD
from paper_2510_06873_b200.inputs import hill_walk, hill_walk_periodic, seeded_heights  # noqa: F401

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


def force_bound(F_ref, dV_gpu, dV_ref, grads, tol_f=TOL_F):
    """End-to-end bound on |F_gpu - F_ref| when the two sides used their OWN dV/ds (reading S):
    F = -sum_d dV/ds_d * ds_d/dr, so a difference delta(dV/ds_d) between the two chains moves every force component by at
    most |delta(dV/ds_d)| * max|ds_d/dr|; on top of that the stage tolerance 1e-5 * max|F|."""
    dd = np.abs(np.atleast_1d(dV_gpu) - np.atleast_1d(dV_ref))
    gmax = np.array([np.abs(g).max() for g in grads])
    return tol_f * np.abs(F_ref).max() + float(np.sum(dd * gmax))


def chained_run(w, precision=None, nsteps=7, grid=None, lazy=False, hills=None, host=False, n_init_hills=40,
                pos_of_step=None, box_of_step=None, seed=5, device_box=False, box_slack=0.0, skin=0.0, check_neighbors=False,
                free_run=True):
    """The library's RUN paths (metad_run = CUDA-graph replay, or metad_step_host with host=True) one step at a time, every
    step checked stage-wise against the oracle fed with the CUDA path's OWN upstream values (reading S, no slack factor):

        s_gpu            vs  oracle CV of the same positions                              1e-6 relative
        V_gpu, dVds_gpu  vs  oracle bias of (the hills the library held BEFORE the step) at s_gpu    1e-6
        F_gpu (one step) vs  oracle forces with dVds_gpu                                  1e-5 max|F|
        deposited hill   ==  (s_gpu bit for bit, w0 exp(-V_gpu / ((gamma - 1) kT)) to 1e-12), earlier hills untouched

    and, beside it, a FREE-RUNNING oracle loop (its own hills): CV 1e-6, hill count, and the accumulated forces within the
    derived bound sum_steps force_bound() (free_run=False skips this second oracle: the 4-million-atom cases).  Returns a dict
    (md, per-step states, launches per step)."""
    import oracle as orc
    import torch
    from paper_2510_06873_b200.metad import MetaD, pinned_array
    precision = w.precision if precision is None else precision
    tdt = torch.float32 if precision == 32 else torch.float64
    pos = positions_for(w, precision)
    o, of = OracleMetaD(w), OracleMetaD(w)          # chained (hills reset from the library every step), free-running
    if hills is None:
        o.build_neighbors(pos.astype(np.float64))
        s0 = o.eval_cv(want_grad=False)
        if getattr(w, "period", None):
            c0 = hill_walk_periodic(seed, s0, w.sigma, n_init_hills, w.period, w.extra["period_lo"])
        else:
            c0 = hill_walk(seed, s0, w.sigma, n_init_hills)
        hills = (c0, seeded_heights(seed, n_init_hills, w.w0))
    if grid is not None:
        o.enable_grid(*grid)
        of.enable_grid(*grid)
    of.set_hills(*hills)
    md = MetaD(w, precision=precision, max_hills=len(hills[1]) + nsteps + 8, grid=grid, lazy_neighbors=lazy, box_slack=box_slack, skin=skin)
    md.set_hills(*hills)
    with torch.cuda.stream(md.stream):
        dpos = torch.tensor(pos, device="cuda", dtype=tdt)
        F = torch.zeros((w.natoms, 3), device="cuda", dtype=tdt)
        dbox = torch.zeros(9, device="cuda", dtype=torch.float64)       # device_box: the library never sees a host box
    md.synchronize()
    if host:
        pos_h = pinned_array(pos.shape, pos.dtype)
        F_h = pinned_array((w.natoms, 3), pos.dtype)
    F_acc, Fo_acc, bound_acc = np.zeros((w.natoms, 3)), np.zeros((w.natoms, 3)), 0.0
    states, per_step_launches = [], None
    box0 = np.array(w.box, dtype=np.float64)
    for k in range(nsteps):
        box = box0 if box_of_step is None else np.asarray(box_of_step(k), dtype=np.float64)
        p = pos if pos_of_step is None else np.ascontiguousarray(pos_of_step(k).astype(pos.dtype))
        p64 = p.astype(np.float64)
        o.w.box = box                                # o.w is of.w is w: the oracle reads the box from the workload
        hc, hh = md.get_hills()
        l0 = md.launch_count()
        if host:
            pos_h[...] = p
            F_h[...] = 0
            cv_h, V_h = md.step_host(pos_h, F_h, box=box)
            Fg = np.array(F_h, dtype=np.float64)
        else:
            with torch.cuda.stream(md.stream):
                dpos.copy_(torch.from_numpy(p))
                F.zero_()
                if device_box:
                    dbox.copy_(torch.from_numpy(box))
            md.synchronize()
            if device_box:
                md.run_dev(dpos, dbox, F, 1)
            else:
                md.run(dpos, F, 1, box=box)
            md.synchronize()
            Fg = F.cpu().numpy().astype(np.float64)
        per_step_launches = md.launch_count() - l0
        st = md.state()
        if host:
            assert np.array_equal(cv_h, st["cv"]) and V_h == st["V"]
        ac, ah = md.get_hills()
        # ---- stage-wise, chained on the library's own values
        o.set_hills(hc, hh)
        o.build_neighbors(p64)
        s_ref = o.eval_cv()
        assert rel(st["cv"], s_ref) <= TOL_CV, (k, st["cv"], s_ref)
        if check_neighbors:                          # the exact rc list at every step, also when a kept rc + skin list is reused
            cnt, lst = md.neighbors()
            assert np.array_equal(cnt, o.count), k
            assert np.array_equal(sorted_rows_fast(cnt, lst), sorted_rows_fast(o.count, o.list)), k
        V_ref, dV_ref = o.bias(st["cv"])
        assert abs(st["V"] - V_ref) <= TOL_CV * max(abs(V_ref), TINY), (k, st["V"], V_ref)
        assert np.abs(st["dVds"] - dV_ref).max() <= TOL_CV * max(np.abs(dV_ref).max(), TINY), (k, st["dVds"], dV_ref)
        F_ref = o.forces(st["dVds"])
        # fp32 force array: half an ulp of the largest component, and never finer than the smallest fp32 denormal
        ulp = max(2.0 ** -24 * np.abs(F_ref).max(), 2.0 ** -149) if precision == 32 else 0.0
        assert np.abs(Fg - F_ref).max() <= TOL_F * np.abs(F_ref).max() + ulp, (k, np.abs(Fg - F_ref).max(), np.abs(F_ref).max())
        due = w.stride > 0 and (k + 1) % w.stride == 0
        assert st["step"] == k + 1 and len(ah) == len(hh) + int(due) == st["nhills"]
        assert np.array_equal(ac[:len(hh)], hc) and np.array_equal(ah[:len(hh)], hh)
        if due:
            assert np.array_equal(ac[-1], st["cv"])
            h_ref = orc.wt_height(w.w0, st["V"], w.kT, w.bias_factor)
            assert abs(ah[-1] - h_ref) <= 1e-12 * h_ref, (k, ah[-1], h_ref)
        F_acc += Fg
        if not free_run:
            states.append(dict(st, s_ref=s_ref, V_ref=V_ref, dV_ref=dV_ref))
            continue
        # ---- free-running oracle loop beside it
        Fo = np.zeros((w.natoms, 3))
        s_f, V_f, dV_f = of.run_step(p64, Fo)
        assert rel(st["cv"], s_f) <= TOL_CV
        bound_acc += force_bound(Fo, st["dVds"], dV_f, of.grads) + ulp
        Fo_acc += Fo
        states.append(dict(st, s_ref=s_ref, V_ref=V_ref, dV_ref=dV_ref, V_free=V_f, dV_free=dV_f))
    assert md.status() == 0, md.status()
    if free_run:
        assert len(of.heights) == states[-1]["nhills"]
        assert rel(md.get_hills()[0], of.centers) <= TOL_CV
        assert np.abs(F_acc - Fo_acc).max() <= bound_acc, (np.abs(F_acc - Fo_acc).max(), bound_acc)
    o.w.box = box0
    return dict(md=md, states=states, launches_per_step=per_step_launches, F=F_acc, F_free=Fo_acc, oracle=of, dpos=dpos,
                hills0=hills)
