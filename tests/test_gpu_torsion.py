"""-m gpu: NEXT-1 (PAPER.md:37 torsion workload) — torsion CVs, nearest-image periodic hill sum and periodic grid of the
CUDA path against the oracle, through the C ABI.  Tolerances as in test_gpu_parity.py."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_2510_06873_b200.inputs import configs, hill_walk_periodic, seeded_heights  # noqa: E402

from gpu_util import TOL_CV, TOL_F, assert_stagewise, chained_run, make_hills, rel, stagewise  # noqa: E402

P = 2.0 * np.pi
LO, HI = np.array([-np.pi, -np.pi]), np.array([np.pi, np.pi])


@pytest.mark.parametrize("precision", [64, 32])
def test_stagewise_parity_t0(precision):
    w = configs.small("t0")
    r = stagewise(w, precision=precision)
    if precision == 32:
        # fp32 inputs: both sides see the same rounded coordinates; the CUDA torsion math is fp64 in both modes
        assert_stagewise(r, tol_f=2e-5)
    else:
        assert_stagewise(r)
    assert r["V_ref"] > 0.1
    assert np.all(np.abs(r["s"]) <= np.pi)


def test_torsion_atoms_across_the_periodic_boundary():
    """The molecule straddles the box faces: minimum-image bonds must give the same angles and forces."""
    w = configs.small("t0")
    w.pos = w.pos + np.array([14.2, -15.3, 15.6])
    w.pos = w.pos - 30.0 * np.floor(w.pos / 30.0)
    r0 = stagewise(configs.small("t0"))
    r = stagewise(w)
    assert_stagewise(r)
    assert rel(r["s"], r0["s"]) <= 1e-9


def test_periodic_hill_sum_wraps():
    """Evaluation points near +-pi with hills on the other side of the seam; s and s + 2 pi k give the same bias."""
    import torch
    import oracle
    from paper_2510_06873_b200.metad import MetaD
    w = configs.small("t0")
    rng = np.random.default_rng(7)
    c = np.stack([rng.uniform(2.6, np.pi, 300) * rng.choice([-1, 1], 300), rng.uniform(-np.pi, np.pi, 300)], axis=1)
    h = seeded_heights(3, 300, w.w0)
    md = MetaD(w, max_hills=400)
    md.set_hills(c, h)
    for s in ([3.1, 0.2], [-3.12, -1.0], [np.pi, np.pi], [-np.pi, 3.0], [3.1 + P, 0.2 - 2 * P]):
        V_ref, dV_ref = oracle.bias_periodic(c, h, w.sigma, w.period, s)
        with torch.cuda.stream(md.stream):
            ds = torch.tensor(np.asarray(s, float), device="cuda")
        V, dV = md.bias(cv=ds)
        md.synchronize()
        assert V_ref > 1e-3
        assert rel(V.cpu().numpy(), V_ref) <= TOL_CV
        assert np.abs(dV.cpu().numpy() - dV_ref).max() <= TOL_CV * np.abs(dV_ref).max()
    assert md.status() == 0


def test_periodic_grid_matches_oracle_periodic_grid():
    import torch
    from oracle.reference import OracleMetaD
    from paper_2510_06873_b200.metad import MetaD
    w = configs.small("t0")
    o = OracleMetaD(w)
    o.build_neighbors(w.pos)
    s_ref = o.eval_cv(want_grad=False)
    centers, heights = make_hills(w, s_ref)
    o.enable_grid(w.grid_n, LO, HI)
    o.set_hills(centers, heights)
    md = MetaD(w, grid=(w.grid_n, LO, HI), max_hills=len(heights) + 8)
    md.set_hills(centers, heights)
    tab = md.grid_table()
    scale = np.abs(o.grid["table"]).reshape(4, -1).max(1)[:, None, None]
    assert (np.abs(tab - o.grid["table"]) / scale).max() <= 1e-10
    rng = np.random.default_rng(0)
    pts = [rng.uniform(-np.pi, np.pi, 2) for _ in range(20)]
    pts += [np.array([np.pi - 1e-9, -np.pi]), np.array([-np.pi, np.pi - 1e-3]), np.array([3.0 + P, -3.1 - P])]
    for s in pts:
        V_ref, dV_ref = o.bias(s)
        with torch.cuda.stream(md.stream):
            ds = torch.tensor(s, device="cuda")
        V, dV = md.bias(cv=ds)
        md.synchronize()
        assert rel(V.cpu().numpy(), V_ref) <= TOL_CV
        assert np.abs(dV.cpu().numpy() - dV_ref).max() <= TOL_CV * np.abs(dV_ref).max() + 1e-12
    assert md.status() == 0           # a periodic dimension has no "outside": no GRID_RANGE bit
    # deposition next to the seam adds the hill to both sides of the table
    w.stride = 1
    o2 = OracleMetaD(w)
    o2.enable_grid(w.grid_n, LO, HI)
    o2.set_hills(centers, heights)
    md2 = MetaD(w, grid=(w.grid_n, LO, HI), max_hills=len(heights) + 8)
    md2.set_hills(centers, heights)
    s = np.array([3.13, -3.1])
    V0, _ = o2.bias(s)
    o2.deposit(s, V0)
    with torch.cuda.stream(md2.stream):
        ds = torch.tensor(s, device="cuda")
    md2.bias(cv=ds)
    md2.deposit(cv=ds)
    tab2 = md2.grid_table()
    assert (np.abs(tab2 - o2.grid["table"]) / scale).max() <= 1e-10


@pytest.mark.parametrize("fused", [False, True])
@pytest.mark.parametrize("use_grid", [False, True])
def test_graph_run_t0_matches_oracle_loop(use_grid, fused):
    """metad_run (CUDA graph, plain metadynamics W = 1.2 kJ/mol, deposition every 2 steps) against the oracle loop, step by
    step (gpu_util.chained_run: stage-wise on the library's own values, and the free-running loop with the derived bound)."""
    w = configs.small("t0")
    w.stride = 2
    nsteps = 9
    r = chained_run(w, nsteps=nsteps, grid=(w.grid_n, LO, HI) if use_grid else None, lazy=fused, n_init_hills=60)
    assert (r["launches_per_step"] == (2 if use_grid else 1)) == fused
    c, h = r["md"].get_hills()
    assert len(h) == 60 + nsteps // 2
    assert np.all(h[60:] == w.w0)                   # plain metadynamics: every deposited hill has height W


def test_create_rejects_bad_torsion_and_period_arguments():
    from paper_2510_06873_b200.metad import MetaD, MetadError
    w = configs.small("t0")
    w.cvs[0].atoms = np.array([4, 6, 6, 14], dtype=np.int32)
    with pytest.raises(MetadError):
        MetaD(w)
    w = configs.small("t0")
    w.cvs[1].atoms = np.array([4, 6, 8, 99], dtype=np.int32)
    with pytest.raises(MetadError):
        MetaD(w)
    w = configs.small("t0")
    with pytest.raises(MetadError):
        MetaD(w, grid=(w.grid_n, LO, HI + 0.1))      # grid span != period


def test_lazy_neighbors_skips_the_unused_list_and_changes_nothing_else():
    import torch
    from paper_2510_06873_b200.metad import MetaD, MetadError
    w = configs.small("t0")
    centers = hill_walk_periodic(5, np.zeros(2), w.sigma, 80, w.period, w.extra["period_lo"])
    heights = seeded_heights(5, 80, w.w0)
    out = []
    for lazy in (False, True):
        md = MetaD(w, max_hills=128, lazy_neighbors=lazy)
        md.set_hills(centers, heights)
        with torch.cuda.stream(md.stream):
            dpos = torch.tensor(w.pos, device="cuda")
            F = torch.zeros((w.natoms, 3), device="cuda", dtype=torch.float64)
        md.synchronize()
        l0 = md.launch_count()
        md.run(dpos, F, 4)
        st = md.state()
        out.append((st["cv"].copy(), st["V"], F.cpu().numpy(), (md.launch_count() - l0) // 4))
        if lazy:
            with pytest.raises(MetadError):
                md.neighbors()
    # lazy_neighbors + torsion-only CVs: metad_run takes the fused one-kernel step (bias.cu); same numbers up to the
    # order of the hill sum
    assert np.array_equal(out[0][0], out[1][0])
    assert abs(out[0][1] - out[1][1]) <= 1e-12 * abs(out[0][1])
    assert np.abs(out[0][2] - out[1][2]).max() <= 1e-12 * np.abs(out[0][2]).max()
    assert out[0][3] >= 4 and out[1][3] == 1                # one launch per step instead of four (22 atoms: one-kernel list
                                                            # build, CVs, hill sum + deposition, forces)
    # a context whose CVs read the list builds it regardless of the flag
    w3 = configs.small("c3")
    md = MetaD(w3, lazy_neighbors=True)
    md.build_neighbors(torch.tensor(w3.pos, device="cuda"))
    cnt, _ = md.neighbors()
    assert cnt.sum() > 0
