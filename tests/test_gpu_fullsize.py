"""-m gpu: parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times.
The oracle finishes configs 1-3 in well under a minute on the box's host cores, so every output
(neighbour sets, per-atom q6, CV, V, dV/ds, every per-atom force) is compared, not a sample.
Config 4 (4.096 M atoms) compares every output as well but is the slow one (~3 min)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_2510_06873_b200.inputs import configs  # noqa: E402

from gpu_util import assert_stagewise, stagewise  # noqa: E402


def test_config1_full_size():
    r = stagewise(configs.config1())
    assert_stagewise(r)


def test_config2_full_size():
    r = stagewise(configs.config2())
    assert_stagewise(r)


@pytest.mark.parametrize("precision", [32, 64])
def test_config3_full_size(precision):
    w = configs.config3()
    r = stagewise(w, precision=precision)
    assert_stagewise(r)
    tol = 2e-6 if precision == 32 else 1e-12
    assert np.abs(r["q6"] - r["q6_ref"]).max() <= tol
    # translation invariance on the GPU result itself: total bias force sums to ~0
    assert np.abs(r["F"].sum(0)).max() <= 1e-5 * np.abs(r["F"]).max() * np.sqrt(w.natoms)


def test_config4_full_size():
    w = configs.config4()
    r = stagewise(w)                      # fp32 pair math, exact hill sum (grid parity: test_gpu_parity)
    assert_stagewise(r)
    assert np.abs(r["q6"] - r["q6_ref"]).max() <= 2e-6


def test_config4_grid_leg_full_size():
    """BASELINE.json configs[4]: "100,000 hills, also evaluated through a 512x512 grid-tabulated bias with bicubic
    interpolation" at ITS size (readings K, M): the separable 16 x 16-node tile build over 100,000 hills against the oracle's
    direct node sums (2.6e10 Gaussian terms on the host cores), 20 lookups, one deposit into the table.  The atoms play no
    part in this leg, so the context sits on the small c4 structure; hill centres walk around the full-size structure's own CV
    values (Q6 = 0.2315, solid-like count = 4.7e5)."""
    import oracle as orc
    import torch
    from paper_2510_06873_b200.inputs import hill_walk, seeded_heights
    from paper_2510_06873_b200.metad import MetaD
    from gpu_util import TOL_CV, rel
    w = configs.small("c4")
    w.sigma = [0.005, 500.0]
    w.stride = 1
    n, sig = 100000, np.array([0.005, 500.0])
    s0 = np.array([0.2315, 4.7e5])
    centers, heights = hill_walk(5, s0, sig, n), seeded_heights(5, n, w.w0)
    lo, hi = s0 - 120 * sig, s0 + 120 * sig
    table = np.zeros((4, 512, 512))
    orc.grid_add(table, lo, hi, centers, heights, sig)
    md = MetaD(w, precision=32, grid=((512, 512), lo, hi), max_hills=n + 8)
    md.set_hills(centers, heights)
    tab = md.grid_table()
    scale = np.abs(table).reshape(4, -1).max(1)[:, None, None]
    assert scale.min() > 0
    assert (np.abs(tab - table) / scale).max() <= 1e-10
    rng = np.random.default_rng(1)
    for k in range(20):
        s = s0 + (rng.random(2) - 0.5) * 120 * sig
        out, V_ref, dV_ref = orc.grid_eval(table, lo, hi, s)
        assert out == 0
        with torch.cuda.stream(md.stream):
            ds = torch.tensor(s, device="cuda")
        V, dV = md.bias(cv=ds)
        md.synchronize()
        assert rel(V.cpu().numpy(), V_ref) <= TOL_CV
        assert np.abs(dV.cpu().numpy() - dV_ref).max() <= TOL_CV * np.abs(dV_ref).max()
    assert md.status() == 0
    # one deposition: the new hill (height by the well-tempered rule from the table's V) lands in the table
    s = s0 + np.array([3.3, -7.1]) * sig
    out, V0, _ = orc.grid_eval(table, lo, hi, s)
    h_new = orc.wt_height(w.w0, V0, w.kT, w.bias_factor)
    orc.grid_add(table, lo, hi, s[None, :], np.array([h_new]), sig)
    with torch.cuda.stream(md.stream):
        ds = torch.tensor(s, device="cuda")
    md.bias(cv=ds)
    md.deposit(cv=ds)
    tab2 = md.grid_table()
    assert (np.abs(tab2 - table) / scale).max() <= 1e-10
    c, h = md.get_hills()
    assert len(h) == n + 1 and rel(h[-1], h_new) <= 1e-9


def test_gan_cv_set_full_size_fp32_tiled():
    """PAPER.md:51 CV set (coordination number + a, b, c) at 1,024,000 atoms in the configuration bench.py --config g0
    times: fp32 pair math on the tiled path (coordination sum fused into the list build)."""
    w = configs.config_g0()
    r = stagewise(w, precision=32)
    assert_stagewise(r)
    fb, fb_ref = r["md"].box_force(), r["o"].box_force(r["dV_ref"])
    assert np.abs(fb - fb_ref).max() <= 1e-12 * np.abs(fb_ref).max()


def test_torsion_workload_full_size():
    """PAPER.md:37 workload in the configuration bench.py --config t0 times (20,000 hills, periodic)."""
    r = stagewise(configs.config_t0())
    assert_stagewise(r)


def test_nearest_hydrogen_workload_full_size():
    """PAPER.md:43 workload in the configuration bench.py --config r0 times (99,999 atoms, one surface oxygen)."""
    r = stagewise(configs.config_r0())
    assert_stagewise(r)
    assert 0.5 < r["s_ref"][0] < 5.0


def test_config3_full_size_is_bit_identical_from_run_to_run():
    """Reading P at the size and in the launch configuration bench.py times (fp32 pair math, tiled build with TMA-staged
    interior tiles, CUDA-graph replay with deposition): two fresh contexts give the same bits in every force component,
    every per-atom q6, the CV, V and the deposited hills."""
    import torch
    from paper_2510_06873_b200.inputs import seeded_heights
    from paper_2510_06873_b200.metad import MetaD
    w = configs.config3()
    w.stride = 2
    pos = w.pos.astype(np.float32)
    centers = (0.23 + 0.002 * np.arange(50))[:, None]
    heights = seeded_heights(11, 50, w.w0)
    out = []
    for rep in range(2):
        md = MetaD(w, precision=32, max_hills=128)
        md.set_hills(centers, heights)
        with torch.cuda.stream(md.stream):
            dpos = torch.tensor(pos, device="cuda")
            F = torch.zeros((w.natoms, 3), device="cuda", dtype=torch.float32)
        md.synchronize()
        md.run(dpos, F, 5)
        st = md.state()
        c, h = md.get_hills()
        assert md.status() == 0
        out.append((F.cpu().numpy(), md.q6(), st["cv"].copy(), st["V"], c, h))
        del md
    assert np.abs(out[0][0]).max() > 0
    for a, b in zip(out[0], out[1]):
        assert np.array_equal(np.asarray(a), np.asarray(b))


def test_config3_full_size_with_a_verlet_skin():
    """params.skin at the size bench.py --skin times (1,024,000 atoms, fp32 pair math): every atom takes a seeded Gaussian step
    of width 0.012 A per step and is re-wrapped into the 255 A box, so pairs across a face and freshly re-wrapped atoms occur
    in the kept list; every step is compared with the oracle, which builds its list from scratch (gpu_util.chained_run: CV,
    V, dV/ds, every force component, the deposited hill)."""
    from paper_2510_06873_b200.inputs import wrap
    from gpu_util import chained_run
    w = configs.config3()
    w.stride = 2
    rng = np.random.default_rng(77)
    frames, p = [], w.pos.copy()
    for k in range(3):
        if k:
            p = wrap(p + rng.standard_normal(p.shape) * 0.012, w.box)
        frames.append(p.copy())
    r = chained_run(w, precision=32, nsteps=3, skin=0.3, pos_of_step=lambda k: frames[k], n_init_hills=30)
    assert r["md"].rebuilds() == 1                # one build, then the list is kept
    assert r["md"].status() == 0


@pytest.mark.parametrize("mode", ["host box", "device box, rescaled every step", "device box + skin"])
def test_config3_full_size_run_paths(mode):
    """The run paths at the size bench.py times (1,024,000 atoms, fp32 pair math, CUDA-graph replay with deposition), every step
    against the oracle (gpu_util.chained_run): metad_run with a host box; metad_run_dev with the box in device memory, rescaled
    with the positions every step as a barostat would (one capture, no graph update); and the same with a Verlet
    skin on top."""
    from gpu_util import chained_run
    w = configs.config3()
    w.stride = 2
    if mode == "host box":
        r = chained_run(w, precision=32, nsteps=2, n_init_hills=30)
    else:
        box0 = w.box.copy()
        frac = np.linalg.solve(box0.reshape(3, 3).T, w.pos.T).T
        scales = [1.0, 1.0006, 0.9996]
        r = chained_run(w, precision=32, nsteps=3, n_init_hills=30, device_box=True, box_slack=0.01,
                        skin=0.3 if "skin" in mode else 0.0,
                        box_of_step=lambda k: box0 * scales[k], pos_of_step=lambda k: frac @ (box0 * scales[k]).reshape(3, 3))
        gi = r["md"].graph_info()
        assert gi["captures"] == 1 and gi["updates"] == 0
    assert r["md"].status() == 0


@pytest.mark.parametrize("case", ["c4 grid", "c4 skin", "g0 lazy", "c3 fp64", "c2 skin", "c1"])
def test_other_workloads_full_size_run_paths(case):
    """metad_run at BASELINE size for the other workloads and modes, every step against the oracle (gpu_util.chained_run):
    c4 (4,096,000 atoms, Q6 mean + solid-like count) through the 512 x 512 grid and, separately, with a Verlet skin over
    moving atoms; the paper's GaN CV set list-free (`lazy_neighbors`); c3 on the generic fp64 kernels; the grouped
    coordination number of c2 with a skin; the chain CVs of c1."""
    from paper_2510_06873_b200.inputs import wrap
    from gpu_util import chained_run
    name = case.split()[0]
    w = {"c4": configs.config4, "g0": configs.config_g0, "c3": configs.config3, "c2": configs.config2, "c1": configs.config1}[name]()
    w.stride = 2
    kw = dict(nsteps=2, n_init_hills=30)
    if "skin" in case:
        rng = np.random.default_rng(3)
        frames, p = [], w.pos.copy()
        for k in range(3):
            if k:
                p = wrap(p + rng.standard_normal(p.shape) * 0.012, w.box)
            frames.append(p.copy())
        kw.update(nsteps=2 if name == "c4" else 3, skin=0.3, pos_of_step=lambda k: frames[k])
    if case == "c4 grid":
        s0 = np.array([0.2315, 4.7e5])                       # the structure's own CV values (test_config4_grid_leg_full_size)
        sig = np.asarray(w.sigma, dtype=np.float64)
        kw.update(grid=((512, 512), s0 - 120 * sig, s0 + 120 * sig))
    precision = {"c4": 32, "g0": 32, "c3": 64, "c2": 64, "c1": 64}[name]
    r = chained_run(w, precision=precision, lazy=(case == "g0 lazy"), free_run=(name != "c4"), **kw)
    assert r["md"].status() == 0
    if "skin" in case:
        assert r["md"].rebuilds() == 1
