"""-m gpu: nearest-neighbour distance CV (reading AA) of the CUDA path against the oracle."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_2510_06873_b200.inputs import CV_MINDIST, CVSpec, configs  # noqa: E402

from gpu_util import assert_stagewise, stagewise  # noqa: E402


def _workload(single):
    """Slab + water of BASELINE.json configs[2] (scaled down), the CV replaced by the paper's surface-O ... nearest-H distance."""
    w = configs.small("c2")
    cv = w.cvs[0]
    A = np.asarray(cv.group_a)[11:12] if single else cv.group_a
    w.cvs = [CVSpec(kind=CV_MINDIST, group_a=A, group_b=cv.group_b)]
    w.sigma = [0.05]
    w.n_hills = 300
    return w


@pytest.mark.parametrize("single", [True, False])
@pytest.mark.parametrize("precision", [64, 32])
def test_stagewise_parity_mindist(single, precision):
    w = _workload(single)
    r = stagewise(w, precision=precision)
    assert_stagewise(r)
    assert 0.5 < r["s_ref"][0] < w.rc
    nz = np.nonzero(np.abs(r["F"]).sum(1))[0]
    assert set(nz.tolist()) == set(r["o"].min_pair)            # only the nearest pair feels the bias


def test_nobody_within_rc_gives_rc_and_no_force():
    import torch
    from paper_2510_06873_b200.metad import MetaD
    w = _workload(True)
    # move the chosen oxygen's hydrogens out of reach: group B = slab atoms only would be empty of H -> use a far subset
    far = np.asarray(w.cvs[0].group_b)
    L = np.diag(w.box.reshape(3, 3))                          # orthorhombic slab box: nearest image by rounding
    dv = w.pos[far] - w.pos[w.cvs[0].group_a[0]]
    d = np.linalg.norm(dv - L * np.round(dv / L), axis=1)
    w.cvs[0].group_b = far[d > 6.0]
    md = MetaD(w)
    dpos = torch.tensor(w.pos, device="cuda")
    F = torch.zeros((w.natoms, 3), device="cuda", dtype=torch.float64)
    torch.cuda.synchronize()
    md.set_hills(np.array([[w.rc]]), np.array([1.0]))
    md.run(dpos, F, 1)
    st = md.state()
    assert st["cv"][0] == w.rc and abs(st["V"] - 1.0) < 1e-12
    assert not F.cpu().numpy().any() and md.status() == 0


@pytest.mark.parametrize("precision", [64, 32])
def test_list_free_variant_matches_the_list_based_one_and_the_oracle(precision):
    """lazy_neighbors + a single centre: no neighbour list is built, group B is scanned directly (k_mindist_brute).  Both
    variants step by step against the oracle loop (gpu_util.chained_run)."""
    from gpu_util import chained_run, positions_for, rel
    from oracle.reference import OracleMetaD
    w = _workload(True)
    w.stride = 2
    o = OracleMetaD(w)
    o.build_neighbors(positions_for(w, precision).astype(np.float64))
    s0 = o.eval_cv(want_grad=False)
    hills = (s0 + np.linspace(0.02, 0.3, 40)[:, None], np.full(40, 1.0))     # one-sided: a non-zero dV/ds at s0
    outs = [chained_run(w, precision=precision, nsteps=5, lazy=lazy, hills=hills) for lazy in (False, True)]
    assert abs(outs[0]["states"][-1]["dVds"][0]) > 0
    assert outs[1]["launches_per_step"] == outs[0]["launches_per_step"] - 6      # the six kernels of the list build are gone
    assert rel(outs[1]["states"][-1]["cv"], outs[0]["states"][-1]["cv"]) <= 1e-7
