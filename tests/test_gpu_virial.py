"""-m gpu: bias virial for NPT (reading AD) of the CUDA path against the oracle's strain derivatives."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_2510_06873_b200.inputs import (CV_COORD, CV_LATTICE, CV_Q6_MEAN, CV_Q6_SOLID, CV_RGYR, CVSpec,  # noqa: E402
                                          configs)

from gpu_util import assert_stagewise, stagewise  # noqa: E402


def _check(w, precision, tol, from_force_bar=False):
    r = stagewise(w, precision=precision, want_virial=True)
    assert_stagewise(r)
    W = r["md"].virial()
    W_ref = r["o"].virial(r["dV_ref"])
    assert np.abs(W_ref).max() > 0
    bound = tol * np.abs(W_ref).max()
    if from_force_bar:
        # DESIGN.md reading AD: N per-atom contributions, each within the force bar 1e-5 max|F| times |d| <= rc
        bound = max(bound, 0.5 * np.sqrt(w.natoms) * 1e-5 * np.abs(r["F_ref"]).max() * w.rc)
    assert np.abs(W - W_ref).max() <= bound, (W, W_ref)
    # rotation-invariant CVs: symmetric virial.  |W - W^T| <= |W - W_ref| + |W_ref^T - W^T| + |W_ref - W_ref^T|
    assert np.abs(W - W.T).max() <= 2 * bound + np.abs(W_ref - W_ref.T).max()
    return r, W


@pytest.mark.parametrize("precision,tol", [(64, 1e-9), (32, 1e-5)])
def test_virial_generic_path_four_cvs(precision, tol):
    """Coordination number + Q6 mean + solid-like count + lattice parameter c in one context (generic kernels)."""
    w = configs.small("c3")
    N = w.natoms
    w.cvs = [CVSpec(kind=CV_COORD, r0=2.4, n=6, m=12, scale=1.0 / N), CVSpec(kind=CV_Q6_MEAN, scale=1.0 / N),
             CVSpec(kind=CV_Q6_SOLID, scale=1.0, q_thresh=0.25, q_width=0.05), CVSpec(kind=CV_LATTICE, n=2)]
    w.sigma = [0.05, 0.005, 20.0, 0.2]
    w.n_hills = 200
    _check(w, precision, tol)


@pytest.mark.parametrize("solid", [False, True])
def test_virial_tiled_q6(solid):
    w = configs.small("c4" if solid else "c3")                 # c4: Q6 mean + solid-like count; c3: Q6 mean only
    r, W = _check(w, 32, 1e-5)
    if not solid:
        assert abs(np.trace(W)) <= 1e-4 * np.abs(W).max()      # Q6 is scale-invariant: traceless virial


def test_virial_tiled_coordination_and_lattice():
    w = configs.small("g0")                                    # PAPER.md:51 CV set: C.N. + a, b, c
    r, W = _check(w, 32, 1e-5)
    assert np.trace(W) != 0.0


@pytest.mark.parametrize("name,precision,tol", [("c1", 64, 1e-9), ("c1", 32, 1e-5), ("t0", 64, 1e-9), ("c2", 64, 1e-9)])
def test_virial_chain_torsion_and_grouped_coordination(name, precision, tol):
    """Rg + native contacts (c1), two torsions (t0, traceless), grouped coordination number on the warp-per-atom sizes (c2)."""
    w = configs.small(name)
    r, W = _check(w, precision, tol)
    if name == "t0":
        assert abs(np.trace(W)) <= 1e-9 * np.abs(W).max()


def test_virial_nearest_distance():
    from paper_2510_06873_b200.inputs import CV_MINDIST
    w = configs.small("c2")
    cv = w.cvs[0]
    w.cvs = [CVSpec(kind=CV_MINDIST, group_a=np.asarray(cv.group_a)[11:12], group_b=cv.group_b)]
    w.sigma = [0.05]
    w.n_hills = 100
    _check(w, 64, 1e-9)


def test_virial_needs_the_flag():
    from paper_2510_06873_b200.metad import MetaD, MetadError
    w = configs.small("c3")
    md = MetaD(w)
    with pytest.raises(MetadError):
        md.virial()


@pytest.mark.parametrize("name", ["c3", "g0", "c4"])
def test_virial_full_size_tiled_fp32(name):
    """The bias virial at the sizes bench.py times (fp32 pair math on the tiled path): Q6 at 1,024,000 atoms (traceless), the
    paper's GaN CV set (coordination number + a, b, c), and Q6 + solid-like count at 4,096,000 atoms."""
    w = {"c3": configs.config3, "g0": configs.config_g0, "c4": configs.config4}[name]()
    r, W = _check(w, 32, 1e-5, from_force_bar=True)
    if name == "c3":
        assert abs(np.trace(W)) <= 1e-5 * np.abs(W).max()     # Q6 is scale-invariant: traceless (no coherent radial residue)
