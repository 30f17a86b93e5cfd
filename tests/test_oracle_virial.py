"""Pins of the oracle's strain derivatives (bias virial for NPT; reading AD): central differences of the CV
itself under a homogeneous deformation of positions and box, on structures with a gap around the cutoff so that no pair
crosses rc during the differentiation."""
import numpy as np

import oracle
from oracle.reference import OracleMetaD
from paper_2510_06873_b200.inputs import CV_COORD, CV_LATTICE, CV_Q6_MEAN, CV_Q6_SOLID, CVSpec, Workload, configs


def _crystal(seed=0):
    """Jittered ideal wurtzite (shells at 3.233 and 3.738 A around rc = 3.6 A: a 0.13 A gap on either side)."""
    pos, _, box = configs.wurtzite(6, 6, 4)
    rng = np.random.default_rng(seed)
    pos = pos + rng.standard_normal(pos.shape) * 0.015
    from paper_2510_06873_b200.inputs import wrap
    return wrap(pos, box), box


def _deform(pos, box, eps):
    M = np.eye(3) + eps
    return pos @ M.T, (box.reshape(3, 3) @ M.T).ravel()


def _cv_values(w, pos, box):
    w2 = Workload(name="x", pos=pos, box=box, rc=w.rc, max_neigh=w.max_neigh, cvs=w.cvs, sigma=w.sigma, n_hills=1)
    o = OracleMetaD(w2)
    o.build_neighbors(pos)
    return o.eval_cv(want_grad=False)


def test_strain_derivatives_match_central_differences():
    pos, box = _crystal()
    N = len(pos)
    cvs = [CVSpec(kind=CV_COORD, r0=2.4, n=6, m=12, scale=1.0 / N), CVSpec(kind=CV_Q6_MEAN, scale=1.0 / N),
           CVSpec(kind=CV_Q6_SOLID, scale=1.0, q_thresh=0.2, q_width=0.05), CVSpec(kind=CV_LATTICE, n=1)]
    w = Workload(name="v", pos=pos, box=box, rc=3.6, max_neigh=32, cvs=cvs, sigma=[1.0] * 4, n_hills=1)
    o = OracleMetaD(w)
    o.build_neighbors(pos)
    assert o.count.min() == 17 and o.count.max() == 17
    o.eval_cv(want_grad=False)
    ana = o.strain_derivatives()
    h = 1e-6
    # the deformed box must stay lower-triangular: eps_yx = eps_zx = eps_zy = 0; the other six components are free
    for a, b in [(0, 0), (1, 1), (2, 2), (0, 1), (0, 2), (1, 2)]:
        eps = np.zeros((3, 3)); eps[a, b] = h
        sp = _cv_values(w, *_deform(pos, box, eps))
        sm = _cv_values(w, *_deform(pos, box, -eps))
        fd = (sp - sm) / (2 * h)
        for d in range(4):
            scale = max(np.abs(ana[d]).max(), 1e-12)
            assert abs(fd[d] - ana[d][a, b]) < 2e-6 * scale + 1e-9, (d, a, b, fd[d], ana[d][a, b])
    # rotation-invariant CVs: symmetric tensors; Q6 is also scale-invariant: zero trace
    for d in range(3):
        assert np.abs(ana[d] - ana[d].T).max() < 1e-10 * max(np.abs(ana[d]).max(), 1e-12)
    assert abs(np.trace(ana[1])) < 1e-12 and abs(np.trace(ana[2])) < 1e-9
    # coordination number: trace = sum_pairs sw'(x) x (Euler), negative
    assert np.trace(ana[0]) < 0
    # lattice parameter: d|b|/d eps = b b^T/|b|
    bvec = box.reshape(3, 3)[1]
    assert np.allclose(ana[3], np.outer(bvec, bvec) / np.linalg.norm(bvec), rtol=1e-14)


def test_virial_of_a_single_pair_by_hand():
    box = np.diag([20.0, 20.0, 20.0]).ravel()
    pos = np.array([[5.0, 5.0, 5.0], [6.2, 6.1, 4.3]])
    cnt, lst, _ = oracle.neighbors(pos, box, 3.0, 4)
    d = pos[1] - pos[0]; r = np.linalg.norm(d)
    x = r / 2.0
    dsw = -6 * x**5 / (1 + x**6) ** 2                       # sw = 1/(1+x^6), m = 2n
    ref = 2 * dsw / (2.0 * r) * np.outer(d, d)              # two ordered pairs
    got = oracle.cv_coord_strain(pos, box, cnt, lst, 2.0, 6, 12, 1.0)
    assert np.allclose(got, ref, rtol=1e-13)


def _fd_strain(w, pos, box, ana, comps=((0, 0), (1, 1), (2, 2), (0, 1), (0, 2), (1, 2)), h=1e-6, tol=2e-6):
    for a, b in comps:
        eps = np.zeros((3, 3)); eps[a, b] = h
        sp = _cv_values(w, *_deform(pos, box, eps))
        sm = _cv_values(w, *_deform(pos, box, -eps))
        fd = (sp - sm) / (2 * h)
        fd = np.where(np.abs(fd) > np.pi / (4 * h), fd - np.sign(fd) * np.pi / h, fd)      # a torsion crossing +-pi
        for d in range(len(ana)):
            scale = max(np.abs(ana[d]).max(), 1e-12)
            assert abs(fd[d] - ana[d][a, b]) < tol * scale + 1e-9, (d, a, b, fd[d], ana[d][a, b])


def test_strain_derivatives_of_the_chain_torsion_and_nearest_distance_cvs():
    # Rg + native contacts on the chain workload (molecule and contacts well inside the box)
    w = configs.small("c1")
    o = OracleMetaD(w); o.build_neighbors(w.pos); o.eval_cv(want_grad=False)
    ana = o.strain_derivatives()
    _fd_strain(w, w.pos, w.box, ana)
    assert np.abs(ana[0] - ana[0].T).max() < 1e-12 and np.abs(ana[1] - ana[1].T).max() < 1e-12
    assert abs(np.trace(ana[0]) - o.s[0]) < 1e-10 * o.s[0]                 # Rg is homogeneous of degree 1 (Euler)
    # torsions: scale- and rotation-invariant -> symmetric, traceless
    w = configs.small("t0")
    o = OracleMetaD(w); o.build_neighbors(w.pos); o.eval_cv(want_grad=False)
    ana = o.strain_derivatives()
    _fd_strain(w, w.pos, w.box, ana)
    for d in range(2):
        assert np.abs(ana[d] - ana[d].T).max() < 1e-12 and abs(np.trace(ana[d])) < 1e-12
    # nearest-neighbour distance: d d^T / |d|, trace = s
    from paper_2510_06873_b200.inputs import CV_MINDIST
    w = configs.small("c2")
    cv = w.cvs[0]
    w.cvs = [CVSpec(kind=CV_MINDIST, group_a=np.asarray(cv.group_a)[11:12], group_b=cv.group_b)]
    w.sigma = [0.05]
    o = OracleMetaD(w); o.build_neighbors(w.pos); o.eval_cv(want_grad=False)
    ana = o.strain_derivatives()
    _fd_strain(w, w.pos, w.box, ana)
    assert abs(np.trace(ana[0]) - o.s[0]) < 1e-12
