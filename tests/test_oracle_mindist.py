"""Pins of orc_cv_mindist ("distance between a surface oxygen atom and its nearest hydrogen atom"; reading AA)."""
import numpy as np

import oracle
from paper_2510_06873_b200.inputs import configs


def _setup():
    w = configs.small("c2")
    cv = w.cvs[0]
    cnt, lst, _ = oracle.neighbors(w.pos, w.box, w.rc, w.max_neigh)
    fl = oracle.make_flags(w.natoms, cv.group_a, cv.group_b)
    return w, cv, cnt, lst, fl


def test_equals_numpy_minimum_over_brute_force_minimum_image_distances():
    w, cv, cnt, lst, fl = _setup()
    s, g, (i, j) = oracle.cv_mindist(w.pos, w.box, cnt, lst, w.rc, fl)
    A, B = np.asarray(cv.group_a), np.asarray(cv.group_b)
    Bm = w.box.reshape(3, 3)
    f = np.linalg.solve(Bm.T, (w.pos[B][None, :, :] - w.pos[A][:, None, :]).reshape(-1, 3).T).T
    f -= np.round(f)                                  # orthorhombic slab box: nearest image by rounding
    d = np.linalg.norm(f @ Bm, axis=1).reshape(len(A), len(B))
    d[A[:, None] == B[None, :]] = np.inf
    assert abs(s - d.min()) < 1e-12
    a, b = np.unravel_index(np.argmin(d), d.shape)
    assert (i, j) == (A[a], B[b])
    assert 0.5 < s < w.rc
    # gradient: only the two atoms of the nearest pair, unit vectors, opposite
    nz = np.nonzero(np.abs(g).sum(1))[0]
    assert set(nz.tolist()) == {i, j}
    assert abs(np.linalg.norm(g[j]) - 1.0) < 1e-12 and np.abs(g[i] + g[j]).max() < 1e-15
    assert np.abs(g[j] - oracle.delta(w.box, w.pos[i], w.pos[j]) / s).max() < 1e-12


def test_gradient_by_central_differences_and_single_centre():
    w, cv, cnt, lst, fl = _setup()
    one = np.asarray(cv.group_a)[7:8]                 # "a surface oxygen atom": group A with one member
    fl1 = oracle.make_flags(w.natoms, one, cv.group_b)
    s, g, (i, j) = oracle.cv_mindist(w.pos, w.box, cnt, lst, w.rc, fl1)
    assert i == one[0]
    h = 1e-6
    for a in (i, j):
        for k in range(3):
            p = w.pos.copy(); p[a, k] += h
            s1 = oracle.cv_mindist(p, w.box, cnt, lst, w.rc, fl1, False)[0]
            p[a, k] -= 2 * h
            s0 = oracle.cv_mindist(p, w.box, cnt, lst, w.rc, fl1, False)[0]
            assert abs((s1 - s0) / (2 * h) - g[a, k]) < 1e-8


def test_constructed_and_degenerate_cases():
    box = np.diag([20.0, 20.0, 20.0]).ravel()
    pos = np.array([[1.0, 1.0, 1.0], [19.5, 1.0, 1.0], [4.0, 1.0, 1.0], [1.0, 3.5, 1.0]])
    cnt, lst, _ = oracle.neighbors(pos, box, 6.0, 8)
    fl = oracle.make_flags(4, [0], [1, 2, 3])
    s, g, pair = oracle.cv_mindist(pos, box, cnt, lst, 6.0, fl)
    assert abs(s - 1.5) < 1e-14 and pair == (0, 1)            # nearest across the periodic boundary
    assert np.allclose(g[1], [-1.0, 0.0, 0.0]) and np.allclose(g[0], [1.0, 0.0, 0.0])
    # tie: atoms 2 and 3 both 2.5 away once atom 1 is out of group B -> smallest index wins
    pos[2] = [3.5, 1.0, 1.0]
    cnt, lst, _ = oracle.neighbors(pos, box, 6.0, 8)
    s, g, pair = oracle.cv_mindist(pos, box, cnt, lst, 6.0, oracle.make_flags(4, [0], [2, 3]))
    assert abs(s - 2.5) < 1e-14 and pair == (0, 2)
    # nobody within rc: s = rc, zero gradient
    cnt, lst, _ = oracle.neighbors(pos, box, 1.0, 8)
    s, g, pair = oracle.cv_mindist(pos, box, cnt, lst, 1.0, oracle.make_flags(4, [0], [2, 3]))
    assert s == 1.0 and pair == (-1, -1) and not g.any()
