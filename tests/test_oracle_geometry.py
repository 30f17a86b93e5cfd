"""Pins for the oracle's neighbour predicate / lists, switching function and coordination CV.
(-m "not gpu"; nothing here touches the CUDA path.)"""
import numpy as np
import pytest

import oracle
from paper_2510_06873_b200.inputs import configs, wrap


def _rand_box_positions(seed, box, n):
    rng = np.random.default_rng(seed)
    return wrap(rng.random((n, 3)) @ np.asarray(box).reshape(3, 3), box)


BOXES = {
    "cubic3cells": (np.array([10.0, 0, 0, 0, 10.0, 0, 0, 0, 10.0]), 3.2),
    "ortho": (np.array([9.0, 0, 0, 0, 11.0, 0, 0, 0, 13.0]), 4.4),
    "hex120": (np.array([12.0, 0, 0, -6.0, 6.0 * np.sqrt(3.0), 0, 0, 0, 9.0]), 4.0),
    "hex60": (np.array([12.0, 0, 0, 6.0, 6.0 * np.sqrt(3.0), 0, 0, 0, 9.0]), 4.0),
    "triclinic": (np.array([11.0, 0, 0, 3.0, 10.0, 0, -2.5, 4.0, 12.0]), 3.5),
}


@pytest.mark.parametrize("name", list(BOXES))
def test_predicate_equals_periodic_image_definition(name):
    """Reading O pin: the sequential min-image predicate finds exactly the pairs whose nearest
    periodic image (brute force over 125 images) is closer than rc."""
    box, rc = BOXES[name]
    code, widths = oracle.box_check(box, rc)
    assert code == 0 and rc < 0.5 * widths.min()
    pos = _rand_box_positions(11, box, 220)
    c_img, l_img, _ = oracle.neighbors(pos, box, rc, 200, "images")
    c_brt, l_brt, _ = oracle.neighbors(pos, box, rc, 200, "brute")
    c_cel, l_cel, _ = oracle.neighbors(pos, box, rc, 200, "cells")
    assert c_img.sum() > 0
    assert np.array_equal(c_img, c_brt) and np.array_equal(l_img, l_brt)
    assert np.array_equal(c_img, c_cel) and np.array_equal(l_img, l_cel)


def test_neighbor_list_is_symmetric_and_excludes_self():
    w = configs.config0()
    c, l, mx = oracle.neighbors(w.pos, w.box, w.rc, w.max_neigh, "cells")
    assert mx <= w.max_neigh
    pairs = {(i, int(j)) for i in range(w.natoms) for j in l[i, :c[i]]}
    assert all((j, i) in pairs for (i, j) in pairs)
    assert all(i != j for (i, j) in pairs)
    # ascending order
    for i in range(w.natoms):
        assert np.all(np.diff(l[i, :c[i]]) > 0)


def test_box_check_rejects_bad_boxes():
    assert oracle.box_check([10, 0, 0, 0, 10, 0, 0, 0, 10], 5.0)[0] == 2     # rc == half width
    assert oracle.box_check([10, 1, 0, 0, 10, 0, 0, 0, 10], 3.0)[0] == 1     # not lower-triangular
    assert oracle.box_check([10, 0, 0, 0, -10, 0, 0, 0, 10], 3.0)[0] == 1
    assert oracle.box_check([10, 0, 0, 0, 10, 0, 0, 0, 10], 4.9)[0] == 0


def test_delta_is_difference_plus_lattice_vector():
    box, _ = BOXES["triclinic"]
    B = box.reshape(3, 3)
    pos = _rand_box_positions(5, box, 50)
    for i in range(0, 50, 7):
        for j in range(50):
            d = oracle.delta(box, pos[i], pos[j])
            n = np.linalg.solve(B.T, d - (pos[j] - pos[i]))
            assert np.allclose(n, np.round(n), atol=1e-9)


# ------------------------------------------------------------------ switching function (reading A)
@pytest.mark.parametrize("n,m,val,slope", [(6, 12, 0.5, -1.5), (8, 16, 0.5, -2.0), (6, 10, 0.6, -1.2)])
def test_switch_limit_at_r0(n, m, val, slope):
    v, d = oracle.switch(1.0, n, m)
    assert v == pytest.approx(val, abs=1e-15) and d == pytest.approx(slope, abs=1e-15)
    # continuity across the Taylor window
    for x in (1 - 3e-6, 1 + 3e-6, 1 - 0.9e-6, 1 + 0.9e-6):
        v, d = oracle.switch(x, n, m)
        assert v == pytest.approx(val + slope * (x - 1), abs=1e-9)
        assert d == pytest.approx(slope, abs=2e-4)


def test_switch_reduces_to_textbook_form_when_m_is_2n():
    # (1-x^n)/(1-x^2n) = 1/(1+x^n): an identity, not the oracle's own formula
    for x in np.linspace(0.05, 2.5, 57):
        v, d = oracle.switch(x, 6, 12)
        assert v == pytest.approx(1.0 / (1.0 + x ** 6), rel=1e-11)
        assert d == pytest.approx(-6 * x ** 5 / (1.0 + x ** 6) ** 2, rel=1e-9, abs=1e-14)


def test_switch_derivative_by_finite_difference():
    for (n, m) in [(6, 12), (6, 10), (4, 9)]:
        for x in (0.3, 0.8, 1.3, 2.0):
            h = 1e-6
            fd = (oracle.switch(x + h, n, m)[0] - oracle.switch(x - h, n, m)[0]) / (2 * h)
            assert oracle.switch(x, n, m)[1] == pytest.approx(fd, rel=1e-7)


# ------------------------------------------------------------------ coordination CV
def test_coordination_of_perfect_sc_lattice(golden):
    """Reading D pin: every atom of the perfect 8^3 a=2.5 lattice has 56 neighbours within 6 A
    (shells 6,12,8,6,24) and the mean coordination is 9.380343874693."""
    g = np.arange(8) * 2.5
    pos = np.stack(np.meshgrid(g, g, g, indexing="ij"), -1).reshape(-1, 3).astype(float)
    box = np.array([20.0, 0, 0, 0, 20.0, 0, 0, 0, 20.0])
    c, l, mx = oracle.neighbors(pos, box, 6.0, 96)
    assert np.all(c == 56)
    s, grad = oracle.cv_coord(pos, box, c, l, 3.0, 6, 12, 1.0 / 512)
    assert s == pytest.approx(golden["cn_sc_lattice"], abs=2e-12)
    # shell-by-shell closed form using the m=2n identity
    shells = [(6, 2.5), (12, 2.5 * 2 ** 0.5), (8, 2.5 * 3 ** 0.5), (6, 5.0), (24, 2.5 * 5 ** 0.5)]
    assert s == pytest.approx(sum(k / (1 + (r / 3.0) ** 6) for k, r in shells), rel=1e-13)
    assert np.abs(grad).max() < 1e-13         # symmetric lattice: zero gradient


def test_coordination_gradient_fd_and_translation_invariance():
    w = configs.config0()
    pos, box = w.pos, w.box
    cv = w.cvs[0]
    c, l, _ = oracle.neighbors(pos, box, w.rc, w.max_neigh)
    s, grad = oracle.cv_coord(pos, box, c, l, cv.r0, cv.n, cv.m, cv.scale)
    assert 9.3 < s < 9.6                      # reading D: outside the [0,8] hill range of config 0
    assert np.abs(grad.sum(0)).max() < 1e-12 * np.abs(grad).max() * len(pos)
    rng = np.random.default_rng(0)
    h = 1e-5
    for i in rng.choice(len(pos), 12, replace=False):
        for a in range(3):
            pp, pm = pos.copy(), pos.copy()
            pp[i, a] += h
            pm[i, a] -= h
            cp, lp, _ = oracle.neighbors(pp, box, w.rc, w.max_neigh)
            cm, lm, _ = oracle.neighbors(pm, box, w.rc, w.max_neigh)
            if not (np.array_equal(cp, c) and np.array_equal(cm, c)):
                continue                      # a pair crossed rc: hard-cutoff delta term (reading B)
            fd = (oracle.cv_coord(pp, box, cp, lp, cv.r0, cv.n, cv.m, cv.scale, want_grad=False)[0]
                  - oracle.cv_coord(pm, box, cm, lm, cv.r0, cv.n, cv.m, cv.scale, want_grad=False)[0]) / (2 * h)
            assert grad[i, a] == pytest.approx(fd, rel=2e-6, abs=3e-9)   # fd rounding ~ eps*s/h


def test_coordination_groups_brute_force():
    """Reading C pin: ordered (i in A, j in B) pairs, overlap allowed, j != i — against a direct
    O(N^2) numpy sum with its own minimum-image arithmetic (cubic box)."""
    rng = np.random.default_rng(3)
    L, N, rc, r0 = 12.0, 150, 4.0, 2.0
    pos = rng.random((N, 3)) * L
    box = np.array([L, 0, 0, 0, L, 0, 0, 0, L])
    A = np.sort(rng.choice(N, 40, replace=False)).astype(np.int32)
    B = np.sort(rng.choice(N, 90, replace=False)).astype(np.int32)
    c, l, _ = oracle.neighbors(pos, box, rc, 64)
    fl = oracle.make_flags(N, A, B)
    s, _ = oracle.cv_coord(pos, box, c, l, r0, 6, 12, 1.0, fl)
    d = pos[None, B] - pos[A, None]
    d -= L * np.round(d / L)
    r = np.linalg.norm(d, axis=-1)
    mask = (r < rc) & (A[:, None] != B[None, :])
    ref = np.sum(1.0 / (1.0 + (r[mask] / r0) ** 6))
    assert s == pytest.approx(ref, rel=1e-12)
