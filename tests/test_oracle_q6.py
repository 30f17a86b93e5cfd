"""Pins for the oracle's Steinhardt q6 (reading E): closed-form shells, a library spherical-harmonic
routine, the two independent routes against each other, invariances and finite differences."""
import numpy as np
import pytest
import scipy.special

import oracle
from paper_2510_06873_b200.inputs import configs

BOX = np.array([60.0, 0, 0, 0, 60.0, 0, 0, 0, 60.0])
C = np.array([30.0, 30.0, 30.0])


def _q6_of_shell(vectors, rc=None, route="p6"):
    v = np.asarray(vectors, dtype=float)
    pos = np.concatenate([C[None], C[None] + v])
    if rc is None:
        rc = 1.05 * np.linalg.norm(v, axis=1).max()
    c, l, _ = oracle.neighbors(pos, BOX, rc, 64, "brute")
    assert c[0] == len(v)
    q = oracle.q6_atoms(pos, BOX, c, l) if route == "p6" else oracle.q6_atoms_ylm(pos, BOX, c, l)[0]
    return q[0]


def fcc12():
    return [(a, b, 0) for a in (1, -1) for b in (1, -1)] + [(a, 0, b) for a in (1, -1) for b in (1, -1)] + \
           [(0, a, b) for a in (1, -1) for b in (1, -1)]


def bcc8():
    return [(a, b, c) for a in (1, -1) for b in (1, -1) for c in (1, -1)]


def sc6(s=1.0):
    return [(s, 0, 0), (-s, 0, 0), (0, s, 0), (0, -s, 0), (0, 0, s), (0, 0, -s)]


def hcp12():
    a = 1.0
    c = np.sqrt(8.0 / 3.0) * a
    inplane = [(a * np.cos(k * np.pi / 3), a * np.sin(k * np.pi / 3), 0.0) for k in range(6)]
    up = [(a * np.cos(k * 2 * np.pi / 3 + np.pi / 6) / np.sqrt(3), a * np.sin(k * 2 * np.pi / 3 + np.pi / 6) / np.sqrt(3), c / 2)
          for k in range(3)]
    down = [(x, y, -z) for (x, y, z) in up]
    return inplane + up + down


def ico12():
    p = (1 + np.sqrt(5)) / 2
    return [(0, a, b * p) for a in (1, -1) for b in (1, -1)] + [(a, b * p, 0) for a in (1, -1) for b in (1, -1)] + \
           [(a * p, 0, b) for a in (1, -1) for b in (1, -1)]


@pytest.mark.parametrize("route", ["p6", "ylm"])
def test_q6_closed_form_shells(golden, route):
    assert _q6_of_shell(fcc12(), route=route) == pytest.approx(golden["q6_fcc12"], abs=1e-4)
    assert _q6_of_shell(bcc8() + sc6(2.0), rc=2.1, route=route) == pytest.approx(golden["q6_bcc14"], abs=1e-4)
    assert _q6_of_shell(sc6(), route=route) == pytest.approx(golden["q6_sc6"], abs=1e-4)
    assert _q6_of_shell(fcc12(), route=route) == pytest.approx(golden["q6_fcc12_6d"], abs=5e-7)
    assert _q6_of_shell(bcc8() + sc6(2.0), rc=2.1, route=route) == pytest.approx(golden["q6_bcc14_6d"], abs=5e-7)
    assert _q6_of_shell(sc6(), route=route) == pytest.approx(np.sqrt(1 / 8), abs=1e-14)
    assert _q6_of_shell(hcp12(), route=route) == pytest.approx(golden["q6_hcp12"], abs=5e-7)
    assert _q6_of_shell(ico12(), route=route) == pytest.approx(golden["q6_ico12"], abs=5e-7)
    assert _q6_of_shell(bcc8(), route=route) == pytest.approx(golden["q6_bcc8"], abs=5e-7)


def test_q6_one_and_two_neighbours(golden):
    assert _q6_of_shell([(0.3, -1.2, 0.7)]) == pytest.approx(1.0, abs=1e-14)
    assert _q6_of_shell([(1, 0, 0), (0, 1.3, 0)]) == pytest.approx(golden["q6_two_90deg"], abs=5e-7)
    for gam in (0.4, 1.1, 2.0, 3.0):
        x = np.cos(gam)
        p6 = (231 * x ** 6 - 315 * x ** 4 + 105 * x ** 2 - 5) / 16
        q = _q6_of_shell([(1, 0, 0), (1.2 * np.cos(gam), 1.2 * np.sin(gam), 0)])
        assert q == pytest.approx(np.sqrt((1 + p6) / 2), abs=1e-13)
    # no neighbours => 0
    pos = np.array([[1.0, 1, 1], [30.0, 30, 30]])
    c, l, _ = oracle.neighbors(pos, BOX, 3.0, 8, "brute")
    assert np.all(oracle.q6_atoms(pos, BOX, c, l) == 0.0)


def test_y6_table_matches_library_spherical_harmonics():
    rng = np.random.default_rng(1)
    for _ in range(40):
        u = rng.standard_normal(3)
        u /= np.linalg.norm(u)
        theta, phi = np.arccos(u[2]), np.arctan2(u[1], u[0])
        ref = np.array([scipy.special.sph_harm_y(6, m, theta, phi) for m in range(7)])
        assert np.allclose(oracle.y6(u), ref, atol=2e-14)
    # sum rule: sum_m |Y6m|^2 = 13/4pi
    y = oracle.y6(u)
    assert abs(y[0]) ** 2 + 2 * np.sum(np.abs(y[1:]) ** 2) == pytest.approx(13 / (4 * np.pi), rel=1e-13)


def test_q6_routes_agree_and_rotation_invariance():
    w = configs.small("c3")
    c, l, mx = oracle.neighbors(w.pos, w.box, w.rc, w.max_neigh)
    assert mx <= w.max_neigh
    qa = oracle.q6_atoms(w.pos, w.box, c, l)
    qb, _ = oracle.q6_atoms_ylm(w.pos, w.box, c, l)
    assert np.abs(qa - qb).max() < 1e-13
    # random rotation of an isolated cluster
    rng = np.random.default_rng(2)
    v = rng.standard_normal((11, 3))
    Q, _ = np.linalg.qr(rng.standard_normal((3, 3)))
    assert _q6_of_shell(v, rc=20.0) == pytest.approx(_q6_of_shell(v @ Q.T, rc=20.0), abs=1e-13)


def test_q6_ideal_wurtzite(golden):
    from paper_2510_06873_b200.inputs.configs import wurtzite
    pos, sp, box = wurtzite(6, 6, 4)
    from paper_2510_06873_b200.inputs import wrap
    pos = wrap(pos, box)
    c, l, _ = oracle.neighbors(pos, box, 3.6, 32)
    assert np.all(c == 17)
    q = oracle.q6_atoms(pos, box, c, l)
    assert np.allclose(q, golden["q6_wurtzite17"], atol=5e-7)
    # distances of the 17: 3@1.949, 1@1.957, 6@3.182, 6@3.190, 1@3.233
    d = np.sort([np.linalg.norm(oracle.delta(box, pos[0], pos[j])) for j in l[0, :17]])
    assert np.allclose(d[[0, 3, 4, 10, 16]], [1.949, 1.957, 3.182, 3.190, 3.233], atol=2e-3)


def test_q6_gradient_fd_and_sum_zero():
    w = configs.small("c3")
    pos, box = w.pos, w.box
    N = len(pos)
    c, l, _ = oracle.neighbors(pos, box, w.rc, w.max_neigh)
    q = oracle.q6_atoms(pos, box, c, l)
    rng = np.random.default_rng(4)
    wts = rng.random(N)                      # arbitrary per-atom weights: E = sum w_i q6_i
    g = oracle.q6_grad(pos, box, c, l, q, wts)
    assert np.abs(g.sum(0)).max() < 1e-11
    h = 1e-5
    checked = 0
    for i in rng.choice(N, 40, replace=False):
        a = int(rng.integers(3))
        pp, pm = pos.copy(), pos.copy()
        pp[i, a] += h
        pm[i, a] -= h
        cp, lp, _ = oracle.neighbors(pp, box, w.rc, w.max_neigh)
        cm, lm, _ = oracle.neighbors(pm, box, w.rc, w.max_neigh)
        if not (np.array_equal(lp, l) and np.array_equal(lm, l)):
            continue
        fd = (np.dot(wts, oracle.q6_atoms(pp, box, cp, lp)) - np.dot(wts, oracle.q6_atoms(pm, box, cm, lm))) / (2 * h)
        assert g[i, a] == pytest.approx(fd, rel=1e-6, abs=1e-8)
        checked += 1
    assert checked >= 20


def test_solid_like_switching_is_the_logistic_of_reading_F(golden):
    """oracle.reference.logistic (BASELINE.json configs[4]: "switching on per-atom q6, threshold 0.35, width 0.05";
    SURVEY.md §8(c)-F): f(q0) = 1/2, f(q0 +- w) = 1/(1 + e^-+1), limits 0 and 1, monotone, symmetric about the threshold,
    f' = df/dq by central differences and f'(q0) = 1/(4 w) — a shifted threshold, another width convention (w vs 2w), a
    flipped sign or a different sigmoid each fail one of these."""
    from oracle.reference import logistic
    q0, w = 0.35, 0.05
    f, df = logistic(np.array([q0, q0 + w, q0 - w]), q0, w)
    assert f[0] == golden["solid_half"]
    assert f[1] == pytest.approx(1.0 / (1.0 + np.exp(-1.0)), abs=1e-15) and f[1] == pytest.approx(golden["solid_plus_w"], abs=1e-12)
    assert f[2] == pytest.approx(1.0 / (1.0 + np.exp(1.0)), abs=1e-15) and f[2] == pytest.approx(golden["solid_minus_w"], abs=1e-12)
    assert df[0] == pytest.approx(1.0 / (4.0 * w), rel=1e-15)
    lim, dlim = logistic(np.array([q0 - 40 * w, q0 + 40 * w, 0.0, 1.0]), q0, w)
    assert lim[0] < 1e-17 and lim[1] == 1.0 and abs(dlim[0]) < 1e-15 and dlim[1] == 0.0
    assert lim[2] == pytest.approx(1.0 / (1.0 + np.exp(7.0)), rel=1e-14)          # a liquid-like atom, q6 = 0
    assert lim[3] == pytest.approx(1.0 / (1.0 + np.exp(-13.0)), rel=1e-14)       # q6 = 1 (one neighbour)
    q = np.linspace(0.0, 1.0, 2001)
    fq, dq = logistic(q, q0, w)
    assert np.all(np.diff(fq) > 0) and np.all(dq > 0)
    # point symmetry about (q0, 1/2) and the central-difference derivative
    d = np.linspace(0.0, 0.3, 301)
    fa, _ = logistic(q0 + d, q0, w)
    fb, _ = logistic(q0 - d, q0, w)
    assert np.abs(fa + fb - 1.0).max() < 1e-15
    h = 1e-6
    fp, _ = logistic(q + h, q0, w)
    fm, _ = logistic(q - h, q0, w)
    assert np.abs((fp - fm) / (2 * h) - dq).max() < 1e-8
    # other parameters: the width really is the e-folding scale of the odds f/(1-f)
    f2, _ = logistic(np.array([0.5, 0.6]), 0.5, 0.1)
    assert f2[0] == 0.5 and f2[1] / (1 - f2[1]) == pytest.approx(np.e, rel=1e-14)
