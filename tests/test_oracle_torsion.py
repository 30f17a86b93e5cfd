"""Pins of the NEXT-1 oracle functions (torsion CV, periodic bias, periodic grid; readings V, W, X) against
things other than themselves: constructed geometries with known dihedrals, invariances, central differences,
numpy restatements of the plain definition, the non-periodic routines on a replicated table."""
import numpy as np
import pytest

import oracle
from oracle.reference import OracleMetaD
from paper_2510_06873_b200.inputs import configs, hill_walk_periodic, seeded_heights

BOX = np.diag([30.0, 30.0, 30.0]).ravel()


def golden():
    import os
    out = {}
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "closed_forms.txt")):
        line = line.split("#")[0].split()
        if len(line) == 2:
            out[line[0]] = float(line[1])
    return out


def four(theta, origin=(5.0, 6.0, 7.0), l1=1.3, l2=1.5, l3=1.1, a1=1.9, a2=2.0):
    """i-j-k-l with the j->k bond along +z, bond angles a1, a2, the far bond rotated by theta about z
    (counterclockwise seen from +z = clockwise looking along j->k)."""
    j = np.zeros(3)
    k = np.array([0, 0, l2])
    i = j + l1 * np.array([np.sin(a1), 0.0, np.cos(a1)])       # in the xz plane, x > 0
    l = k + l3 * np.array([np.sin(a2) * np.cos(theta), np.sin(a2) * np.sin(theta), -np.cos(a2)])
    return np.array([i, j, k, l]) + np.asarray(origin)


@pytest.mark.parametrize("theta", [0.0, np.pi / 3, np.pi / 2, 2.5, -np.pi / 3, -2.0, np.pi])
def test_constructed_dihedral(theta):
    phi, _ = oracle.cv_torsion(four(theta), BOX, [0, 1, 2, 3], False)
    assert abs(np.angle(np.exp(1j * (phi - theta)))) < 1e-12


def test_golden_values():
    g = golden()
    assert abs(oracle.cv_torsion(four(0.0), BOX, [0, 1, 2, 3], False)[0] - g["torsion_cis"]) < 1e-12
    assert abs(abs(oracle.cv_torsion(four(np.pi), BOX, [0, 1, 2, 3], False)[0]) - g["torsion_trans"]) < 1e-11
    assert abs(oracle.cv_torsion(four(np.pi / 3), BOX, [0, 1, 2, 3], False)[0] - g["torsion_gauche"]) < 1e-11
    assert abs(oracle.pdiff(-3.0, 3.0, 2 * np.pi) - g["hill_wrap_delta"]) < 1e-11


def test_numpy_restatement_and_invariances():
    rng = np.random.default_rng(1)
    for _ in range(20):
        p = rng.random((4, 3)) * 4 + 10
        b1, b2, b3 = p[1] - p[0], p[2] - p[1], p[3] - p[2]
        n1, n2 = np.cross(b1, b2), np.cross(b2, b3)
        # textbook: cos phi = n1.n2/(|n1||n2|), sign = sign(b1 . n2)
        ref = np.arccos(np.clip(n1 @ n2 / np.linalg.norm(n1) / np.linalg.norm(n2), -1, 1)) * np.sign(b1 @ n2)
        phi = oracle.cv_torsion(p, BOX, [0, 1, 2, 3], False)[0]
        assert abs(phi - ref) < 1e-9
        # reversal i-j-k-l -> l-k-j-i keeps phi; mirror image flips its sign
        assert abs(oracle.cv_torsion(p, BOX, [3, 2, 1, 0], False)[0] - phi) < 1e-12
        q = p.copy(); q[:, 0] = 30.0 - q[:, 0]
        assert abs(oracle.cv_torsion(q, BOX, [0, 1, 2, 3], False)[0] + phi) < 1e-12
        # rotation + translation, then wrapped into the periodic box: minimum-image bonds give the same angle
        Q, _ = np.linalg.qr(rng.standard_normal((3, 3)))
        if np.linalg.det(Q) < 0:
            Q[:, 0] = -Q[:, 0]
        r = (p - p.mean(0)) @ Q.T + np.array([29.5, 0.3, 15.0])
        r = r - 30.0 * np.floor(r / 30.0)
        assert abs(oracle.cv_torsion(r, BOX, [0, 1, 2, 3], False)[0] - phi) < 1e-11


def test_gradient_by_central_differences_and_sum_rules():
    rng = np.random.default_rng(2)
    for _ in range(10):
        p = rng.random((4, 3)) * 3 + 10
        phi, g = oracle.cv_torsion(p, BOX, [0, 1, 2, 3])
        h = 1e-6
        fd = np.zeros((4, 3))
        for a in range(4):
            for c in range(3):
                q = p.copy(); q[a, c] += h
                f1 = oracle.cv_torsion(q, BOX, [0, 1, 2, 3], False)[0]
                q[a, c] -= 2 * h
                f0 = oracle.cv_torsion(q, BOX, [0, 1, 2, 3], False)[0]
                fd[a, c] = np.angle(np.exp(1j * (f1 - f0))) / (2 * h)
        assert np.abs(fd - g).max() < 1e-7 * max(1.0, np.abs(g).max())
        assert np.abs(g.sum(0)).max() < 1e-12 * max(1.0, np.abs(g).max())            # translation invariance
        assert np.abs(np.cross(p, g).sum(0)).max() < 1e-10 * max(1.0, np.abs(g).max())  # rotation invariance


def test_periodic_bias_single_hill_periodicity_and_limit():
    P = 2 * np.pi
    g = golden()
    sig, w = g["paper_sigma_rad"], g["paper_w_kjmol"]
    V, dV = oracle.bias_periodic([[3.0]], [w], [sig], [P], [-3.0])
    d = 2 * np.pi - 6.0
    assert abs(d - g["hill_wrap_delta"]) < 1e-11
    assert abs(V - w * np.exp(-d * d / (2 * sig * sig))) < 1e-14
    assert abs(dV[0] + V * d / sig**2) < 1e-13
    rng = np.random.default_rng(3)
    c = rng.uniform(-np.pi, np.pi, (50, 2)); h = rng.random(50) + 0.1
    s = np.array([2.9, -3.0])
    V0, dV0 = oracle.bias_periodic(c, h, [sig, 0.2], [P, P], s)
    V1, dV1 = oracle.bias_periodic(c, h, [sig, 0.2], [P, P], s + [P, -3 * P])
    assert abs(V0 - V1) < 1e-12 * V0 and np.abs(dV0 - dV1).max() < 1e-10 * np.abs(dV0).max()
    # numpy restatement of the definition
    d = s - c; d -= P * np.round(d / P)
    e = h * np.exp(-0.5 * ((d[:, 0] / sig) ** 2 + (d[:, 1] / 0.2) ** 2))
    assert abs(V0 - e.sum()) < 1e-13 * e.sum()
    assert np.abs(dV0 - [-(e * d[:, 0]).sum() / sig**2, -(e * d[:, 1]).sum() / 0.04]).max() < 1e-12
    # period 0 = the non-periodic routine; hills all nearer than P/2 = the non-periodic routine
    Va, dVa = oracle.bias_periodic(c, h, [sig, 0.2], [0.0, 0.0], s)
    Vb, dVb = oracle.bias(c, h, [sig, 0.2], s)
    assert abs(Va - Vb) < 1e-14 * abs(Vb) and np.abs(dVa - dVb).max() < 1e-13 * np.abs(dVb).max()
    c2 = c * 0.2
    assert np.allclose(oracle.bias_periodic(c2, h, [sig, 0.2], [P, P], [0.1, -0.2])[0], oracle.bias(c2, h, [sig, 0.2], [0.1, -0.2])[0], rtol=1e-14)
    # mixed: only dimension 0 periodic
    Vm, _ = oracle.bias_periodic(c, h, [sig, 0.2], [P, 0.0], s)
    d = s - c; d[:, 0] -= P * np.round(d[:, 0] / P)
    assert abs(Vm - (h * np.exp(-0.5 * ((d[:, 0] / sig) ** 2 + (d[:, 1] / 0.2) ** 2))).sum()) < 1e-13


def test_periodic_grid_equals_replicated_nonperiodic_grid_and_reproduces_nodes():
    P = 2 * np.pi
    rng = np.random.default_rng(4)
    c = rng.uniform(-np.pi, np.pi, (30, 2)); h = rng.random(30) + 0.1
    sig = [0.35, 0.35]
    n0, n1 = 24, 20
    lo, hi = np.array([-np.pi, -np.pi]), np.array([np.pi, np.pi])
    tp = np.zeros((4, n0, n1))
    oracle.grid_add_p(tp, lo, hi, [1, 1], c, h, sig)
    # node values are the analytic periodic hill sum and its derivatives
    for (i, j) in [(0, 0), (5, 19), (23, 7)]:
        s = lo + np.array([i * P / n0, j * P / n1])
        V, dV = oracle.bias_periodic(c, h, sig, [P, P], s)
        assert abs(tp[0, i, j] - V) < 1e-13 and abs(tp[1, i, j] - dV[0]) < 1e-12 and abs(tp[2, i, j] - dV[1]) < 1e-12
        out, Vg, dVg = oracle.grid_eval_p(tp, lo, hi, [1, 1], s)
        assert out == 0 and abs(Vg - V) < 1e-13 and np.abs(dVg - dV).max() < 1e-12
    # replicate: non-periodic table with n+1 nodes over the closed period (node n = node 0)
    tr = np.zeros((4, n0 + 1, n1 + 1))
    tr[:, :n0, :n1] = tp; tr[:, n0, :n1] = tp[:, 0, :]; tr[:, :n0, n1] = tp[:, :, 0]; tr[:, n0, n1] = tp[:, 0, 0]
    for _ in range(40):
        s = rng.uniform(-np.pi, np.pi, 2)
        o1, V1, dV1 = oracle.grid_eval_p(tp, lo, hi, [1, 1], s)
        o2, V2, dV2 = oracle.grid_eval(tr, lo, hi, s)
        assert o1 == 0 and o2 == 0 and abs(V1 - V2) < 1e-13 and np.abs(dV1 - dV2).max() < 1e-12
        o3, V3, dV3 = oracle.grid_eval_p(tp, lo, hi, [1, 1], s + [3 * P, -P])       # no "outside" on a periodic dimension
        assert o3 == 0 and abs(V3 - V1) < 1e-11 and np.abs(dV3 - dV1).max() < 1e-10
    # incremental add == one-shot build
    t2 = np.zeros_like(tp)
    oracle.grid_add_p(t2, lo, hi, [1, 1], c, h, sig, 0, 11)
    oracle.grid_add_p(t2, lo, hi, [1, 1], c, h, sig, 11, 30)
    assert np.abs(t2 - tp).max() < 1e-13
    # non-periodic flags = the reading-M routine
    ta, tb = np.zeros((4, n0, n1)), np.zeros((4, n0, n1))
    oracle.grid_add_p(ta, lo, hi, [0, 0], c, h, sig); oracle.grid_add(tb, lo, hi, c, h, sig)
    assert np.array_equal(ta, tb)
    assert oracle.grid_eval_p(ta, lo, hi, [0, 0], [4.0, 0.0])[0] == 1


def test_t0_step_forces_match_finite_differences_of_the_bias():
    """End to end on the alanine-dipeptide-shaped workload: F = -dV/dr by central differences of V(Phi(r), Psi(r))."""
    w = configs.small("t0")
    o = OracleMetaD(w)
    o.build_neighbors(w.pos)
    s = o.eval_cv()
    assert np.all(np.abs(s) <= np.pi)
    c = hill_walk_periodic(5, s, w.sigma, w.n_hills, w.period, w.extra["period_lo"])
    o.set_hills(c, seeded_heights(5, w.n_hills, w.w0))
    V, dV = o.bias(s)
    assert V > 0.1
    F = o.forces(dV)
    assert np.abs(F.sum(0)).max() < 1e-12 * np.abs(F).max()
    h = 1e-5
    touched = sorted(set(np.concatenate([cv.atoms for cv in w.cvs]).tolist()))
    for a in touched:
        for k in range(3):
            vals = []
            for sgn in (1, -1):
                p = w.pos.copy(); p[a, k] += sgn * h
                o2 = OracleMetaD(w); o2.build_neighbors(p); s2 = o2.eval_cv(want_grad=False)
                o2.set_hills(c, o.heights)
                vals.append(o2.bias(s2)[0])
            fd = -(vals[0] - vals[1]) / (2 * h)
            assert abs(fd - F[a, k]) < 1e-6 * np.abs(F).max() + 1e-9
    untouched = [i for i in range(w.natoms) if i not in touched]
    assert np.all(F[untouched] == 0.0)
