"""Pins of orc_cv_lattice ("triaxial lattice parameters as CVs"; reading AB)."""
import numpy as np

import oracle
from paper_2510_06873_b200.inputs import configs


def test_lengths_of_known_cells_and_box_gradient():
    cubic = np.diag([20.0, 20.0, 20.0]).ravel()
    for k in range(3):
        s, g = oracle.cv_lattice(cubic, k)
        assert s == 20.0 and g[k, k] == 1.0 and np.count_nonzero(g) == 1
    # wurtzite supercell of BASELINE.json configs[3] (reading Q): a = b = 80 * 3.19, c = 40 * 5.19, gamma = 120 degrees
    w = configs.small("c3")
    B = w.box.reshape(3, 3)
    a, b, c = (oracle.cv_lattice(w.box, k)[0] for k in range(3))
    assert abs(a - 12 * 3.19) < 1e-12 and abs(b - 12 * 3.19) < 1e-12 and abs(c - 8 * 5.19) < 1e-12
    assert abs(np.degrees(np.arccos(B[0] @ B[1] / (a * b))) - 120.0) < 1e-10
    # gradient with respect to every box element by central differences
    rng = np.random.default_rng(0)
    box = np.array([11.0, 0, 0, -3.0, 9.5, 0, 1.2, -2.1, 13.0]) + 0.0
    for k in range(3):
        s, g = oracle.cv_lattice(box, k)
        assert abs(s - np.linalg.norm(box.reshape(3, 3)[k])) < 1e-14
        fd = np.zeros(9)
        for e in range(9):
            p = box.copy(); p[e] += 1e-5
            q = box.copy(); q[e] -= 1e-5
            fd[e] = (oracle.cv_lattice(p, k)[0] - oracle.cv_lattice(q, k)[0]) / 2e-5
        assert np.abs(fd.reshape(3, 3) - g).max() < 1e-8
    del rng
