"""Pins of orc_reweight (NEXT-2, reading Z) against things other than itself."""
import numpy as np

import oracle

KT = 0.0083144626 * 300.0


def test_zero_bias_is_the_normalised_histogram():
    rng = np.random.default_rng(0)
    traj = rng.normal(0.3, 0.8, (5000, 2))
    lo, hi, nb = [-2.0, -1.5], [2.0, 2.5], [16, 10]
    P, F = oracle.reweight(traj, np.zeros((1, 2)), [0.0], [0.3, 0.3], None, KT, nb, lo, hi)
    Hn, _, _ = np.histogram2d(traj[:, 0], traj[:, 1], bins=nb, range=[[lo[0], hi[0]], [lo[1], hi[1]]])
    vol = (hi[0] - lo[0]) / nb[0] * (hi[1] - lo[1]) / nb[1]
    inside = (traj[:, 0] >= lo[0]) & (traj[:, 0] < hi[0]) & (traj[:, 1] >= lo[1]) & (traj[:, 1] < hi[1])
    # numpy puts points exactly on the last edge into the last bin; none here
    assert np.abs(P - Hn / (len(traj) * vol)).max() < 1e-12
    assert abs(P.sum() * vol - inside.mean()) < 1e-12          # frames outside count in the denominator only
    assert np.all(np.isinf(F[Hn == 0])) and np.allclose(F[Hn > 0], -KT * np.log(P[Hn > 0]))


def test_flat_biased_ensemble_gives_minus_the_bias():
    """A converged run samples the biased ensemble uniformly ("the FES is flatten"): one frame at every
    bin centre => P_unbias ~ e^{beta V}, i.e. F(s) = -V(s) + const exactly."""
    rng = np.random.default_rng(1)
    c = rng.uniform(-1, 1, (40, 1)); h = rng.random(40) + 0.2
    nb, lo, hi = 50, -1.5, 1.5
    s = lo + (np.arange(nb) + 0.5) * (hi - lo) / nb
    P, F = oracle.reweight(s[:, None], c, h, [0.2], None, KT, [nb], [lo], [hi])
    V = np.array([oracle.bias(c, h, [0.2], [x])[0] for x in s])
    d = F[:, 0] + V
    assert np.abs(d - d[0]).max() < 1e-10
    assert abs(P.sum() * (hi - lo) / nb - 1.0) < 1e-12
    # every frame visited twice: same averages
    P2, F2 = oracle.reweight(np.concatenate([s, s])[:, None], c, h, [0.2], None, KT, [nb], [lo], [hi])
    assert np.allclose(P, P2, rtol=1e-13) and np.allclose(F, F2, rtol=1e-12, atol=1e-12)


def test_weights_follow_the_definition_two_frames():
    """Two frames, one hill: P ratios are e^{beta (V1 - V2)} by hand."""
    c, h, sig = [[0.0]], [2.0], [0.5]
    s1, s2 = 0.1, 0.9
    P, _ = oracle.reweight([[s1], [s2]], c, h, sig, None, KT, [2], [0.0], [1.0])
    V1, V2 = 2.0 * np.exp(-s1**2 / 0.5), 2.0 * np.exp(-s2**2 / 0.5)
    w1, w2 = np.exp(V1 / KT), np.exp(V2 / KT)
    assert np.allclose(P[:, 0], np.array([w1, w2]) / (w1 + w2) / 0.5, rtol=1e-13)


def test_periodic_dimension_wraps_frames_and_hills():
    P_ = 2 * np.pi
    rng = np.random.default_rng(2)
    c = rng.uniform(-np.pi, np.pi, (30, 2)); h = rng.random(30) + 0.1
    traj = rng.uniform(-np.pi, np.pi, (2000, 2))
    shifted = traj + rng.integers(-2, 3, traj.shape) * P_
    a = oracle.reweight(traj, c, h, [0.35, 0.35], [P_, P_], KT, [12, 9], [-np.pi, -np.pi], [np.pi, np.pi])
    b = oracle.reweight(shifted, c, h, [0.35, 0.35], [P_, P_], KT, [12, 9], [-np.pi, -np.pi], [np.pi, np.pi])
    assert np.allclose(a[0], b[0], rtol=1e-9)
    assert abs(a[0].sum() * (P_ / 12) * (P_ / 9) - 1.0) < 1e-12
    # numpy restatement
    w = np.array([np.exp(oracle.bias_periodic(c, h, [0.35, 0.35], [P_, P_], s)[0] / KT) for s in traj])
    i0 = np.floor((traj[:, 0] + np.pi) / (P_ / 12)).astype(int); i1 = np.floor((traj[:, 1] + np.pi) / (P_ / 9)).astype(int)
    ref = np.zeros((12, 9)); np.add.at(ref, (i0, i1), w)
    assert np.allclose(a[0], ref / (w.sum() * (P_ / 12) * (P_ / 9)), rtol=1e-12)
