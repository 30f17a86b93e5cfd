"""-m gpu: NEXT-2 — batched bias and reweighting of the CUDA path against the oracle."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle  # noqa: E402
from paper_2510_06873_b200.inputs import configs, hill_walk, hill_walk_periodic, seeded_heights  # noqa: E402

from gpu_util import TOL_CV, rel  # noqa: E402

P2 = 2.0 * np.pi


def _ctx(w, centers, heights):
    from paper_2510_06873_b200.metad import MetaD
    md = MetaD(w, max_hills=len(heights) + 8)
    md.set_hills(centers, heights)
    return md


def test_bias_batch_matches_oracle_point_by_point():
    import torch
    for name in ("t0", "c0'", "c4"):
        w = configs.config0(shifted=True) if name == "c0'" else configs.small(name)
        rng = np.random.default_rng(11)
        if w.period:
            c = hill_walk_periodic(5, np.zeros(2), w.sigma, 700, w.period, w.extra["period_lo"])
            pts = rng.uniform(-4.0, 4.0, (3001, 2))
        elif name == "c4":
            c = hill_walk(5, [0.23, 400.0], w.sigma, 700)
            pts = c[rng.integers(0, 700, 3001)] + rng.standard_normal((3001, 2)) * np.asarray(w.sigma)
        else:
            c = np.asarray(w.hill_centers)
            pts = rng.uniform(4.5, 13.5, (3001, 1))
        h = seeded_heights(5, len(c), w.w0)
        md = _ctx(w, c, h)
        with torch.cuda.stream(md.stream):
            dp = torch.tensor(pts, device="cuda")
        V = md.bias_batch(dp)
        md.synchronize()
        V = V.cpu().numpy()
        per = w.period if w.period else np.zeros(w.ncv)
        ref = np.array([oracle.bias_periodic(c, h, w.sigma, per, s)[0] for s in pts])
        big = ref > 1e-12 * ref.max()
        assert big.sum() > 100
        assert np.abs(V[big] - ref[big]).max() / 1.0 <= TOL_CV * ref.max()
        assert (np.abs(V[big] - ref[big]) / ref[big]).max() <= TOL_CV
        assert md.status() == 0


@pytest.mark.parametrize("name", ["t0", "c0'"])
def test_reweight_matches_oracle(name):
    import torch
    w = configs.config0(shifted=True) if name == "c0'" else configs.small(name)
    rng = np.random.default_rng(12)
    T = 20011
    if name == "t0":
        c = hill_walk_periodic(5, np.zeros(2), w.sigma, 400, w.period, w.extra["period_lo"])
        traj = hill_walk_periodic(6, np.zeros(2), [1.0, 1.0], T, w.period, w.extra["period_lo"], step_frac=0.3)
        traj = traj + rng.integers(-1, 2, traj.shape) * P2            # unwrapped frames must be wrapped by the library
        nb, lo, hi = [36, 30], [-np.pi, -np.pi], [np.pi, np.pi]
        h = seeded_heights(5, len(c), w.w0)
    else:
        c = np.asarray(w.hill_centers)
        traj = rng.uniform(4.0, 14.0, (T, 1))                          # some frames outside the histogram range
        nb, lo, hi = [64], [5.0], [13.0]
        h = 3.0 * seeded_heights(5, len(c), w.w0)
    md = _ctx(w, c, h)
    with torch.cuda.stream(md.stream):
        dt = torch.tensor(traj, device="cuda")
    md.synchronize()
    P, F = md.reweight(dt, nb, lo, hi)
    P_ref, F_ref = oracle.reweight(traj, c, h, w.sigma, w.period, w.kT, nb, lo, hi)
    assert P.shape == P_ref.shape
    # per-bin 128-bit sums relative to the bin's own largest weight: EVERY visited bin is resolved, however improbable
    ok = P_ref > 0
    assert ok.sum() > 10 and np.array_equal(P > 0, ok)
    assert (np.abs(P[ok] - P_ref[ok]) / P_ref[ok]).max() <= TOL_CV
    assert np.abs(F[ok] - F_ref[ok]).max() <= TOL_CV * w.kT * np.abs(np.log(P_ref[ok])).max()
    assert np.all(np.isinf(F[~ok]))
    assert np.abs(F[ok] - F_ref[ok]).max() <= TOL_CV * w.kT * 10
    assert np.array_equal(np.isinf(F), P == 0.0)
    # run-to-run bit-identical (integer atomics)
    Pb, Fb = md.reweight(dt, nb, lo, hi)
    assert np.array_equal(P, Pb) and np.array_equal(F, Fb)
    assert md.status() == 0


def test_reweight_argument_errors():
    import torch
    from paper_2510_06873_b200.metad import MetadError
    w = configs.small("t0")
    md = _ctx(w, np.zeros((1, 2)), np.ones(1))
    dt = torch.zeros((4, 2), device="cuda", dtype=torch.float64)
    with pytest.raises(MetadError):
        md.reweight(dt, [8, 8], [-np.pi, -np.pi], [np.pi, 3.0])        # span != period
    with pytest.raises(MetadError):
        md.reweight(dt, [0, 8], [-np.pi, -np.pi], [np.pi, np.pi])


@pytest.mark.parametrize("fused", [False, True])
def test_recorded_trajectory_is_reweighted_on_the_device(fused):
    """The CV frames of a run stay on the GPU (params.traj_capacity) and feed metad_reweight_recorded; the same frames,
    read back step by step, go through the oracle."""
    import torch
    from paper_2510_06873_b200 import metad
    from paper_2510_06873_b200.metad import MetaD
    w = configs.small("t0")
    w.stride = 3
    rng = np.random.default_rng(31)
    c = hill_walk_periodic(5, np.array([-1.4, -0.9]), w.sigma, 60, w.period, w.extra["period_lo"])
    h = seeded_heights(5, 60, w.w0)
    md = MetaD(w, max_hills=128, traj_capacity=40, lazy_neighbors=fused)
    md.set_hills(c, h)
    F = torch.zeros((w.natoms, 3), device="cuda", dtype=torch.float64)
    frames = []
    for k in range(25):
        pos = w.pos + rng.standard_normal(w.pos.shape) * 0.08
        dpos = torch.tensor(pos, device="cuda")
        torch.cuda.synchronize()
        md.run(dpos, F, 1)
        frames.append(md.state()["cv"].copy())
    frames = np.array(frames)
    nb, lo, hi = [96, 80], [-np.pi, -np.pi], [np.pi, np.pi]
    P, Fe, n = md.reweight_recorded(nb, lo, hi)
    assert n == 25
    cc, hh = md.get_hills()
    assert len(hh) == 60 + 25 // 3
    P_ref, F_ref = oracle.reweight(frames, cc, hh, w.sigma, w.period, w.kT, nb, lo, hi)
    assert np.abs(P - P_ref).max() <= 1e-9 * P_ref.max()
    ok = P_ref > 1e-5 * P_ref.max()
    assert ok.sum() >= 1 and (np.abs(P[ok] - P_ref[ok]) / P_ref[ok]).max() <= TOL_CV
    # capacity: frames beyond it are dropped and flagged
    md.run(dpos, F, 20)
    _, _, n2 = md.reweight_recorded(nb, lo, hi)
    assert n2 == 40 and md.status() & metad.DEV_TRAJ_FULL
    md.reset_steps()
    md.run(dpos, F, 2)
    assert md.reweight_recorded(nb, lo, hi)[2] == 2


def test_reweight_resolves_bins_tens_of_kT_below_the_most_probable_one():
    """A deep bias (one 150 kT hill): frames on its flank carry weights 40-140 kT below the frames at its top.  A sum
    quantised against the GLOBAL maximum would flush those bins to P = 0, F = +inf (2^-40 fixed point: everything more than
    27.7 kT down); per-bin sums relative to the bin's own maximum keep them: F against the oracle in every visited bin, to 1e-6
    of its own value, and the weight of 70,000 frames in one bin does not overflow."""
    import torch
    w = configs.config0(shifted=True)
    kT = w.kT
    c, h = np.array([[9.0]]), np.array([150.0 * kT])
    w.sigma = [0.5]
    rng = np.random.default_rng(3)
    traj = np.concatenate([rng.uniform(9.0 - 2.4, 9.0 + 2.4, (30000, 1)), np.full((70000, 1), 9.01)])
    nb, lo, hi = [48], [6.6], [11.4]
    md = _ctx(w, c, h)
    with torch.cuda.stream(md.stream):
        dt = torch.tensor(traj, device="cuda")
    md.synchronize()
    P, F = md.reweight(dt, nb, lo, hi)
    P2_, F2_ = md.reweight(dt, nb, lo, hi)
    assert np.array_equal(P, P2_) and np.array_equal(F, F2_)                      # bit-identical repeats
    P_ref, F_ref = oracle.reweight(traj, c, h, w.sigma, None, kT, nb, lo, hi)
    assert np.all(P_ref > 0) and np.all(np.isfinite(F))
    depth = (F_ref - F_ref.min()) / kT
    assert depth.max() > 100 and np.count_nonzero((depth > 40) & (depth < 60)) >= 2
    assert np.abs(F - F_ref).max() <= TOL_CV * np.abs(F_ref).max()
    assert (np.abs(P - P_ref) / P_ref).max() <= TOL_CV
    assert abs(P.sum() * (hi[0] - lo[0]) / nb[0] - 1.0) <= 1e-12                   # every frame is inside: P integrates to 1
