"""-m gpu: Verlet-skin reuse of the neighbour list (params.skin) — atoms move every step, the
library keeps its rc + skin list until an atom has moved skin / 2 (decided on the device, inside the captured graph), and
every step must still give the exact rc neighbour sets, CVs, bias and forces of the oracle, which rebuilds its list from
scratch every step (gpu_util.chained_run)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_2510_06873_b200.inputs import CV_MINDIST, CVSpec, configs, wrap  # noqa: E402

from gpu_util import chained_run  # noqa: E402


def _walk(w, nsteps, sigma, seed=31, hop=None):
    """Seeded random walk of every atom (Gaussian steps of width sigma, re-wrapped into the box); `hop`: atoms that are pushed
    across a box face at step 3, so that their periodic image changes while the kept list still holds them."""
    rng = np.random.default_rng(seed)
    frames, p = [], w.pos.copy()
    for k in range(nsteps):
        if k:
            p = p + rng.standard_normal(p.shape) * sigma
        if hop is not None and k == 3:
            B = w.box.reshape(3, 3)
            frac = np.linalg.solve(B.T, p[hop].T).T
            frac[:, 0] = np.where(frac[:, 0] < 0.5, 1.0 - 1e-4, 1e-4)          # next to the a-face, on the other side of it
            p[hop] = frac @ B
        p = wrap(p, w.box)
        frames.append(p.copy())
    return frames


@pytest.mark.parametrize("name,precision", [("c3", 32), ("c3", 64), ("c4", 32), ("c2", 64), ("c2", 32), ("c0'", 64)])
def test_skin_reuse_matches_the_exact_list_every_step(name, precision):
    w = configs.config0(shifted=True) if name == "c0'" else configs.small(name)
    w.stride = 3
    nsteps, skin = 14, 0.3
    B = w.box.reshape(3, 3)
    frac0 = np.linalg.solve(B.T, w.pos.T).T
    hop = np.argsort(np.minimum(frac0[:, 0], 1.0 - frac0[:, 0]))[:6]          # the six atoms nearest to an a-face
    frames = _walk(w, nsteps, 0.012, hop=None if name == "c0'" else hop)
    w.max_neigh = {"c3": 32, "c4": 32, "c2": 64, "c0'": 128}[name]
    hills = (w.hill_centers, w.hill_heights) if name == "c0'" else None
    r = chained_run(w, precision=precision, nsteps=nsteps, skin=skin, check_neighbors=True, hills=hills,
                    pos_of_step=lambda k: frames[k])
    md = r["md"]
    nb = md.rebuilds()
    assert 1 <= nb < nsteps, nb                   # the list was kept over most steps ...
    gi = md.graph_info()
    # ... decided on the device: kernel nodes + ONE conditional node (the build kernels are its body), nothing that touches the host
    assert gi["captures"] == 1 and gi["conditional"] == 1 and gi["nodes"] == gi["kernel"] + 1
    assert gi["memcpy"] == gi["memset"] == gi["host"] == gi["other"] == 0
    # the same walk without a skin: same physics, a build every step
    r0 = chained_run(w, precision=precision, nsteps=nsteps, skin=0.0, hills=r["hills0"], pos_of_step=lambda k: frames[k])
    assert r0["md"].rebuilds() == nsteps
    for a, b in zip(r["states"], r0["states"]):
        assert abs(a["cv"][0] - b["cv"][0]) <= 2e-6 * abs(b["cv"][0])


def test_skin_with_the_nearest_distance_cv_and_a_jump():
    """MINDIST reads the list too; one atom jumps by more than the skin in a single step: the displacement check must force a
    rebuild in that very step."""
    w = configs.small("c2")
    cv = w.cvs[0]
    w.cvs = [CVSpec(kind=CV_MINDIST, group_a=np.asarray(cv.group_a)[11:12], group_b=cv.group_b)]
    w.sigma = [0.05]
    w.stride = 2
    w.max_neigh = 96
    frames = _walk(w, 8, 0.01)
    j = int(np.asarray(cv.group_b)[5])
    for k in range(5, 8):
        frames[k][j] = wrap((frames[k][j] + np.array([0.0, 1.1, 0.4]))[None, :], w.box)[0]
    r = chained_run(w, nsteps=8, skin=0.4, check_neighbors=True, pos_of_step=lambda k: frames[k])
    assert 2 <= r["md"].rebuilds() < 8


def test_skin_rejects_a_box_too_small_for_rc_plus_skin():
    from paper_2510_06873_b200 import metad
    from paper_2510_06873_b200.metad import MetaD, MetadError
    import torch
    w = configs.config0()                         # L = 20, rc = 6: rc + skin must stay below 10
    md = MetaD(w, skin=4.5)
    with pytest.raises(MetadError) as e:
        md.build_neighbors(torch.tensor(w.pos, device="cuda"))
    assert e.value.code == metad.ERR_BOX
    with pytest.raises(MetadError):
        MetaD(w, skin=-0.1)
