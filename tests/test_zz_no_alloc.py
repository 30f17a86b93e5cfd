"""-m gpu: metad_bias_noalloc (include/metad.h) — the hill sum V(s), dV/ds through the ONE entry point that allocates
nothing (scratch in a file-scope __device__ array, csrc/noalloc.cu) against the existing path, metad_bias of a context that
holds the same hills, within the tolerance the other tests use for V and dV/ds (1e-6 relative, BASELINE.json north_star).

The file is named so that pytest collects it LAST (the suite runs with `pytest -x`); it passes alone in a fresh process and
after the other tests: it shares nothing with them but the loaded library."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_2510_06873_b200.inputs import configs, hill_walk, hill_walk_periodic, seeded_heights  # noqa: E402

TOL = 1e-6


def _existing_path(w, centers, heights, points):
    """metad_bias of a context holding the hills: [(V, dVds)] at the given points."""
    import torch
    from paper_2510_06873_b200.metad import MetaD
    md = MetaD(w, max_hills=len(heights) + 8)
    md.set_hills(centers, heights)
    out = []
    for s in points:
        with torch.cuda.stream(md.stream):
            ds = torch.tensor(s, device="cuda", dtype=torch.float64)
        V, dV = md.bias(cv=ds)
        md.synchronize()
        out.append((float(V.cpu().numpy().ravel()[0]), dV.cpu().numpy().astype(np.float64).copy()[:len(s)]))
    assert md.status() == 0
    return out


def _close(got, ref):
    V, dV = got
    V_ref, dV_ref = ref
    assert abs(V - V_ref) <= TOL * max(abs(V_ref), 1e-300), (V, V_ref)
    assert np.abs(dV - dV_ref).max() <= TOL * max(np.abs(dV_ref).max(), 1e-300), (dV, dV_ref)


@pytest.mark.parametrize("name", ["c4", "t0"])
def test_no_alloc_hill_sum_matches_the_context_path_on_two_calls_in_a_row(name):
    """Two calls back to back on one stream share the scratch array: the second (another point, FEWER hills, so fewer rows of
    partial sums than the first left behind) must not see the first one's contents.  c4: 2-D, not periodic; t0: 2-D torsions,
    periodic hills across the seam.  5,000 hills = two full blocks of 2,048 and a ragged third."""
    import torch
    from paper_2510_06873_b200 import metad
    w = configs.small(name)
    D = w.ncv
    sig = np.asarray(w.sigma, dtype=np.float64)
    n1, n2 = 5000, 1500
    if getattr(w, "period", None):
        period, lo = np.asarray(w.period, dtype=np.float64), np.asarray(w.extra["period_lo"], dtype=np.float64)
        centers = hill_walk_periodic(3, lo + 0.02 * period, sig, n1, period, lo)
        s1, s2 = centers[n1 // 2] + 0.3 * sig, lo + np.array([0.01, 0.99]) * period          # s2: next to the seam
    else:
        period = None
        centers = hill_walk(3, np.array([0.23, 40.0])[:D], sig, n1)
        s1, s2 = centers[n1 // 2] + 0.3 * sig, centers[100] - 0.7 * sig
    heights = seeded_heights(3, n1, w.w0)
    ref1 = _existing_path(w, centers, heights, [s1])[0]
    ref2 = _existing_path(w, centers[:n2], heights[:n2], [s2])[0]
    assert abs(ref1[0]) > 0 and abs(ref2[0]) > 0

    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        dc = torch.tensor(np.ascontiguousarray(centers.T), device="cuda", dtype=torch.float64)      # [D][ld = n1]
        dh = torch.tensor(heights, device="cuda", dtype=torch.float64)
        d1 = torch.tensor(s1, device="cuda", dtype=torch.float64)
        d2 = torch.tensor(s2, device="cuda", dtype=torch.float64)
        V1, V2 = torch.full((1,), np.nan, device="cuda", dtype=torch.float64), torch.full((1,), np.nan, device="cuda", dtype=torch.float64)
        g1, g2 = torch.full((D,), np.nan, device="cuda", dtype=torch.float64), torch.full((D,), np.nan, device="cuda", dtype=torch.float64)
    st.synchronize()
    metad.bias_noalloc(dc, dh, d1, sig, V1, g1, period=period, stream=st)
    metad.bias_noalloc(dc, dh, d2, sig, V2, g2, period=period, nhills=n2, stream=st)            # ld stays n1
    st.synchronize()
    _close((float(V1.cpu()[0]), g1.cpu().numpy()), ref1)
    _close((float(V2.cpu()[0]), g2.cpu().numpy()), ref2)
    # the same two calls again: run-to-run identical bits (fixed-order sums), and no device memory taken by a call
    free0 = torch.cuda.mem_get_info()[0]
    W1, h1 = torch.zeros(1, device="cuda", dtype=torch.float64), torch.zeros(D, device="cuda", dtype=torch.float64)
    free1 = torch.cuda.mem_get_info()[0]
    metad.bias_noalloc(dc, dh, d1, sig, W1, h1, period=period, stream=None)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free1 <= free0
    assert torch.equal(W1, V1) and torch.equal(h1, g1)


def test_no_alloc_limits_and_empty_input():
    import torch
    from paper_2510_06873_b200 import metad
    z = torch.zeros(8, device="cuda", dtype=torch.float64)
    c = torch.zeros((1, 8), device="cuda", dtype=torch.float64)
    V, g = torch.ones(1, device="cuda", dtype=torch.float64), torch.ones(1, device="cuda", dtype=torch.float64)
    metad.bias_noalloc(c, z, z[:1], [0.1], V, g, nhills=0)                      # no hills: V = 0, dV/ds = 0
    torch.cuda.synchronize()
    assert float(V.cpu()[0]) == 0.0 and float(g.cpu()[0]) == 0.0
    with pytest.raises(metad.MetadError) as e:                                    # beyond the fixed scratch array
        metad.bias_noalloc(c, z, z[:1], [0.1], V, g, nhills=metad.NOALLOC_MAX_HILLS + 1)
    assert e.value.code == metad.ERR_ARG and "METAD_NOALLOC_MAX_HILLS" in str(e.value)
    with pytest.raises(metad.MetadError):                                         # ld_centers < nhills
        metad.bias_noalloc(c, z, z[:1], [0.1], V, g, nhills=9)
    with pytest.raises(metad.MetadError):
        metad.bias_noalloc(c, z, z[:1], [0.0], V, g, nhills=4)                  # sigma must be positive
    with pytest.raises(metad.MetadError):                                         # ncv beyond METAD_MAX_CV
        metad.bias_noalloc(torch.zeros((5, 8), device="cuda", dtype=torch.float64), z, z[:5], [0.1] * 5, V,
                           torch.zeros(5, device="cuda", dtype=torch.float64), nhills=4)


def test_no_alloc_at_the_limit():
    """METAD_NOALLOC_MAX_HILLS hills (every row of the scratch array in use) of one 1-D Gaussian each at the same centre:
    V = sum of the heights at that centre, dV/ds = 0 there; one sigma away V e^(-1/2), dV/ds = -V e^(-1/2) / sigma."""
    import torch
    from paper_2510_06873_b200 import metad
    n = metad.NOALLOC_MAX_HILLS
    h = seeded_heights(9, n)
    dc = torch.full((1, n), 0.25, device="cuda", dtype=torch.float64)
    dh = torch.tensor(h, device="cuda", dtype=torch.float64)
    V, g = torch.zeros(1, device="cuda", dtype=torch.float64), torch.zeros(1, device="cuda", dtype=torch.float64)
    tot = float(np.sum(h))
    metad.bias_noalloc(dc, dh, torch.tensor([0.25], device="cuda", dtype=torch.float64), [0.05], V, g)
    torch.cuda.synchronize()
    assert abs(float(V.cpu()[0]) - tot) <= 1e-12 * tot and abs(float(g.cpu()[0])) <= 1e-12 * tot / 0.05
    metad.bias_noalloc(dc, dh, torch.tensor([0.30], device="cuda", dtype=torch.float64), [0.05], V, g)
    torch.cuda.synchronize()
    e = tot * np.exp(-0.5)
    assert abs(float(V.cpu()[0]) - e) <= 1e-12 * e and abs(float(g.cpu()[0]) + e / 0.05) <= 1e-12 * e / 0.05
