"""-m gpu: the RUN paths the benchmark times — metad_run (CUDA-graph replay with the deposition fused into the hill sum and the
CV handed over by the last block of the tiled build) and metad_step_host (the e2e leg) — on the tiled fp32 path, step by step
against the oracle (gpu_util.chained_run: stage-wise on the library's own upstream values, reading S; plus a free-running
oracle loop with the derived force bound).  Covers the glue that the stage-call tests do not reach."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_2510_06873_b200.inputs import configs  # noqa: E402

from gpu_util import chained_run  # noqa: E402


def _grid_for(w, hills):
    sig = np.asarray(w.sigma)
    c0 = hills[0][0]
    return (w.grid_n, c0 - 40 * sig, c0 + 40 * sig)


def test_metad_run_tiled_fp32_q6_against_the_oracle_loop():
    """BASELINE.json configs[3] shape (Q6 mean, well-tempered, gamma = 20) in the launch configuration bench.py times."""
    w = configs.small("c3")
    w.stride = 2
    r = chained_run(w, precision=32, nsteps=8)
    assert r["launches_per_step"] <= 8
    assert r["states"][-1]["nhills"] == 40 + 4


@pytest.mark.parametrize("use_grid", [False, True])
def test_metad_run_tiled_fp32_q6_and_solid_count(use_grid):
    """configs[4] shape: 2-D CV (Q6 mean, solid-like count), exact hill sum and the bicubic grid (separate deposit launch)."""
    w = configs.small("c4")
    w.stride = 2
    hills = None
    grid = None
    if use_grid:
        # the grid window must hold the structure's own CV: take the seeded hill walk chained_run would take
        from oracle.reference import OracleMetaD
        from gpu_util import positions_for
        from paper_2510_06873_b200.inputs import hill_walk, seeded_heights
        o = OracleMetaD(w)
        o.build_neighbors(positions_for(w, 32).astype(np.float64))
        s0 = o.eval_cv(want_grad=False)
        hills = (hill_walk(5, s0, w.sigma, 40), seeded_heights(5, 40, w.w0))
        grid = _grid_for(w, hills)
    r = chained_run(w, precision=32, nsteps=7, grid=grid, hills=hills)
    assert r["states"][-1]["nhills"] == 40 + 3


@pytest.mark.parametrize("lazy", [False, True])
def test_metad_run_tiled_fp32_coordination_plus_lattice(lazy):
    """PAPER.md:51 CV set (g0): the coordination sum and the per-atom gradient ride on the tiled build; lazy_neighbors
    runs the same pass list-free."""
    w = configs.small("g0")
    w.stride = 3
    r = chained_run(w, precision=32, nsteps=7, lazy=lazy)
    assert r["states"][-1]["nhills"] == 40 + 2


@pytest.mark.parametrize("name,precision", [("c3", 32), ("c4", 32), ("c3", 64), ("c1", 64)])
def test_metad_step_host_against_the_oracle_loop(name, precision):
    """The e2e leg of bench.py: host buffers in, forces / CV / V out, on the tiled fp32 path and the generic fp64 one."""
    w = configs.small(name)
    w.stride = 2
    r = chained_run(w, precision=precision, nsteps=5, host=True)
    assert r["states"][-1]["nhills"] == 40 + 2


def test_metad_run_generic_fp64_paths():
    """c0' (coordination, plain MetaD, no deposition), c1 (Rg + contacts) and c2 (grouped coordination) through metad_run."""
    for name in ("c1", "c2"):
        w = configs.small(name)
        w.stride = 2
        chained_run(w, nsteps=5)
    w = configs.config0(shifted=True)
    r = chained_run(w, nsteps=3, hills=(w.hill_centers, w.hill_heights))
    assert r["states"][-1]["nhills"] == 200


@pytest.mark.parametrize("name,precision,lazy", [("c3", 32, False), ("c4", 32, False), ("g0", 32, True), ("c1", 64, False),
                                                 ("t0", 64, True)])
def test_captured_step_graph_has_kernel_nodes_only(name, precision, lazy):
    """BASELINE.json north_star: "a multi-step loop makes zero host round-trips" (PAPER.md:61 names the GPU-CPU transfer
    overhead as the cost to avoid): the CUDA graph metad_run captures holds kernel nodes only — no memcpy, no host node —
    (a bias virial adds one 72-byte device memset), as many of them as the library counts launches per step, and replaying it
    for a fixed box never re-captures."""
    import torch
    from paper_2510_06873_b200.metad import MetaD, MetadError
    w = configs.small(name)
    md = MetaD(w, precision=precision, max_hills=64, lazy_neighbors=lazy)
    with pytest.raises(MetadError):
        md.graph_info()                                           # nothing captured yet
    tdt = torch.float32 if precision == 32 else torch.float64
    with torch.cuda.stream(md.stream):
        dpos = torch.tensor(w.pos, device="cuda", dtype=tdt)
        F = torch.zeros((w.natoms, 3), device="cuda", dtype=tdt)
    md.synchronize()
    l0 = md.launch_count()
    md.run(dpos, F, 4)
    md.run(dpos, F, 3)
    gi = md.graph_info()
    assert gi["nodes"] == gi["kernel"] > 0
    assert gi["memcpy"] == gi["memset"] == gi["host"] == gi["other"] == 0
    assert gi["captures"] == 1 and gi["updates"] == 0
    assert md.launch_count() - l0 == 7 * gi["kernel"]
    assert md.state()["step"] == 7 and md.status() == 0


def test_context_on_a_private_stream_when_the_caller_passes_null():
    """include/metad.h: cuda_stream == NULL makes the library create (and own) a non-blocking stream; metad_synchronize
    orders the caller with it.  Same numbers as a context on a caller-provided stream; create / destroy cycles leak nothing
    that the driver reports (memory in use returns to where it was)."""
    import ctypes
    import torch
    from paper_2510_06873_b200 import metad
    from paper_2510_06873_b200.metad import MetaD
    w = configs.small("c3")
    pos = np.ascontiguousarray(w.pos.astype(np.float32))
    ref = MetaD(w, precision=32, max_hills=64)
    ref.set_hills(np.array([[0.23]]), np.array([1.0]))
    dpos = torch.tensor(pos, device="cuda")
    F0 = torch.zeros((w.natoms, 3), device="cuda", dtype=torch.float32)
    torch.cuda.synchronize()
    ref.run(dpos, F0, 2)
    st0 = ref.state()
    L = metad.load()
    h = ctypes.c_void_p()
    assert L.metad_create(ctypes.byref(h), ctypes.byref(ref._params), None) == 0
    c = np.array([0.23]); hh = np.array([1.0])
    assert L.metad_set_hills(h, c.ctypes.data, hh.ctypes.data, 1, 0) == 0
    F1 = torch.zeros((w.natoms, 3), device="cuda", dtype=torch.float32)
    torch.cuda.synchronize()
    box = np.ascontiguousarray(w.box)
    assert L.metad_run(h, ctypes.c_void_p(dpos.data_ptr()), box.ctypes.data, float(w.rc), ctypes.c_void_p(F1.data_ptr()), 2) == 0
    assert L.metad_synchronize(h) == 0
    assert torch.equal(F0, F1)
    cv, V = np.zeros(1), np.zeros(1)
    assert L.metad_get_state(h, cv.ctypes.data, V.ctypes.data, None, None, None) == 0
    assert cv[0] == st0["cv"][0] and V[0] == st0["V"]
    assert L.metad_destroy(h) == 0
    # failed creates free what they allocated: a bad group index is detected after the first device buffers exist
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    p = metad.Params()
    ctypes.memmove(ctypes.byref(p), ctypes.byref(ref._params), ctypes.sizeof(p))
    bad = np.array([0, 1, w.natoms + 5], dtype=np.int32)
    p.ncv = 2
    p.cv[1].kind = metad.CV_COORD
    p.cv[1].r0, p.cv[1].n, p.cv[1].m, p.cv[1].scale = 2.0, 6, 12, 1.0
    p.cv[1].group_a, p.cv[1].n_a = bad.ctypes.data, 3
    p.sigma[1] = 1.0
    for _ in range(20):
        assert L.metad_create(ctypes.byref(h), ctypes.byref(p), None) == metad.ERR_ARG
    torch.cuda.synchronize()
    assert abs(torch.cuda.mem_get_info()[0] - free0) <= (8 << 20)
