"""-m gpu: the CV set of the paper's GaN workload — coordination number + the three lattice parameters (
reading AB) — CUDA path against the oracle, including the bias force on the cell."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_2510_06873_b200.inputs import CV_COORD, CV_LATTICE, CVSpec, configs  # noqa: E402

from gpu_util import TOL_CV, TOL_F, assert_stagewise, chained_run, rel, stagewise  # noqa: E402


def _workload():
    w = configs.small("c3")                     # GaN-shaped: wurtzite nucleus in random liquid, triclinic (hexagonal) box
    w.cvs = [CVSpec(kind=CV_COORD, r0=2.4, n=6, m=12, scale=1.0 / w.natoms),
             CVSpec(kind=CV_LATTICE, n=0), CVSpec(kind=CV_LATTICE, n=1), CVSpec(kind=CV_LATTICE, n=2)]
    w.sigma = [0.05, 0.1, 0.1, 0.15]
    w.n_hills = 200
    w.precision = 64
    return w


@pytest.mark.parametrize("precision", [64, 32])
def test_coordination_plus_lattice_parameters(precision):
    w = _workload()
    r = stagewise(w, precision=precision)
    assert_stagewise(r)
    B = w.box.reshape(3, 3)
    assert np.allclose(r["s"][1:], np.linalg.norm(B, axis=1), rtol=1e-14)
    fb = r["md"].box_force()
    fb_ref = r["o"].box_force(r["dV_ref"])
    assert np.abs(fb_ref).max() > 0
    assert np.abs(fb - fb_ref).max() <= 1e-12 * np.abs(fb_ref).max()
    # the lattice dimensions put no force on the atoms: F equals the coordination-number term alone
    F_cn = -r["dV_ref"][0] * r["o"].grads[0]
    assert np.abs(r["F_ref"] - F_cn).max() <= 1e-15 * np.abs(F_cn).max()


@pytest.mark.parametrize("n,m", [(6, 12), (8, 16), (4, 8), (2, 4), (5, 10), (6, 10)])
def test_tiled_coordination_switching_exponents(n, m):
    """The tiled fp32 coordination path (k_tile_build<2> + k_force_add) evaluates sw = 1 / (1 + x^n) for even n with m = 2n
    from r^2 alone (n = 6 special-cased, other even n by square-and-multiply, n = 2 with exponent 0), odd n and m != 2n through
    the general form with a square root (reading A): every branch against the oracle, CV and per-atom forces."""
    w = _workload()
    w.cvs = [CVSpec(kind=CV_COORD, r0=2.4, n=n, m=m, scale=1.0 / w.natoms)]
    w.sigma = [0.05]
    r = stagewise(w, precision=32)
    assert_stagewise(r)
    assert np.abs(r["F_ref"]).max() > 0
    assert np.abs(r["F"].sum(axis=0)).max() <= 1e-3 * np.abs(r["F_ref"]).max()      # translation invariance (reading N), fp32 sums


@pytest.mark.parametrize("drop", [0, 1, 2, 3])
def test_tiled_coordination_force_update_unaligned_and_ragged(drop):
    """k_force_add4 adds the per-atom gradient to F with 128-bit accesses, four atoms per thread; a ragged tail (N not a
    multiple of 4, nor of the 32-atom list slabs) and a caller's F that is not 16-byte aligned (scalar k_force_add) must give
    the same forces: both against the oracle, on top of a non-zero F."""
    import torch
    w = _workload()
    n = w.natoms - drop
    w.pos = np.ascontiguousarray(w.pos[:n])
    assert w.natoms == n
    w.cvs = [CVSpec(kind=CV_COORD, r0=2.4, n=6, m=12, scale=1.0 / n)]
    w.sigma = [0.05]
    r = stagewise(w, precision=32)
    assert_stagewise(r)
    md, fmax = r["md"], np.abs(r["F_ref"]).max()
    dV_in = torch.tensor(r["dV_ref"], device="cuda", dtype=torch.float64)
    for offset in (0, 1):                                    # offset 1 float: F is 4 bytes off a 16-byte boundary
        with torch.cuda.stream(md.stream):
            buf = torch.full((3 * n + 4,), 0.25, device="cuda", dtype=torch.float32)
        F = buf[offset:offset + 3 * n].view(n, 3)
        assert (F.data_ptr() % 16 == 0) == (offset == 0)
        md.synchronize()
        md.apply_forces(F, dVds=dV_in)
        md.synchronize()
        out = buf.cpu().numpy().astype(np.float64)
        assert np.abs(out[offset:offset + 3 * n].reshape(n, 3) - 0.25 - r["F_ref"]).max() <= TOL_F * fmax + 2 ** -24
        assert np.all(out[:offset] == 0.25) and np.all(out[offset + 3 * n:] == 0.25)      # nothing written outside F


def test_lazy_neighbors_runs_the_tiled_coordination_pass_list_free():
    """params.lazy_neighbors on the paper's GaN CV set: the fp32 tiled build accumulates the coordination sum and
    the per-atom gradient and stores no list — same CV, V and forces bit for bit as with the list, metad_get_neighbors says so;
    with the virial wanted the list is built regardless (its force kernel walks it)."""
    import torch
    from paper_2510_06873_b200.metad import MetaD, MetadError
    w = _workload()
    pos = np.ascontiguousarray(w.pos.astype(np.float32))
    outs = []
    for lazy, vir in ((False, False), (True, False), (True, True)):
        md = MetaD(w, precision=32, max_hills=64, lazy_neighbors=lazy, want_virial=vir)
        s0 = np.array([5.4, *np.linalg.norm(w.box.reshape(3, 3), axis=1)])
        md.set_hills(np.array([s0 + [0.03, 0.05, -0.02, 0.04]]), np.array([1.5]))
        with torch.cuda.stream(md.stream):
            dpos = torch.tensor(pos, device="cuda")
            F = torch.zeros((w.natoms, 3), device="cuda", dtype=torch.float32)
        md.synchronize()
        md.run(dpos, F, 3)
        st = md.state()
        assert md.status() == 0
        outs.append((st["cv"].copy(), st["V"], F.cpu().numpy()))
        if lazy and not vir:
            with pytest.raises(MetadError):
                md.neighbors()
        else:
            cnt, _ = md.neighbors()
            assert cnt.sum() > 0
    assert np.abs(outs[0][2]).max() > 0
    for o in outs[1:]:
        assert np.array_equal(o[0], outs[0][0]) and o[1] == outs[0][1]
    assert np.array_equal(outs[1][2], outs[0][2])
    assert np.abs(outs[2][2] - outs[0][2]).max() <= 1e-5 * np.abs(outs[0][2]).max()      # k_coord_force_g: other summation order


def test_lattice_only_context_and_bad_axis():
    import torch
    from paper_2510_06873_b200.metad import MetaD, MetadError
    w = _workload()
    w.cvs = w.cvs[1:]
    w.sigma = w.sigma[1:]
    md = MetaD(w)
    dpos = torch.tensor(w.pos, device="cuda")
    F = torch.zeros((w.natoms, 3), device="cuda", dtype=torch.float64)
    torch.cuda.synchronize()
    s0 = np.linalg.norm(w.box.reshape(3, 3), axis=1)
    md.set_hills(np.array([s0 + [0.05, -0.02, 0.1]]), np.array([2.0]))
    md.run(dpos, F, 1)
    st = md.state()
    assert np.allclose(st["cv"], s0, rtol=1e-14) and not F.cpu().numpy().any()
    d = s0 - (s0 + [0.05, -0.02, 0.1])
    V = 2.0 * np.exp(-0.5 * np.sum((d / np.asarray(w.sigma)) ** 2))
    assert abs(st["V"] - V) <= 1e-12 * V
    fb = md.box_force()
    ref = np.zeros((3, 3))
    for k in range(3):
        ref[k] = -(-V * d[k] / w.sigma[k] ** 2) * w.box.reshape(3, 3)[k] / s0[k]
    assert np.abs(fb - ref).max() <= 1e-12 * np.abs(ref).max()
    w.cvs[0].n = 3
    with pytest.raises(MetadError):
        MetaD(w)


def test_changing_box_every_step_updates_the_graph():
    """NPT-like loop: positions and box are rescaled every step; metad_run must follow the new box (kernel
    arguments, cell grid and tile counts change) and match the oracle loop step by step (gpu_util.chained_run)."""
    w = _workload()
    w.stride = 2
    frac = np.linalg.solve(w.box.reshape(3, 3).T, w.pos.T).T
    box0 = w.box.copy()
    scales = [1.0, 1.004, 0.97, 1.08, 1.0801, 0.9]      # 0.97 / 1.08 / 0.9 change the cell counts
    # hills that cover the whole excursion of the lattice parameters (widths 0.1 A): a few wide-spread seeded centres
    s0 = np.array([5.4, *np.linalg.norm(box0.reshape(3, 3), axis=1)])
    rng = np.random.default_rng(8)
    centers = s0 * (1.0 + 0.1 * (rng.random((30, 4)) - 0.5))
    r = chained_run(w, nsteps=len(scales), hills=(centers, np.full(30, 1.0)),
                    box_of_step=lambda k: box0 * scales[k], pos_of_step=lambda k: frac @ (box0 * scales[k]).reshape(3, 3))
    assert r["states"][-1]["nhills"] == 30 + 3
    assert np.array_equal(w.box, box0)


@pytest.mark.parametrize("precision", [64, 32])
def test_device_resident_box_one_capture_no_graph_update(precision):
    """NEXT-3 (PAPER.md:51 NPT; PAPER.md:61 on GPU-CPU transfers): the box lives in device memory and changes every step —
    metad_run_dev captures its CUDA graph ONCE, never updates it, and every step matches the oracle (gpu_util.chained_run) on
    the generic fp64 kernels and on the tiled fp32 path; a box that shrinks below the frozen cell grid raises METAD_DEV_BOX,
    metad_reset_box re-derives the grid."""
    import torch
    from paper_2510_06873_b200 import metad
    w = _workload()
    w.stride = 2
    frac = np.linalg.solve(w.box.reshape(3, 3).T, w.pos.T).T
    box0 = w.box.copy()
    scales = [1.0, 1.004, 0.985, 1.02, 1.03, 0.975, 1.0]
    s0 = np.array([5.4, *np.linalg.norm(box0.reshape(3, 3), axis=1)])
    rng = np.random.default_rng(8)
    centers = s0 * (1.0 + 0.04 * (rng.random((30, 4)) - 0.5))
    r = chained_run(w, precision=precision, nsteps=len(scales), hills=(centers, np.full(30, 1.0)), device_box=True, box_slack=0.03,
                    box_of_step=lambda k: box0 * scales[k], pos_of_step=lambda k: frac @ (box0 * scales[k]).reshape(3, 3))
    md = r["md"]
    gi = md.graph_info()
    assert gi["captures"] == 1 and gi["updates"] == 0
    assert gi["nodes"] == gi["kernel"] and gi["memcpy"] == 0 and gi["host"] == 0
    assert md.status() == 0
    # a box 8 % smaller than the one the grid was frozen for: cells narrower than rc -> sticky bit, no error code
    tdt = torch.float32 if precision == 32 else torch.float64
    with torch.cuda.stream(md.stream):
        dbox = torch.tensor(box0 * 0.92, device="cuda", dtype=torch.float64)
        dpos = torch.tensor(frac @ (box0 * 0.92).reshape(3, 3), device="cuda", dtype=tdt)
        F = torch.zeros((w.natoms, 3), device="cuda", dtype=tdt)
    md.synchronize()
    md.build_neighbors_dev(dpos, dbox)
    assert md.status() & metad.DEV_BOX
    md.reset_box()
    md.run_dev(dpos, dbox, F, 1)
    assert md.graph_info()["captures"] == 2
