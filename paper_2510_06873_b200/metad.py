"""Thin Python binding over the C ABI of include/metad.h (libmetad_b200.so).

Argument marshalling only: every step of the hot path runs in the CUDA kernels of csrc/.
PyTorch is used for device memory and streams.  There is NO CPU fallback: loading fails loudly if
the library has not been built, and metad_create fails if there is no CUDA device.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmetad_b200.so")

MAX_CV = 4
OK, ERR_ARG, ERR_BOX, ERR_STATE, ERR_CUDA, ERR_NOMEM = range(6)
DEV_NEIGH_OVERFLOW, DEV_HILL_OVERFLOW, DEV_GRID_RANGE, DEV_NONFINITE, DEV_POS_RANGE, DEV_TRAJ_FULL, DEV_BOX = 1, 2, 4, 8, 16, 32, 64
CV_COORD, CV_Q6_MEAN, CV_Q6_SOLID, CV_RGYR, CV_CONTACTS, CV_TORSION, CV_MINDIST, CV_LATTICE = range(8)

_P = ctypes.c_void_p
_I = ctypes.c_int
_D = ctypes.c_double


class CvDesc(ctypes.Structure):
    _fields_ = [("kind", _I), ("n", _I), ("m", _I), ("r0", _D), ("scale", _D),
                ("group_a", _P), ("n_a", _I), ("group_b", _P), ("n_b", _I),
                ("pairs", _P), ("pair_r0", _P), ("npairs", _I),
                ("chain", _P), ("nchain", _I), ("mass", _P),
                ("q_thresh", _D), ("q_width", _D), ("torsion", _I * 4)]


class Params(ctypes.Structure):
    _fields_ = [("natoms", _I), ("precision", _I), ("max_neigh", _I), ("ncv", _I),
                ("cv", CvDesc * MAX_CV), ("sigma", _D * MAX_CV), ("w0", _D), ("kT", _D),
                ("bias_factor", _D), ("max_hills", _I), ("stride", _I), ("grid_n", _I * 2),
                ("grid_lo", _D * 2), ("grid_hi", _D * 2), ("force_scale", _D), ("period", _D * MAX_CV), ("traj_capacity", _I), ("lazy_neighbors", _I), ("want_virial", _I), ("skin", _D), ("box_slack", _D), ("fill_fraction", _D), ("c_window_lo", _D)]


EXPORTS = ["metad_create", "metad_destroy", "metad_build_neighbors", "metad_eval_cv", "metad_bias",
           "metad_apply_forces", "metad_deposit", "metad_run", "metad_build_neighbors_dev", "metad_run_dev", "metad_reset_box", "metad_step_host", "metad_host_alloc", "metad_host_free", "metad_status",
           "metad_get_state", "metad_get_neighbors", "metad_get_q6", "metad_set_hills", "metad_get_hills",
           "metad_get_grid", "metad_get_box_force", "metad_get_virial", "metad_bias_batch", "metad_reweight", "metad_reweight_recorded", "metad_reset_steps", "metad_set_timing", "metad_get_timing", "metad_launch_count", "metad_synchronize", "metad_get_rebuilds", "metad_graph_info", "metad_fma_peak", "metad_bias_noalloc", "metad_cv_owned_sum", "metad_version", "metad_last_error"]

_lib = None


def load():
    """dlopen the CUDA library; raises if it is missing (no fallback)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} not found: run `python -m paper_2510_06873_b200.build` "
                           "(or __graft_entry__.build()); this package has no CPU fallback")
    L = ctypes.CDLL(LIB_PATH)
    L.metad_create.argtypes = [ctypes.POINTER(_P), ctypes.POINTER(Params), _P]
    L.metad_destroy.argtypes = [_P]
    L.metad_build_neighbors.argtypes = [_P, _P, _P, _D]
    L.metad_eval_cv.argtypes = [_P, _P]
    L.metad_bias.argtypes = [_P, _P, _P, _P]
    L.metad_apply_forces.argtypes = [_P, _P, _P]
    L.metad_deposit.argtypes = [_P, _P, _P]
    L.metad_run.argtypes = [_P, _P, _P, _D, _P, _I]
    L.metad_step_host.argtypes = [_P, _P, _P, _D, _P, _P, _P]
    L.metad_build_neighbors_dev.argtypes = [_P, _P, _P, _D]
    L.metad_run_dev.argtypes = [_P, _P, _P, _D, _P, _I]
    L.metad_reset_box.argtypes = [_P]
    L.metad_host_alloc.argtypes = [ctypes.POINTER(_P), ctypes.c_size_t]
    L.metad_host_free.argtypes = [_P]
    L.metad_status.argtypes = [_P, _P]
    L.metad_get_state.argtypes = [_P, _P, _P, _P, _P, _P]
    L.metad_get_neighbors.argtypes = [_P, _P, _P]
    L.metad_get_q6.argtypes = [_P, _P]
    L.metad_set_hills.argtypes = [_P, _P, _P, _I, _I]
    L.metad_get_hills.argtypes = [_P, _P, _P, _I, _P, _I]
    L.metad_get_grid.argtypes = [_P, _P]
    L.metad_reset_steps.argtypes = [_P]
    L.metad_get_box_force.argtypes = [_P, _P]
    L.metad_get_virial.argtypes = [_P, _P]
    L.metad_bias_batch.argtypes = [_P, _P, _I, _P]
    L.metad_reweight.argtypes = [_P, _P, _I, _P, _P, _P, _P, _P]
    L.metad_reweight_recorded.argtypes = [_P, _P, _P, _P, _P, _P, _P]
    L.metad_set_timing.argtypes = [_P, _I]
    L.metad_get_timing.argtypes = [_P, _P, _P]
    L.metad_launch_count.argtypes = [_P]
    L.metad_launch_count.restype = ctypes.c_longlong
    L.metad_synchronize.argtypes = [_P]
    L.metad_get_rebuilds.argtypes = [_P, _P]
    L.metad_graph_info.argtypes = [_P, _P]
    L.metad_fma_peak.argtypes = [_I, _P, _P]
    L.metad_cv_owned_sum.argtypes = [_P, _P, _P]
    L.metad_bias_noalloc.argtypes = [_P, _I, _P, _I, _I, _P, _P, _P, _P, _P, _P]
    L.metad_version.restype = ctypes.c_char_p
    L.metad_last_error.restype = ctypes.c_char_p
    _lib = L
    return L


def fma_peak(kind):
    """Measured scalar-pipe FMA throughput of the current device in TFLOP/s (metad_fma_peak): kind 'f32', 'f32x2' or 'f64'."""
    t, ms = ctypes.c_double(0), ctypes.c_double(0)
    _check(load().metad_fma_peak({"f32": 0, "f32x2": 1, "f64": 2}[kind], ctypes.byref(t), ctypes.byref(ms)))
    return t.value, ms.value


NOALLOC_MAX_HILLS = 1048576       # include/metad.h: METAD_NOALLOC_MAX_HILLS


def bias_noalloc(centers, heights, cv, sigma, V, dVds, period=None, nhills=None, stream=None):
    """metad_bias_noalloc: V(s), dV/ds of the caller's own hill arrays with no context and no allocation (argument
    marshalling only).  centers: CUDA float64 tensor [ncv, ld]; heights: CUDA float64 [>= nhills]; cv: CUDA float64 [ncv];
    V (1) and dVds (ncv): CUDA float64 outputs owned by the caller; stream: a torch.cuda.Stream or None (default stream)."""
    ncv = int(cv.numel())
    for t in (centers, heights, cv, V, dVds):
        assert t.is_cuda and t.is_contiguous() and t.element_size() == 8
    ld = int(centers.shape[1]) if centers.dim() == 2 else int(centers.numel())
    n = int(heights.numel()) if nhills is None else int(nhills)
    sg = np.ascontiguousarray(sigma, dtype=np.float64)
    assert len(sg) == ncv
    pr = None if period is None else np.ascontiguousarray(period, dtype=np.float64)
    _check(load().metad_bias_noalloc(_ptr(centers), ld, _ptr(heights), n, ncv, sg.ctypes.data,
                                     None if pr is None else pr.ctypes.data, _ptr(cv), _ptr(V), _ptr(dVds),
                                     None if stream is None else ctypes.c_void_p(stream.cuda_stream)))
    return V, dVds


class MetadError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"metad error {code}: {msg}")
        self.code = code


def _check(code):
    if code != OK:
        raise MetadError(code, load().metad_last_error().decode())


def _ptr(t):
    return ctypes.c_void_p(t.data_ptr())


class _PinnedBlock:
    """Owner of one metad_host_alloc allocation (freed when the last array viewing it goes away)."""

    def __init__(self, nbytes):
        self.ptr = ctypes.c_void_p()
        _check(load().metad_host_alloc(ctypes.byref(self.ptr), nbytes))
        self.nbytes = nbytes

    def __del__(self):
        if getattr(self, "ptr", None) and self.ptr.value and _lib is not None:
            _lib.metad_host_free(self.ptr)
            self.ptr = ctypes.c_void_p()


def pinned_array(shape, dtype):
    """numpy array in page-locked host memory from metad_host_alloc: the buffers metad_step_host copies at full PCIe rate."""
    dtype = np.dtype(dtype)
    n = int(np.prod(shape))
    blk = _PinnedBlock(max(n * dtype.itemsize, 1))
    buf = (ctypes.c_char * blk.nbytes).from_address(blk.ptr.value)
    buf._owner = blk                                   # keeps the allocation alive as long as the buffer is referenced
    return np.frombuffer(buf, dtype=dtype, count=n).reshape(shape)


class MetaD:
    """One context.  `workload` is a paper_2510_06873_b200.inputs.Workload (or anything with the same
    fields); tensors passed to the methods are torch CUDA tensors (float64, or float32 for pos/F when
    precision == 32)."""

    def __init__(self, workload, max_hills=None, precision=None, grid=None, force_scale=1.0, stream=None, want_virial=False, lazy_neighbors=False, traj_capacity=0,
                 box_slack=0.0, skin=0.0, fill_fraction=0.0, c_window_lo=0.0):
        import torch
        self.torch = torch
        L = load()
        w = workload
        self.N, self.D = w.natoms, w.ncv
        self.precision = int(precision if precision is not None else w.precision)
        self.dtype = torch.float32 if self.precision == 32 else torch.float64
        self.np_dtype = np.float32 if self.precision == 32 else np.float64
        self.box = np.ascontiguousarray(w.box, dtype=np.float64)
        self.rc = float(w.rc)
        self.max_neigh = int(w.max_neigh)
        self.stream = stream if stream is not None else torch.cuda.Stream()
        p = Params()
        p.natoms, p.precision, p.max_neigh, p.ncv = self.N, self.precision, self.max_neigh, self.D
        self._keep = []
        for d, cv in enumerate(w.cvs):
            c = p.cv[d]
            c.kind, c.n, c.m, c.r0, c.scale = int(cv.kind), int(cv.n), int(cv.m), float(cv.r0), float(cv.scale)
            c.q_thresh, c.q_width = float(cv.q_thresh), float(cv.q_width)
            for name, cnt, arr, dt in (("group_a", "n_a", cv.group_a, np.int32), ("group_b", "n_b", cv.group_b, np.int32),
                                       ("chain", "nchain", cv.chain, np.int32)):
                if arr is not None:
                    a = np.ascontiguousarray(arr, dtype=dt)
                    self._keep.append(a)
                    setattr(c, name, a.ctypes.data)
                    setattr(c, cnt, len(a))
            if cv.pairs is not None:
                a = np.ascontiguousarray(cv.pairs, dtype=np.int32)
                b = np.ascontiguousarray(cv.pair_r0, dtype=np.float64)
                self._keep += [a, b]
                c.pairs, c.pair_r0, c.npairs = a.ctypes.data, b.ctypes.data, len(b)
            if getattr(cv, "atoms", None) is not None:
                for k in range(4):
                    c.torsion[k] = int(cv.atoms[k])
            p.sigma[d] = float(w.sigma[d])
            per = getattr(w, "period", None)
            p.period[d] = float(per[d]) if per else 0.0
        p.w0, p.kT, p.bias_factor = float(w.w0), float(w.kT), float(w.bias_factor)
        self.max_hills = int(max_hills if max_hills is not None else max(w.n_hills + 1024, 1024))
        p.max_hills, p.stride = self.max_hills, int(w.stride)
        if grid is not None:
            n, lo, hi = grid
            p.grid_n[0], p.grid_n[1] = int(n[0]), int(n[1])
            p.grid_lo[0], p.grid_lo[1] = float(lo[0]), float(lo[1])
            p.grid_hi[0], p.grid_hi[1] = float(hi[0]), float(hi[1])
            self.grid_n = (int(n[0]), int(n[1]))
        else:
            self.grid_n = None
        p.force_scale = float(force_scale)
        p.want_virial = 1 if want_virial else 0
        p.lazy_neighbors = 1 if lazy_neighbors else 0
        p.traj_capacity = int(traj_capacity)
        p.box_slack = float(box_slack)
        p.fill_fraction = float(fill_fraction)
        p.c_window_lo = float(c_window_lo)
        p.skin = float(skin)
        self._params = p
        h = _P()
        _check(L.metad_create(ctypes.byref(h), ctypes.byref(p), _P(self.stream.cuda_stream)))
        self._h = h
        dev = torch.device("cuda")
        self.cv = torch.zeros(self.D, dtype=torch.float64, device=dev)
        self.V = torch.zeros(1, dtype=torch.float64, device=dev)
        self.dVds = torch.zeros(self.D, dtype=torch.float64, device=dev)

    def close(self):
        if getattr(self, "_h", None):
            load().metad_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- the five hot-path calls (enqueue only)
    def build_neighbors(self, pos, box=None, rc=None):
        assert pos.dtype == self.dtype and pos.is_cuda and pos.is_contiguous()
        box = self.box if box is None else np.ascontiguousarray(box, dtype=np.float64)
        _check(load().metad_build_neighbors(self._h, _ptr(pos), box.ctypes.data, float(self.rc if rc is None else rc)))

    def eval_cv(self, out=None):
        out = self.cv if out is None else out
        _check(load().metad_eval_cv(self._h, _ptr(out)))
        return out

    def bias(self, cv=None, V=None, dVds=None):
        cv = self.cv if cv is None else cv
        V = self.V if V is None else V
        dVds = self.dVds if dVds is None else dVds
        _check(load().metad_bias(self._h, _ptr(cv), _ptr(V), _ptr(dVds)))
        return V, dVds

    def cv_owned_sum(self, owned, cv=None):
        """metad_cv_owned_sum: the Q6 CVs summed over the atoms flagged in `owned` (CUDA uint8 tensor, natoms)."""
        assert owned.is_cuda and owned.is_contiguous() and owned.element_size() == 1 and owned.numel() == self.N
        cv = self.cv if cv is None else cv
        _check(load().metad_cv_owned_sum(self._h, _ptr(owned), _ptr(cv)))
        return cv

    def apply_forces(self, F, dVds=None):
        assert F.dtype == self.dtype and F.is_cuda and F.is_contiguous()
        dVds = self.dVds if dVds is None else dVds
        _check(load().metad_apply_forces(self._h, _ptr(dVds), _ptr(F)))
        return F

    def deposit(self, cv=None, V=None):
        _check(load().metad_deposit(self._h, _ptr(self.cv if cv is None else cv), _ptr(self.V if V is None else V)))

    # ---- graph loop / host path
    def run(self, pos, F, nsteps, box=None, rc=None):
        box = self.box if box is None else np.ascontiguousarray(box, dtype=np.float64)
        _check(load().metad_run(self._h, _ptr(pos), box.ctypes.data, float(self.rc if rc is None else rc), _ptr(F),
                                int(nsteps)))

    def build_neighbors_dev(self, pos, d_box, rc=None):
        """Box in device memory (torch float64 CUDA tensor of 9 elements)."""
        assert pos.dtype == self.dtype and pos.is_cuda and d_box.is_cuda and d_box.dtype == self.torch.float64
        _check(load().metad_build_neighbors_dev(self._h, _ptr(pos), _ptr(d_box), float(self.rc if rc is None else rc)))

    def run_dev(self, pos, d_box, F, nsteps, rc=None):
        assert d_box.is_cuda and d_box.dtype == self.torch.float64 and d_box.numel() == 9
        _check(load().metad_run_dev(self._h, _ptr(pos), _ptr(d_box), float(self.rc if rc is None else rc), _ptr(F), int(nsteps)))

    def reset_box(self):
        _check(load().metad_reset_box(self._h))

    def step_host(self, pos_host, F_host, box=None, rc=None):
        """pos_host / F_host: pinned CPU torch tensors (or numpy arrays) of the context's dtype."""
        box = self.box if box is None else np.ascontiguousarray(box, dtype=np.float64)
        cv = np.zeros(self.D)
        V = np.zeros(1)
        pp = pos_host.data_ptr() if hasattr(pos_host, "data_ptr") else pos_host.ctypes.data
        fp = F_host.data_ptr() if hasattr(F_host, "data_ptr") else F_host.ctypes.data
        _check(load().metad_step_host(self._h, _P(pp), box.ctypes.data, float(self.rc if rc is None else rc), _P(fp),
                                      cv.ctypes.data, V.ctypes.data))
        return cv, V[0]

    # ---- getters (synchronising)
    def synchronize(self):
        self.stream.synchronize()

    def status(self):
        b = ctypes.c_uint(0)
        _check(load().metad_status(self._h, ctypes.byref(b)))
        return b.value

    def state(self):
        cv, V, dV = np.zeros(self.D), np.zeros(1), np.zeros(self.D)
        st, nh = ctypes.c_int(0), ctypes.c_int(0)
        _check(load().metad_get_state(self._h, cv.ctypes.data, V.ctypes.data, dV.ctypes.data, ctypes.byref(st),
                                      ctypes.byref(nh)))
        return {"cv": cv, "V": V[0], "dVds": dV, "step": st.value, "nhills": nh.value}

    def neighbors(self):
        torch = self.torch
        cnt = torch.empty(self.N, dtype=torch.int32, device="cuda")
        lst = torch.empty((self.N, self.max_neigh), dtype=torch.int32, device="cuda")
        _check(load().metad_get_neighbors(self._h, _ptr(cnt), _ptr(lst)))
        self.synchronize()
        return cnt.cpu().numpy(), lst.cpu().numpy()

    def q6(self):
        q = self.torch.empty(self.N, dtype=self.dtype, device="cuda")
        _check(load().metad_get_q6(self._h, _ptr(q)))
        self.synchronize()
        return q.cpu().numpy().astype(np.float64)

    def set_hills(self, centers, heights):
        c = np.ascontiguousarray(centers, dtype=np.float64).reshape(-1, self.D)
        h = np.ascontiguousarray(heights, dtype=np.float64)
        assert len(c) == len(h)
        _check(load().metad_set_hills(self._h, c.ctypes.data, h.ctypes.data, len(h), 0))

    def get_hills(self):
        n = ctypes.c_int(0)
        _check(load().metad_get_hills(self._h, None, None, 0, ctypes.byref(n), 0))
        c, h = np.zeros((max(n.value, 1), self.D)), np.zeros(max(n.value, 1))
        _check(load().metad_get_hills(self._h, c.ctypes.data, h.ctypes.data, n.value, ctypes.byref(n), 0))
        return c[:n.value], h[:n.value]

    def grid_table(self):
        t = self.torch.empty((4,) + self.grid_n, dtype=self.torch.float64, device="cuda")
        _check(load().metad_get_grid(self._h, _ptr(t)))
        self.synchronize()
        return t.cpu().numpy()

    def box_force(self):
        """Bias force on the box rows (3,3) of the last apply_forces (lattice-parameter CVs)."""
        t = self.torch.empty(9, dtype=self.torch.float64, device="cuda")
        _check(load().metad_get_box_force(self._h, _ptr(t)))
        self.synchronize()
        return t.cpu().numpy().reshape(3, 3)

    def virial(self):
        """Bias virial W (3,3) of the last apply_forces (needs want_virial=True; PAPER.md:51 NPT, reading AD)."""
        t = self.torch.empty(9, dtype=self.torch.float64, device="cuda")
        _check(load().metad_get_virial(self._h, _ptr(t)))
        self.synchronize()
        return t.cpu().numpy().reshape(3, 3)

    def bias_batch(self, points):
        """V_b at many CV points (torch float64 CUDA tensor [T, ncv]) -> tensor [T]."""
        torch = self.torch
        T = int(points.shape[0])
        with torch.cuda.stream(self.stream):
            V = torch.empty(T, dtype=torch.float64, device="cuda")
        _check(load().metad_bias_batch(self._h, _ptr(points), T, _ptr(V)))
        return V

    def reweight(self, traj, nbins, lo, hi):
        """(P, F) on the bins, numpy arrays of shape (nb0, nb1)."""
        torch = self.torch
        T = int(traj.shape[0])
        nb = (ctypes.c_int * 2)(int(nbins[0]), int(nbins[1]) if self.D > 1 else 1)
        lo2 = (ctypes.c_double * 2)(float(lo[0]), float(lo[1]) if self.D > 1 else 0.0)
        hi2 = (ctypes.c_double * 2)(float(hi[0]), float(hi[1]) if self.D > 1 else 1.0)
        with torch.cuda.stream(self.stream):
            P = torch.empty((nb[0], nb[1]), dtype=torch.float64, device="cuda")
            F = torch.empty((nb[0], nb[1]), dtype=torch.float64, device="cuda")
        _check(load().metad_reweight(self._h, _ptr(traj), T, nb, lo2, hi2, _ptr(P), _ptr(F)))
        return P.cpu().numpy(), F.cpu().numpy()

    def reweight_recorded(self, nbins, lo, hi):
        """(P, F, nframes) from the CV frames recorded on the device (needs traj_capacity > 0)."""
        torch = self.torch
        nb = (ctypes.c_int * 2)(int(nbins[0]), int(nbins[1]) if self.D > 1 else 1)
        lo2 = (ctypes.c_double * 2)(float(lo[0]), float(lo[1]) if self.D > 1 else 0.0)
        hi2 = (ctypes.c_double * 2)(float(hi[0]), float(hi[1]) if self.D > 1 else 1.0)
        with torch.cuda.stream(self.stream):
            P = torch.empty((nb[0], nb[1]), dtype=torch.float64, device="cuda")
            F = torch.empty((nb[0], nb[1]), dtype=torch.float64, device="cuda")
        n = ctypes.c_int(0)
        _check(load().metad_reweight_recorded(self._h, nb, lo2, hi2, _ptr(P), _ptr(F), ctypes.byref(n)))
        return P.cpu().numpy(), F.cpu().numpy(), n.value

    def reset_steps(self):
        _check(load().metad_reset_steps(self._h))

    def set_timing(self, on=True):
        _check(load().metad_set_timing(self._h, int(bool(on))))

    def get_timing(self):
        a, b = ctypes.c_float(0), ctypes.c_float(0)
        _check(load().metad_get_timing(self._h, ctypes.byref(a), ctypes.byref(b)))
        return a.value, b.value

    def launch_count(self):
        return int(load().metad_launch_count(self._h))

    def rebuilds(self):
        """Neighbour-list builds executed so far (with a skin: fewer than steps)."""
        n = ctypes.c_int(0)
        _check(load().metad_get_rebuilds(self._h, ctypes.byref(n)))
        return n.value

    def graph_info(self):
        """Node counts of the captured step graph (metad_graph_info)."""
        k = (ctypes.c_int * 9)()
        _check(load().metad_graph_info(self._h, k))
        names = ("nodes", "kernel", "memcpy", "memset", "host", "other", "captures", "updates", "conditional")
        return dict(zip(names, (int(x) for x in k)))
