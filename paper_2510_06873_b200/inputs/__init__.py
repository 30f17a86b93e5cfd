"""Seeded synthetic inputs shaped like BASELINE.json's five configs.

This module serves BOTH the CPU oracle tests and the CUDA tests / bench, and holds none of the
method's arithmetic: it only places atoms, picks index groups / contact pairs and draws the
random numbers the method consumes (hill-centre walks).  It imports neither ``oracle`` nor the
CUDA binding.  Everything is a pure function of (config index, seed).

Box convention: 9 doubles, rows a=(ax,0,0), b=(bx,by,0), c=(cx,cy,cz) (lower-triangular).
Positions are wrapped into the primary cell (fractional coordinates in [0,1)).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass, field
from typing import Optional

import numpy as np

BASE_SEED = 2510068730  # + config index
_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = os.path.join(_HERE, "libmetad_inputs.so")

# CV kinds (mirrors include/metad.h; plain integers, no arithmetic)
CV_COORD, CV_Q6_MEAN, CV_Q6_SOLID, CV_RGYR, CV_CONTACTS, CV_TORSION, CV_MINDIST, CV_LATTICE = 0, 1, 2, 3, 4, 5, 6, 7


def build_native(force: bool = False) -> str:
    """Compile gen.c (RSA placement helper) into libmetad_inputs.so next to this file."""
    src = os.path.join(_HERE, "gen.c")
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(src):
        subprocess.check_call(["gcc", "-O2", "-shared", "-fPIC", "-o", _LIB, src, "-lm"])
    return _LIB


_lib = None


def _native():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build_native())
        _lib.gen_rsa.restype = ctypes.c_long
        _lib.gen_rsa.argtypes = [ctypes.c_long, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p,
                                 ctypes.c_void_p, ctypes.c_void_p, ctypes.c_double, ctypes.c_double,
                                 ctypes.c_void_p, ctypes.c_long, ctypes.c_uint64, ctypes.c_void_p,
                                 ctypes.c_long]
    return _lib


def rsa(n_new, box, min_sep, seed, existing=None, periodic=(1, 1, 1), flo=(0, 0, 0), fhi=(1, 1, 1),
        sphere_center=(0, 0, 0), sphere_r=0.0, max_trials=None):
    """Random sequential addition of n_new points (see gen.c).  Returns (n_new,3) float64."""
    box = np.ascontiguousarray(box, dtype=np.float64)
    ex = np.zeros((0, 3)) if existing is None else np.ascontiguousarray(existing, dtype=np.float64)
    out = np.empty((n_new, 3), dtype=np.float64)
    per = np.asarray(periodic, dtype=np.int32)
    lo = np.asarray(flo, dtype=np.float64)
    hi = np.asarray(fhi, dtype=np.float64)
    sc = np.asarray(sphere_center, dtype=np.float64)
    if max_trials is None:
        max_trials = 400 * n_new + 100000
    placed = _native().gen_rsa(n_new, box.ctypes.data, per.ctypes.data, lo.ctypes.data, hi.ctypes.data,
                               sc.ctypes.data, float(sphere_r), float(min_sep), ex.ctypes.data, len(ex),
                               int(seed), out.ctypes.data, int(max_trials))
    if placed != n_new:
        raise RuntimeError(f"RSA placed only {placed} of {n_new} points")
    return out


def wrap(pos, box):
    """Wrap cartesian positions into the primary cell of a lower-triangular row box."""
    box = np.asarray(box, dtype=np.float64).reshape(3, 3)
    s = np.empty_like(pos)
    s[:, 2] = pos[:, 2] / box[2, 2]
    s[:, 1] = (pos[:, 1] - s[:, 2] * box[2, 1]) / box[1, 1]
    s[:, 0] = (pos[:, 0] - s[:, 1] * box[1, 0] - s[:, 2] * box[2, 0]) / box[0, 0]
    s -= np.floor(s)
    s[s >= 1.0] = 0.0
    return s @ box


@dataclass
class CVSpec:
    kind: int
    r0: float = 1.0
    n: int = 6
    m: int = 12
    scale: float = 1.0
    group_a: Optional[np.ndarray] = None   # int32 indices, None = all atoms
    group_b: Optional[np.ndarray] = None
    pairs: Optional[np.ndarray] = None     # (P,2) int32        (CONTACTS)
    pair_r0: Optional[np.ndarray] = None   # (P,) float64       (CONTACTS)
    chain: Optional[np.ndarray] = None     # ordered int32      (RGYR)
    q_thresh: float = 0.35
    q_width: float = 0.05
    atoms: Optional[np.ndarray] = None     # 4 int32 indices i-j-k-l (TORSION)


@dataclass
class Workload:
    name: str
    pos: np.ndarray            # (N,3) float64, wrapped
    box: np.ndarray            # (9,) float64
    rc: float
    max_neigh: int
    cvs: list
    sigma: list
    n_hills: int
    w0: float = 1.0
    kT: float = 0.0083144626 * 300.0   # kJ/mol at 300 K
    bias_factor: float = 1.0           # <=1: plain metadynamics
    stride: int = 10
    precision: int = 64
    hill_centers: Optional[np.ndarray] = None   # (H, D) when the config fixes them (c0)
    hill_heights: Optional[np.ndarray] = None
    grid_n: tuple = (0, 0)
    period: Optional[list] = None               # per CV dimension; 0 = not periodic (torsions: 2 pi)
    species: Optional[np.ndarray] = None
    extra: dict = field(default_factory=dict)

    @property
    def natoms(self):
        return len(self.pos)

    @property
    def ncv(self):
        return len(self.cvs)


def hill_walk(seed, s0, sigma, n_hills, step_frac=0.5, span=100.0):
    """Scripted CV path for hill centres: start at s0, seeded reflecting random
    walk with per-dimension step step_frac*sigma_d inside [s0-span*sigma, s0+span*sigma].
    Pure random-number bookkeeping — the well-tempered heights are computed by whoever replays it."""
    rng = np.random.default_rng(seed)
    s0 = np.atleast_1d(np.asarray(s0, dtype=np.float64))
    sigma = np.atleast_1d(np.asarray(sigma, dtype=np.float64))
    D = len(s0)
    steps = rng.standard_normal((n_hills, D)) * (step_frac * sigma)
    lo, hi = s0 - span * sigma, s0 + span * sigma
    out = np.empty((n_hills, D))
    cur = s0.copy()
    for k in range(n_hills):
        out[k] = cur
        cur = cur + steps[k]
        for d in range(D):
            if cur[d] > hi[d]:
                cur[d] = 2 * hi[d] - cur[d]
            if cur[d] < lo[d]:
                cur[d] = 2 * lo[d] - cur[d]
    return out


def seeded_heights(seed, n_hills, w0=1.0):
    """Synthetic hill heights in (0.05*w0, w0] for stage-wise tests that do not replay deposition."""
    rng = np.random.default_rng(seed + 77)
    return w0 * (0.05 + 0.95 * rng.random(n_hills))


def hill_walk_periodic(seed, s0, sigma, n_hills, period, lo, step_frac=0.5):
    """Scripted CV path on a periodic domain: seeded random walk with per-dimension step
    step_frac*sigma_d, wrapped into [lo_d, lo_d + period_d).  Random-number bookkeeping only."""
    rng = np.random.default_rng(seed)
    s0 = np.atleast_1d(np.asarray(s0, dtype=np.float64))
    sigma = np.atleast_1d(np.asarray(sigma, dtype=np.float64))
    period = np.atleast_1d(np.asarray(period, dtype=np.float64))
    lo = np.atleast_1d(np.asarray(lo, dtype=np.float64))
    steps = rng.standard_normal((n_hills, len(s0))) * (step_frac * sigma)
    path = s0 + np.concatenate([np.zeros((1, len(s0))), np.cumsum(steps[:-1], axis=0)])
    out = lo + np.mod(path - lo, period)
    out[out >= lo + period] = np.broadcast_to(lo, out.shape)[out >= lo + period]
    return out
