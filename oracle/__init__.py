"""CPU oracle (TEST INFRASTRUCTURE, NOT PRODUCT) — ctypes access to oracle/metad_oracle.c.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package.  It never imports the CUDA binding, and the CUDA binding never imports it.
All arithmetic is in metad_oracle.c (fp64, -ffp-contract=off); this file only marshals numpy arrays.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "metad_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
                               "-o", _LIB, _SRC, "-lm"])
    return _LIB


_lib = None
_P = ctypes.c_void_p
_I = ctypes.c_int
_D = ctypes.c_double


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        L.orc_num_threads.restype = _I
        L.orc_set_threads.argtypes = [_I]
        L.orc_box_check.restype = _I
        L.orc_box_check.argtypes = [_P, _D, _P]
        L.orc_delta.argtypes = [_P, _P, _P, _P]
        for f in (L.orc_neighbors_brute, L.orc_neighbors_images, L.orc_neighbors_cells):
            f.restype = _I
            f.argtypes = [_I, _P, _P, _D, _I, _P, _P]
        L.orc_switch.restype = _D
        L.orc_switch.argtypes = [_D, _I, _I, _P]
        L.orc_cv_coord.restype = _D
        L.orc_cv_coord.argtypes = [_I, _P, _P, _P, _P, _I, _P, _D, _I, _I, _D, _P]
        L.orc_q6_atoms.argtypes = [_I, _P, _P, _P, _P, _I, _P]
        L.orc_q6_grad.argtypes = [_I, _P, _P, _P, _P, _I, _P, _P, _P]
        L.orc_y6.argtypes = [_P, _P]
        L.orc_q6_atoms_ylm.argtypes = [_I, _P, _P, _P, _P, _I, _P, _P]
        L.orc_cv_rgyr.restype = _D
        L.orc_cv_rgyr.argtypes = [_I, _P, _P, _P, _P, _P]
        L.orc_cv_contacts.restype = _D
        L.orc_cv_contacts.argtypes = [_I, _I, _P, _P, _I, _I, _D, _P, _P, _P]
        L.orc_bias.argtypes = [_I, _I, _P, _P, _P, _P, _P, _P]
        L.orc_wt_height.restype = _D
        L.orc_wt_height.argtypes = [_D, _D, _D, _D]
        L.orc_grid_add.argtypes = [_I, _I, _P, _P, _I, _I, _P, _P, _P, _P]
        L.orc_grid_eval.restype = _I
        L.orc_grid_eval.argtypes = [_I, _I, _P, _P, _P, _P, _P, _P]
        L.orc_apply_forces.argtypes = [_I, _I, _P, _P, _D, _P]
        L.orc_cv_torsion.restype = _D
        L.orc_cv_torsion.argtypes = [_P, _P, _P, _P]
        L.orc_pdiff.restype = _D
        L.orc_pdiff.argtypes = [_D, _D, _D]
        L.orc_wrap.restype = _D
        L.orc_wrap.argtypes = [_D, _D, _D]
        L.orc_bias_periodic.argtypes = [_I, _I, _P, _P, _P, _P, _P, _P, _P]
        L.orc_grid_add_p.argtypes = [_I, _I, _P, _P, _P, _I, _I, _P, _P, _P, _P]
        L.orc_reweight.argtypes = [_I, _I, _P, _I, _P, _P, _P, _P, _D, _P, _P, _P, _P, _P]
        L.orc_cv_mindist.restype = _D
        L.orc_cv_mindist.argtypes = [_I, _P, _P, _P, _P, _I, _P, _D, _P, _P]
        L.orc_cv_lattice.restype = _D
        L.orc_cv_lattice.argtypes = [_P, _I, _P]
        L.orc_cv_coord_strain.argtypes = [_I, _P, _P, _P, _P, _I, _P, _D, _I, _I, _D, _P]
        L.orc_q6_strain.argtypes = [_I, _P, _P, _P, _P, _I, _P, _P, _P]
        L.orc_cv_lattice_strain.argtypes = [_P, _I, _P]
        L.orc_cv_rgyr_strain.argtypes = [_I, _P, _P, _P, _P, _P]
        L.orc_cv_contacts_strain.argtypes = [_I, _P, _P, _I, _I, _D, _P, _P, _P]
        L.orc_cv_mindist_strain.argtypes = [_I, _P, _P, _P, _P, _I, _P, _D, _P]
        L.orc_cv_torsion_strain.argtypes = [_P, _P, _P, _P]
        L.orc_grid_eval_p.restype = _I
        L.orc_grid_eval_p.argtypes = [_I, _I, _P, _P, _P, _P, _P, _P, _P]
        _lib = L
    return _lib


def _f(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _i(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def _p(a):
    return None if a is None else a.ctypes.data


def num_threads():
    return lib().orc_num_threads()


def set_threads(n):
    lib().orc_set_threads(int(n))


def box_check(box, rc):
    w = np.zeros(3)
    rcode = lib().orc_box_check(_p(_f(box)), float(rc), _p(w))
    return rcode, w


def delta(box, ri, rj):
    d = np.zeros(3)
    box, ri, rj = _f(box), _f(ri), _f(rj)
    lib().orc_delta(_p(box), _p(ri), _p(rj), _p(d))
    return d


def neighbors(pos, box, rc, maxn, method="cells"):
    """Returns (count[N] int32, list[N,maxn] int32 row-major ascending j, max_count)."""
    pos, box = _f(pos), _f(box)
    N = len(pos)
    count = np.zeros(N, dtype=np.int32)
    lst = np.full((N, maxn), -1, dtype=np.int32)
    fn = {"cells": lib().orc_neighbors_cells, "brute": lib().orc_neighbors_brute,
          "images": lib().orc_neighbors_images}[method]
    mx = fn(N, _p(pos), _p(box), float(rc), int(maxn), _p(count), _p(lst))
    if mx < 0:
        raise ValueError("invalid box / cutoff")
    return count, lst, mx


def switch(x, n, m):
    d = ctypes.c_double(0.0)
    v = lib().orc_switch(float(x), int(n), int(m), ctypes.addressof(d))
    return v, d.value


def make_flags(N, group_a, group_b):
    """bit0 = in A, bit1 = in B; None = all atoms (reading C)."""
    if group_a is None and group_b is None:
        return None
    fl = np.zeros(N, dtype=np.uint8)
    if group_a is None:
        fl |= 1
    else:
        fl[np.asarray(group_a)] |= 1
    if group_b is None:
        fl |= 2
    else:
        fl[np.asarray(group_b)] |= 2
    return fl


def cv_coord(pos, box, count, lst, r0, n, m, scale, flags=None, want_grad=True):
    pos, box = _f(pos), _f(box)
    N = len(pos)
    grad = np.zeros((N, 3)) if want_grad else None
    s = lib().orc_cv_coord(N, _p(pos), _p(box), _p(count), _p(lst), lst.shape[1], _p(flags),
                           float(r0), int(n), int(m), float(scale), _p(grad))
    return s, grad


def q6_atoms(pos, box, count, lst):
    pos, box = _f(pos), _f(box)
    q = np.zeros(len(pos))
    lib().orc_q6_atoms(len(pos), _p(pos), _p(box), _p(count), _p(lst), lst.shape[1], _p(q))
    return q


def q6_grad(pos, box, count, lst, q6, w):
    pos, box, q6, w = _f(pos), _f(box), _f(q6), _f(w)
    g = np.zeros((len(pos), 3))
    lib().orc_q6_grad(len(pos), _p(pos), _p(box), _p(count), _p(lst), lst.shape[1], _p(q6), _p(w), _p(g))
    return g


def y6(u):
    u = _f(u)
    y = np.zeros(14)
    lib().orc_y6(_p(u), _p(y))
    return y[0::2] + 1j * y[1::2]


def q6_atoms_ylm(pos, box, count, lst):
    pos, box = _f(pos), _f(box)
    q = np.zeros(len(pos))
    y = np.zeros((len(pos), 14))
    lib().orc_q6_atoms_ylm(len(pos), _p(pos), _p(box), _p(count), _p(lst), lst.shape[1], _p(q), _p(y))
    return q, y[:, 0::2] + 1j * y[:, 1::2]


def cv_rgyr(pos, box, chain, mass=None, want_grad=True):
    pos, box, chain = _f(pos), _f(box), _i(chain)
    mass = None if mass is None else _f(mass)
    g = np.zeros((len(chain), 3)) if want_grad else None
    rg = lib().orc_cv_rgyr(len(chain), _p(chain), _p(mass), _p(pos), _p(box), _p(g))
    return rg, g


def cv_contacts(pos, box, pairs, pair_r0, n, m, scale, want_grad=True):
    pos, box, pairs, pair_r0 = _f(pos), _f(box), _i(pairs), _f(pair_r0)
    g = np.zeros((len(pos), 3)) if want_grad else None
    q = lib().orc_cv_contacts(len(pos), len(pairs), _p(pairs), _p(pair_r0), int(n), int(m), float(scale),
                              _p(pos), _p(box), _p(g))
    return q, g


def bias(centers, heights, sigma, s):
    centers, heights, sigma, s = _f(centers), _f(heights), _f(sigma), _f(np.atleast_1d(s))
    D = len(sigma)
    H = len(heights)
    centers = centers.reshape(H, D)
    V = ctypes.c_double(0.0)
    dV = np.zeros(D)
    lib().orc_bias(D, H, _p(centers), _p(heights), _p(sigma), _p(s), ctypes.addressof(V), _p(dV))
    return V.value, dV


def wt_height(w0, V, kT, gamma):
    return lib().orc_wt_height(float(w0), float(V), float(kT), float(gamma))


def grid_add(table, lo, hi, centers, heights, sigma, k0=0, k1=None):
    """table: float64 [4,n0,n1], modified in place."""
    lo, hi, centers, heights, sigma = _f(lo), _f(hi), _f(centers), _f(heights), _f(sigma)
    if k1 is None:
        k1 = len(heights)
    assert table.dtype == np.float64 and table.flags.c_contiguous and table.shape[0] == 4
    lib().orc_grid_add(table.shape[1], table.shape[2], _p(lo), _p(hi), int(k0), int(k1), _p(centers),
                       _p(heights), _p(sigma), _p(table))
    return table


def grid_eval(table, lo, hi, s):
    lo, hi, s = _f(lo), _f(hi), _f(s)
    V = ctypes.c_double(0.0)
    dV = np.zeros(2)
    out = lib().orc_grid_eval(table.shape[1], table.shape[2], _p(lo), _p(hi), _p(table), _p(s),
                              ctypes.addressof(V), _p(dV))
    return out, V.value, dV


def apply_forces(F, dVds, grads, force_scale=1.0):
    """F (N,3) float64 modified in place; grads (D,N,3)."""
    grads, dVds = _f(grads), _f(np.atleast_1d(dVds))
    assert F.dtype == np.float64 and F.flags.c_contiguous
    lib().orc_apply_forces(len(F), len(dVds), _p(dVds), _p(grads), float(force_scale), _p(F))
    return F


# ---- NEXT-1: torsion CV, periodic bias (readings V, W, X)
def cv_torsion(pos, box, idx, want_grad=True):
    """phi in (-pi, pi] of atoms idx[0..3]; grad (4,3) = d phi / d r of those four atoms."""
    pos, box, idx = _f(pos), _f(box), _i(idx)
    g = np.zeros((4, 3)) if want_grad else None
    phi = lib().orc_cv_torsion(_p(idx), _p(pos), _p(box), _p(g))
    return phi, g


def pdiff(x, c, period):
    return lib().orc_pdiff(float(x), float(c), float(period))


def wrap(x, lo, period):
    return lib().orc_wrap(float(x), float(lo), float(period))


def bias_periodic(centers, heights, sigma, period, s):
    centers, heights, sigma, period, s = _f(centers), _f(heights), _f(sigma), _f(period), _f(np.atleast_1d(s))
    D, H = len(sigma), len(heights)
    centers = centers.reshape(H, D)
    V = ctypes.c_double(0.0)
    dV = np.zeros(D)
    lib().orc_bias_periodic(D, H, _p(centers), _p(heights), _p(sigma), _p(period), _p(s), ctypes.addressof(V), _p(dV))
    return V.value, dV


def grid_add_p(table, lo, hi, periodic, centers, heights, sigma, k0=0, k1=None):
    lo, hi, centers, heights, sigma, periodic = _f(lo), _f(hi), _f(centers), _f(heights), _f(sigma), _i(periodic)
    if k1 is None:
        k1 = len(heights)
    assert table.dtype == np.float64 and table.flags.c_contiguous and table.shape[0] == 4
    lib().orc_grid_add_p(table.shape[1], table.shape[2], _p(lo), _p(hi), _p(periodic), int(k0), int(k1), _p(centers),
                         _p(heights), _p(sigma), _p(table))
    return table


def grid_eval_p(table, lo, hi, periodic, s):
    lo, hi, s, periodic = _f(lo), _f(hi), _f(s), _i(periodic)
    V = ctypes.c_double(0.0)
    dV = np.zeros(2)
    out = lib().orc_grid_eval_p(table.shape[1], table.shape[2], _p(lo), _p(hi), _p(periodic), _p(table), _p(s),
                                ctypes.addressof(V), _p(dV))
    return out, V.value, dV


# ---- NEXT-2: free-energy reconstruction by reweighting (reading Z)
def reweight(traj, centers, heights, sigma, period, kT, nbins, lo, hi):
    """Returns (P, F), each (nb0, nb1) (nb1 = 1 for a 1-D CV)."""
    sigma = _f(np.atleast_1d(sigma))
    D = len(sigma)
    traj = _f(traj).reshape(-1, D)
    heights = _f(heights)
    centers = _f(centers).reshape(len(heights), D)
    period = _f(np.zeros(D) if period is None else np.atleast_1d(period))
    nb = _i(list(np.atleast_1d(nbins)) + [1] * (2 - D))
    lo2, hi2 = _f(list(np.atleast_1d(lo)) + [0.0] * (2 - D)), _f(list(np.atleast_1d(hi)) + [1.0] * (2 - D))
    P = np.zeros((int(nb[0]), int(nb[1])))
    F = np.zeros_like(P)
    lib().orc_reweight(D, len(traj), _p(traj), len(heights), _p(centers), _p(heights), _p(sigma), _p(period), float(kT),
                       _p(nb), _p(lo2), _p(hi2), _p(P), _p(F))
    return P, F


# ---- NEXT-2b: distance to the nearest atom of a group (reading AA)
def cv_mindist(pos, box, count, lst, rc, flags=None, want_grad=True):
    """Returns (s, grad (N,3) or None, (i, j) of the nearest pair or (-1, -1))."""
    pos, box = _f(pos), _f(box)
    N = len(pos)
    grad = np.zeros((N, 3)) if want_grad else None
    pair = np.zeros(2, dtype=np.int32)
    s = lib().orc_cv_mindist(N, _p(pos), _p(box), _p(count), _p(lst), lst.shape[1], _p(flags), float(rc), _p(grad), _p(pair))
    return s, grad, (int(pair[0]), int(pair[1]))


# ---- NEXT-3: lattice-parameter CV (reading AB)
def cv_lattice(box, axis):
    """Returns (|h_axis|, d s / d box as (3,3))."""
    box = _f(box)
    g = np.zeros(9)
    s = lib().orc_cv_lattice(_p(box), int(axis), _p(g))
    return s, g.reshape(3, 3)


# ---- NEXT-3b: strain derivatives d s / d eps (3,3) for the bias virial (PAPER.md:51 NPT; reading AD)
def cv_coord_strain(pos, box, count, lst, r0, n, m, scale, flags=None):
    pos, box = _f(pos), _f(box)
    out = np.zeros(9)
    lib().orc_cv_coord_strain(len(pos), _p(pos), _p(box), _p(count), _p(lst), lst.shape[1], _p(flags), float(r0), int(n), int(m),
                              float(scale), _p(out))
    return out.reshape(3, 3)


def q6_strain(pos, box, count, lst, q6, w):
    pos, box, q6, w = _f(pos), _f(box), _f(q6), _f(w)
    out = np.zeros(9)
    lib().orc_q6_strain(len(pos), _p(pos), _p(box), _p(count), _p(lst), lst.shape[1], _p(q6), _p(w), _p(out))
    return out.reshape(3, 3)


def cv_lattice_strain(box, axis):
    box = _f(box)
    out = np.zeros(9)
    lib().orc_cv_lattice_strain(_p(box), int(axis), _p(out))
    return out.reshape(3, 3)


def cv_rgyr_strain(pos, box, chain, mass=None):
    pos, box, chain = _f(pos), _f(box), _i(chain)
    mass = None if mass is None else _f(mass)
    out = np.zeros(9)
    lib().orc_cv_rgyr_strain(len(chain), _p(chain), _p(mass), _p(pos), _p(box), _p(out))
    return out.reshape(3, 3)


def cv_contacts_strain(pos, box, pairs, pair_r0, n, m, scale):
    pos, box, pairs, pair_r0 = _f(pos), _f(box), _i(pairs), _f(pair_r0)
    out = np.zeros(9)
    lib().orc_cv_contacts_strain(len(pairs), _p(pairs), _p(pair_r0), int(n), int(m), float(scale), _p(pos), _p(box), _p(out))
    return out.reshape(3, 3)


def cv_mindist_strain(pos, box, count, lst, rc, flags=None):
    pos, box = _f(pos), _f(box)
    out = np.zeros(9)
    lib().orc_cv_mindist_strain(len(pos), _p(pos), _p(box), _p(count), _p(lst), lst.shape[1], _p(flags), float(rc), _p(out))
    return out.reshape(3, 3)


def cv_torsion_strain(pos, box, idx):
    pos, box, idx = _f(pos), _f(box), _i(idx)
    out = np.zeros(9)
    lib().orc_cv_torsion_strain(_p(idx), _p(pos), _p(box), _p(out))
    return out.reshape(3, 3)
