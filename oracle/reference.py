"""Step-level oracle (TEST INFRASTRUCTURE, NOT PRODUCT): composes the primitives of
metad_oracle.c into the per-step order of reading U:
    neighbours -> CVs -> V, dV/ds from the hills deposited so far -> forces -> deposit with that V.
Plain fp64 numpy + the C primitives; no blocking, fusion or reordering.
"""
from __future__ import annotations

import numpy as np

from . import (cv_contacts_strain, cv_coord_strain, cv_lattice_strain, cv_mindist_strain, cv_rgyr_strain,
               cv_torsion_strain, q6_strain, apply_forces, bias, bias_periodic, cv_contacts, cv_coord, cv_lattice, cv_mindist, cv_rgyr, cv_torsion, grid_add, grid_add_p,
               grid_eval, grid_eval_p, make_flags, neighbors, q6_atoms, q6_grad, wt_height)

# CV kinds — restated (not imported) so the oracle depends on nothing of the product.
COORD, Q6_MEAN, Q6_SOLID, RGYR, CONTACTS, TORSION, MINDIST, LATTICE = 0, 1, 2, 3, 4, 5, 6, 7


def logistic(q, q0, width):
    """Solid-like switching on per-atom q6 (BASELINE.json configs[4]; reading F):
    f(q) = 1/(1+exp(-(q-q0)/width)), f' = f(1-f)/width."""
    f = 1.0 / (1.0 + np.exp(-(q - q0) / width))
    return f, f * (1.0 - f) / width


class OracleMetaD:
    def __init__(self, w, neighbor_method="cells"):
        self.w = w
        self.N = w.natoms
        self.D = w.ncv
        self.sigma = np.asarray(w.sigma, dtype=np.float64)
        self.centers = np.zeros((0, self.D))
        self.heights = np.zeros(0)
        self.step = 0
        self.method = neighbor_method
        self.grid = None
        per = getattr(w, "period", None)
        self.period = np.zeros(self.D) if per is None else np.asarray(per, dtype=np.float64)   # reading W
        self.periodic = bool(np.any(self.period > 0))

    # -- a1
    def build_neighbors(self, pos):
        self.pos = np.ascontiguousarray(pos, dtype=np.float64)
        self.count, self.list, self.max_count = neighbors(self.pos, self.w.box, self.w.rc,
                                                          self.w.max_neigh, self.method)
        return self.count, self.list

    # -- a2..a4: CV values and gradients d s_d / d r  (D, N, 3)
    def eval_cv(self, want_grad=True):
        w, pos, box = self.w, self.pos, self.w.box
        s = np.zeros(self.D)
        grads = np.zeros((self.D, self.N, 3)) if want_grad else None
        q6 = None
        box_grads = np.zeros((self.D, 3, 3))          # d s_d / d box (lattice CVs only; reading AB)
        for d, cv in enumerate(w.cvs):
            if cv.kind == COORD:
                fl = make_flags(self.N, cv.group_a, cv.group_b)
                s[d], g = cv_coord(pos, box, self.count, self.list, cv.r0, cv.n, cv.m, cv.scale, fl, want_grad)
            elif cv.kind in (Q6_MEAN, Q6_SOLID):
                if q6 is None:
                    q6 = q6_atoms(pos, box, self.count, self.list)
                    self.q6 = q6
                if cv.kind == Q6_MEAN:
                    s[d] = cv.scale * np.sum(q6)
                    wts = np.full(self.N, cv.scale)
                else:
                    f, df = logistic(q6, cv.q_thresh, cv.q_width)
                    s[d] = cv.scale * np.sum(f)
                    wts = cv.scale * df
                g = q6_grad(pos, box, self.count, self.list, q6, wts) if want_grad else None
            elif cv.kind == RGYR:
                s[d], gc = cv_rgyr(pos, box, cv.chain, None, want_grad)
                g = None
                if want_grad:
                    g = np.zeros((self.N, 3))
                    np.add.at(g, np.asarray(cv.chain), gc)
            elif cv.kind == CONTACTS:
                s[d], g = cv_contacts(pos, box, cv.pairs, cv.pair_r0, cv.n, cv.m, cv.scale, want_grad)
            elif cv.kind == LATTICE:
                s[d], box_grads[d] = cv_lattice(box, cv.n)
                g = np.zeros((self.N, 3)) if want_grad else None
            elif cv.kind == MINDIST:
                fl = make_flags(self.N, cv.group_a, cv.group_b)
                s[d], g, self.min_pair = cv_mindist(pos, box, self.count, self.list, w.rc, fl, want_grad)
            elif cv.kind == TORSION:
                s[d], g4 = cv_torsion(pos, box, cv.atoms, want_grad)
                g = None
                if want_grad:
                    g = np.zeros((self.N, 3))
                    np.add.at(g, np.asarray(cv.atoms), g4)
            else:
                raise ValueError(cv.kind)
            if want_grad:
                grads[d] = g
        self.s, self.grads = s, grads
        self.box_grads = box_grads
        return s

    # -- a5 / a5g
    def set_hills(self, centers, heights):
        self.centers = np.array(centers, dtype=np.float64).reshape(-1, self.D)
        self.heights = np.array(heights, dtype=np.float64)
        if self.grid is not None:
            self.grid["table"][:] = 0.0
            self._grid_add(0, len(self.heights))

    def enable_grid(self, n, lo, hi):
        self.grid = {"lo": np.asarray(lo, float), "hi": np.asarray(hi, float),
                     "table": np.zeros((4, n[0], n[1]))}
        if len(self.heights):
            self._grid_add(0, len(self.heights))

    def _grid_add(self, k0, k1):
        g = self.grid
        if self.periodic:
            grid_add_p(g["table"], g["lo"], g["hi"], (self.period > 0).astype(np.int32), self.centers, self.heights,
                       self.sigma, k0, k1)
        else:
            grid_add(g["table"], g["lo"], g["hi"], self.centers, self.heights, self.sigma, k0, k1)

    def bias(self, s, use_grid=None):
        use_grid = (self.grid is not None) if use_grid is None else use_grid
        if use_grid:
            if self.periodic:
                out, V, dV = grid_eval_p(self.grid["table"], self.grid["lo"], self.grid["hi"],
                                         (self.period > 0).astype(np.int32), s)
            else:
                out, V, dV = grid_eval(self.grid["table"], self.grid["lo"], self.grid["hi"], s)
            if out == 0:
                return V, dV
        if len(self.heights) == 0:
            return 0.0, np.zeros(self.D)
        if self.periodic:
            return bias_periodic(self.centers, self.heights, self.sigma, self.period, s)
        return bias(self.centers, self.heights, self.sigma, s)

    # -- a6
    def forces(self, dVds, F=None, force_scale=1.0):
        if F is None:
            F = np.zeros((self.N, 3))
        return apply_forces(F, dVds, self.grads, force_scale)

    def box_force(self, dVds, force_scale=1.0):
        """F_h = -force_scale * sum_d dVds_d * d s_d / d h  (reading AB)."""
        return -force_scale * np.tensordot(np.atleast_1d(dVds), self.box_grads, axes=1)

    def strain_derivatives(self):
        """d s_d / d eps (D, 3, 3) of the CVs of the last eval_cv (reading AD); NaN for CV kinds without one here."""
        w, pos, box = self.w, self.pos, self.w.box
        out = np.full((self.D, 3, 3), np.nan)
        for d, cv in enumerate(w.cvs):
            if cv.kind == COORD:
                fl = make_flags(self.N, cv.group_a, cv.group_b)
                out[d] = cv_coord_strain(pos, box, self.count, self.list, cv.r0, cv.n, cv.m, cv.scale, fl)
            elif cv.kind == Q6_MEAN:
                out[d] = q6_strain(pos, box, self.count, self.list, self.q6, np.full(self.N, cv.scale))
            elif cv.kind == Q6_SOLID:
                _, df = logistic(self.q6, cv.q_thresh, cv.q_width)
                out[d] = q6_strain(pos, box, self.count, self.list, self.q6, cv.scale * df)
            elif cv.kind == LATTICE:
                out[d] = cv_lattice_strain(box, cv.n)
            elif cv.kind == RGYR:
                out[d] = cv_rgyr_strain(pos, box, cv.chain)
            elif cv.kind == CONTACTS:
                out[d] = cv_contacts_strain(pos, box, cv.pairs, cv.pair_r0, cv.n, cv.m, cv.scale)
            elif cv.kind == MINDIST:
                out[d] = cv_mindist_strain(pos, box, self.count, self.list, w.rc, make_flags(self.N, cv.group_a, cv.group_b))
            elif cv.kind == TORSION:
                out[d] = cv_torsion_strain(pos, box, cv.atoms)
        return out

    def virial(self, dVds, force_scale=1.0):
        """W = -force_scale * sum_d dVds_d * d s_d / d eps (reading AD)."""
        return -force_scale * np.tensordot(np.atleast_1d(dVds), self.strain_derivatives(), axes=1)

    # -- a7 (readings I, J, U): every `stride` steps append (s, w0*exp(-V/((gamma-1)kT)))
    def deposit(self, s, V):
        w = self.w
        self.step += 1
        if w.stride > 0 and self.step % w.stride == 0:
            h = wt_height(w.w0, V, w.kT, w.bias_factor)
            self.centers = np.concatenate([self.centers, np.asarray(s, float).reshape(1, self.D)])
            self.heights = np.append(self.heights, h)
            if self.grid is not None:
                k = len(self.heights)
                self._grid_add(k - 1, k)
            return h
        return None

    def run_step(self, pos, F):
        self.build_neighbors(pos)
        s = self.eval_cv()
        V, dV = self.bias(s)
        self.forces(dV, F)
        self.deposit(s, V)
        return s, V, dV


def replay_heights(centers, sigma, w0, kT, gamma):
    """Well-tempered heights along a scripted centre path (reading K): hill k gets
    w0*exp(-V_{k-1}(s_k)/((gamma-1)kT)) with V_{k-1} the bias of hills 0..k-1."""
    centers = np.asarray(centers, dtype=np.float64)
    H, D = centers.shape
    heights = np.zeros(H)
    for k in range(H):
        V = bias(centers[:k], heights[:k], sigma, centers[k])[0] if k else 0.0
        heights[k] = wt_height(w0, V, kT, gamma)
    return heights
