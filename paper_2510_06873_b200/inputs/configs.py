"""Builders for the five BASELINE.json workloads (and scaled-down variants for quick tests).

Recipes: SURVEY.md §8(d) / DESIGN.md "Input recipe".  No method arithmetic here.
"""
from __future__ import annotations

import numpy as np

from . import (BASE_SEED, CV_LATTICE, CV_MINDIST, CV_COORD, CV_Q6_MEAN, CV_Q6_SOLID, CV_RGYR, CV_CONTACTS, CV_TORSION, CVSpec, Workload,
               hill_walk_periodic, rsa, wrap)


def _cubic(L):
    return np.array([L, 0, 0, 0, L, 0, 0, 0, L], dtype=np.float64)


# ----------------------------------------------------------------------------------------- c0
def config0(seed=BASE_SEED + 0, shifted=False, n_side=8, a=2.5):
    """512 atoms, 8x8x8 simple cubic a=2.5 in L=20, Gaussian jitter 0.1; mean coordination number,
    r0=3, n=6, m=12, rc=6; 200 hills U[0,8], height 1, width 0.05 (BASELINE.json configs[0]).
    shifted=True is the supplementary c0' of SURVEY §8(c)-D: same seeded centres moved by +5 so
    that they cover the actual CV value (~9.45) and V = O(1)."""
    rng = np.random.default_rng(seed)
    L = n_side * a
    g = np.arange(n_side) * a
    pos = np.stack(np.meshgrid(g, g, g, indexing="ij"), axis=-1).reshape(-1, 3).astype(np.float64)
    pos = pos + rng.standard_normal(pos.shape) * 0.1
    box = _cubic(L)
    pos = wrap(pos, box)
    centers = rng.random((200, 1)) * 8.0
    if shifted:
        centers = centers + 5.0
    N = len(pos)
    cv = CVSpec(kind=CV_COORD, r0=3.0, n=6, m=12, scale=1.0 / N)
    return Workload(name="c0'" if shifted else "c0", pos=pos, box=box, rc=6.0, max_neigh=96, cvs=[cv],
                    sigma=[0.05], n_hills=200, w0=1.0, bias_factor=1.0, stride=0, precision=64,
                    hill_centers=centers, hill_heights=np.ones(200))


# ----------------------------------------------------------------------------------------- c1
def _random_unit(rng):
    v = rng.standard_normal(3)
    return v / np.linalg.norm(v)


def _chain_walk(rng, n, step, excl, start):
    """Self-avoiding walk: fixed step length, reject a trial if closer than excl to any chain atom
    >= 3 bonds away; after 1000 failed trials back up 10 atoms."""
    pts = np.empty((n, 3))
    pts[0] = start
    k = 1
    fails = 0
    while k < n:
        trial = pts[k - 1] + step * _random_unit(rng)
        ok = True
        if k >= 3:
            d2 = np.sum((pts[:k - 2] - trial) ** 2, axis=1)
            ok = bool(np.all(d2 >= excl * excl))
        if ok:
            pts[k] = trial
            k += 1
            fails = 0
        else:
            fails += 1
            if fails >= 1000:
                k = max(1, k - 10)
                fails = 0
    return pts


def config1(seed=BASE_SEED + 1, natoms=20000, nchain=1000, npairs=5000, n_hills=5000):
    """Chain (seeded self-avoiding walk, 1.5 A steps, 3 A excluded volume) + uniform random solvent
    at 0.1 atoms/A^3; CVs = radius of gyration and native-contact fraction (BASELINE.json configs[1])."""
    rng = np.random.default_rng(seed)
    L = (natoms / 0.1) ** (1.0 / 3.0)
    box = _cubic(L)
    chain_xyz = _chain_walk(rng, nchain, 1.5, 3.0, np.full(3, 0.5 * L))
    solvent = rng.random((natoms - nchain, 3)) * L
    # contact pairs: j-i >= 3, initial (unwrapped) distance < cap; raise cap by 1 A until enough
    ii, jj = np.triu_indices(nchain, k=3)
    dist = np.linalg.norm(chain_xyz[ii] - chain_xyz[jj], axis=1)
    cap = 12.0
    while np.count_nonzero(dist < cap) < npairs:
        cap += 1.0
    cand = np.flatnonzero(dist < cap)
    pick = np.sort(rng.choice(cand, size=npairs, replace=False))
    pairs = np.stack([ii[pick], jj[pick]], axis=1).astype(np.int32)
    ref = dist[pick]
    pos = wrap(np.concatenate([chain_xyz, solvent]), box)
    chain = np.arange(nchain, dtype=np.int32)
    cvs = [CVSpec(kind=CV_RGYR, chain=chain),
           CVSpec(kind=CV_CONTACTS, n=6, m=12, pairs=pairs, pair_r0=1.5 * ref, scale=1.0 / npairs)]
    return Workload(name="c1", pos=pos, box=box, rc=6.0, max_neigh=160, cvs=cvs, sigma=[0.2, 0.02],
                    n_hills=n_hills, w0=1.0, bias_factor=10.0, stride=10, precision=64,
                    extra={"pair_ref": ref, "contact_cap": cap})


# ----------------------------------------------------------------------------------------- c2
def config2(seed=BASE_SEED + 2, ncell=40, n_water=20533, n_hills=20000):
    """Rocksalt slab (a=4.2, 6 layers) + water-like O,H,H layer + vacuum; CV = coordination count
    between top-layer slab anions and all H (r0=1.2, n=6, m=12, rc=3) (BASELINE.json configs[2]).
    ncell=40 gives 38,400 slab atoms + 3*20,533 = 99,999 atoms (100,000 is not reachable with whole
    molecules)."""
    rng = np.random.default_rng(seed)
    a = 4.2
    h = a / 2
    nx = 2 * ncell
    Lxy = ncell * a
    z0 = 1.0
    ix, iy, iz = np.meshgrid(np.arange(nx), np.arange(nx), np.arange(6), indexing="ij")
    slab = np.stack([ix * h, iy * h, z0 + iz * h], axis=-1).reshape(-1, 3).astype(np.float64)
    slab_species = ((ix + iy + iz) % 2).reshape(-1).astype(np.int32)      # 0 cation, 1 anion
    top = (iz.reshape(-1) == 5)
    z_top = z0 + 5 * h
    w_lo, w_hi = z_top + 2.0, z_top + 2.0 + 22.05
    Lz = w_hi + 15.0
    box = np.array([Lxy, 0, 0, 0, Lxy, 0, 0, 0, Lz], dtype=np.float64)
    O = rsa(n_water, box, 2.5, seed, periodic=(1, 1, 0), flo=(0, 0, w_lo / Lz), fhi=(1, 1, w_hi / Lz))
    # H positions: O-H 0.96 A, H-O-H 104.5 deg, random orientation
    u = rng.standard_normal((n_water, 3))
    u /= np.linalg.norm(u, axis=1, keepdims=True)
    v = rng.standard_normal((n_water, 3))
    v -= np.sum(v * u, axis=1, keepdims=True) * u
    v /= np.linalg.norm(v, axis=1, keepdims=True)
    half = np.deg2rad(104.5) / 2
    H1 = O + 0.96 * (np.cos(half) * u + np.sin(half) * v)
    H2 = O + 0.96 * (np.cos(half) * u - np.sin(half) * v)
    water = np.stack([O, H1, H2], axis=1).reshape(-1, 3)
    water_species = np.tile(np.array([2, 3, 3], dtype=np.int32), n_water)
    pos = wrap(np.concatenate([slab, water]), box)
    species = np.concatenate([slab_species, water_species])
    group_a = np.flatnonzero(np.concatenate([top & (slab_species == 1), np.zeros(3 * n_water, bool)])).astype(np.int32)
    group_b = np.flatnonzero(species == 3).astype(np.int32)
    cv = CVSpec(kind=CV_COORD, r0=1.2, n=6, m=12, scale=1.0, group_a=group_a, group_b=group_b)
    return Workload(name="c2", pos=pos, box=box, rc=3.0, max_neigh=48, cvs=[cv], sigma=[0.5],
                    n_hills=n_hills, w0=1.0, bias_factor=1.0, stride=10, precision=64, species=species)


# ------------------------------------------------------------------------------------ c3 / c4
def wurtzite(ncx, ncy, ncz, a=3.19, c=5.19, u=0.377):
    """Primitive hexagonal wurtzite cells (4 atoms) -> positions, species (0 Ga, 1 N), triclinic box."""
    box = np.array([ncx * a, 0, 0, -0.5 * ncy * a, 0.5 * np.sqrt(3.0) * ncy * a, 0, 0, 0, ncz * c])
    basis = np.array([[1 / 3, 2 / 3, 0.0], [2 / 3, 1 / 3, 0.5], [1 / 3, 2 / 3, u], [2 / 3, 1 / 3, 0.5 + u]])
    sp = np.array([0, 0, 1, 1], dtype=np.int32)
    i, j, k = np.meshgrid(np.arange(ncx), np.arange(ncy), np.arange(ncz), indexing="ij")
    cell = np.stack([i, j, k], axis=-1).reshape(-1, 1, 3).astype(np.float64)
    frac = (cell + basis[None]) / np.array([ncx, ncy, ncz], dtype=np.float64)
    frac = frac.reshape(-1, 3)
    species = np.tile(sp, ncx * ncy * ncz)
    pos = frac @ box.reshape(3, 3)
    return pos, species, box


def gan_nucleus(ncx, ncy, ncz, sphere_r, seed, min_sep=1.8):
    """Wurtzite crystal; every atom outside a central sphere is replaced by a seeded random
    position (RSA, min separation 1.8 A) at the same density (BASELINE.json configs[3],[4])."""
    pos, species, box = wurtzite(ncx, ncy, ncz)
    B = box.reshape(3, 3)
    centre = 0.5 * (B[0] + B[1] + B[2])
    inside = np.sum((pos - centre) ** 2, axis=1) < sphere_r * sphere_r
    crystal = pos[inside]
    n_liq = int(np.count_nonzero(~inside))
    liquid = rsa(n_liq, box, min_sep, seed, existing=wrap(crystal, box), sphere_center=centre,
                 sphere_r=sphere_r)
    allpos = np.concatenate([crystal, liquid])
    allsp = np.concatenate([species[inside], species[~inside]])
    # shuffle so that the input order is not already spatially sorted (an MD code's order is arbitrary)
    perm = np.random.default_rng(seed + 1).permutation(len(allpos))
    return wrap(allpos[perm], box), allsp[perm], box


def config3(seed=BASE_SEED + 3, cells=(80, 80, 40), sphere_r=30.0, n_hills=10000, precision=64):
    """GaN-shaped nucleation, 1,024,000 atoms; CV = global mean Steinhardt Q6, rc=3.6;
    10,000 well-tempered hills, width 0.005, bias factor 20 (BASELINE.json configs[3])."""
    pos, species, box = gan_nucleus(*cells, sphere_r, seed)
    N = len(pos)
    cv = CVSpec(kind=CV_Q6_MEAN, scale=1.0 / N)
    return Workload(name="c3", pos=pos, box=box, rc=3.6, max_neigh=32, cvs=[cv], sigma=[0.005],
                    n_hills=n_hills, w0=1.0, bias_factor=20.0, stride=10, precision=precision,
                    species=species)


def config4(seed=BASE_SEED + 4, cells=(160, 160, 40), sphere_r=50.0, n_hills=100000, grid=(512, 512)):
    """4,096,000-atom GaN-shaped system; CVs = mean Q6 and solid-like count (logistic on per-atom q6,
    threshold 0.35, width 0.05); 100,000 hills; 512x512 grid; fp32 pair math (BASELINE.json configs[4])."""
    pos, species, box = gan_nucleus(*cells, sphere_r, seed)
    N = len(pos)
    cvs = [CVSpec(kind=CV_Q6_MEAN, scale=1.0 / N),
           CVSpec(kind=CV_Q6_SOLID, scale=1.0, q_thresh=0.35, q_width=0.05)]
    return Workload(name="c4", pos=pos, box=box, rc=3.6, max_neigh=32, cvs=cvs, sigma=[0.005, 500.0],
                    n_hills=n_hills, w0=1.0, bias_factor=20.0, stride=10, precision=32, grid_n=grid,
                    species=species)


# ----------------------------------------------------------------------------------------- t0
def config_t0(seed=BASE_SEED + 10, natoms=22, n_hills=20000, grid=(256, 256), n_solvent=0):
    """Alanine-dipeptide-shaped torsion workload (Phi(C-N-Ca-C), Psi(N-Ca-C-N), sigma = 0.35 rad,
    W = 1.2 kJ/mol, plain metadynamics; reading Y): a 22-atom chain (seeded self-avoiding walk, 1.5 A bonds,
    2.2 A exclusion) centred in a cubic box L = 30 A (optionally plus uniform solvent atoms); Phi = atoms 4-6-8-14,
    Psi = 6-8-14-16 (the usual 0-based backbone indices of the 22-atom molecule); hill centres = seeded walk on the
    torus [-pi, pi)^2 started at the structure's own (Phi, Psi) (reading K), seeded heights; 256 x 256 periodic grid."""
    rng = np.random.default_rng(seed)
    L = 30.0
    box = _cubic(L)
    chain = _chain_walk(rng, natoms, 1.5, 2.2, np.full(3, 0.5 * L))
    solvent = rng.random((n_solvent, 3)) * L
    pos = wrap(np.concatenate([chain, solvent]), box)
    cvs = [CVSpec(kind=CV_TORSION, atoms=np.array([4, 6, 8, 14], dtype=np.int32)),
           CVSpec(kind=CV_TORSION, atoms=np.array([6, 8, 14, 16], dtype=np.int32))]
    sigma = [0.35, 0.35]
    P = 2.0 * np.pi
    return Workload(name="t0", pos=pos, box=box, rc=6.0, max_neigh=64, cvs=cvs, sigma=sigma, n_hills=n_hills, w0=1.2,
                    bias_factor=1.0, stride=10, precision=64, grid_n=tuple(grid), period=[P, P],
                    extra={"period_lo": [-np.pi, -np.pi]})


# ----------------------------------------------------------------------------------------- r0
def config_r0(seed=BASE_SEED + 2, ncell=40, n_water=20533, n_hills=20000):
    """The CV of the paper's second workload ("the distance between a surface oxygen atom and its nearest
    hydrogen atom", well-tempered metadynamics) on the slab + water structure of BASELINE.json configs[2] (same seed, same
    atoms): 1-D CV = distance from ONE top-layer anion (the middle one of group A) to its nearest H within rc = 5 A (the
    water layer starts 2 A above the slab, so 3 A does not always reach a hydrogen); bias factor 10, width 0.05 A,
    20,000 hills."""
    w = config2(seed=seed, ncell=ncell, n_water=n_water, n_hills=n_hills)
    cv = w.cvs[0]
    A = np.asarray(cv.group_a)
    w.name = "r0"
    w.cvs = [CVSpec(kind=CV_MINDIST, group_a=A[len(A) // 2:len(A) // 2 + 1], group_b=cv.group_b)]
    w.sigma = [0.05]
    w.bias_factor = 10.0
    w.rc = 5.0
    w.max_neigh = 128
    return w


# ----------------------------------------------------------------------------------------- g0
def config_g0(seed=BASE_SEED + 3, cells=(80, 80, 40), sphere_r=30.0, n_hills=10000):
    """The CV set of the paper's own GaN runs ("the coordination number (C.N.) and the triaxial lattice
    parameters as CVs") on the GaN-shaped structure of BASELINE.json configs[3] (same seed, same atoms): 4-D CV =
    mean coordination number (r0 = 2.4 A between the first and second wurtzite shells, n = 6, m = 12, rc = 3.6 A) and
    the lengths of the three box rows; well-tempered, bias factor 20; widths (0.02, 0.1, 0.1, 0.1)."""
    w = config3(seed=seed, cells=cells, sphere_r=sphere_r, n_hills=n_hills)
    w.name = "g0"
    w.cvs = [CVSpec(kind=CV_COORD, r0=2.4, n=6, m=12, scale=1.0 / w.natoms),
             CVSpec(kind=CV_LATTICE, n=0), CVSpec(kind=CV_LATTICE, n=1), CVSpec(kind=CV_LATTICE, n=2)]
    w.sigma = [0.02, 0.1, 0.1, 0.1]
    return w


def small(name):
    """Scaled-down variants with the same structure, for the CPU suite and quick GPU parity."""
    if name == "c1":
        return config1(natoms=4000, nchain=200, npairs=600, n_hills=300)
    if name == "c2":
        return config2(ncell=8, n_water=800, n_hills=500)
    if name == "c3":
        return config3(cells=(12, 12, 8), sphere_r=9.0, n_hills=400)
    if name == "c4":
        w = config4(cells=(14, 12, 8), sphere_r=10.0, n_hills=600, grid=(64, 64))
        w.sigma = [0.005, 20.0]
        return w
    if name == "c0":
        return config0()
    if name == "t0":
        return config_t0(n_hills=500, grid=(48, 40))
    if name == "g0":
        return config_g0(cells=(12, 12, 8), sphere_r=9.0, n_hills=400)
    if name == "r0":
        return config_r0(ncell=8, n_water=800, n_hills=500)
    raise KeyError(name)


BUILDERS = {"c0": config0, "c1": config1, "c2": config2, "c3": config3, "c4": config4, "t0": config_t0, "g0": config_g0, "r0": config_r0}
