"""Seeded synthetic Ni-cluster inputs (BASELINE.json configs C1..C5).

This module is the ONE piece of code the CPU oracle's tests and the CUDA path's
tests/bench share.  It holds none of the method's arithmetic (no Sutton-Chen
density, energy, force or integrator): it only lays atoms out in space and draws
Maxwell-Boltzmann velocities.  The paper uses no public dataset; its workloads
are free Ni clusters ("initial geometry ... icosahedral symmetry",
benchmark sizes up to >1e4 atoms PAPER.md:139).  BASELINE.json's five configs
stand in for them; the recipes below are the readings Q12..Q16 of SURVEY.md
section 8(c)/(d), restated in DESIGN.md.

All randomness is numpy ``default_rng(seed)`` (PCG64); draw order is part of the
definition: positions first (jitter / rejection candidates), then velocities.
"""
from __future__ import annotations

import math
from dataclasses import dataclass

import numpy as np

# Units: Angstrom, fs, eV, u, K.  Generator-side literals (the oracle and the
# CUDA library carry their own copies; nothing is imported across).
_KB_EV_PER_K = 8.617333262e-5          # CODATA-2018
_ACC = 9.648533215665e-3               # (eV/A/u) -> A/fs^2
NI_MASS_U = 58.69                      # BASELINE.json configs[0]
NI_A_FCC = 3.52                        # PAPER.md:71 (a = 3.52 A)

# Sutton-Chen Ni parameters.
NI_PARAMS = dict(n=9, m=6, eps=1.5707e-2, c=39.432, a=3.52, mass=NI_MASS_U)


@dataclass
class Workload:
    name: str
    pos: np.ndarray          # (N, 3) float64, Angstrom
    vel: np.ndarray          # (N, 3) float64, Angstrom/fs
    temperature: float       # K, the Maxwell-Boltzmann draw temperature
    seed: int

    @property
    def n_atoms(self) -> int:
        return int(self.pos.shape[0])


# --------------------------------------------------------------------------- #
# velocities
# --------------------------------------------------------------------------- #
def maxwell_boltzmann(rng: np.random.Generator, n_atoms: int, temperature: float,
                      mass: float = NI_MASS_U) -> np.ndarray:
    """Each component N(0, sigma_v^2), sigma_v = sqrt(kB T ACC / m) A/fs; then the
    mean velocity is subtracted (COM momentum removed).  No rescale to exact T
    (reading Q15)."""
    sigma_v = math.sqrt(_KB_EV_PER_K * temperature * _ACC / mass)
    v = rng.standard_normal((n_atoms, 3)) * sigma_v
    if n_atoms > 0:
        v -= v.mean(axis=0, keepdims=True)
    return np.ascontiguousarray(v)


# --------------------------------------------------------------------------- #
# C1: Mackay icosahedron
# --------------------------------------------------------------------------- #
def _icosahedron_axes() -> np.ndarray:
    phi = (1.0 + math.sqrt(5.0)) / 2.0
    norm = math.sqrt(1.0 + phi * phi)
    verts = []
    for s1 in (1.0, -1.0):
        for s2 in (1.0, -1.0):
            base = (0.0, s1 * 1.0, s2 * phi)
            for rot in range(3):                       # cyclic permutations
                verts.append(tuple(base[(k - rot) % 3] for k in range(3)))
    v = np.array(verts, dtype=np.float64) / norm
    assert v.shape == (12, 3)
    return v


def mackay_icosahedron(n_shells: int, d: float = 2.49) -> np.ndarray:
    """Mackay icosahedron with ``n_shells`` shells around a central atom; radial
    inter-shell spacing ``d`` (centre -> first-shell vertex), reading Q12.
    Shell s holds 10 s^2 + 2 atoms: points d*(i A + j B + l C), i+j+l = s, over the
    20 triangular faces (A, B, C unit vertex vectors), de-duplicated at 1e-6 A.
    Canonical order: by shell, then by (x, y, z) rounded to 1e-6."""
    axes = _icosahedron_axes()
    edge = 2.0 / math.sqrt(1.0 + ((1.0 + math.sqrt(5.0)) / 2.0) ** 2)   # 1.0514622...
    faces = []
    for p in range(12):
        for q in range(p + 1, 12):
            for r in range(q + 1, 12):
                dpq = np.linalg.norm(axes[p] - axes[q])
                dpr = np.linalg.norm(axes[p] - axes[r])
                dqr = np.linalg.norm(axes[q] - axes[r])
                if max(abs(dpq - edge), abs(dpr - edge), abs(dqr - edge)) < 1e-9:
                    faces.append((p, q, r))
    assert len(faces) == 20
    shells = [np.zeros((1, 3))]
    for s in range(1, n_shells + 1):
        seen = {}
        for (p, q, r) in faces:
            for i in range(s + 1):
                for j in range(s + 1 - i):
                    l = s - i - j
                    pt = d * (i * axes[p] + j * axes[q] + l * axes[r])
                    key = tuple(np.round(pt / 1e-6).astype(np.int64).tolist())
                    seen.setdefault(key, pt)
        keys = sorted(seen.keys())
        assert len(keys) == 10 * s * s + 2, (s, len(keys))
        shells.append(np.array([seen[k] for k in keys]))
    return np.ascontiguousarray(np.concatenate(shells, axis=0))


# --------------------------------------------------------------------------- #
# C2, C4, C5: fcc N-nearest sites
# --------------------------------------------------------------------------- #
def fcc_half_lattice_indices(n_atoms: int) -> np.ndarray:
    """The ``n_atoms`` fcc sites nearest the origin (cluster centred on an atom),
    as half-lattice integers (i, j, k) with i + j + k even; ties broken by the key
    (q = i^2 + j^2 + k^2, i, j, k) ascending (reading Q13)."""
    if n_atoms <= 0:
        return np.zeros((0, 3), dtype=np.int64)
    # sites in a sphere of half-lattice radius R: ~ (4/3) pi R^3 / 2
    r = (2.0 * n_atoms * 3.0 / (4.0 * math.pi)) ** (1.0 / 3.0)
    lim = int(math.ceil(r)) + 3
    while True:
        ax = np.arange(-lim, lim + 1, dtype=np.int64)
        i, j, k = np.meshgrid(ax, ax, ax, indexing="ij")
        i = i.ravel(); j = j.ravel(); k = k.ravel()
        keep = ((i + j + k) & 1) == 0
        i, j, k = i[keep], j[keep], k[keep]
        q = i * i + j * j + k * k
        inside = q <= lim * lim            # only complete shells are trustworthy
        i, j, k, q = i[inside], j[inside], k[inside], q[inside]
        if i.size >= n_atoms:
            break
        lim += 4
    order = np.lexsort((k, j, i, q))       # primary key last
    order = order[:n_atoms]
    return np.stack([i[order], j[order], k[order]], axis=1)


def fcc_sphere(n_atoms: int, a_fcc: float = NI_A_FCC) -> np.ndarray:
    """Unjittered fcc N-nearest-site cluster, positions (a/2) * (i, j, k)."""
    return np.ascontiguousarray(fcc_half_lattice_indices(n_atoms).astype(np.float64) * (0.5 * a_fcc))


def fcc_cluster(n_atoms: int, temperature: float, seed: int, jitter: float = 0.05,
                name: str | None = None) -> Workload:
    """fcc N-nearest sites + uniform(-jitter, +jitter) per coordinate, then
    Maxwell-Boltzmann velocities (drawn after the jitter), readings Q13/Q14."""
    rng = np.random.default_rng(seed)
    pos = fcc_sphere(n_atoms)
    if jitter > 0.0:
        pos = pos + rng.uniform(-jitter, jitter, size=(n_atoms, 3))
    vel = maxwell_boltzmann(rng, n_atoms, temperature)
    return Workload(name or f"Ni{n_atoms}-fcc", np.ascontiguousarray(pos), vel, temperature, seed)


# --------------------------------------------------------------------------- #
# C3: liquid droplet
# --------------------------------------------------------------------------- #
def liquid_droplet_positions(rng: np.random.Generator, n_atoms: int, density: float = 0.080,
                             min_sep: float = 1.8, batch: int = 4096) -> np.ndarray:
    """Seeded sequential rejection (reading Q16): candidates uniform in the cube
    [-R, R]^3, R = (3N / (4 pi density))^(1/3); a candidate is kept iff |p| <= R and
    it is >= min_sep from every atom kept so far.  Candidates are drawn in batches
    of ``batch`` (rng.uniform(-R, R, (batch, 3))) and consumed in order."""
    radius = (3.0 * n_atoms / (4.0 * math.pi * density)) ** (1.0 / 3.0)
    cell = min_sep
    ncell = int(math.ceil(2.0 * radius / cell)) + 2
    grid: dict[tuple[int, int, int], list[int]] = {}
    kept = np.empty((n_atoms, 3), dtype=np.float64)
    n_kept = 0
    min_sep2 = min_sep * min_sep
    r2max = radius * radius
    while n_kept < n_atoms:
        cand = rng.uniform(-radius, radius, size=(batch, 3))
        for p in cand:
            if p[0] * p[0] + p[1] * p[1] + p[2] * p[2] > r2max:
                continue
            cx = int((p[0] + radius) // cell) + 1
            cy = int((p[1] + radius) // cell) + 1
            cz = int((p[2] + radius) // cell) + 1
            ok = True
            for ax in (cx - 1, cx, cx + 1):
                for ay in (cy - 1, cy, cy + 1):
                    for az in (cz - 1, cz, cz + 1):
                        for idx in grid.get((ax, ay, az), ()):
                            q = kept[idx]
                            d0 = p[0] - q[0]; d1 = p[1] - q[1]; d2 = p[2] - q[2]
                            if d0 * d0 + d1 * d1 + d2 * d2 < min_sep2:
                                ok = False
                                break
                        if not ok:
                            break
                    if not ok:
                        break
                if not ok:
                    break
            if not ok:
                continue
            kept[n_kept] = p
            grid.setdefault((cx, cy, cz), []).append(n_kept)
            n_kept += 1
            if n_kept == n_atoms:
                break
    assert ncell > 0
    return kept


def liquid_droplet(n_atoms: int = 8000, temperature: float = 2000.0, seed: int = 3001) -> Workload:
    rng = np.random.default_rng(seed)
    pos = liquid_droplet_positions(rng, n_atoms)
    vel = maxwell_boltzmann(rng, n_atoms, temperature)
    return Workload(f"Ni{n_atoms}-liquid", pos, vel, temperature, seed)


# --------------------------------------------------------------------------- #
# the five BASELINE.json configs
# --------------------------------------------------------------------------- #
def config_c1(seed: int = 1001) -> Workload:
    """C1: Ni147 Mackay icosahedron, 1000 K."""
    rng = np.random.default_rng(seed)
    pos = mackay_icosahedron(3, 2.49)
    vel = maxwell_boltzmann(rng, pos.shape[0], 1000.0)
    return Workload("Ni147-mackay", pos, vel, 1000.0, seed)


def mackay_cluster(n_shells: int, temperature: float, seed: int) -> Workload:
    """Mackay icosahedron with n_shells shells (10 s^2 + 2 atoms per shell: 147, 309, 561, 923, 1415, 2057
    atoms for 3..8 shells), Maxwell-Boltzmann velocities.  8 shells = the paper's Ni2057."""
    rng = np.random.default_rng(seed)
    pos = mackay_icosahedron(n_shells, 2.49)
    vel = maxwell_boltzmann(rng, pos.shape[0], temperature)
    return Workload(f"Ni{pos.shape[0]}-mackay", pos, vel, temperature, seed)


def config_c2(seed: int = 2001) -> Workload:
    """C2: Ni1415 fcc N-nearest sites, jitter +-0.05 A, 2000 K."""
    return fcc_cluster(1415, 2000.0, seed, name="Ni1415-fcc")


def config_c3(seed: int = 3001, n_atoms: int = 8000) -> Workload:
    """C3: Ni8000 liquid droplet, 2000 K."""
    return liquid_droplet(n_atoms, 2000.0, seed)


def config_c4(seed: int = 4001, n_atoms: int = 65536) -> Workload:
    """C4: Ni65536 fcc cluster, 1200 K."""
    return fcc_cluster(n_atoms, 1200.0, seed, name=f"Ni{n_atoms}-fcc")


def config_c5(k: int) -> Workload:
    """C5 sweep member: N = 4^k (k = 5..10), 1500 K, seed 5000 + k."""
    n_atoms = 4 ** k
    return fcc_cluster(n_atoms, 1500.0, 5000 + k, name=f"Ni{n_atoms}-fcc-sweep")
