"""Pins for oracle/sc_oracle.c against things other than itself (all CPU, -m "not gpu").

Each test says which pin of SURVEY.md section 8(c) it implements and what mistake in
the oracle it would catch.  Equations: PAPER.md:65 (Eq. 1), PAPER.md:69 (Eq. 2),
parameters PAPER.md:71, two sweeps PAPER.md:127, Verlet dt = 1 fs PAPER.md:145.
"""
import json
import math
from pathlib import Path

import mpmath as mp
import numpy as np
import pytest

from paper_1210_3559_b200 import workloads as W

GOLD = json.loads((Path(__file__).parent / "golden" / "survey_pins.json").read_text())
EPS, C, A, N_EXP, M_EXP, MASS = 1.5707e-2, 39.432, 3.52, 9, 6, 58.69


def rel(a, b):
    return abs(a - b) / max(abs(b), 1e-300)


def rel_l2(a, b):
    return float(np.linalg.norm(np.asarray(a) - np.asarray(b)) / max(np.linalg.norm(b), 1e-300))


# --------------------------------------------------------------------------- #
# independent brute force in mpmath (50 digits): Eq. (1)-(2) typed from the paper,
# forces by high-precision numerical differentiation (no force formula involved)
# --------------------------------------------------------------------------- #
def mp_energy(pos, n=N_EXP, m=M_EXP, eps=EPS, c=C, a=A, r_cut=None):
    mp.mp.dps = 50
    N = len(pos)
    total = mp.mpf(0)
    for i in range(N):
        pair = mp.mpf(0)
        rho = mp.mpf(0)
        for j in range(N):
            if j == i:
                continue
            r = mp.sqrt(sum((mp.mpf(pos[i][k]) - mp.mpf(pos[j][k])) ** 2 for k in range(3)))
            if r_cut is not None and not (r < r_cut):
                continue
            pair += (mp.mpf(a) / r) ** n
            rho += (mp.mpf(a) / r) ** m
        total += pair / 2 - mp.mpf(c) * mp.sqrt(rho)
    return mp.mpf(eps) * total


def mp_forces(pos, **kw):
    mp.mp.dps = 50
    pos = [[mp.mpf(float(x)) for x in p] for p in pos]
    N = len(pos)
    F = np.zeros((N, 3))
    h = mp.mpf(10) ** -20
    for i in range(N):
        for k in range(3):
            p1 = [row[:] for row in pos]; p1[i][k] += h
            p2 = [row[:] for row in pos]; p2[i][k] -= h
            F[i, k] = float(-(mp_energy(p1, **kw) - mp_energy(p2, **kw)) / (2 * h))
    return F


def test_bruteforce_mpmath_energy_and_forces(oracle_ld):
    """Brute force on tiny inputs: catches a dropped term, wrong sign or index, or a missing
    rho_j contribution in the force (the 'implicit many-body' term)."""
    rng = np.random.default_rng(7)
    pos = rng.uniform(-2.5, 2.5, (5, 3))
    # keep atoms apart so that no term dominates
    pos += 1.3 * np.arange(5)[:, None] * np.array([1.0, 0.3, -0.2])
    P = oracle_ld.params()
    rho, F, (U, Up, Ue) = oracle_ld.energy_forces(pos, P)
    U_mp = float(mp_energy(pos.tolist()))
    assert rel(U, U_mp) < 1e-15
    assert abs((Up + Ue) - U) < 1e-15 * abs(U)
    F_mp = mp_forces(pos.tolist())
    assert rel_l2(F, F_mp) < 1e-14


def test_bruteforce_mpmath_other_exponents_and_cutoff(oracle_ld):
    """Generic integer (n, m) and the strict cutoff, against mpmath."""
    rng = np.random.default_rng(11)
    pos = rng.uniform(0, 6.0, (6, 3))
    for (n, m) in ((12, 6), (10, 8), (7, 3)):
        P = oracle_ld.params(n=n, m=m, eps=0.02, c=30.0, a=3.0)
        _, F, (U, _, _) = oracle_ld.energy_forces(pos, P)
        assert rel(U, float(mp_energy(pos.tolist(), n=n, m=m, eps=0.02, c=30.0, a=3.0))) < 1e-14
        assert rel_l2(F, mp_forces(pos.tolist(), n=n, m=m, eps=0.02, c=30.0, a=3.0)) < 1e-13
    P = oracle_ld.params(r_cut=4.0)
    _, F, (U, _, _) = oracle_ld.energy_forces(pos, P)
    assert rel(U, float(mp_energy(pos.tolist(), r_cut=4.0))) < 1e-14
    # away from the cutoff discontinuity the force is still minus the gradient
    assert rel_l2(F, mp_forces(pos.tolist(), r_cut=4.0)) < 1e-13


# --------------------------------------------------------------------------- #
# P1: dimer closed form
# --------------------------------------------------------------------------- #
def dimer_closed(r):
    mp.mp.dps = 40
    u = mp.mpf(A) / mp.mpf(r)
    E = mp.mpf(EPS) * (u ** N_EXP - 2 * mp.mpf(C) * u ** (mp.mpf(M_EXP) / 2))
    mdEdr = mp.mpf(EPS) * (N_EXP * u ** N_EXP - mp.mpf(C) * M_EXP * u ** (mp.mpf(M_EXP) / 2)) / mp.mpf(r)
    return float(E), float(mdEdr), float(u ** M_EXP)


@pytest.mark.parametrize("r", [3.52, 2.49, 2.0, 2.04134498312021, 7.7])
def test_dimer_closed_form(oracle_ld, r):
    """E(r) = eps [u^n - 2 c u^(m/2)], radial force -dE/dr = eps [n u^n - c m u^(m/2)] / r."""
    pos = np.array([[0.1, -0.2, 0.3], [0.1 + r, -0.2, 0.3]])
    rho, F, (U, _, _) = oracle_ld.energy_forces(pos, oracle_ld.params())
    E, mdEdr, rho_cf = dimer_closed(np.float64(0.1 + r) - 0.1)   # the separation as stored
    assert rel(U, E) < 5e-15
    assert rel(rho[0], rho_cf) < 5e-15 and rho[0] == rho[1]
    # -dE/dr > 0 is repulsive: atom 1 (at +x) is pushed to +x, atom 0 to -x
    assert abs(F[1, 0] - mdEdr) < 5e-14 * max(1.0, abs(mdEdr))
    assert abs(F[0, 0] + mdEdr) < 5e-14 * max(1.0, abs(mdEdr))
    assert np.all(F[:, 1:] == 0)


def test_dimer_golden_values(oracle_ld):
    g = GOLD["dimer"]
    P = oracle_ld.params()
    E_at = lambda r: oracle_ld.energy(np.array([[0, 0, 0], [r, 0, 0.0]]), P)
    assert rel(E_at(A), g["E_at_a"]) < 1e-12
    assert rel(E_at(g["r_eq"]), g["E_r_eq"]) < 1e-12
    r_eq = A * (N_EXP / (C * M_EXP)) ** (1.0 / (N_EXP - M_EXP / 2))
    assert rel(r_eq, g["r_eq"]) < 1e-13
    _, F, _ = oracle_ld.energy_forces(np.array([[0, 0, 0], [r_eq, 0, 0.0]]), P)
    assert np.abs(F).max() < 1e-12                                  # equilibrium
    rho, F, (U, _, _) = oracle_ld.energy_forces(np.array([[0, 0, 0], [2.49, 0, 0.0]]), P)
    assert rel(U, g["r249"]["E"]) < 1e-12 and rel(rho[0], g["r249"]["rho"]) < 1e-12
    assert rel(np.linalg.norm(F[0]), g["r249"]["F_norm"]) < 1e-12
    assert F[0, 0] > 0 and F[1, 0] < 0                              # attractive at 2.49 A
    _, F, (U, _, _) = oracle_ld.energy_forces(np.array([[0, 0, 0], [2.0, 0, 0.0]]), P)
    assert rel(U, g["r200"]["E"]) < 1e-12
    assert rel(F[1, 0], g["r200"]["minus_dEdr"]) < 1e-12            # repulsive below r_eq


# --------------------------------------------------------------------------- #
# P2-P4: all-equivalent and high-symmetry clusters
# --------------------------------------------------------------------------- #
def equivalent_cluster_energy(N, k, r):
    mp.mp.dps = 40
    u = mp.mpf(A) / mp.mpf(r)
    return float(mp.mpf(EPS) * (mp.mpf(N) * k / 2 * u ** N_EXP - N * mp.mpf(C) * mp.sqrt(k) * u ** (mp.mpf(M_EXP) / 2)))


def test_triangle_and_tetrahedron(oracle_ld):
    r = 2.49
    tri = np.array([[0, 0, 0], [r, 0, 0], [r / 2, r * math.sqrt(3) / 2, 0]])
    U = oracle_ld.energy(tri, oracle_ld.params())
    assert rel(U, equivalent_cluster_energy(3, 2, r)) < 1e-14
    assert rel(U, GOLD["triangle_r249_E"]) < 1e-12
    s = r / math.sqrt(2)
    tet = np.array([[s, 0, 0], [0, s, 0], [0, 0, s], [s, s, s]]) - np.array([s / 2, s / 2, s / 2])
    rho, F, (U, _, _) = oracle_ld.energy_forces(tet, oracle_ld.params())
    assert rel(U, equivalent_cluster_energy(4, 3, r)) < 1e-14
    assert rel(U, GOLD["tetrahedron_r249"]["E"]) < 1e-12
    for i in range(4):
        assert rel(np.linalg.norm(F[i]), GOLD["tetrahedron_r249"]["F_norm"]) < 1e-12
        assert np.dot(F[i], -tet[i]) > 0                            # toward the centroid


def test_icosahedron13(oracle_ld):
    """13-atom icosahedron, centre-vertex R: vertex sees 5 at 1.0514622 R, 5 at 1.7013016 R,
    1 at 2 R and the centre at R."""
    R = 2.49
    pos = W.mackay_icosahedron(1, R)
    assert pos.shape == (13, 3)
    rho, F, (U, _, _) = oracle_ld.energy_forces(pos, oracle_ld.params())
    mp.mp.dps = 40
    phi = (1 + mp.sqrt(5)) / 2
    e1 = 2 / mp.sqrt(1 + phi ** 2)                                   # edge / R
    e2 = e1 * phi                                                    # second-neighbour / R
    u = lambda x: mp.mpf(A) / (mp.mpf(R) * x)
    rho_c = 12 * u(1) ** 6
    rho_v = u(1) ** 6 + 5 * u(e1) ** 6 + 5 * u(e2) ** 6 + u(2) ** 6
    pair = (12 * u(1) ** 9 + 12 * (u(1) ** 9 + 5 * u(e1) ** 9 + 5 * u(e2) ** 9 + u(2) ** 9)) / 2
    E = mp.mpf(EPS) * (pair - mp.mpf(C) * (mp.sqrt(rho_c) + 12 * mp.sqrt(rho_v)))
    assert rel(rho[0], float(rho_c)) < 1e-14
    assert all(rel(x, float(rho_v)) < 1e-13 for x in rho[1:])
    assert rel(U, float(E)) < 1e-14
    g = GOLD["icosahedron13_R249"]
    assert rel(U, g["E"]) < 1e-12 and rel(rho[0], g["rho_centre"]) < 1e-12
    assert rel(rho[1], g["rho_vertex"]) < 1e-12
    assert np.abs(F[0]).max() < 1e-13
    for i in range(1, 13):
        radial = np.dot(F[i], pos[i]) / np.linalg.norm(pos[i])
        assert rel(radial, g["vertex_radial_force"]) < 1e-11
        assert np.linalg.norm(F[i] - radial * pos[i] / np.linalg.norm(pos[i])) < 1e-13


def test_cuboctahedron13(oracle_ld):
    pos = W.fcc_sphere(13)
    rho, _, (U, _, _) = oracle_ld.energy_forces(pos, oracle_ld.params())
    assert rho[0] == 96.0                                           # 12 * (sqrt 2)^6, exact
    assert rel(U, GOLD["cuboctahedron13_a352"]["E"]) < 1e-11


# --------------------------------------------------------------------------- #
# P5, P6: Ni147 Mackay and fcc N-nearest-site clusters (surveyor's independent numbers)
# --------------------------------------------------------------------------- #
def test_mackay147(oracle_ld):
    g = GOLD["mackay147_radial249"]
    pos = W.mackay_icosahedron(3, 2.49)
    assert pos.shape == (147, 3)
    d = np.linalg.norm(pos[:, None] - pos[None], axis=-1) + 1e9 * np.eye(147)
    assert abs(d.min() - 2.49) < 1e-12                              # reading Q12: radial spacing
    rho, F, (U, _, _) = oracle_ld.energy_forces(pos, oracle_ld.params())
    assert rel(U, g["E"]) < 1e-12
    assert rel(U, g["E_if_edge_reading"]) > 1e-3                    # the other reading is told apart
    orbits = sorted(set(np.round(rho, 7)))
    assert len(orbits) == 7
    assert np.allclose(orbits, g["rho_orbits"], rtol=0, atol=2e-7)
    fn = sorted(set(np.round(np.linalg.norm(F, axis=1), 7)))
    assert len(fn) == 7 and np.allclose(fn, g["force_norm_orbits"], rtol=0, atol=2e-7)
    assert np.abs(F.sum(0)).max() < 1e-13


@pytest.mark.parametrize("key", ["1409", "1415", "1433"])
def test_fcc_nearest_sites(oracle_ld, key):
    g = GOLD["fcc_nearest_sites_unjittered"][key]
    pos = W.fcc_sphere(int(key))
    rho, _, (U, _, _) = oracle_ld.energy_forces(pos, oracle_ld.params())
    assert rel(U, g["E"]) < 1e-12
    if "rho0" in g:
        assert rel(rho[0], g["rho0"]) < 1e-12
    if "sum_pos" in g:
        assert np.allclose(pos.sum(0), g["sum_pos"], atol=1e-9)


def test_fcc1415_cutoff10(oracle_ld):
    g = GOLD["fcc_nearest_sites_unjittered"]["1415_rc10"]
    pos = W.fcc_sphere(1415)
    rho, _, (U, _, _) = oracle_ld.energy_forces(pos, oracle_ld.params(r_cut=10.0))
    assert rel(U, g["E"]) < 1e-12 and rel(rho[0], g["rho0"]) < 1e-12
    d0 = np.linalg.norm(pos - pos[0], axis=1)
    assert int(((d0 < 10.0) & (d0 > 0)).sum()) == g["neighbours0"]


# --------------------------------------------------------------------------- #
# P7: bulk limit -- textbook fcc lattice sums (Lennard-Jones A6 = 14.45392, A12 = 12.13188
# in nearest-neighbour units; Kittel / Ashcroft-Mermin): S_k = A_k * 2^(k/2) in units of a
# --------------------------------------------------------------------------- #
def test_bulk_lattice_sum_and_cohesive_energy(oracle_ld):
    n_atoms = 16384
    pos = W.fcc_sphere(n_atoms)
    rho0 = oracle_ld.density_rows(pos, oracle_ld.params(), [0])[0]
    S6_textbook = 14.45392 * 8.0
    # a finite sphere of radius R misses the tail: integral_R^inf 4 pi r^2 (4/a^3) (a/r)^6 dr
    R = np.linalg.norm(pos, axis=1).max()
    tail = 4 * math.pi * (4 / A ** 3) * A ** 6 / (3 * R ** 3)
    assert rho0 < S6_textbook
    assert abs(rho0 + tail - S6_textbook) < 2e-3 * tail + 2e-5 * S6_textbook
    # n = 12 sum through the generic-exponent path: rho with m := 12
    rho12 = oracle_ld.density_rows(pos, oracle_ld.params(n=13, m=12), [0])[0]
    assert rel(rho12, 12.13188 * 64.0) < 1e-6
    # centre atom's energy -> cohesive energy eps [S9/2 - c sqrt(S6)] = -4.4401 eV
    g = GOLD["bulk"]
    rho9 = oracle_ld.density_rows(pos, oracle_ld.params(n=10, m=9), [0])[0]
    assert rel(rho9, g["S9"]) < 1e-6
    e_atom = EPS * (rho9 / 2 - C * math.sqrt(rho0 + tail))
    assert abs(e_atom - g["E_coh"]) < 2e-4
    # SC fit condition: a = 3.52 is the zero-pressure lattice constant, n S9 / (m sqrt S6) = c
    assert abs(N_EXP * rho9 / (M_EXP * math.sqrt(rho0 + tail)) - C) < 2e-3


def test_fcc16384_energy_per_atom(oracle_plain):
    pos = W.fcc_sphere(16384)
    U = oracle_plain.energy(pos, oracle_plain.params())
    assert abs(U / 16384 - GOLD["fcc_nearest_sites_unjittered"]["16384"]["E_per_atom"]) < 2e-6


# --------------------------------------------------------------------------- #
# P8-P11: gradient, Newton 3, torque, invariances, homogeneity
# --------------------------------------------------------------------------- #
def random_cluster(rng, n, spread=2.2):
    base = W.fcc_sphere(n)
    return base + rng.uniform(-0.25, 0.25, base.shape) * spread / 2.2


@pytest.mark.parametrize("n_atoms,r_cut", [(4, 0.0), (8, 0.0), (19, 0.0), (19, 4.4)])
def test_force_is_minus_gradient_central_differences(oracle_ld, n_atoms, r_cut):
    rng = np.random.default_rng(100 + n_atoms)
    pos = random_cluster(rng, n_atoms)
    P = oracle_ld.params(r_cut=r_cut)
    _, F, _ = oracle_ld.energy_forces(pos, P)
    h = 1e-5
    G = np.zeros_like(F)
    for i in range(n_atoms):
        for k in range(3):
            p1 = pos.copy(); p1[i, k] += h
            p2 = pos.copy(); p2[i, k] -= h
            G[i, k] = -(oracle_ld.energy(p1, P) - oracle_ld.energy(p2, P)) / (2 * h)
    assert rel_l2(F, G) < 2e-9


def test_newton_third_law_and_zero_torque(oracle_ld):
    rng = np.random.default_rng(5)
    for n_atoms, r_cut in ((7, 0.0), (200, 0.0), (200, 6.0)):
        pos = random_cluster(rng, n_atoms)
        _, F, _ = oracle_ld.energy_forces(pos, oracle_ld.params(r_cut=r_cut))
        scale = np.linalg.norm(F, axis=1).sum()
        assert np.abs(F.sum(0)).max() < 1e-14 * scale
        lever = np.abs(pos).max()
        assert np.abs(np.cross(pos, F).sum(0)).max() < 1e-14 * scale * lever


def random_rotation(rng):
    q, r = np.linalg.qr(rng.standard_normal((3, 3)))
    q *= np.sign(np.diag(r))
    if np.linalg.det(q) < 0:
        q[:, 0] *= -1
    return q


def test_rigid_motion_and_permutation_invariance(oracle_ld):
    rng = np.random.default_rng(17)
    pos = random_cluster(rng, 60)
    P = oracle_ld.params()
    rho, F, (U, _, _) = oracle_ld.energy_forces(pos, P)
    Q = random_rotation(rng)
    t = np.array([3.1, -7.7, 12.9])
    rho2, F2, (U2, _, _) = oracle_ld.energy_forces(pos @ Q.T + t, P)
    assert rel(U2, U) < 1e-13
    assert np.allclose(rho2, rho, rtol=1e-13, atol=0)
    assert rel_l2(F2, F @ Q.T) < 1e-12
    perm = rng.permutation(60)
    rho3, F3, (U3, _, _) = oracle_ld.energy_forces(pos[perm], P)
    assert rel(U3, U) < 1e-14
    assert np.allclose(rho3, rho[perm], rtol=1e-15, atol=0)
    assert rel_l2(F3, F[perm]) < 1e-14


def test_homogeneity(oracle_ld):
    """Scaling r and a together leaves rho and U/eps unchanged; scaling r alone scales rho
    by lambda^-m (exact identities of Eq. (1)-(2))."""
    rng = np.random.default_rng(23)
    pos = random_cluster(rng, 30)
    lam = 2.0                                                       # power of two: exact in binary
    rho, F, (U, _, _) = oracle_ld.energy_forces(pos, oracle_ld.params())
    rho2, F2, (U2, _, _) = oracle_ld.energy_forces(pos * lam, oracle_ld.params(a=A * lam))
    assert np.array_equal(rho2, rho) and U2 == U
    assert np.array_equal(F2 * lam, F)
    rho3 = oracle_ld.density(pos * lam, oracle_ld.params())
    assert np.allclose(rho3 * lam ** M_EXP, rho, rtol=1e-15)
    # eps is an overall factor
    _, F4, (U4, _, _) = oracle_ld.energy_forces(pos, oracle_ld.params(eps=2 * EPS))
    assert U4 == 2 * U and np.array_equal(F4, 2 * F)


def test_long_double_and_binary64_builds_agree(oracle_ld, oracle_plain):
    assert oracle_ld.lib.oracle_real_bits() == 128 and oracle_plain.lib.oracle_real_bits() == 64
    w = W.config_c2()
    P = oracle_ld.params()
    rho, F, (U, _, _) = oracle_ld.energy_forces(w.pos, P)
    rho2, F2, (U2, _, _) = oracle_plain.energy_forces(w.pos, P)
    assert rel(U2, U) < 1e-13
    assert rel_l2(F2, F) < 1e-12
    assert np.allclose(rho2, rho, rtol=1e-13)


def test_row_subset_entry_points_match_full(oracle_ld):
    w = W.config_c2()
    for r_cut in (0.0, 10.0):
        P = oracle_ld.params(r_cut=r_cut)
        rho, F, _ = oracle_ld.energy_forces(w.pos, P)
        rows = np.array([0, 1, 17, 700, 1414])
        assert np.array_equal(oracle_ld.density_rows(w.pos, P, rows), rho[rows])
        Fr, ps = oracle_ld.forces_rows(w.pos, P, rho, rows)
        assert rel_l2(Fr, F[rows]) < 1e-15


# --------------------------------------------------------------------------- #
# P15: cutoff consistency
# --------------------------------------------------------------------------- #
def test_cutoff_beyond_diameter_is_all_pairs_bit_for_bit(oracle_ld):
    w = W.config_c1()
    r0 = oracle_ld.energy_forces(w.pos, oracle_ld.params())
    r1 = oracle_ld.energy_forces(w.pos, oracle_ld.params(r_cut=100.0))
    assert np.array_equal(r0[0], r1[0]) and np.array_equal(r0[1], r1[1]) and r0[2] == r1[2]


def test_cutoff_numpy_bruteforce_and_isolated_atom(oracle_ld):
    rng = np.random.default_rng(3)
    pos = random_cluster(rng, 120)
    pos = np.vstack([pos, [[60.0, 0, 0]]])                          # an evaporated atom (Q9)
    rc = 5.0
    rho, F, (U, _, _) = oracle_ld.energy_forces(pos, oracle_ld.params(r_cut=rc))
    d = pos[:, None] - pos[None]
    r = np.sqrt((d ** 2).sum(-1)); np.fill_diagonal(r, np.inf)
    mask = r < rc
    u = np.where(mask, A / r, 0.0)
    rho_np = (u ** 6).sum(1)
    assert np.allclose(rho, rho_np, rtol=1e-13)
    assert rho[-1] == 0.0 and np.all(F[-1] == 0.0)
    U_np = EPS * ((u ** 9).sum() / 2 - C * np.sqrt(rho_np).sum())
    assert rel(U, U_np) < 1e-13
    assert oracle_ld.count_pairs(pos, rc) == int(mask.sum())
    assert np.all(np.isfinite(F))


# --------------------------------------------------------------------------- #
# kinetic energy, units, integrator
# --------------------------------------------------------------------------- #
def test_kinetic_energy_and_unit_conversion(oracle_ld):
    """ACC = (e / u) * 1e-10 from CODATA-2018 e and u (retyped here, not imported)."""
    e_C, u_kg, kB_J = 1.602176634e-19, 1.66053906660e-27, 1.380649e-23
    acc = e_C / u_kg * 1e10 * 1e10 * 1e-30       # eV/(A u): 1/A -> 1/m, m -> A, s^-2 -> fs^-2
    v = np.array([[1e-2, 0, 0], [-1e-2, 0, 0], [0, 2e-2, 0], [0, -2e-2, 0.0]])
    ke, T = oracle_ld.kinetic(v, MASS)
    ke_expect = 0.5 * MASS * (2 * 1e-4 + 2 * 4e-4) / acc
    assert rel(ke, ke_expect) < 1e-12
    assert rel(T, 2 * ke_expect / ((kB_J / e_C) * (3 * 4 - 3))) < 1e-9
    assert oracle_ld.kinetic(np.zeros((1, 3)), MASS) == (0.0, 0.0)  # N = 1: T := 0 (Q5)
    # one velocity-Verlet step of a dimer at rest moves each atom by (dt^2 / 2) ACC F / m
    pos = np.array([[0, 0, 0], [2.49, 0, 0.0]])
    _, F, _ = oracle_ld.energy_forces(pos, oracle_ld.params())
    out = oracle_ld.run(pos, np.zeros((2, 3)), oracle_ld.params(), dt=1.0, nsteps=1)
    assert rel(out["pos"][0, 0], 0.5 * acc * F[0, 0] / MASS) < 1e-12


def test_maxwell_boltzmann_generator_statistics():
    w = W.fcc_cluster(20000, 1500.0, seed=9)
    assert np.abs(w.vel.mean(0)).max() < 1e-18 + 1e-16
    sigma = math.sqrt(8.617333262e-5 * 1500.0 * 9.648533215665e-3 / MASS)
    assert abs(w.vel.std() / sigma - 1) < 0.01


def test_nve_energy_conservation_dt_scaling_and_reversal(oracle_plain):
    """P12: Ni147 at 1000 K; velocity-Verlet energy error is O(dt^2) and the map is
    time-reversible.  Catches a wrong half-kick, a stale force, a wrong ACC or mass."""
    w = W.config_c1()
    P = oracle_plain.params()
    out = oracle_plain.run(w.pos, w.vel, P, dt=1.0, nsteps=1000)
    etot = out["epot"] + out["ekin"]
    exc1 = np.abs(etot - etot[0]).max()
    assert exc1 / abs(etot[0]) < 2e-5
    _, T0 = oracle_plain.kinetic(w.vel)
    assert 850 < T0 < 1150
    out_h = oracle_plain.run(w.pos, w.vel, P, dt=0.5, nsteps=2000)
    etot_h = out_h["epot"] + out_h["ekin"]
    exc2 = np.abs(etot_h - etot_h[0]).max()
    assert 3.5 < exc1 / exc2 < 4.5
    fwd = oracle_plain.run(w.pos, w.vel, P, dt=1.0, nsteps=100)
    back = oracle_plain.run(fwd["pos"], -fwd["vel"], P, dt=1.0, nsteps=100)
    assert np.abs(back["pos"] - w.pos).max() < 1e-10
    assert np.abs(back["vel"] + w.vel).max() < 1e-12


def test_rescale_thermostat_hits_target_every_step(oracle_ld):
    """P14: after each step T equals T_target(k) = T_start + (T_end - T_start) k / nsteps."""
    w = W.config_c1()
    nsteps = 40
    out = oracle_ld.run(w.pos, w.vel, oracle_ld.params(), dt=1.0, nsteps=nsteps, thermo_kind=1,
                        T_start=1000.0, T_end=600.0)
    kB = 8.617333262e-5
    T = 2 * out["ekin"] / (kB * (3 * 147 - 3))
    target = 1000.0 + (600.0 - 1000.0) * np.arange(nsteps + 1) / nsteps
    assert np.allclose(T[1:], target[1:], rtol=1e-13)
    _, T_end = oracle_ld.kinetic(out["vel"])
    assert rel(T_end, 600.0) < 1e-13


def test_trajectory_sensitivity_headroom(oracle_plain):
    """P13: a 1e-12 A perturbation stays far below the 1e-8 A / 100-step parity bound."""
    w = W.config_c1()
    P = oracle_plain.params()
    a = oracle_plain.run(w.pos, w.vel, P, 1.0, 100)
    p2 = w.pos.copy(); p2[5, 0] += 1e-12
    b = oracle_plain.run(p2, w.vel, P, 1.0, 100)
    assert np.abs(a["pos"] - b["pos"]).max() < 1e-10


# --------------------------------------------------------------------------- #
# input generators (structure only -- no method arithmetic)
# --------------------------------------------------------------------------- #
def test_generators_shapes_and_structure():
    assert [W.mackay_icosahedron(s).shape[0] for s in (0, 1, 2, 3)] == [1, 13, 55, 147]
    idx = W.fcc_half_lattice_indices(1415)
    assert idx.shape == (1415, 3) and np.all((idx.sum(1) % 2) == 0)
    q = (idx ** 2).sum(1)
    assert np.all(np.diff(q) >= 0) and len({tuple(r) for r in idx.tolist()}) == 1415
    w = W.config_c2()
    assert np.abs(w.pos - W.fcc_sphere(1415)).max() <= 0.05
    w2 = W.config_c2()
    assert np.array_equal(w.pos, w2.pos) and np.array_equal(w.vel, w2.vel)   # seeded
    liq = W.liquid_droplet(600, 2000.0, seed=3001)
    d = np.linalg.norm(liq.pos[:, None] - liq.pos[None], axis=-1) + 1e9 * np.eye(600)
    assert d.min() >= 1.8
    R = (3 * 600 / (4 * math.pi * 0.080)) ** (1 / 3)
    assert np.linalg.norm(liq.pos, axis=1).max() <= R
