"""Pins of the oracle's energy-shifted cutoff (cut_shift = 1, reading Q21) against what the
mathematics fixes: the closed-form dimer, continuity of U where plain truncation jumps, the exact relation to
the all-pairs sums when the cutoff exceeds the diameter, an mpmath restatement of the definition, F = -grad U
by central differences, and the NVE energy of a hot droplet that plain truncation random-walks."""
import math

import numpy as np
import pytest

from paper_1210_3559_b200 import workloads as W

EPS, C, A, N_EXP, M_EXP = 1.5707e-2, 39.432, 3.52, 9, 6


def dimer(r):
    return np.array([[0.0, 0.0, 0.0], [r, 0.0, 0.0]])


def test_dimer_closed_form_and_continuity(oracle_ld):
    rc = 6.0
    P1 = oracle_ld.params(r_cut=rc, cut_shift=1)
    P0 = oracle_ld.params(r_cut=rc, cut_shift=0)
    for r in (2.2, 3.0, 4.5, 5.9):
        psi = (A / r) ** M_EXP - (A / rc) ** M_EXP
        phi = (A / r) ** N_EXP - (A / rc) ** N_EXP
        u = EPS * (phi - 2.0 * C * math.sqrt(psi))
        dudr = EPS * (-N_EXP * A ** N_EXP / r ** (N_EXP + 1) + C * M_EXP * A ** M_EXP / r ** (M_EXP + 1) / math.sqrt(psi))
        rho, f, (e, ep, ee) = oracle_ld.energy_forces(dimer(r), P1)
        assert e == pytest.approx(u, rel=1e-13)
        assert rho[0] == pytest.approx(psi, rel=1e-13) and rho[1] == pytest.approx(psi, rel=1e-13)
        assert f[1, 0] == pytest.approx(-dudr, rel=1e-12) and f[0, 0] == pytest.approx(dudr, rel=1e-12)
        assert abs(f[0, 1]) + abs(f[0, 2]) == 0.0
    # just inside the cutoff: the shifted energy goes to the value beyond it (0), the truncated one does not
    d = 1e-10
    e1 = oracle_ld.energy_forces(dimer(rc * (1 - d)), P1)[2][0]
    e0 = oracle_ld.energy_forces(dimer(rc * (1 - d)), P0)[2][0]
    assert abs(e1) < 1e-5 and abs(e0) > 0.2                   # sqrt(psi) ~ sqrt(6 (a/rc)^6 d): small but not linear in d
    for P in (P0, P1):
        rho, f, (e, _, _) = oracle_ld.energy_forces(dimer(rc * (1 + d)), P)
        assert e == 0.0 and np.all(rho == 0.0) and np.all(f == 0.0)
        rho, f, (e, _, _) = oracle_ld.energy_forces(dimer(rc), P)          # strict <: exactly at r_c is outside
        assert e == 0.0 and np.all(rho == 0.0)


def test_energy_is_continuous_when_a_pair_crosses_the_cutoff(oracle_ld):
    """An fcc cluster with one atom pushed radially through the cutoff sphere of another: across the crossing
    plain truncation jumps by ~eps (a/rc)^m-sized terms, the shifted energy changes only by its slope."""
    rc = 7.0
    pos = W.fcc_cluster(200, 0.0, seed=5).pos.copy()
    i = 0
    d = np.linalg.norm(pos - pos[i], axis=1)
    j = int(np.argmin(np.abs(d - rc)))                          # the atom nearest to the cutoff sphere of i
    u = (pos[j] - pos[i]) / d[j]
    h = 1e-7

    def energy(shift, r):
        p = pos.copy()
        p[j] = pos[i] + u * r
        return oracle_ld.energy_forces(p, oracle_ld.params(r_cut=rc, cut_shift=shift))[2][0]

    jump0 = abs(energy(0, rc + h) - energy(0, rc - h))
    jump1 = abs(energy(1, rc + h) - energy(1, rc - h))
    slope = abs(energy(1, rc - h) - energy(1, rc - 3 * h)) / (2 * h)
    assert jump0 > 1e-5                                          # eps c (a/rc)^6 / sqrt(rho) and eps (a/rc)^9 terms
    assert jump1 < 10 * slope * 2 * h + 1e-12 and jump1 < 1e-4 * jump0


def test_cutoff_beyond_diameter_is_all_pairs_minus_constants(oracle_ld):
    w = W.fcc_cluster(60, 300.0, seed=9)
    n = w.n_atoms
    rc = 100.0
    rho_a, f_a, (e_a, ep_a, ee_a) = oracle_ld.energy_forces(w.pos, oracle_ld.params())
    rho_s, f_s, (e_s, ep_s, ee_s) = oracle_ld.energy_forces(w.pos, oracle_ld.params(r_cut=rc, cut_shift=1))
    assert np.allclose(rho_s, rho_a - (n - 1) * (A / rc) ** M_EXP, rtol=1e-14, atol=0)
    assert ep_s == pytest.approx(ep_a - EPS * 0.5 * n * (n - 1) * (A / rc) ** N_EXP, rel=1e-14)
    assert ee_s == pytest.approx(-EPS * C * np.sqrt(rho_s).sum(), rel=1e-14)
    # cut_shift = 0 with the same cutoff is the all-pairs result itself
    rho_0, f_0, (e_0, _, _) = oracle_ld.energy_forces(w.pos, oracle_ld.params(r_cut=rc, cut_shift=0))
    assert np.array_equal(rho_0, rho_a) and np.array_equal(f_0, f_a) and e_0 == e_a
    # and cut_shift without a cutoff changes nothing
    rho_n, f_n, (e_n, _, _) = oracle_ld.energy_forces(w.pos, oracle_ld.params(cut_shift=1))
    assert np.array_equal(rho_n, rho_a) and np.array_equal(f_n, f_a) and e_n == e_a


def test_mpmath_restatement_with_pairs_cut(oracle_ld):
    mp = pytest.importorskip("mpmath")
    mp.mp.dps = 50
    rng = np.random.default_rng(21)
    pos = W.fcc_sphere(19) + rng.normal(scale=0.1, size=(19, 3))
    rc = 4.2                                                     # cuts the second shell
    kw = dict(n=8, m=5, eps=0.02, c=30.0, a=3.3)
    P = oracle_ld.params(r_cut=rc, cut_shift=1, **kw)
    rho, f, (e, ep, ee) = oracle_ld.energy_forces(pos, P)
    a, eps, c = mp.mpf(kw["a"]), mp.mpf(kw["eps"]), mp.mpf(kw["c"])
    x = [[mp.mpf(float(v)) for v in row] for row in pos]
    tot = mp.mpf(0)
    n_cut = 0
    for i in range(19):
        rho_i, pair_i = mp.mpf(0), mp.mpf(0)
        for j in range(19):
            if j == i:
                continue
            r = mp.sqrt(sum((x[i][k] - x[j][k]) ** 2 for k in range(3)))
            if r < rc:
                rho_i += (a / r) ** kw["m"] - (a / mp.mpf(rc)) ** kw["m"]
                pair_i += (a / r) ** kw["n"] - (a / mp.mpf(rc)) ** kw["n"]
            else:
                n_cut += 1
        assert float(rho_i) == pytest.approx(rho[i], rel=1e-14)
        tot += eps * (pair_i / 2 - c * mp.sqrt(rho_i))
    assert 0 < n_cut < 19 * 18
    assert float(tot) == pytest.approx(e, rel=1e-14)


@pytest.mark.parametrize("shift", [0, 1])
def test_force_is_minus_gradient(oracle_ld, shift):
    w = W.liquid_droplet(120, 0.0, seed=4)
    P = oracle_ld.params(r_cut=5.5, cut_shift=shift)
    _, f, _ = oracle_ld.energy_forces(w.pos, P)
    h = 1e-5
    rng = np.random.default_rng(0)
    d2 = ((w.pos[:, None, :] - w.pos[None, :, :]) ** 2).sum(axis=2)
    assert np.abs(np.sqrt(d2[d2 > 0]) - 5.5).min() > 10 * h      # no pair crosses within the stencil
    for i in rng.choice(120, size=6, replace=False):
        for k in range(3):
            pp, pm = w.pos.copy(), w.pos.copy()
            pp[i, k] += h
            pm[i, k] -= h
            g = (oracle_ld.energy_forces(pp, P)[2][0] - oracle_ld.energy_forces(pm, P)[2][0]) / (2 * h)
            assert f[i, k] == pytest.approx(-g, rel=2e-7, abs=1e-9)


def test_nve_energy_with_and_without_the_shift(oracle_ld):
    """Hot droplet (equilibrated first), pairs cross the cutoff all the time: the total energy of the truncated
    model random-walks by a jump per crossing; the shifted model conserves it as well as the all-pairs model
    does at the same time step."""
    w = W.liquid_droplet(150, 1800.0, seed=11)
    eq = oracle_ld.run(w.pos, w.vel, oracle_ld.params(), dt=1.0, nsteps=300, thermo_kind=1, T_start=1800.0, T_end=1800.0)
    out = {}
    for key, kw in (("all", {}), (0, dict(r_cut=6.0, cut_shift=0)), (1, dict(r_cut=6.0, cut_shift=1))):
        r = oracle_ld.run(eq["pos"], eq["vel"], oracle_ld.params(**kw), dt=1.0, nsteps=600)
        tot = r["epot"] + r["ekin"]
        out[key] = np.abs(tot - tot[0]).max()
    assert out[1] < 2 * out["all"] + 1e-3, out                   # measured: 4.7e-3 against 4.2e-3 eV
    assert out[0] > 30 * out[1], out                             # measured: 0.56 eV
