"""SC_OPT_CUTOFF_SHIFT = 1 (energy-shifted cutoff, Q21) on the list path against the
oracle's cut_shift = 1 definition: densities, forces and energy within the cutoff path's tolerances, the
in-range pair count exact, plain truncation untouched to the bit, trajectories, and the NVE energy that the
shift is there to conserve."""
import numpy as np
import pytest

from paper_1210_3559_b200 import workloads as W

pytestmark = pytest.mark.gpu

FORCE_TOL = {0: 1e-10, 1: 1e-5}
ENERGY_TOL = {0: 1e-12, 1: 1e-7}
RHO_TOL = {0: 1e-12, 1: 2e-6}


def make(scmd, pos, vel, shift, **kw):
    import torch
    sc = scmd.SuttonChen(len(pos), **kw)
    sc.sc_set_option(scmd.SC_OPT_CUTOFF_SHIFT, shift)
    sc.sc_set_state(torch.as_tensor(np.ascontiguousarray(pos), device="cuda"),
                    None if vel is None else torch.as_tensor(np.ascontiguousarray(vel), device="cuda"))
    return sc


def evaluate(sc):
    return sc.sc_density().cpu().numpy(), sc.sc_forces().cpu().numpy(), sc.sc_energy()


@pytest.mark.parametrize("precision", [0, 1])
@pytest.mark.parametrize("case", ["fcc4001-rc7", "liquid3000-rc6", "ni1415-rc10", "generic-exponents", "isolated"])
def test_sweeps_against_oracle(scmd, oracle_ld, case, precision):
    params = {}
    if case == "fcc4001-rc7":
        pos, rc = W.fcc_cluster(4001, 900.0, seed=31).pos, 7.0
    elif case == "liquid3000-rc6":
        pos, rc = W.liquid_droplet(3000, 0.0, seed=32).pos, 6.0
    elif case == "ni1415-rc10":
        pos, rc = W.config_c2().pos, 10.0
    elif case == "generic-exponents":
        pos, rc = W.fcc_cluster(900, 600.0, seed=33).pos, 6.5
        params = dict(n=12, m=5, eps=0.02, c=30.0, a=3.3)
    else:                                                        # two far atoms: no neighbour in range -> rho = 0 exactly
        pos = np.vstack([W.fcc_cluster(300, 300.0, seed=34).pos, [[80.0, 0.0, 0.0]], [[0.0, -90.0, 5.0]]])
        rc = 6.0
    P = oracle_ld.params(r_cut=rc, cut_shift=1, **params)
    rho_o, f_o, (e_o, _, _) = oracle_ld.energy_forces(pos, P)
    sc = make(scmd, pos, None, 1, r_cut=rc, skin=0.8, precision=precision, **params)
    rho, f, e = evaluate(sc)
    assert sc.sc_stats()["n_pairs_in_cut"] == oracle_ld.count_pairs(pos, rc)
    nz = rho_o > 0
    assert np.array_equal(rho[~nz], rho_o[~nz])
    assert np.max(np.abs(rho[nz] - rho_o[nz]) / rho_o[nz]) < RHO_TOL[precision]
    assert np.linalg.norm(f - f_o) < FORCE_TOL[precision] * np.linalg.norm(f_o)
    assert abs(e - e_o) < ENERGY_TOL[precision] * abs(e_o)
    # the shift is not a rounding-level change: the truncated model differs by far more than the tolerance
    e_t = oracle_ld.energy_forces(pos, oracle_ld.params(r_cut=rc, cut_shift=0, **params))[2][0]
    assert abs(e_t - e_o) > 1e-4 * abs(e_o)
    # switching the option off again gives the truncated model, bit for bit what a fresh context gives
    sc.sc_set_option(scmd.SC_OPT_CUTOFF_SHIFT, 0)
    rho0, f0, e0 = evaluate(sc)
    ref = make(scmd, pos, None, 0, r_cut=rc, skin=0.8, precision=precision, **params)
    rho1, f1, e1 = evaluate(ref)
    assert np.array_equal(rho0, rho1) and np.array_equal(f0, f1) and e0 == e1
    assert abs(e0 - e_t) < ENERGY_TOL[precision] * abs(e_t)
    sc.close()
    ref.close()


@pytest.mark.parametrize("tpa", [8, 32])
def test_trajectory_against_oracle(scmd, oracle_ld, tpa):
    """100 steps with rebuilds, FP64: positions within 1e-8 A of the oracle's shifted model."""
    w = W.fcc_cluster(1200, 1200.0, seed=35)
    P = oracle_ld.params(r_cut=6.5, cut_shift=1)
    ref = oracle_ld.run(w.pos, w.vel, P, dt=1.0, nsteps=100)
    sc = make(scmd, w.pos, w.vel, 1, r_cut=6.5, skin=0.4)
    sc.sc_set_option(scmd.SC_OPT_LANES_PER_ROW, tpa)
    sc.sc_step(1.0, 100)
    pos, vel = sc.sc_get_state()
    assert sc.sc_stats()["n_rebuilds"] >= 2
    assert np.abs(pos.cpu().numpy() - ref["pos"]).max() < 1e-8
    assert abs(sc.sc_energy() - ref["epot"][-1]) < 1e-11 * abs(ref["epot"][-1])
    sc.close()


@pytest.mark.parametrize("precision", [0, 1])
def test_nve_energy_is_conserved_with_the_shift(scmd, precision):
    """Hot liquid droplet, 4000 steps, r_cut = 6 A: thousands of pairs cross the cutoff.  Plain truncation
    random-walks the total energy; with the shift it stays within the integrator's own error."""
    import torch
    from paper_1210_3559_b200.binding import rescale_thermostat
    w = W.liquid_droplet(2000, 1800.0, seed=36)
    drift = {}
    for shift in (0, 1):
        sc = make(scmd, w.pos, w.vel, shift, r_cut=6.0, skin=0.6, precision=precision)
        sc.sc_set_option(scmd.SC_OPT_ENERGY_EVERY_STEP, 1)
        sc.sc_step(1.0, 500, rescale_thermostat(1800.0, 1800.0))           # settle the random start
        e0 = sc.sc_energy() + sc.sc_kinetic()[0]
        worst = 0.0
        for _ in range(8):
            sc.sc_step(1.0, 500)
            worst = max(worst, abs(sc.sc_energy() + sc.sc_kinetic()[0] - e0))
        drift[shift] = worst
        sc.close()
    assert drift[1] < 0.5 and drift[0] > 10 * drift[1], drift


def test_option_validation_and_all_pairs_ignore(scmd, oracle_ld):
    import torch
    w = W.fcc_cluster(500, 300.0, seed=37)
    sc = make(scmd, w.pos, None, 1)                               # no cutoff: accepted, changes nothing
    rho, f, e = evaluate(sc)
    ref = make(scmd, w.pos, None, 0)
    rho1, f1, e1 = evaluate(ref)
    assert np.array_equal(rho, rho1) and np.array_equal(f, f1) and e == e1
    for bad in (-1, 2):
        with pytest.raises(scmd.ScError) as err:
            sc.sc_set_option(scmd.SC_OPT_CUTOFF_SHIFT, bad)
        assert err.value.status == scmd.SC_ERR_INVALID
    sc.close()
    ref.close()
