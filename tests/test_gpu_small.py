"""The one-launch step loop (csrc/sc_small.cuh: whole sc_step in one cooperative kernel, grid barriers
between the phases of a step) against the CPU oracle and against the multi-launch path, through the
C ABI.  SC_OPT_PERSISTENT = 1 forces it (N <= 6144), 2 forbids it, 0 lets the library choose."""
import numpy as np
import pytest

from paper_1210_3559_b200 import workloads as W

pytestmark = pytest.mark.gpu
TRAJ_TOL = 1e-8            # Angstrom (BASELINE.json: 100-step trajectories, FP64)


def make(scmd, w, persistent, **kw):
    import torch
    sc = scmd.SuttonChen(w.n_atoms, **kw)
    sc.sc_set_option(scmd.SC_OPT_PERSISTENT, persistent)
    sc.sc_set_state(torch.as_tensor(w.pos, device="cuda"), torch.as_tensor(w.vel, device="cuda"))
    return sc


def state(sc):
    pos, vel = sc.sc_get_state()
    return pos.cpu().numpy(), vel.cpu().numpy()


@pytest.mark.parametrize("n_atoms", [1, 2, 3, 33, 147, 149, 600, 2607, 4100, 6144])
def test_nve_against_oracle_and_launch_count(scmd, oracle_ld, n_atoms):
    """rows per CTA 1 .. 42, threads per row 512 .. 8, ragged last CTA; one launch for the whole loop."""
    w = W.fcc_cluster(n_atoms, 1200.0, seed=900 + n_atoms)
    nsteps = 30 if n_atoms <= 2607 else 8
    ref = oracle_ld.run(w.pos, w.vel, oracle_ld.params(), dt=1.0, nsteps=nsteps)
    sc = make(scmd, w, 1)
    sc.sc_forces()                                          # forces at t = 0 (multi-launch sweeps)
    before = sc.sc_launch_count()
    sc.sc_step(1.0, nsteps)
    assert sc.sc_launch_count() - before == 1
    pos, vel = state(sc)
    assert np.abs(pos - ref["pos"]).max() < TRAJ_TOL
    assert np.abs(vel - ref["vel"]).max() < 1e-10
    if n_atoms > 1:
        assert abs(sc.sc_energy() - ref["epot"][-1]) <= 1e-11 * abs(ref["epot"][-1])
        assert abs(sc.sc_kinetic()[0] - ref["ekin"][-1]) <= 1e-10 * abs(ref["ekin"][-1])
    # forces, densities and energy left behind by the loop = a fresh evaluation at the final positions
    P = oracle_ld.params()
    rho_o, f_o, (e_o, _, _) = oracle_ld.energy_forces(ref["pos"], P)
    f = sc.sc_forces().cpu().numpy()
    rho = sc.sc_density().cpu().numpy()
    if n_atoms > 1:
        assert np.linalg.norm(f - f_o) <= 1e-9 * np.linalg.norm(f_o)
        assert np.max(np.abs(rho - rho_o) / rho_o) < 1e-10
    else:
        assert np.all(f == 0.0) and np.all(rho == 0.0)
    sc.close()


def test_both_paths_agree_and_default_choice(scmd):
    """Same trajectory from the one-launch loop and from the multi-launch path (summation orders differ:
    agreement to rounding, not to the bit); the default picks the one-launch loop at N = 1415."""
    w = W.config_c2()
    out = {}
    for mode in (0, 1, 2):
        sc = make(scmd, w, mode)
        sc.sc_forces()
        before = sc.sc_launch_count()
        sc.sc_step(1.0, 50)
        launches = sc.sc_launch_count() - before
        out[mode] = (state(sc), sc.sc_energy(), launches)
        sc.close()
    assert out[0][2] == 1 and out[1][2] == 1 and out[2][2] > 50
    assert np.array_equal(out[0][0][0], out[1][0][0])                       # same kernel, same bits
    assert np.abs(out[1][0][0] - out[2][0][0]).max() < 1e-10
    assert abs(out[1][1] - out[2][1]) < 1e-11 * abs(out[2][1])


def test_rescale_ramp_across_paths(scmd, oracle_ld):
    """Rescale thermostat: 25 steps in the one-launch loop, 15 through the multi-launch path, 20 in the
    loop again = one 60-step oracle run per leg (each sc_step call has its own ramp)."""
    from paper_1210_3559_b200.binding import rescale_thermostat
    w = W.config_c1()
    P = oracle_ld.params()
    legs = [(25, 1000.0, 800.0, 1), (15, 800.0, 900.0, 2), (20, 900.0, 500.0, 1)]
    pos, vel = w.pos, w.vel
    for n, a, b, _ in legs:
        ref = oracle_ld.run(pos, vel, P, dt=1.0, nsteps=n, thermo_kind=1, T_start=a, T_end=b)
        pos, vel = ref["pos"], ref["vel"]
    sc = make(scmd, w, 1)
    for n, a, b, mode in legs:
        sc.sc_set_option(scmd.SC_OPT_PERSISTENT, mode)
        sc.sc_step(1.0, n, rescale_thermostat(a, b))
    ke, T = sc.sc_kinetic()
    assert abs(T - 500.0) < 1e-9
    gpos, gvel = state(sc)
    assert np.abs(gpos - pos).max() < TRAJ_TOL
    assert np.abs(gvel - vel).max() < 1e-10
    sc.close()


@pytest.mark.parametrize("n_atoms", [2, 147, 1415, 4100])
def test_mixed_precision_in_one_launch(scmd, oracle_ld, n_atoms):
    """Mixed path (binary32 pair arithmetic on split coordinates): forces / energy left by the loop within
    BASELINE.json's mixed tolerances of the oracle at the oracle's own positions after a few steps, trajectory
    within 1e-5 A over 100 steps at N = 1415 (as the multi-launch mixed path), and the packed records of the
    multi-launch sweeps are refreshed (a forced re-evaluation agrees)."""
    w = W.config_c2() if n_atoms == 1415 else W.fcc_cluster(n_atoms, 1200.0, seed=900 + n_atoms)
    nsteps = 100 if n_atoms == 1415 else 10
    P = oracle_ld.params()
    ref = oracle_ld.run(w.pos, w.vel, P, dt=1.0, nsteps=nsteps)
    sc = make(scmd, w, 1, precision=scmd.SC_PREC_MIXED)
    sc.sc_forces()
    before = sc.sc_launch_count()
    sc.sc_step(1.0, nsteps)
    assert sc.sc_launch_count() - before == 1
    pos, vel = state(sc)
    assert np.abs(pos - ref["pos"]).max() < 1e-5
    # forces / energy left by the loop against the oracle at the ORACLE's final positions (the two trajectories are
    # within 1e-5 A, which moves a force by < 1e-6 of its size: inside the mixed tolerance)
    rho_o, f_o, (e_o, _, _) = oracle_ld.energy_forces(ref["pos"], P)
    f = sc.sc_forces().cpu().numpy()
    assert np.linalg.norm(f - f_o) <= 1e-5 * np.linalg.norm(f_o)
    assert abs(sc.sc_energy() - e_o) <= 1e-7 * abs(e_o)
    # multi-launch sweeps from the refreshed records: one more step there = one more oracle step (stale records
    # would be off by the ~0.05 A the atoms moved inside the loop)
    sc.sc_set_option(scmd.SC_OPT_PERSISTENT, 2)
    sc.sc_step(1.0, 1)
    ref2 = oracle_ld.run(ref["pos"], ref["vel"], P, dt=1.0, nsteps=1)
    pos2, _ = state(sc)
    assert np.abs(pos2 - ref2["pos"]).max() < 1e-5
    sc.close()


def test_langevin_in_one_launch(scmd, oracle_ld):
    from paper_1210_3559_b200.binding import langevin_thermostat
    w = W.fcc_cluster(555, 900.0, seed=12)
    ref = oracle_ld.run(w.pos, w.vel, oracle_ld.params(), dt=1.0, nsteps=60, thermo_kind=2, T_start=900.0, T_end=700.0,
                        gamma=0.01, seed=99)
    sc = make(scmd, w, 1)
    sc.sc_step(1.0, 60, langevin_thermostat(900.0, 700.0, 0.01, 99))
    pos, vel = state(sc)
    assert np.abs(pos - ref["pos"]).max() < TRAJ_TOL
    assert np.abs(vel - ref["vel"]).max() < 1e-10
    sc.close()


def test_generic_exponents_in_one_launch(scmd, oracle_ld):
    w = W.fcc_cluster(300, 600.0, seed=3)
    kw = dict(n=12, m=5, eps=0.02, c=30.0, a=3.3)
    ref = oracle_ld.run(w.pos, w.vel, oracle_ld.params(**kw), dt=1.0, nsteps=40)
    sc = make(scmd, w, 1, **kw)
    sc.sc_step(1.0, 40)
    pos, _ = state(sc)
    assert np.abs(pos - ref["pos"]).max() < TRAJ_TOL
    sc.close()


def test_forced_beyond_capacity_falls_back(scmd):
    """N above the shared-memory capacity of the loop: option 1 is a request, the multi-launch path runs."""
    w = W.fcc_cluster(7000, 300.0, seed=4)
    sc = make(scmd, w, 1)
    sc.sc_forces()
    before = sc.sc_launch_count()
    sc.sc_step(1.0, 2)
    assert sc.sc_launch_count() - before > 2
    sc.close()
