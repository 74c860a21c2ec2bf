"""libscmd's Langevin thermostat (reading Q18) against the CPU oracle, through the C ABI."""
import math

import numpy as np
import pytest

from paper_1210_3559_b200 import workloads as W

pytestmark = pytest.mark.gpu
TRAJ_TOL = 1e-8                  # Angstrom over 100 steps (BASELINE.json, FP64 path)
GAMMA = 0.01                     # 1/fs = 10 ps^-1


def run_gpu(scmd, w, nsteps_list, T0, T1, seed, gamma=GAMMA, dt=1.0, step0=None, **kw):
    import torch
    from paper_1210_3559_b200.binding import langevin_thermostat
    sc = scmd.SuttonChen(w.n_atoms, **kw)
    sc.sc_set_state(torch.as_tensor(w.pos, device="cuda"), torch.as_tensor(w.vel, device="cuda"))
    if step0 is not None:
        sc.sc_set_option(scmd.SC_OPT_LANGEVIN_STEP, step0)
    for n, a, b in nsteps_list:
        sc.sc_step(dt, n, langevin_thermostat(a, b, gamma, seed))
    pos, vel = sc.sc_get_state()
    out = dict(pos=pos.cpu().numpy(), vel=vel.cpu().numpy(), epot=sc.sc_energy(), ekin=sc.sc_kinetic()[0])
    sc.close()
    return out


def test_langevin_trajectory_c1(scmd, oracle_ld):
    w = W.config_c1()
    ref = oracle_ld.run(w.pos, w.vel, oracle_ld.params(), dt=1.0, nsteps=100, thermo_kind=2, T_start=1000.0, T_end=400.0,
                        gamma=GAMMA, seed=2057)
    out = run_gpu(scmd, w, [(100, 1000.0, 400.0)], None, None, 2057)
    assert np.abs(out["pos"] - ref["pos"]).max() < TRAJ_TOL
    assert np.abs(out["vel"] - ref["vel"]).max() < 1e-10
    assert abs(out["epot"] - ref["epot"][-1]) / abs(ref["epot"][-1]) < 1e-10
    assert abs(out["ekin"] - ref["ekin"][-1]) / abs(ref["ekin"][-1]) < 1e-9


def test_langevin_split_calls_and_resume_c2(scmd, oracle_ld):
    """Ni1415: 40 + 60 steps in two calls at constant T = one 100-step oracle run; a fresh context resumed
    at generator step 40 reproduces the second leg."""
    w = W.config_c2()
    P = oracle_ld.params()
    ref = oracle_ld.run(w.pos, w.vel, P, dt=1.0, nsteps=100, thermo_kind=2, T_start=900.0, T_end=900.0, gamma=GAMMA,
                        seed=(1 << 40) + 7)
    out = run_gpu(scmd, w, [(40, 900.0, 900.0), (60, 900.0, 900.0)], None, None, (1 << 40) + 7)
    assert np.abs(out["pos"] - ref["pos"]).max() < TRAJ_TOL
    mid = oracle_ld.run(w.pos, w.vel, P, dt=1.0, nsteps=40, thermo_kind=2, T_start=900.0, T_end=900.0, gamma=GAMMA,
                        seed=(1 << 40) + 7)
    w2 = W.Workload(name="resume", pos=mid["pos"], vel=mid["vel"], temperature=900.0, seed=0)
    out2 = run_gpu(scmd, w2, [(60, 900.0, 900.0)], None, None, (1 << 40) + 7, step0=40)
    assert np.abs(out2["pos"] - ref["pos"]).max() < TRAJ_TOL


@pytest.mark.parametrize("precision", [0, 1])
def test_langevin_with_cutoff_uses_callers_atom_index(scmd, oracle_ld, precision):
    """The cutoff path reorders atoms internally; the noise of an atom must follow its index in the caller's
    order, so the trajectory equals the oracle's (which never reorders).  skin 0.15 forces rebuilds."""
    w = W.config_c2()
    P = oracle_ld.params(r_cut=7.0)
    ref = oracle_ld.run(w.pos, w.vel, P, dt=1.0, nsteps=60, thermo_kind=2, T_start=2000.0, T_end=1500.0, gamma=GAMMA, seed=99)
    out = run_gpu(scmd, w, [(60, 2000.0, 1500.0)], None, None, 99, r_cut=7.0, skin=0.15, precision=precision)
    tol = TRAJ_TOL if precision == 0 else 2e-4
    assert np.abs(out["pos"] - ref["pos"]).max() < tol


def test_langevin_limits_and_errors(scmd):
    import torch
    from paper_1210_3559_b200.binding import langevin_thermostat
    w = W.config_c1()
    # gamma = 0 is NVE bit for bit
    a = run_gpu(scmd, w, [(20, 700.0, 700.0)], None, None, 5, gamma=0.0)
    sc = scmd.SuttonChen(147)
    sc.sc_set_state(torch.as_tensor(w.pos, device="cuda"), torch.as_tensor(w.vel, device="cuda"))
    sc.sc_step(1.0, 20)
    pos, vel = sc.sc_get_state()
    assert np.array_equal(pos.cpu().numpy(), a["pos"]) and np.array_equal(vel.cpu().numpy(), a["vel"])
    with pytest.raises(scmd.ScError):
        sc.sc_step(1.0, 1, langevin_thermostat(300.0, 300.0, -1.0, 1))
    with pytest.raises(scmd.ScError):
        sc.sc_step(1.0, 1, langevin_thermostat(-5.0, 300.0, 0.01, 1))
    with pytest.raises(scmd.ScError):
        sc.sc_set_option(scmd.SC_OPT_LANGEVIN_STEP, -1)
    # the generator step is readable (exact resume without the caller counting): one-launch loop and multi-launch path
    assert sc.sc_get_option(scmd.SC_OPT_LANGEVIN_STEP) == 0
    sc.sc_step(1.0, 7, langevin_thermostat(300.0, 300.0, 0.01, 1))
    assert sc.sc_get_option(scmd.SC_OPT_LANGEVIN_STEP) == 7
    sc.sc_set_option(scmd.SC_OPT_PERSISTENT, 2)
    sc.sc_step(1.0, 5, langevin_thermostat(300.0, 300.0, 0.01, 1))
    assert sc.sc_get_option(scmd.SC_OPT_LANGEVIN_STEP) == 12
    sc.sc_step(1.0, 3)                                                  # NVE steps do not advance it
    assert sc.sc_get_option(scmd.SC_OPT_LANGEVIN_STEP) == 12
    sc.close()


def test_langevin_equipartition_free_particles(scmd):
    """65,536 non-interacting atoms (spacing 50 A, r_cut 5 A): <v^2> per component -> kB T ACC / m."""
    import torch
    from paper_1210_3559_b200.binding import langevin_thermostat
    n = 65536
    g = np.arange(n)
    pos = np.stack([(g % 64) * 50.0, ((g // 64) % 64) * 50.0, (g // 4096) * 50.0], axis=1).astype(np.float64)
    sc = scmd.SuttonChen(n, r_cut=5.0, skin=1.0)
    sc.sc_set_state(torch.as_tensor(pos, device="cuda"), torch.zeros(n, 3, dtype=torch.float64, device="cuda"))
    sc.sc_step(1.0, 12, langevin_thermostat(1000.0, 1000.0, 0.5, 11))
    _, vel = sc.sc_get_state()
    var = float(vel.var())
    expect = 8.617333262e-5 * 1000.0 * 9.648533215665e-3 / 58.69 * (1 - math.exp(-2 * 0.5 * 12))
    assert abs(var / expect - 1) < 4 * math.sqrt(2 / (3 * n))
    ke, T = sc.sc_kinetic()
    assert abs(T / 1000.0 - 1) < 0.02
    sc.close()
