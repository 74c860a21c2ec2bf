"""Parity of the mixed-precision all-pairs sweeps (binary32 pair arithmetic on split coordinates,
binary64 accumulation) against the CPU oracle.  Tolerances from BASELINE.json north_star: relative L2
force error <= 1e-5, relative energy error <= 1e-7."""
import numpy as np
import pytest

from paper_1210_3559_b200 import workloads as W

pytestmark = pytest.mark.gpu

FORCE_TOL = 1e-5
ENERGY_TOL = 1e-7
RHO_TOL = 2e-6      # per element: ~6 roundings of 2^-24 per term, terms all positive


def rel(a, b):
    return abs(a - b) / max(abs(b), 1e-300)


def rel_l2(a, b):
    return float(np.linalg.norm(np.asarray(a) - np.asarray(b)) / max(np.linalg.norm(b), 1e-300))


def gpu_eval(scmd, pos, vel=None, options=None, **params):
    import torch
    sc = scmd.SuttonChen(len(pos), precision=scmd.SC_PREC_MIXED, **params)
    for k, v in (options or {}).items():
        sc.sc_set_option(k, v)
    d_pos = torch.as_tensor(np.ascontiguousarray(pos), device="cuda")
    d_vel = None if vel is None else torch.as_tensor(np.ascontiguousarray(vel), device="cuda")
    sc.sc_set_state(d_pos, d_vel)
    rho = sc.sc_density().cpu().numpy()
    f = sc.sc_forces().cpu().numpy()
    e = sc.sc_energy()
    return sc, rho, f, e


def check_eval(scmd, oracle, pos, options=None, energy_tol=ENERGY_TOL, **params):
    P = oracle.params(**params)
    rho_o, f_o, (e_o, _, _) = oracle.energy_forces(pos, P)
    sc, rho, f, e = gpu_eval(scmd, pos, options=options, **params)
    sc.close()
    assert np.all(np.isfinite(f))
    errs = (float(np.max(np.abs(rho - rho_o) / rho_o)), rel_l2(f, f_o), rel(e, e_o))
    assert errs[0] < RHO_TOL and errs[1] < FORCE_TOL and errs[2] < energy_tol, errs
    return errs


def test_c2_ni1415_mixed(scmd, oracle_ld):
    check_eval(scmd, oracle_ld, W.config_c2().pos)


def test_c1_ni147_mixed(scmd, oracle_ld):
    """The perfect icosahedron: forces are small differences of large symmetric sums; still in tolerance."""
    check_eval(scmd, oracle_ld, W.config_c1().pos)


def test_c3_ni8000_liquid_mixed(scmd, oracle_ld):
    check_eval(scmd, oracle_ld, W.config_c3().pos)


def test_far_from_origin(scmd, oracle_ld):
    """The whole cluster displaced by (3000, -2000, 1000) A: split coordinates keep the displacement
    exact where plain binary32 positions (ulp 2.4e-4 A at 3000 A) would be useless."""
    w = W.config_c2()
    check_eval(scmd, oracle_ld, w.pos + np.array([3000.0, -2000.0, 1000.0]))


@pytest.mark.parametrize("it,tpr,warps", [(1, 1, 1), (1, 32, 8), (2, 1, 8), (2, 4, 3), (2, 32, 2), (4, 1, 8),
                                           (4, 4, 5), (1, 8, 7), (2, 16, 4), (1, 2, 6)])
def test_tile_shapes_ragged_mixed(scmd, oracle_ld, it, tpr, warps):
    w = W.fcc_cluster(2607, 1500.0, seed=77)
    opts = {scmd.SC_OPT_ROWS_PER_THREAD: it, scmd.SC_OPT_LANES_PER_ROW: tpr, scmd.SC_OPT_WARPS_PER_CTA: warps}
    check_eval(scmd, oracle_ld, w.pos, options=opts)


@pytest.mark.parametrize("n_atoms", [1, 2, 3, 33, 511, 513])
def test_small_and_boundary_sizes_mixed(scmd, oracle_ld, n_atoms):
    w = W.fcc_cluster(n_atoms, 300.0, seed=500 + n_atoms)
    if n_atoms == 1:
        sc, rho, f, e = gpu_eval(scmd, w.pos)
        sc.close()
        assert rho[0] == 0.0 and np.all(f == 0.0) and e == 0.0
        return
    # 1e-7 on the energy is BASELINE.json's bound for its mixed configs (N >= 1415), where the per-term
    # binary32 roundings (a few 2^-24 each) average out over ~N * 100 significant terms; a dimer has ONE
    # term, so the bound for tiny clusters is the per-term one: 8 roundings * 2^-24 ~ 5e-7
    check_eval(scmd, oracle_ld, w.pos, energy_tol=ENERGY_TOL if n_atoms >= 500 else 5e-7)


@pytest.mark.parametrize("n,m", [(12, 6), (10, 8), (7, 3)])
def test_generic_exponents_mixed(scmd, oracle_ld, n, m):
    w = W.fcc_cluster(700, 300.0, seed=31)
    check_eval(scmd, oracle_ld, w.pos, n=n, m=m, eps=0.02, c=30.0, a=3.3, energy_tol=2e-7)


@pytest.mark.parametrize("n_atoms,kw", [(8192, {}), (9001, {}), (8333, dict(n=12, m=6, eps=0.02, c=30.0, a=3.3)),
                                        (13400, {}),
                                        (2048, {}), (4609, {}), (5003, {})])   # smallest carved size, the default's lower end
def test_newton3_sweeps_mixed(scmd, oracle_ld, n_atoms, kw):
    """The Newton's-third-law sweeps in mixed precision (binary32 rotation on split records, binary64 sums):
    BASELINE.json's mixed tolerances, and agreement with the one-sided mixed sweeps."""
    w = W.fcc_cluster(n_atoms, 1500.0, seed=83)
    P = oracle_ld.params(**kw)
    rho_o, f_o, (e_o, _, _) = oracle_ld.energy_forces(w.pos, P)
    out = {}
    for mode in (1, 2):
        sc, rho, f, e = gpu_eval(scmd, w.pos, options={scmd.SC_OPT_NEWTON3: mode}, **kw)
        sc.close()
        assert float(np.max(np.abs(rho - rho_o) / rho_o)) < RHO_TOL
        assert rel_l2(f, f_o) < FORCE_TOL and rel(e, e_o) < ENERGY_TOL
        out[mode] = (f, e)
    assert rel_l2(out[1][0], out[2][0]) < 5e-6


def test_nve_drift_and_trajectory_mixed(scmd, oracle_ld):
    """Ni1415 at 2000 K, 100 NVE steps: total energy conserved to the velocity-Verlet level and the
    trajectory stays within 1e-5 A of the binary64 oracle (the 1e-8 A bound is the FP64 path's)."""
    import torch
    w = W.config_c2()
    ref = oracle_ld.run(w.pos, w.vel, oracle_ld.params(), dt=1.0, nsteps=100)
    sc = scmd.SuttonChen(1415, precision=scmd.SC_PREC_MIXED)
    sc.sc_set_state(torch.as_tensor(w.pos, device="cuda"), torch.as_tensor(w.vel, device="cuda"))
    e0 = sc.sc_energy() + sc.sc_kinetic()[0]
    sc.sc_step(1.0, 100)
    e1 = sc.sc_energy() + sc.sc_kinetic()[0]
    assert abs(e1 - e0) / abs(e0) < 2e-5
    pos, _ = sc.sc_get_state()
    assert np.abs(pos.cpu().numpy() - ref["pos"]).max() < 1e-5
    assert rel(e1, ref["epot"][-1] + ref["ekin"][-1]) < 1e-6
    sc.close()


def test_c4_ni65536_full_size_mixed(scmd, oracle_ld):
    """BASELINE.json config 4 at full size in the launch configuration bench.py times."""
    w = W.config_c4()
    rho_o, f_o, (e_o, _, _) = oracle_ld.energy_forces(w.pos, oracle_ld.params())
    sc, rho, f, e = gpu_eval(scmd, w.pos)
    sc.close()
    errs = (float(np.max(np.abs(rho - rho_o) / rho_o)), rel_l2(f, f_o), rel(e, e_o))
    print("mixed N=65536 errors (rho max, force L2, energy):", errs)
    assert errs[0] < RHO_TOL and errs[1] < FORCE_TOL and errs[2] < ENERGY_TOL, errs


def test_split_records_refreshed_by_the_one_launch_loop(scmd, oracle_ld):
    """Mixed N = 2057 (the one-launch loop by default): after sc_step, switching the sweeps to Newton's third law
    (which read the RecF split records) and re-evaluating WITHOUT new positions must see the stepped positions."""
    import torch
    w = W.mackay_cluster(8, 1000.0, 1001)
    sc = scmd.SuttonChen(w.n_atoms, precision=scmd.SC_PREC_MIXED)
    sc.sc_set_state(torch.as_tensor(w.pos, device="cuda"), torch.as_tensor(w.vel, device="cuda"))
    assert sc.sc_get_option(scmd.SC_INFO_STEP_PATH) == 2
    sc.sc_step(1.0, 25)
    pos, _ = sc.sc_get_state()
    sc.sc_set_option(scmd.SC_OPT_NEWTON3, 1)                           # invalidates forces, repacks nothing
    f = sc.sc_forces().cpu().numpy()
    e = sc.sc_energy()
    sc.close()
    _, f_o, (e_o, _, _) = oracle_ld.energy_forces(pos.cpu().numpy(), oracle_ld.params())
    assert rel_l2(f, f_o) < FORCE_TOL and rel(e, e_o) < ENERGY_TOL
