"""Parity of the CUDA path (through the C ABI) against the CPU oracle, element by element on the
same seeded inputs.  FP64 tolerances from BASELINE.json north_star: relative L2 force error
<= 1e-10, relative energy error <= 1e-12, 100-step trajectories within 1e-8 A."""
import math

import numpy as np
import pytest

from paper_1210_3559_b200 import workloads as W

pytestmark = pytest.mark.gpu

FORCE_TOL = 1e-10
ENERGY_TOL = 1e-12
RHO_TOL = 1e-12          # per-element relative; derived: ~sqrt(N) * 2^-53 accumulation + 2 ulp per term
TRAJ_TOL = 1e-8          # Angstrom, 100 steps


def rel(a, b):
    return abs(a - b) / max(abs(b), 1e-300)


def rel_l2(a, b):
    return float(np.linalg.norm(np.asarray(a) - np.asarray(b)) / max(np.linalg.norm(b), 1e-300))


def gpu_eval(scmd, pos, vel=None, options=None, **params):
    import torch
    sc = scmd.SuttonChen(len(pos), **params)
    for k, v in (options or {}).items():
        sc.sc_set_option(k, v)
    d_pos = torch.as_tensor(np.ascontiguousarray(pos), device="cuda")
    d_vel = None if vel is None else torch.as_tensor(np.ascontiguousarray(vel), device="cuda")
    sc.sc_set_state(d_pos, d_vel)
    rho = sc.sc_density().cpu().numpy()
    f = sc.sc_forces().cpu().numpy()
    e = sc.sc_energy()
    return sc, rho, f, e


def check_eval(scmd, oracle, pos, options=None, **params):
    oparams = {k: v for k, v in params.items()}
    P = oracle.params(**oparams)
    rho_o, f_o, (e_o, _, _) = oracle.energy_forces(pos, P)
    sc, rho, f, e = gpu_eval(scmd, pos, options=options, **params)
    sc.close()
    assert np.all(np.isfinite(f))
    assert np.max(np.abs(rho - rho_o) / np.maximum(np.abs(rho_o), 1e-300)) < RHO_TOL
    assert rel_l2(f, f_o) < FORCE_TOL
    assert rel(e, e_o) < ENERGY_TOL
    return rel_l2(f, f_o), rel(e, e_o)


# --------------------------------------------------------------------------- #
def test_device_reciprocals(scmd):
    """The hand-rolled FP64 1/x and x^-1/2 (MUFU seed + cubic refinement) over the r^2 range of
    any cluster this library accepts are within 2 ulp; the seeds are better than 2^-19."""
    err = scmd.probe_reciprocal(0.5, 1.0e7, 1 << 22)
    assert err["rcp_seed"] < 2.0 ** -19 and err["rsqrt_seed"] < 2.0 ** -19
    assert err["rcp"] < 4.5e-16 and err["rsqrt"] < 4.5e-16


def test_c1_ni147_mackay(scmd, oracle_ld):
    w = W.config_c1()
    check_eval(scmd, oracle_ld, w.pos)


def test_c2_ni1415(scmd, oracle_ld):
    w = W.config_c2()
    check_eval(scmd, oracle_ld, w.pos)


def test_c3_ni8000_liquid(scmd, oracle_ld):
    w = W.config_c3()
    check_eval(scmd, oracle_ld, w.pos)


@pytest.mark.parametrize("it,tpr,warps", [(1, 1, 1), (1, 32, 8), (2, 1, 8), (2, 4, 3), (2, 32, 2), (4, 1, 8),
                                           (4, 4, 5), (1, 8, 7), (2, 16, 4), (1, 2, 6)])
def test_tile_shapes_ragged(scmd, oracle_ld, it, tpr, warps):
    """Every (rows/thread, lanes/row, warps) family on N = 2600: 6 tiles of 512 with a ragged
    tail of 40, rows not a multiple of any rows-per-CTA > 8."""
    w = W.fcc_cluster(2600 + 7, 1500.0, seed=77)
    opts = {scmd.SC_OPT_ROWS_PER_THREAD: it, scmd.SC_OPT_LANES_PER_ROW: tpr, scmd.SC_OPT_WARPS_PER_CTA: warps}
    check_eval(scmd, oracle_ld, w.pos, options=opts)


@pytest.mark.parametrize("n_atoms,kw", [(8192, {}), (9001, {}), (8333, dict(n=12, m=6, eps=0.02, c=30.0, a=3.3)),
                                        (12345, dict(n=7, m=3, eps=0.02, c=30.0, a=3.3)),
                                        (2048, {}), (4097, {}), (5003, {})])   # smallest carved size, the default's lower end
def test_newton3_sweeps(scmd, oracle_ld, n_atoms, kw):
    """Every unordered pair once, its term added to both atoms (csrc/sc_allpairs_n3.cuh): block-aligned and ragged
    sizes (dummy rows and records, diagonal chunks), (9, 6) and generic exponents; same tolerances as the one-sided
    sweeps, and the two agree with each other to rounding."""
    w = W.fcc_cluster(n_atoms, 1500.0, seed=81)
    on = {scmd.SC_OPT_NEWTON3: 1}
    check_eval(scmd, oracle_ld, w.pos, options=on, **kw)
    a = gpu_eval(scmd, w.pos, options=on, **kw)
    b = gpu_eval(scmd, w.pos, options={scmd.SC_OPT_NEWTON3: 2}, **kw)
    a2 = gpu_eval(scmd, w.pos, options=on, **kw)
    for sc in (a[0], b[0], a2[0]):
        sc.close()
    assert rel_l2(a[2], b[2]) < 1e-12 and rel(a[3], b[3]) < 1e-13
    assert np.array_equal(a[1], a2[1]) and np.array_equal(a[2], a2[2]) and a[3] == a2[3]      # bit-reproducible


@pytest.mark.parametrize("precision", [0, 1])
@pytest.mark.parametrize("n_atoms,pieces", [(2048, 16), (2051, 1), (5003, -1), (5003, 3), (5003, 16), (9001, 2),
                                            (9001, -1), (20011, 1), (20011, 16)])
def test_newton3_plans(scmd, oracle_ld, n_atoms, pieces, precision):
    """SC_OPT_NEWTON3_PIECES: the triangle cut into pieces of equal cost (k per SM; several tiles per CTA at the narrow
    end, several CTAs per row block at the wide end, slivers, one-chunk tiles) and the (row block x j segment) grid of
    round 1, both precisions at BASELINE.json's tolerances; invalid values are refused."""
    import torch
    w = W.fcc_cluster(n_atoms, 1500.0, seed=85)
    P = oracle_ld.params()
    rho_o, f_o, (e_o, _, _) = oracle_ld.energy_forces(w.pos, P)
    sc = scmd.SuttonChen(n_atoms, precision=precision)
    sc.sc_set_option(scmd.SC_OPT_NEWTON3, 1)
    sc.sc_set_option(scmd.SC_OPT_NEWTON3_PIECES, pieces)
    assert sc.sc_get_option(scmd.SC_OPT_NEWTON3_PIECES) == pieces
    assert sc.sc_get_option(scmd.SC_INFO_STEP_PATH) == (2 if n_atoms <= 2960 else 1)  # sc_step at the two small sizes: one-launch loop
    sc.sc_set_state(torch.as_tensor(w.pos, device="cuda"))
    rho, f, e = sc.sc_density().cpu().numpy(), sc.sc_forces().cpu().numpy(), sc.sc_energy()
    tol = (RHO_TOL, FORCE_TOL, ENERGY_TOL) if precision == 0 else (2e-6, 1e-5, 1e-7)
    assert np.max(np.abs(rho - rho_o) / rho_o) < tol[0]
    assert rel_l2(f, f_o) < tol[1]
    assert rel(e, e_o) < tol[2]
    # the plan can change under a live context: next evaluation uses the new one, same results to rounding
    sc.sc_set_option(scmd.SC_OPT_NEWTON3_PIECES, 0)
    f2, e2 = sc.sc_forces().cpu().numpy(), sc.sc_energy()
    assert rel_l2(f2, f) < (1e-12 if precision == 0 else 1e-6) and rel(e2, e) < (1e-13 if precision == 0 else 1e-7)
    for bad in (-2, 17):
        with pytest.raises(scmd.ScError):
            sc.sc_set_option(scmd.SC_OPT_NEWTON3_PIECES, bad)
    sc.close()


@pytest.mark.parametrize("precision", [0, 1])
def test_newton3_six_warp_ctas(scmd, oracle_ld, precision):
    """SC_OPT_WARPS_PER_CTA <= 6 with the Newton's-third-law sweeps: CTAs of six warps (two row sets of three warps, the
    pair hand-over on three pairs of named barriers), two CTAs per SM."""
    import torch
    w = W.fcc_cluster(7003, 1500.0, seed=88)
    rho_o, f_o, (e_o, _, _) = oracle_ld.energy_forces(w.pos, oracle_ld.params())
    sc = scmd.SuttonChen(w.n_atoms, precision=precision)
    sc.sc_set_option(scmd.SC_OPT_NEWTON3, 1)
    sc.sc_set_option(scmd.SC_OPT_WARPS_PER_CTA, 6)
    sc.sc_set_state(torch.as_tensor(w.pos, device="cuda"))
    rho, f, e = sc.sc_density().cpu().numpy(), sc.sc_forces().cpu().numpy(), sc.sc_energy()
    sc.close()
    tol = (RHO_TOL, FORCE_TOL, ENERGY_TOL) if precision == 0 else (2e-6, 1e-5, 1e-7)
    assert np.max(np.abs(rho - rho_o) / rho_o) < tol[0]
    assert rel_l2(f, f_o) < tol[1]
    assert rel(e, e_o) < tol[2]


def test_newton3_trajectory(scmd, oracle_ld):
    """100 velocity-Verlet steps at N = 8192 through the Newton's-third-law sweeps: positions within 1e-8 A."""
    import torch
    w = W.fcc_cluster(8192, 1200.0, seed=82)
    ref = oracle_ld.run(w.pos, w.vel, oracle_ld.params(), dt=1.0, nsteps=100)
    sc = scmd.SuttonChen(8192)
    sc.sc_set_option(scmd.SC_OPT_NEWTON3, 1)
    sc.sc_set_state(torch.as_tensor(w.pos, device="cuda"), torch.as_tensor(w.vel, device="cuda"))
    sc.sc_step(1.0, 100)
    pos, _ = sc.sc_get_state()
    assert np.abs(pos.cpu().numpy() - ref["pos"]).max() < TRAJ_TOL
    assert rel(sc.sc_energy(), ref["epot"][-1]) < 1e-10
    sc.close()


@pytest.mark.parametrize("precision", [0, 1])
@pytest.mark.parametrize("n_atoms", [2961, 5003, 12288])
def test_newton3_step_loop(scmd, oracle_ld, n_atoms, precision):
    """n3_loop_kernel (csrc/sc_n3_loop.cuh): NVE sc_step calls through the Newton's-third-law sweeps in one cooperative
    launch.  Same device functions, same sums in the same order as the four launches per step (SC_OPT_PERSISTENT = 2),
    so positions, velocities, forces and energies agree bit for bit, also over split calls; and against the oracle."""
    import torch
    w = W.fcc_cluster(n_atoms, 1200.0, seed=86)
    out = {}
    for mode in (0, 2):
        sc = scmd.SuttonChen(n_atoms, precision=precision)
        sc.sc_set_option(scmd.SC_OPT_PERSISTENT, mode)
        assert sc.sc_get_option(scmd.SC_INFO_STEP_PATH) == 1
        sc.sc_set_state(torch.as_tensor(w.pos, device="cuda"), torch.as_tensor(w.vel, device="cuda"))
        sc.sc_forces()
        before = sc.sc_launch_count()
        sc.sc_step(1.0, 7)
        used = sc.sc_launch_count() - before
        assert used == 5 if mode == 0 else used >= 4 * 7   # first half kick + drift, the loop, three scalar reductions
        sc.sc_step(1.0, 1)
        sc.sc_step(1.0, 12)
        pos, vel = sc.sc_get_state()
        out[mode] = (pos.cpu().numpy(), vel.cpu().numpy(), sc.sc_forces().cpu().numpy(), sc.sc_energy(), sc.sc_kinetic()[0],
                     sc.sc_density().cpu().numpy())
        sc.close()
    for a, b in zip(out[0], out[2]):
        assert np.array_equal(a, b)
    ref = oracle_ld.run(w.pos, w.vel, oracle_ld.params(), dt=1.0, nsteps=20)
    assert np.abs(out[0][0] - ref["pos"]).max() < (TRAJ_TOL if precision == 0 else 1e-5)
    assert rel(out[0][3], ref["epot"][-1]) < (1e-10 if precision == 0 else 1e-7)
    assert rel(out[0][4], ref["ekin"][-1]) < (1e-10 if precision == 0 else 1e-6)


@pytest.mark.parametrize("precision", [0, 1])
def test_newton3_step_loop_rescale(scmd, oracle_ld, precision):
    """Velocity rescaling inside n3_loop_kernel (BASELINE.json config 3's cooling ramp runs through it): two ramps and
    an NVE leg in separate calls against the oracle's runs, the temperature on target after every call, and the
    separate-launch path (SC_OPT_PERSISTENT = 2) to rounding."""
    import torch
    from paper_1210_3559_b200.binding import rescale_thermostat
    n_atoms = 2500
    w = W.fcc_cluster(n_atoms, 2000.0, seed=87)
    P = oracle_ld.params()
    legs = [(25, 1, 2000.0, 1800.0), (10, 1, 1800.0, 1850.0), (5, 0, 0.0, 0.0)]
    pos, vel = w.pos, w.vel
    for n, kind, a, b in legs:
        ref = oracle_ld.run(pos, vel, P, dt=1.0, nsteps=n, thermo_kind=kind, T_start=a, T_end=b)
        pos, vel = ref["pos"], ref["vel"]
    out = {}
    for mode in (0, 2):
        sc = scmd.SuttonChen(n_atoms, precision=precision)
        sc.sc_set_option(scmd.SC_OPT_PERSISTENT, mode)
        sc.sc_set_state(torch.as_tensor(w.pos, device="cuda"), torch.as_tensor(w.vel, device="cuda"))
        sc.sc_forces()
        for n, kind, a, b in legs:
            before = sc.sc_launch_count()
            sc.sc_step(1.0, n, rescale_thermostat(a, b) if kind else None)
            if mode == 0:
                assert sc.sc_launch_count() - before <= 7      # kick + drift, the loop, 3 reductions, the pending scale
            if kind:
                assert abs(sc.sc_kinetic()[1] - b) < 1e-9
        gpos, gvel = sc.sc_get_state()
        out[mode] = (gpos.cpu().numpy(), gvel.cpu().numpy(), sc.sc_energy())
        sc.close()
    assert np.abs(out[0][0] - pos).max() < (TRAJ_TOL if precision == 0 else 1e-5)
    assert np.abs(out[0][1] - vel).max() < (1e-10 if precision == 0 else 1e-6)
    assert rel(out[0][2], ref["epot"][-1]) < (1e-10 if precision == 0 else 1e-7)
    assert np.abs(out[0][0] - out[2][0]).max() < (1e-12 if precision == 0 else 1e-7)


def test_step_path_queries(scmd):
    """SC_INFO_STEP_PATH / SC_INFO_ONE_LAUNCH tell which kernels a context runs as configured (bench.py asks them
    instead of repeating the library's thresholds)."""
    cases = [  # (N, kwargs, options, path, one_launch)
        (147, {}, {}, 2, 1), (2960, {}, {}, 2, 1), (2961, {}, {}, 1, 1), (16384, dict(precision=1), {}, 1, 1),
        (16385, {}, {}, 1, 0), (5003, {}, {scmd.SC_OPT_PERSISTENT: 2}, 1, 0), (5003, {}, {scmd.SC_OPT_NEWTON3: 2}, 0, 0),
        (5003, {}, {scmd.SC_OPT_NEWTON3_PIECES: -1}, 1, 0), (1415, {}, {scmd.SC_OPT_PERSISTENT: 2}, 0, 0),
        (3001, dict(r_cut=8.0, skin=1.0), {}, 3, 0),
    ]
    for n, kw, opts, path, one in cases:
        sc = scmd.SuttonChen(n, **kw)
        for k, v in opts.items():
            sc.sc_set_option(k, v)
        assert sc.sc_get_option(scmd.SC_INFO_STEP_PATH) == path, (n, kw, opts)
        assert sc.sc_get_option(scmd.SC_INFO_ONE_LAUNCH) == one, (n, kw, opts)
        sc.close()


@pytest.mark.parametrize("n_atoms", [1, 2, 3, 31, 33, 511, 512, 513, 1025])
def test_small_and_boundary_sizes(scmd, oracle_ld, n_atoms):
    """Degenerate and tile-boundary sizes.  N = 1: rho = 0, F = 0, U = 0 (reading Q9)."""
    w = W.fcc_cluster(n_atoms, 300.0, seed=500 + n_atoms)
    if n_atoms == 1:
        sc, rho, f, e = gpu_eval(scmd, w.pos)
        sc.close()
        assert rho[0] == 0.0 and np.all(f == 0.0) and e == 0.0
        return
    check_eval(scmd, oracle_ld, w.pos)


def test_dimer_closed_form_on_gpu(scmd):
    eps, c, a = 1.5707e-2, 39.432, 3.52
    r = 2.49
    sc, rho, f, e = gpu_eval(scmd, np.array([[0.0, 0, 0], [r, 0, 0]]))
    sc.close()
    u = a / r
    assert rel(e, eps * (u ** 9 - 2 * c * u ** 3)) < 1e-14
    assert rel(f[1, 0], eps * (9 * u ** 9 - 6 * c * u ** 3) / r) < 1e-13
    assert f[0, 0] == -f[1, 0] and rel(rho[0], u ** 6) < 1e-15


@pytest.mark.parametrize("n,m", [(12, 6), (10, 8), (7, 3), (9, 5)])
def test_generic_exponents(scmd, oracle_ld, n, m):
    w = W.fcc_cluster(700, 300.0, seed=31)
    check_eval(scmd, oracle_ld, w.pos, n=n, m=m, eps=0.02, c=30.0, a=3.3)


def test_bitwise_deterministic_and_state_roundtrip(scmd):
    import torch
    w = W.config_c2()
    sc, rho, f, e = gpu_eval(scmd, w.pos, w.vel)
    pos2, vel2 = sc.sc_get_state()
    assert np.array_equal(pos2.cpu().numpy(), w.pos) and np.array_equal(vel2.cpu().numpy(), w.vel)
    sc.close()
    _, rho2, f2, e2 = gpu_eval(scmd, w.pos, w.vel)
    assert np.array_equal(rho, rho2) and np.array_equal(f, f2) and e == e2


def test_trajectory_100_steps_c1(scmd, oracle_ld):
    import torch
    w = W.config_c1()
    ref = oracle_ld.run(w.pos, w.vel, oracle_ld.params(), dt=1.0, nsteps=100)
    sc = scmd.SuttonChen(147)
    sc.sc_set_state(torch.as_tensor(w.pos, device="cuda"), torch.as_tensor(w.vel, device="cuda"))
    sc.sc_step(1.0, 100)
    pos, vel = sc.sc_get_state()
    assert np.abs(pos.cpu().numpy() - ref["pos"]).max() < TRAJ_TOL
    assert np.abs(vel.cpu().numpy() - ref["vel"]).max() < 1e-10
    assert rel(sc.sc_energy(), ref["epot"][-1]) < 1e-10
    ke, T = sc.sc_kinetic()
    assert rel(ke, ref["ekin"][-1]) < 1e-10
    sc.close()


def test_trajectory_100_steps_c2_split_calls(scmd, oracle_ld):
    """Ni1415 at 2000 K; the GPU run is split 37 + 63 to check that sc_step composes."""
    import torch
    w = W.config_c2()
    ref = oracle_ld.run(w.pos, w.vel, oracle_ld.params(), dt=1.0, nsteps=100)
    sc = scmd.SuttonChen(1415)
    sc.sc_set_state(torch.as_tensor(w.pos, device="cuda"), torch.as_tensor(w.vel, device="cuda"))
    sc.sc_step(1.0, 37)
    sc.sc_step(1.0, 63)
    pos, _ = sc.sc_get_state()
    assert np.abs(pos.cpu().numpy() - ref["pos"]).max() < TRAJ_TOL
    sc.close()


def test_nve_energy_conservation_and_reversal(scmd):
    import torch
    w = W.config_c1()
    sc = scmd.SuttonChen(147)
    sc.sc_set_state(torch.as_tensor(w.pos, device="cuda"), torch.as_tensor(w.vel, device="cuda"))
    e0 = sc.sc_energy() + sc.sc_kinetic()[0]
    worst = 0.0
    for _ in range(10):
        sc.sc_step(1.0, 100)
        worst = max(worst, abs(sc.sc_energy() + sc.sc_kinetic()[0] - e0))
    assert worst / abs(e0) < 2e-5
    # time reversal: 100 steps forward from the start, flip v, 100 steps
    sc.sc_set_state(torch.as_tensor(w.pos, device="cuda"), torch.as_tensor(w.vel, device="cuda"))
    sc.sc_step(1.0, 100)
    pos, vel = sc.sc_get_state()
    sc.sc_set_state(pos, -vel)
    sc.sc_step(1.0, 100)
    pos, vel = sc.sc_get_state()
    assert np.abs(pos.cpu().numpy() - w.pos).max() < 1e-10
    sc.close()


def test_rescale_thermostat_ramp(scmd, oracle_ld):
    import torch
    from paper_1210_3559_b200.binding import rescale_thermostat
    w = W.config_c1()
    ref = oracle_ld.run(w.pos, w.vel, oracle_ld.params(), dt=1.0, nsteps=40, thermo_kind=1, T_start=1000.0, T_end=600.0)
    sc = scmd.SuttonChen(147)
    sc.sc_set_state(torch.as_tensor(w.pos, device="cuda"), torch.as_tensor(w.vel, device="cuda"))
    sc.sc_step(1.0, 40, rescale_thermostat(1000.0, 600.0))
    ke, T = sc.sc_kinetic()
    assert rel(T, 600.0) < 1e-12
    pos, vel = sc.sc_get_state()
    assert np.abs(pos.cpu().numpy() - ref["pos"]).max() < TRAJ_TOL
    assert np.abs(vel.cpu().numpy() - ref["vel"]).max() < 1e-10
    sc.close()


def test_host_entry_points(scmd, oracle_ld):
    w = W.config_c2()
    P = oracle_ld.params()
    rho_o, f_o, (e_o, _, _) = oracle_ld.energy_forces(w.pos, P)
    sc = scmd.SuttonChen(1415)
    f = np.empty((1415, 3)); rho = np.empty(1415)
    e = sc.sc_eval_host(w.pos, f, rho)
    assert rel_l2(f, f_o) < FORCE_TOL and rel(e, e_o) < ENERGY_TOL
    assert np.max(np.abs(rho - rho_o) / rho_o) < RHO_TOL
    ref = oracle_ld.run(w.pos, w.vel, P, dt=1.0, nsteps=20)
    pos, vel = w.pos.copy(), w.vel.copy()
    out = sc.sc_step_host(pos, vel, 1.0, 20)
    assert np.abs(pos - ref["pos"]).max() < TRAJ_TOL
    assert rel(out["epot"], ref["epot"][-1]) < 1e-10 and rel(out["ekin"], ref["ekin"][-1]) < 1e-10
    assert sc.sc_launch_count() > 0
    sc.close()


def test_error_paths(scmd):
    import torch
    sc = scmd.SuttonChen(10)
    with pytest.raises(scmd.ScError) as ei:
        sc.sc_energy()
    assert ei.value.status == 4                                       # SC_ERR_STATE: no positions
    pos = torch.as_tensor(W.fcc_sphere(10), device="cuda")
    sc.sc_set_state(pos)
    with pytest.raises(scmd.ScError) as ei:
        sc.sc_step(1.0, 1)
    assert ei.value.status == 4                                       # velocities never set
    sc.sc_set_state(pos, torch.zeros_like(pos))
    with pytest.raises(scmd.ScError) as ei:
        sc.sc_step(-1.0, 1)
    assert ei.value.status == 1
    bad = pos.clone(); bad[3] = bad[7]                                 # coincident atoms (Q10)
    sc.sc_set_state(bad)
    with pytest.raises(scmd.ScError) as ei:
        sc.sc_energy()
    assert ei.value.status == 5
    sc.close()
    with pytest.raises(scmd.ScError):
        scmd.SuttonChen(10, n=6, m=9)


@pytest.fixture(scope="module")
def c4_oracle(oracle_ld):
    w = W.config_c4()
    rho, f, (e, _, _) = oracle_ld.energy_forces(w.pos, oracle_ld.params())
    return w, rho, f, e


def test_c4_ni65536_full_size(scmd, c4_oracle):
    """BASELINE.json config 4 at full size, in the launch configuration bench.py times, against
    the complete oracle evaluation (every row, not a sample)."""
    import torch
    w, rho_o, f_o, e_o = c4_oracle
    sc, rho, f, e = gpu_eval(scmd, w.pos)
    assert np.max(np.abs(rho - rho_o) / rho_o) < RHO_TOL
    assert rel_l2(f, f_o) < FORCE_TOL
    assert rel(e, e_o) < ENERGY_TOL
    assert sc.sc_stats()["n_pairs_in_cut"] == 65536 * 65535
    sc.close()
