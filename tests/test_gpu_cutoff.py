"""Parity of the cutoff variant (cell binning, Verlet rows with a skin, list-driven sweeps; SURVEY
section 8a rows a5-a7) against the CPU oracle's all-pairs-with-filter definition (reading Q7: a pair
counts iff r2 < r_c^2, strict, r2 formed in binary64).  Integer results (in-range pair count) are
bit-exact; floating point within BASELINE.json's tolerances."""
import numpy as np
import pytest

from paper_1210_3559_b200 import workloads as W

pytestmark = pytest.mark.gpu

FORCE_TOL = {0: 1e-10, 1: 1e-5}
ENERGY_TOL = {0: 1e-12, 1: 1e-7}
RHO_TOL = {0: 1e-12, 1: 2e-6}
TRAJ_TOL = 1e-8


def rel(a, b):
    return abs(a - b) / max(abs(b), 1e-300)


def rel_l2(a, b):
    return float(np.linalg.norm(np.asarray(a) - np.asarray(b)) / max(np.linalg.norm(b), 1e-300))


def gpu_eval(scmd, pos, vel=None, options=None, **kw):
    import torch
    sc = scmd.SuttonChen(len(pos), **kw)
    for k, v in (options or {}).items():
        sc.sc_set_option(k, v)
    d_pos = torch.as_tensor(np.ascontiguousarray(pos), device="cuda")
    d_vel = None if vel is None else torch.as_tensor(np.ascontiguousarray(vel), device="cuda")
    sc.sc_set_state(d_pos, d_vel)
    rho = sc.sc_density().cpu().numpy()
    f = sc.sc_forces().cpu().numpy()
    e = sc.sc_energy()
    return sc, rho, f, e


def check(scmd, oracle, pos, r_cut, skin=1.0, precision=0, options=None, **params):
    P = oracle.params(r_cut=r_cut, **params)
    rho_o, f_o, (e_o, _, _) = oracle.energy_forces(pos, P)
    npairs_o = oracle.count_pairs(pos, r_cut)
    sc, rho, f, e = gpu_eval(scmd, pos, options=options, r_cut=r_cut, skin=skin, precision=precision, **params)
    stats = sc.sc_stats()
    sc.close()
    assert stats["n_pairs_in_cut"] == npairs_o                          # integer work: bit-exact
    assert stats["n_rebuilds"] == 1
    assert np.all(np.isfinite(f))
    nz = rho_o > 0
    assert np.array_equal(rho[~nz], rho_o[~nz])                         # isolated atoms: exactly 0 (Q9)
    if nz.any():
        assert np.max(np.abs(rho[nz] - rho_o[nz]) / rho_o[nz]) < RHO_TOL[precision]
    if np.linalg.norm(f_o) > 0:
        assert rel_l2(f, f_o) < FORCE_TOL[precision]
    else:
        assert np.all(f == 0.0)
    if e_o != 0.0:
        assert rel(e, e_o) < ENERGY_TOL[precision]
    else:
        assert e == 0.0
    return stats


@pytest.mark.parametrize("precision", [0, 1])
def test_c2_ni1415_rc10(scmd, oracle_ld, precision):
    w = W.config_c2()
    stats = check(scmd, oracle_ld, w.pos, 10.0, precision=precision)
    assert 380 <= stats["max_neighbours"] <= 640                        # fcc: 530 sites within 11 A


@pytest.mark.parametrize("precision", [0, 1])
def test_c3_ni8000_liquid_rc10(scmd, oracle_ld, precision):
    w = W.config_c3()
    check(scmd, oracle_ld, w.pos, 10.0, precision=precision)


@pytest.mark.parametrize("tpa", [4, 8, 16, 32])
@pytest.mark.parametrize("precision", [0, 1])
def test_lanes_per_atom_ragged(scmd, oracle_ld, tpa, precision):
    """Every lanes-per-atom family on N = 2607 (not a multiple of 32 or of the atoms per CTA)."""
    w = W.fcc_cluster(2607, 1500.0, seed=77)
    check(scmd, oracle_ld, w.pos, 10.0, precision=precision, options={scmd.SC_OPT_LANES_PER_ROW: tpa})


@pytest.mark.parametrize("n_atoms", [1, 2, 3, 31, 33, 257])
def test_small_sizes(scmd, oracle_ld, n_atoms):
    w = W.fcc_cluster(n_atoms, 300.0, seed=600 + n_atoms)
    check(scmd, oracle_ld, w.pos, 6.0, skin=0.5)


@pytest.mark.parametrize("r_cut,skin", [(2.0, 0.0), (2.0, 0.3), (3.0, 1.0), (4.4, 0.0), (7.7, 2.0), (60.0, 1.0)])
def test_cutoff_radii(scmd, oracle_ld, r_cut, skin):
    """r_c below the nearest-neighbour distance (everything exactly zero), between shells, and beyond
    the cluster diameter (= all pairs); skin 0 makes list radius = cutoff."""
    w = W.fcc_cluster(900, 300.0, seed=5)
    stats = check(scmd, oracle_ld, w.pos, r_cut, skin=skin)
    if r_cut == 60.0:
        assert stats["n_pairs_in_cut"] == 900 * 899


def test_evaporated_atoms_and_generic_exponents(scmd, oracle_ld):
    """Atoms far outside the cluster are clamped into boundary cells (rho = 0, F = 0 exactly)."""
    w = W.fcc_cluster(700, 300.0, seed=31)
    pos = w.pos.copy()
    pos[5] = [9000.0, -20.0, 3.0]
    pos[77] = [-40.0, 1.0e5, 0.0]
    pos[300] = [12.0, 13.0, -4000.0]
    check(scmd, oracle_ld, pos, 8.0)
    check(scmd, oracle_ld, pos, 7.0, n=12, m=6, eps=0.02, c=30.0, a=3.3)
    check(scmd, oracle_ld, pos, 7.0, n=7, m=3, eps=0.02, c=30.0, a=3.3, precision=1)


def test_capacity_overflow_is_reported_and_recoverable(scmd, oracle_ld):
    """A row longer than its capacity is reported (never truncated); raising the capacity, or new positions, clears
    the condition: the next evaluation rebuilds the rows and is correct."""
    import torch
    w = W.config_c2()
    P = oracle_ld.params(r_cut=10.0)
    _, f_o, (e_o, _, _) = oracle_ld.energy_forces(w.pos, P)
    sc = scmd.SuttonChen(1415, r_cut=10.0, skin=1.0)
    cap_max = sc.sc_get_option(scmd.SC_INFO_NEIGHBOUR_CAPACITY_MAX)
    sc.sc_set_option(scmd.SC_OPT_NEIGHBOUR_CAPACITY, 64)
    assert sc.sc_get_option(scmd.SC_INFO_NEIGHBOUR_CAPACITY) == 64
    sc.sc_set_state(torch.as_tensor(w.pos, device="cuda"))
    with pytest.raises(scmd.ScError) as ei:
        sc.sc_energy()
    assert ei.value.status == 6                                        # SC_ERR_CAPACITY
    with pytest.raises(scmd.ScError):
        sc.sc_set_option(scmd.SC_OPT_NEIGHBOUR_CAPACITY, 1 << 20)      # beyond what the workspace holds
    sc.sc_set_option(scmd.SC_OPT_NEIGHBOUR_CAPACITY, 0)                # back to what the workspace was sized for
    assert sc.sc_get_option(scmd.SC_INFO_NEIGHBOUR_CAPACITY) == cap_max
    assert rel(sc.sc_energy(), e_o) < 1e-12 and rel_l2(sc.sc_forces().cpu().numpy(), f_o) < 1e-10
    assert sc.sc_stats()["n_rebuilds"] == 2
    # overflow again, then sparser positions (2 atoms per row at most) under the same small capacity
    sc.sc_set_option(scmd.SC_OPT_NEIGHBOUR_CAPACITY, 64)
    with pytest.raises(scmd.ScError):
        sc.sc_energy()
    far = w.pos * 4.0
    sc.sc_set_state(torch.as_tensor(far, device="cuda"))
    assert rel(sc.sc_energy(), oracle_ld.energy(far, P)) < 1e-12
    sc.close()


def test_dense_system_needs_a_create_time_capacity(scmd, oracle_ld):
    """1.9 x the fcc density (lattice compressed to 0.807 a): the default rows (1.3 x fcc) overflow; a context created
    with the capacity sc_stats reported evaluates it (sc_create_ex / sc_create_options.neighbour_capacity)."""
    import torch
    pos = W.fcc_cluster(3000, 300.0, seed=41).pos * 0.807
    P = oracle_ld.params(r_cut=10.0)
    _, f_o, (e_o, _, _) = oracle_ld.energy_forces(pos, P)
    sc = scmd.SuttonChen(3000, r_cut=10.0, skin=1.0)
    sc.sc_set_state(torch.as_tensor(pos, device="cuda"))
    with pytest.raises(scmd.ScError) as ei:
        sc.sc_energy()
    assert ei.value.status == 6
    sc.close()
    sc = scmd.SuttonChen(3000, r_cut=10.0, skin=1.0, neighbour_capacity=1100)
    assert sc.sc_get_option(scmd.SC_INFO_NEIGHBOUR_CAPACITY) == 1120    # rounded up to a multiple of 32
    sc.sc_set_state(torch.as_tensor(pos, device="cuda"))
    assert rel(sc.sc_energy(), e_o) < 1e-12 and rel_l2(sc.sc_forces().cpu().numpy(), f_o) < 1e-10
    stats = sc.sc_stats()
    assert 672 < stats["max_neighbours"] <= 1100 and stats["n_pairs_in_cut"] == oracle_ld.count_pairs(pos, 10.0)
    sc.close()


def test_bitwise_deterministic_and_caller_order(scmd):
    """Two contexts give identical bits (the cell sort is canonical, no floating-point atomics), and
    a shuffled input gives the shuffled output."""
    w = W.config_c2()
    _, rho1, f1, e1 = gpu_eval(scmd, w.pos, w.vel, r_cut=10.0, skin=1.0)
    sc, rho2, f2, e2 = gpu_eval(scmd, w.pos, w.vel, r_cut=10.0, skin=1.0)
    assert np.array_equal(rho1, rho2) and np.array_equal(f1, f2) and e1 == e2
    pos, vel = sc.sc_get_state()
    assert np.array_equal(pos.cpu().numpy(), w.pos) and np.array_equal(vel.cpu().numpy(), w.vel)
    sc.close()
    shuffle = np.random.default_rng(3).permutation(1415)
    _, rho3, f3, e3 = gpu_eval(scmd, w.pos[shuffle], r_cut=10.0, skin=1.0)
    assert np.max(np.abs(rho3 - rho1[shuffle]) / rho1[shuffle]) < 1e-13
    assert rel_l2(f3, f1[shuffle]) < 1e-12 and rel(e3, e1) < 1e-13


@pytest.mark.parametrize("skin", [1.0, 0.15])
def test_trajectory_100_steps_with_rebuilds(scmd, oracle_ld, skin):
    """Ni1415 at 2000 K, r_c = 10 A: 100 NVE steps against the oracle's filtered all-pairs run.  With
    skin 0.15 A the rows are rebuilt (and the internal order re-sorted) many times on the way."""
    import torch
    w = W.config_c2()
    P = oracle_ld.params(r_cut=10.0)
    ref = oracle_ld.run(w.pos, w.vel, P, dt=1.0, nsteps=100)
    sc = scmd.SuttonChen(1415, r_cut=10.0, skin=skin)
    sc.sc_set_state(torch.as_tensor(w.pos, device="cuda"), torch.as_tensor(w.vel, device="cuda"))
    sc.sc_step(1.0, 41)
    sc.sc_step(1.0, 59)
    pos, vel = sc.sc_get_state()
    assert np.abs(pos.cpu().numpy() - ref["pos"]).max() < TRAJ_TOL
    assert np.abs(vel.cpu().numpy() - ref["vel"]).max() < 1e-10
    assert rel(sc.sc_energy(), ref["epot"][-1]) < 1e-10
    assert rel(sc.sc_kinetic()[0], ref["ekin"][-1]) < 1e-10
    stats = sc.sc_stats()
    assert stats["n_rebuilds"] >= (10 if skin < 0.5 else 1)
    # forces come back in the caller's order
    f = sc.sc_forces().cpu().numpy()
    _, f_o, _ = oracle_ld.energy_forces(ref["pos"], P)
    assert rel_l2(f, f_o) < 1e-7                                        # positions differ by ~1e-12 A
    # re-seeding positions only keeps the velocities, in the caller's order
    sc.sc_set_state(pos)
    _, vel2 = sc.sc_get_state()
    assert np.array_equal(vel2.cpu().numpy(), vel.cpu().numpy())
    sc.close()


def test_rescale_thermostat_with_cutoff(scmd, oracle_ld):
    import torch
    from paper_1210_3559_b200.binding import rescale_thermostat
    w = W.config_c2()
    P = oracle_ld.params(r_cut=8.0)
    ref = oracle_ld.run(w.pos, w.vel, P, dt=1.0, nsteps=30, thermo_kind=1, T_start=2000.0, T_end=1500.0)
    sc = scmd.SuttonChen(1415, r_cut=8.0, skin=0.2)
    sc.sc_set_state(torch.as_tensor(w.pos, device="cuda"), torch.as_tensor(w.vel, device="cuda"))
    sc.sc_step(1.0, 30, rescale_thermostat(2000.0, 1500.0))
    assert rel(sc.sc_kinetic()[1], 1500.0) < 1e-12
    pos, vel = sc.sc_get_state()
    assert np.abs(pos.cpu().numpy() - ref["pos"]).max() < TRAJ_TOL
    assert np.abs(vel.cpu().numpy() - ref["vel"]).max() < 1e-10
    sc.close()


def test_host_entry_points_with_cutoff(scmd, oracle_ld):
    w = W.config_c2()
    P = oracle_ld.params(r_cut=10.0)
    rho_o, f_o, (e_o, _, _) = oracle_ld.energy_forces(w.pos, P)
    sc = scmd.SuttonChen(1415, r_cut=10.0, skin=1.0)
    f = np.empty((1415, 3)); rho = np.empty(1415)
    e = sc.sc_eval_host(w.pos, f, rho)
    assert rel_l2(f, f_o) < 1e-10 and rel(e, e_o) < 1e-12
    assert np.max(np.abs(rho - rho_o) / rho_o) < 1e-12
    ref = oracle_ld.run(w.pos, w.vel, P, dt=1.0, nsteps=20)
    pos, vel = w.pos.copy(), w.vel.copy()
    out = sc.sc_step_host(pos, vel, 1.0, 20)
    assert np.abs(pos - ref["pos"]).max() < TRAJ_TOL and np.abs(vel - ref["vel"]).max() < 1e-10
    assert rel(out["epot"], ref["epot"][-1]) < 1e-10
    sc.close()


@pytest.fixture(scope="module")
def c4_cut_oracle(oracle_ld):
    w = W.config_c4()
    P = oracle_ld.params(r_cut=10.0)
    rho, f, (e, _, _) = oracle_ld.energy_forces(w.pos, P)
    return w, rho, f, e, oracle_ld.count_pairs(w.pos, 10.0)


@pytest.mark.parametrize("precision", [0, 1])
def test_c4_ni65536_rc10_full_size(scmd, c4_cut_oracle, precision):
    """BASELINE.json config 4, cutoff variant, at full size against the complete oracle evaluation."""
    w, rho_o, f_o, e_o, npairs = c4_cut_oracle
    sc, rho, f, e = gpu_eval(scmd, w.pos, r_cut=10.0, skin=1.0, precision=precision)
    stats = sc.sc_stats()
    sc.close()
    assert stats["n_pairs_in_cut"] == npairs
    assert np.max(np.abs(rho - rho_o) / rho_o) < RHO_TOL[precision]
    assert rel_l2(f, f_o) < FORCE_TOL[precision]
    assert rel(e, e_o) < ENERGY_TOL[precision]


# the largest sweep sizes (N = 262144 and 2^20) are in tests/test_gpu_large.py
