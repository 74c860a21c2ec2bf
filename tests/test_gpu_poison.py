"""The library allocates nothing: its whole workspace is the caller's.  Handing it a workspace whose every byte is
0xFF (NaN as binary64 and binary32, -1 as integers) proves that no kernel reads workspace memory the library has not
written itself -- partial sums of the Newton's-third-law sweeps, neighbour rows and their padding, staging buffers
of the one-launch loop.  (compute-sanitizer's initcheck is not available on this pool.)"""
import numpy as np
import pytest

from paper_1210_3559_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("n_atoms,kw,opts", [
    (149, {}, {}), (1415, dict(precision=1), {}),                          # one-launch loop
    (7003, {}, {}), (7003, {}, {"SC_OPT_NEWTON3": 2}),                     # Newton's third law / one-sided, FP64
    (16391, dict(precision=1), {}), (7003, dict(precision=1), {"SC_OPT_NEWTON3": 2}),   # mixed: Newton's third law / one-sided
    (4101, {}, {}), (2051, {}, {"SC_OPT_NEWTON3": 1, "SC_OPT_PERSISTENT": 2}),   # Newton's third law: the step loop in one launch / smallest carved size, separate launches
    (2967, {}, {}), (2967, dict(precision=1), {}),                         # ... at its default's lower end (2961), both precisions
    (4611, dict(precision=1), {}), (3001, dict(precision=1), {"SC_OPT_NEWTON3": 2}),   # mixed: Newton's third law; one-sided packed sweeps
    (16391, {}, {}),                                                       # just above the one-launch range: four launches per step
    (3001, dict(r_cut=8.0, skin=1.0), {}), (3001, dict(r_cut=8.0, skin=1.0, precision=1), {}),
])
def test_poisoned_workspace(scmd, oracle_ld, n_atoms, kw, opts):
    import torch
    from paper_1210_3559_b200.binding import rescale_thermostat
    w = W.fcc_cluster(n_atoms, 1200.0, seed=17)
    P = oracle_ld.params(r_cut=kw.get("r_cut", 0.0))
    rho_o, f_o, (e_o, _, _) = oracle_ld.energy_forces(w.pos, P)
    sc = scmd.SuttonChen(n_atoms, poison=True, **kw)
    for k, v in opts.items():
        sc.sc_set_option(getattr(scmd, k), v)
    sc.sc_set_state(torch.as_tensor(w.pos, device="cuda"), torch.as_tensor(w.vel, device="cuda"))
    mixed = kw.get("precision", 0) == 1
    e = sc.sc_energy()
    f = sc.sc_forces().cpu().numpy()
    rho = sc.sc_density().cpu().numpy()
    assert np.all(np.isfinite(f)) and np.all(np.isfinite(rho))
    assert abs(e - e_o) <= (1e-7 if mixed else 1e-12) * abs(e_o)
    assert np.linalg.norm(f - f_o) <= (1e-5 if mixed else 1e-10) * np.linalg.norm(f_o)
    sc.sc_step(1.0, 3)
    sc.sc_step(1.0, 2, rescale_thermostat(1200.0, 1100.0))
    pos, vel = sc.sc_get_state()
    ke, T = sc.sc_kinetic()
    counts, n_ref, _ = sc.sc_rdf(6.0, 0.4, 40)
    assert np.all(np.isfinite(pos.cpu().numpy())) and np.all(np.isfinite(vel.cpu().numpy()))
    assert np.isfinite(sc.sc_energy()) and abs(T - 1100.0) < 1e-6 and n_ref > 0 and counts.sum() > 0
    sc.close()
