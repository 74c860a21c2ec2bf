"""Row split of the all-pairs path (include/scmd.h: sc_step_rows) against the CPU oracle.

One GPU is all this pool has, so the ranks of a split are run ONE AFTER THE OTHER on it, each with its own libscmd
context (its own row range) and its own all-atoms arrays, and the all-gathers are done by copying the owners' rows
between those arrays -- the data flow of RowSplitSuttonChen.step with the collective written out.  No kernel waits on
another.  The test with real NCCL ranks runs only where two GPUs are visible."""
import os
import socket
import subprocess
import sys
from pathlib import Path

import numpy as np
import pytest

from paper_1210_3559_b200 import workloads as W

pytestmark = pytest.mark.gpu
ROOT = Path(__file__).resolve().parent.parent


def rel_l2(a, b):
    return float(np.linalg.norm(np.asarray(a) - np.asarray(b)) / max(np.linalg.norm(b), 1e-300))


class EmulatedSplit:
    def __init__(self, scmd, w, world, **kw):
        import torch
        from paper_1210_3559_b200.distributed import row_range
        self.n, self.world = w.n_atoms, world
        self.ranges = [row_range(self.n, r, world) for r in range(world)]
        self.ctx = [scmd.SuttonChen(self.n, row_begin=b, row_end=e, **kw) for b, e, _ in self.ranges]
        pad = world * self.ranges[0][2]
        self.pos = [torch.zeros(pad, 3, dtype=torch.float64, device="cuda") for _ in range(world)]
        self.rho = [torch.zeros(pad, dtype=torch.float64, device="cuda") for _ in range(world)]
        d_pos, d_vel = torch.as_tensor(w.pos, device="cuda"), torch.as_tensor(w.vel, device="cuda")
        for r in range(world):
            self.pos[r][: self.n].copy_(d_pos)
            self.ctx[r].sc_set_state(self.pos[r][: self.n].contiguous(), d_vel)
        self.evaluate(0.0)

    def gather(self, bufs):                       # the all-gather, written out: every rank receives every owner's rows
        for r, (b, e, _) in enumerate(self.ranges):
            for q in range(self.world):
                if q != r:
                    bufs[q][b:e].copy_(bufs[r][b:e])

    def evaluate(self, dt, th=None):
        for r in range(self.world):
            self.ctx[r].sc_step_rows(1, dt, self.pos[r], self.rho[r], th)
        self.gather(self.rho)
        for r in range(self.world):
            self.ctx[r].sc_step_rows(2, dt, self.pos[r], self.rho[r], th)

    def step(self, dt, nsteps, th=None):
        for _ in range(nsteps):
            for r in range(self.world):
                self.ctx[r].sc_step_rows(0, dt, self.pos[r], self.rho[r], th)
            self.gather(self.pos)
            self.evaluate(dt, th)

    def forces(self):
        f = np.zeros((self.n, 3))
        for r, (b, e, _) in enumerate(self.ranges):
            f[b:e] = self.ctx[r].sc_forces().cpu().numpy()[b:e]
        return f

    def velocities(self):
        v = np.zeros((self.n, 3))
        for r, (b, e, _) in enumerate(self.ranges):
            v[b:e] = self.ctx[r].sc_get_state()[1].cpu().numpy()[b:e]
        return v

    def energy(self):
        return sum(c.sc_energy() for c in self.ctx)

    def kinetic(self):
        return sum(c.sc_kinetic()[0] for c in self.ctx)

    def close(self):
        for c in self.ctx:
            c.close()


@pytest.mark.parametrize("n_atoms,world,precision", [(3001, 2, 0), (3001, 3, 0), (8192, 4, 0), (3001, 2, 1), (257, 8, 0)])
def test_row_split_against_oracle(scmd, oracle_ld, n_atoms, world, precision):
    """Forces, energy (sum of the ranks' shares) and a 20-step NVE trajectory: FP64 at the FP64 tolerances (the sums of
    a row do not depend on how the rows are split: the trajectory is the one-GPU one to rounding), mixed at the mixed ones."""
    w = W.fcc_cluster(n_atoms, 1200.0, seed=300 + n_atoms)
    P = oracle_ld.params()
    rho_o, f_o, (e_o, _, _) = oracle_ld.energy_forces(w.pos, P)
    sp = EmulatedSplit(scmd, w, world, precision=precision)
    ftol, etol, xtol = (1e-10, 1e-12, 1e-8) if precision == 0 else (1e-5, 1e-7, 1e-5)
    assert rel_l2(sp.forces(), f_o) < ftol
    assert abs(sp.energy() - e_o) < etol * abs(e_o)
    rho = sp.rho[0][:n_atoms].cpu().numpy()                         # after the exchange every rank holds all densities
    assert np.max(np.abs(rho - rho_o) / rho_o) < (1e-12 if precision == 0 else 2e-6)
    for r in range(1, world):
        assert np.array_equal(sp.rho[r][:n_atoms].cpu().numpy(), rho)
    ref = oracle_ld.run(w.pos, w.vel, P, dt=1.0, nsteps=20)
    sp.step(1.0, 20)
    for r in range(world):                                          # every rank ends with ALL positions, bit-identical
        assert np.array_equal(sp.pos[r][:n_atoms].cpu().numpy(), sp.pos[0][:n_atoms].cpu().numpy())
    assert np.abs(sp.pos[0][:n_atoms].cpu().numpy() - ref["pos"]).max() < xtol
    assert np.abs(sp.velocities() - ref["vel"]).max() < (1e-10 if precision == 0 else 1e-7)
    assert abs(sp.energy() - ref["epot"][-1]) < (1e-10 if precision == 0 else 1e-6) * abs(ref["epot"][-1])
    assert abs(sp.kinetic() - ref["ekin"][-1]) < (1e-10 if precision == 0 else 1e-6) * ref["ekin"][-1]
    sp.close()


def test_row_split_equals_one_gpu_bitwise_and_langevin(scmd, oracle_ld):
    """The rows of a split are computed by the same kernels in the same order as on one GPU with the one-sided sweeps:
    forces agree to the bit.  The Langevin update is local to an atom (counter = atom index): the split trajectory is
    the oracle's."""
    import torch
    from paper_1210_3559_b200.binding import langevin_thermostat
    w = W.fcc_cluster(2500, 900.0, seed=11)
    one = scmd.SuttonChen(2500, newton3_storage=2)
    one.sc_set_option(scmd.SC_OPT_PERSISTENT, 2)
    one.sc_set_state(torch.as_tensor(w.pos, device="cuda"), torch.as_tensor(w.vel, device="cuda"))
    f1 = one.sc_forces().cpu().numpy()
    one.close()
    sp = EmulatedSplit(scmd, w, 1)                                   # one rank owning all rows: the same launch shapes
    assert np.array_equal(sp.forces(), f1)
    sp.close()
    sp = EmulatedSplit(scmd, w, 3)
    assert rel_l2(sp.forces(), f1) < 1e-14                           # other row blocks per launch, same sums per row
    th = langevin_thermostat(900.0, 900.0, 0.01, 77)
    ref = oracle_ld.run(w.pos, w.vel, oracle_ld.params(), dt=1.0, nsteps=15, thermo_kind=2, T_start=900.0, T_end=900.0,
                        gamma=0.01, seed=77)
    sp.step(1.0, 15, th)
    assert np.abs(sp.pos[1][:2500].cpu().numpy() - ref["pos"]).max() < 1e-8
    assert np.abs(sp.velocities() - ref["vel"]).max() < 1e-10
    sp.close()


def test_row_split_argument_errors(scmd):
    import torch
    from paper_1210_3559_b200.binding import rescale_thermostat
    w = W.fcc_cluster(100, 300.0, seed=1)
    with pytest.raises(scmd.ScError):
        scmd.SuttonChen(100, r_cut=6.0, skin=1.0, row_begin=0, row_end=50)        # the split is all pairs only
    with pytest.raises(scmd.ScError):
        scmd.SuttonChen(100, row_begin=10, row_end=101)
    sc = scmd.SuttonChen(100, row_begin=50, row_end=100)
    pos = torch.zeros(100, 3, dtype=torch.float64, device="cuda"); rho = torch.zeros(100, dtype=torch.float64, device="cuda")
    pos.copy_(torch.as_tensor(w.pos))
    sc.sc_set_state(pos, torch.as_tensor(w.vel, device="cuda"))
    for bad in (lambda: sc.sc_step(1.0, 1), lambda: sc.sc_energy(), lambda: sc.sc_step_rows(0, 1.0, pos, rho),
                lambda: sc.sc_step_rows(2, 1.0, pos, rho, rescale_thermostat(300.0, 300.0)), lambda: sc.sc_step_rows(3, 1.0, pos, rho)):
        with pytest.raises(scmd.ScError):
            bad()
    sc.close()
    full = scmd.SuttonChen(100)
    full.sc_set_state(pos)
    with pytest.raises(scmd.ScError):
        full.sc_step_rows(1, 0.0, pos, rho)                                       # not a rank of a split
    full.close()


def test_row_split_world1_through_the_driver_class(scmd, oracle_ld):
    """RowSplitSuttonChen itself at world = 1 (no process group needed): the same answers as the oracle."""
    import torch
    w = W.fcc_cluster(1500, 1000.0, seed=5)
    rs = scmd.RowSplitSuttonChen(1500, 0, 1)
    rs.set_state(torch.as_tensor(w.pos, device="cuda"), torch.as_tensor(w.vel, device="cuda"))
    P = oracle_ld.params()
    ref = oracle_ld.run(w.pos, w.vel, P, dt=1.0, nsteps=10)
    assert abs(rs.energy() - ref["epot"][0]) < 1e-12 * abs(ref["epot"][0])
    rs.step(1.0, 10)
    assert np.abs(rs.positions().cpu().numpy() - ref["pos"]).max() < 1e-8
    ke, temp = rs.kinetic()
    assert abs(ke - ref["ekin"][-1]) < 1e-10 * ref["ekin"][-1] and temp > 0
    rs.close()


_NCCL_WORKER = r'''
import os, sys, json
import numpy as np, torch, torch.distributed as dist
sys.path.insert(0, sys.argv[1])
import paper_1210_3559_b200 as scmd
from paper_1210_3559_b200 import workloads as W
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
torch.cuda.set_device(rank)
dist.init_process_group("nccl", device_id=torch.device("cuda", rank))
w = W.fcc_cluster(6001, 1200.0, seed=9)
rs = scmd.RowSplitSuttonChen(6001, rank, world)
rs.set_state(torch.as_tensor(w.pos, device="cuda"), torch.as_tensor(w.vel, device="cuda"))
rs.step(1.0, 10)
f = rs.gather_forces().cpu().numpy()
if rank == 0:
    np.save(sys.argv[2], np.concatenate([rs.positions().cpu().numpy(), f]))
    print(json.dumps({"energy": rs.energy(), "ke": rs.kinetic()[0]}))
else:
    rs.energy(); rs.kinetic()
dist.barrier(); dist.destroy_process_group()
'''


def test_row_split_nccl_two_gpus(scmd, oracle_ld, tmp_path):
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs (this pool has one): the single-GPU emulation above covers the kernels, "
                    "tests/test_rowsplit_dist.py the collectives")
    script, out = tmp_path / "worker.py", tmp_path / "out.npy"
    script.write_text(_NCCL_WORKER)
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]
    res = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr",
                          "127.0.0.1", "--master-port", str(port), str(script), str(ROOT), str(out)], capture_output=True,
                         text=True, timeout=900)
    assert res.returncode == 0, res.stderr[-3000:]
    w = W.fcc_cluster(6001, 1200.0, seed=9)
    ref = oracle_ld.run(w.pos, w.vel, oracle_ld.params(), dt=1.0, nsteps=10)
    _, f_o, _ = oracle_ld.energy_forces(ref["pos"], oracle_ld.params())
    got = np.load(out)
    assert np.abs(got[:6001] - ref["pos"]).max() < 1e-8 and rel_l2(got[6001:], f_o) < 1e-7
