"""Host side of the row split over several GPUs (paper_1210_3559_b200/distributed.py) on CPU:
the partition arithmetic, and the exchange schedule of RowSplitSuttonChen under world_size-2 gloo with a stand-in for
libscmd's per-rank calls that the test builds from the ORACLE's row functions (so the orchestration -- which phase
reads what, which rows each all-gather carries -- is checked against a single-process oracle run)."""
import os
import socket
import sys
from pathlib import Path

import numpy as np
import pytest

ROOT = Path(__file__).resolve().parent.parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

ACC, MASS = 9.648533215665e-3, 58.69


def test_row_range_partition():
    from paper_1210_3559_b200.distributed import row_range
    for n in (1, 2, 7, 64, 65, 1000, 65536, 262144):
        for world in (1, 2, 3, 4, 8):
            ranges = [row_range(n, r, world) for r in range(world)]
            chunk = ranges[0][2]
            assert chunk == -(-n // world) and all(c == chunk for _, _, c in ranges)
            assert ranges[0][0] == 0 and max(e for _, e, _ in ranges) == n
            covered = np.zeros(n, dtype=int)
            for b, e, _ in ranges:
                assert 0 <= b <= e <= n and e - b <= chunk and b == min(n, ranges.index((b, e, chunk)) * chunk)
                covered[b:e] += 1
            assert np.all(covered == 1)                                    # every row exactly once
    with pytest.raises(ValueError):
        row_range(10, 3, 3)
    with pytest.raises(ValueError):
        row_range(0, 0, 1)


class OracleRank:
    """Stand-in for one libscmd row-split context, same calls, numpy + the oracle's row functions."""

    def __init__(self, n_atoms, row_begin, row_end, **params):
        from oracle.sc_oracle import Oracle
        self.o = Oracle("ld")
        self.P = self.o.params()
        self.n, self.b, self.e = n_atoms, row_begin, row_end
        self.rows = np.arange(row_begin, row_end, dtype=np.int64)
        self.calls = []

    def sc_set_state(self, pos, vel):
        self.pos, self.vel = pos.numpy().copy(), vel.numpy().copy()
        self.force = np.zeros_like(self.pos)

    def sc_step_rows(self, phase, dt, pos_all, rho_all, thermostat=None):
        self.calls.append(phase)
        hk = 0.5 * dt * ACC / MASS
        if phase == 0:
            self.vel[self.rows] += hk * self.force[self.rows]
            self.pos[self.rows] += dt * self.vel[self.rows]
            pos_all[self.b:self.e] = __import__("torch").from_numpy(self.pos[self.rows])
        elif phase == 1:
            self.pos = pos_all[: self.n].numpy().copy()
            rho_all[self.b:self.e] = __import__("torch").from_numpy(self.o.density_rows(self.pos, self.P, self.rows))
        else:
            rho = rho_all[: self.n].numpy().copy()
            f, ps = self.o.forces_rows(self.pos, self.P, rho, self.rows)
            self.force[self.rows] = f
            self.e_share = 1.5707e-2 * (0.5 * ps.sum() - 39.432 * np.sqrt(rho[self.rows]).sum())
            if dt > 0:
                self.vel[self.rows] += hk * f

    def sc_energy(self):
        return float(self.e_share)

    def sc_kinetic(self):
        return 0.5 * MASS * float((self.vel[self.rows] ** 2).sum()) / ACC, 0.0

    def sc_forces(self):
        return __import__("torch").from_numpy(self.force)

    def sc_get_state(self):
        import torch
        return torch.from_numpy(self.pos), torch.from_numpy(self.vel)

    def close(self):
        pass


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, str(ROOT))
    from paper_1210_3559_b200.distributed import RowSplitSuttonChen
    from paper_1210_3559_b200 import workloads as W
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = W.fcc_cluster(45, 900.0, seed=7)                                   # 45 atoms over 2 ranks: 23 + 22 rows
    rs = RowSplitSuttonChen(45, rank, world, backend=OracleRank)
    rs.set_state(torch.from_numpy(w.pos), torch.from_numpy(w.vel))
    e0 = rs.energy()
    rs.step(1.0, 5)
    ke, temp = rs.kinetic()
    f = rs.gather_forces().numpy().copy()
    q.put((rank, rs.begin, rs.end, e0, rs.energy(), ke, temp, rs.positions().numpy().copy(), f, rs.exchanges,
           list(rs.ctx.calls)))
    dist.barrier()
    dist.destroy_process_group()


def test_rowsplit_schedule_gloo_world2(oracle_ld):
    import torch.multiprocessing as mp
    from paper_1210_3559_b200 import workloads as W
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted((q.get(timeout=300) for _ in range(2)), key=lambda g: g[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    w = W.fcc_cluster(45, 900.0, seed=7)
    P = oracle_ld.params()
    ref = oracle_ld.run(w.pos, w.vel, P, dt=1.0, nsteps=5)
    _, f_ref, _ = oracle_ld.energy_forces(ref["pos"], P)
    assert (got[0][1], got[0][2], got[1][1], got[1][2]) == (0, 23, 23, 45)
    for g in got:
        assert abs(g[3] - ref["epot"][0]) < 1e-12 * abs(ref["epot"][0])   # U at t = 0: all-reduce of the two shares
        assert abs(g[4] - ref["epot"][-1]) < 1e-12 * abs(ref["epot"][-1])
        assert abs(g[5] - ref["ekin"][-1]) < 1e-12 * ref["ekin"][-1]
        assert np.abs(g[7] - ref["pos"]).max() < 1e-13                    # every rank ends with ALL positions
        assert np.abs(g[8] - f_ref).max() < 1e-12 * np.abs(f_ref).max()
        assert g[9] == 1 + 2 * 5 + 1                                      # rho at t = 0; positions + rho per step; forces
        assert g[10] == [1, 2] + [0, 1, 2] * 5                            # the phases, in order
    assert np.array_equal(got[0][7], got[1][7])                           # bit-identical replicas of the positions
