"""Row split of the all-pairs path over several GPUs (include/scmd.h: sc_step_rows).

One process per GPU.  Every rank holds all N positions and owns a contiguous range of atoms; per velocity-Verlet step
the two sweeps of PAPER.md:127 need one exchange each -- the positions after the drift (N x 24 B) and the densities
after sweep 1 (N x 8 B) -- as NCCL all-gathers over NVLink / NVSwitch on torch.distributed's communicator, and the
scalars (U, KE) one all-reduce when somebody asks.  There is no force reduction: a rank computes complete rows (the
one-sided sweeps), which is why the Newton's-third-law kernels are not used here (their reaction terms would have to
cross GPUs).  Marshalling and collectives only: every arithmetic step runs in libscmd's kernels.

The paper's own multi-card use is replicas -- "up to 15 independent simulations" per temperature --
which is what `bench.py --gpus N` runs by default; this split is the strong-scaling alternative for one large cluster
(`bench.py --parallel rows`).
"""
from __future__ import annotations

_KB_EV_PER_K = 8.617333262e-5      # CODATA-2018, as in include/scmd.h
_ACC = 9.648533215665e-3


def row_range(n_atoms: int, rank: int, world: int) -> tuple[int, int, int]:
    """Contiguous rows of `rank`: (begin, end, chunk) with chunk = ceil(N / world) rows per rank (the last ranks may get
    fewer, or none when world > N); all-gather buffers hold world * chunk rows so that every rank sends `chunk`."""
    if n_atoms < 1 or world < 1 or not 0 <= rank < world:
        raise ValueError("row_range: need n_atoms >= 1 and 0 <= rank < world")
    chunk = -(-n_atoms // world)
    begin = min(n_atoms, rank * chunk)
    return begin, min(n_atoms, begin + chunk), chunk


class RowSplitSuttonChen:
    """All pairs, one cluster, `world` GPUs.  `backend`: a factory (n_atoms, row_begin, row_end, **params) -> object
    with the SuttonChen methods used below; None = libscmd on the current CUDA device.  `group`: a torch.distributed
    process group (None = the default one)."""

    def __init__(self, n_atoms: int, rank: int, world: int, *, device=None, group=None, backend=None, **params):
        import torch
        self.torch = torch
        self.n_atoms, self.rank, self.world, self.group = int(n_atoms), int(rank), int(world), group
        self.begin, self.end, self.chunk = row_range(self.n_atoms, self.rank, self.world)
        if self.end <= self.begin:
            raise ValueError("row split: more ranks than atoms")
        if backend is None:
            from .binding import SuttonChen
            self.device = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
            self.ctx = SuttonChen(self.n_atoms, row_begin=self.begin, row_end=self.end, device=self.device, **params)
        else:
            self.device = torch.device("cpu") if device is None else torch.device(device)
            self.ctx = backend(self.n_atoms, self.begin, self.end, **params)
        pad = self.world * self.chunk
        self.pos_all = torch.zeros(pad, 3, dtype=torch.float64, device=self.device)
        self.rho_all = torch.zeros(pad, dtype=torch.float64, device=self.device)
        self.mass = float(params.get("mass", 58.69))
        self.exchanges = 0                                   # all-gathers issued (for the tests and the bench)

    # -- collectives -------------------------------------------------------------------------
    def _all_gather_rows(self, buf, width: int):
        """In place: every rank contributes its own `chunk` rows of `buf` ([world * chunk, width])."""
        if self.world == 1:
            return
        import torch.distributed as dist
        flat = buf.view(-1)
        n = self.chunk * width
        mine = flat[self.rank * n:(self.rank + 1) * n].clone()
        dist.all_gather_into_tensor(flat, mine, group=self.group)
        self.exchanges += 1

    def _all_reduce_sum(self, values):
        t = self.torch.tensor(values, dtype=self.torch.float64, device=self.device)
        if self.world > 1:
            import torch.distributed as dist
            dist.all_reduce(t, op=dist.ReduceOp.SUM, group=self.group)
        return [float(v) for v in t.tolist()]

    # -- the path -----------------------------------------------------------------------------
    def set_state(self, pos, vel):
        """pos, vel: [N, 3] float64 tensors on this rank's device, the same on every rank."""
        self.pos_all[: self.n_atoms].copy_(pos)
        self.ctx.sc_set_state(self.pos_all[: self.n_atoms].contiguous(), vel.contiguous())
        self._evaluate(0.0, None)

    def _evaluate(self, dt: float, thermostat):
        self.ctx.sc_step_rows(1, dt, self.pos_all, self.rho_all, thermostat)     # sweep 1 over the own rows
        self._all_gather_rows(self.rho_all, 1)
        self.ctx.sc_step_rows(2, dt, self.pos_all, self.rho_all, thermostat)     # sweep 2 [+ second half kick]

    def step(self, dt_fs: float, nsteps: int, thermostat=None):
        for _ in range(int(nsteps)):
            self.ctx.sc_step_rows(0, dt_fs, self.pos_all, self.rho_all, thermostat)   # half kick + drift, own rows
            self._all_gather_rows(self.pos_all, 3)
            self._evaluate(dt_fs, thermostat)

    def energy(self) -> float:
        """Potential energy of the whole cluster (all-reduce of the ranks' shares)."""
        return self._all_reduce_sum([self.ctx.sc_energy()])[0]

    def kinetic(self):
        """-> (KE in eV, T in K) of the whole cluster; T = 2 KE / (kB (3N - 3))."""
        ke = self._all_reduce_sum([self.ctx.sc_kinetic()[0]])[0]
        ndof = 3 * self.n_atoms - 3
        return ke, (2.0 * ke / (_KB_EV_PER_K * ndof) if ndof > 0 else 0.0)

    def own_forces(self):
        """[rows, 3] forces of this rank's atoms (device tensor)."""
        return self.ctx.sc_forces()[self.begin:self.end]

    def gather_forces(self):
        """[N, 3] forces of all atoms on every rank (an all-gather: analysis / tests, not part of the step)."""
        buf = self.torch.zeros(self.world * self.chunk, 3, dtype=self.torch.float64, device=self.device)
        buf[self.begin:self.end].copy_(self.own_forces())
        self._all_gather_rows(buf, 3)
        return buf[: self.n_atoms]

    def positions(self):
        return self.pos_all[: self.n_atoms]

    def own_velocities(self):
        return self.ctx.sc_get_state()[1][self.begin:self.end]

    def close(self):
        self.ctx.close()
