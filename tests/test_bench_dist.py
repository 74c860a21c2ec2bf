"""Host-side multi-process logic of bench.py on CPU: world_size-2 gloo (replicas
only; the timing reduction is the one collective).  Also the workload-name parser and the reference arm."""
import json
import os
import socket
import subprocess
import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, q):
    import torch.distributed as dist
    sys.path.insert(0, str(ROOT))
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    # rank r timed 10 + 5 r ms over (100 + r) units: max of the times, sum of the units
    ms, units = bench.aggregate(10.0 + 5.0 * rank, 100.0 + rank, world, backend_device="cpu")
    assert bench.dist_env() == (rank, rank, world)
    # replicas draw different seeds per rank
    w = bench.Spec("Ni1415-fcc-allpairs-fp64").generate(rank)
    q.put((rank, ms, units, w.seed, float(w.pos[0, 0])))
    dist.barrier()
    dist.destroy_process_group()


def test_aggregate_max_time_sum_units_gloo_world2():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [g[1] for g in got] == [15.0, 15.0]
    assert [g[2] for g in got] == [201.0, 201.0]
    assert got[0][3] != got[1][3] and got[0][4] != got[1][4]


def test_workload_names():
    sys.path.insert(0, str(ROOT))
    import bench
    s = bench.Spec("Ni65536-fcc-cutoff10-mixed")
    assert (s.n_atoms, s.kind, s.r_cut, s.skin, s.prec) == (65536, "fcc", 10.0, 1.0, "mixed")
    s = bench.Spec(bench.DEFAULT_WORKLOAD)
    assert (s.n_atoms, s.r_cut, s.prec) == (65536, 0.0, "fp64")
    with pytest.raises(SystemExit):
        bench.Spec("Ni10-bcc-allpairs-fp64")


def test_reference_arm_prints_one_json_line_and_other_ranks_stay_silent():
    env = dict(os.environ, OMP_NUM_THREADS="4")
    out = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "0",
                          "--workload", "Ni1415-fcc-allpairs-fp64"], capture_output=True, text=True, env=env, timeout=600)
    assert out.returncode == 0, out.stderr
    lines = [l for l in out.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["value"] > 0 and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["config"]["workload"] == "Ni1415-fcc-allpairs-fp64"
    out = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "0"],
                         capture_output=True, text=True, env=dict(env, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1"), timeout=60)
    assert out.returncode == 0 and out.stdout.strip() == ""
