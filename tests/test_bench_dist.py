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


def test_gpus_flag_starts_the_ranks_itself(monkeypatch):
    """`python bench.py --gpus N` outside torchrun re-executes itself under torch.distributed.run with N ranks
    (one per GPU) on 127.0.0.1; under torchrun it must find WORLD_SIZE == N."""
    sys.path.insert(0, str(ROOT))
    import bench
    calls = []

    class Done:
        returncode = 0

    def fake_run(cmd, env=None, **kw):
        calls.append((cmd, env))
        return Done()

    monkeypatch.setattr(bench.subprocess, "run", fake_run)
    for k in ("WORLD_SIZE", "RANK", "LOCAL_RANK"):
        monkeypatch.delenv(k, raising=False)
    with pytest.raises(SystemExit) as ei:
        bench.main(["--gpus", "4", "--steps", "7", "--warmup", "3"])
    assert ei.value.code == 0 and len(calls) == 1
    cmd, env = calls[0]
    assert cmd[:3] == [sys.executable, "-m", "torch.distributed.run"]
    assert "--nproc-per-node=4" in cmd and "--nnodes=1" in cmd
    assert cmd[cmd.index("--master-addr") + 1] == "127.0.0.1"
    assert cmd[-6:] == ["--gpus", "4", "--steps", "7", "--warmup", "3"] and cmd[-7].endswith("bench.py")
    assert "NCCL_DEBUG" in env
    # under torchrun with the wrong world size: refuse rather than mislabel the line
    monkeypatch.setenv("WORLD_SIZE", "2"); monkeypatch.setenv("RANK", "0"); monkeypatch.setenv("LOCAL_RANK", "0")
    with pytest.raises(SystemExit) as ei:
        bench.main(["--gpus", "4"])
    assert "WORLD_SIZE" in str(ei.value.code)


def test_reference_arm_under_torchrun_world2():
    """The driver's launch of the reference arm at N = 2: torchrun starts two ranks, rank 0 alone runs and prints."""
    env = dict(os.environ, OMP_NUM_THREADS="4")
    for k in ("WORLD_SIZE", "RANK", "LOCAL_RANK"):
        env.pop(k, None)
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(_free_port()), str(ROOT / "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
           "--warmup", "0", "--workload", "Ni1415-fcc-allpairs-fp64"]
    out = subprocess.run(cmd, capture_output=True, text=True, env=env, timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.strip().startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["config"]["n_atoms"] == 1415
    assert set(d["config"]) >= {"workload", "n_atoms", "pairs_per_step", "r_cut", "skin", "parallelism", "step"}
