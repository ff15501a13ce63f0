"""Host-side logic of the N > 1 bench launch ("replicas only") on CPU with gloo."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = bench.max_over_ranks(10.0 + 5.0 * rank, world, "cpu")
    A0 = (np.arange(12, dtype=np.float64).reshape(3, 4) + 1j).astype(np.complex64)
    A = bench.replica_launch_field(A0, rank, 170805324)
    out.put((rank, ms, np.abs(A).tolist(), bool(np.array_equal(A, A0))))
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_and_replica_fields_world2():
    torch = pytest.importorskip("torch")
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, ms0, abs0, same0), (r1, ms1, abs1, same1) = res
    assert ms0 == ms1 == 15.0                      # both ranks see the slowest rank's time
    assert same0 and not same1                     # rank 0 keeps the configuration's field, rank 1 gets new phases
    assert np.allclose(abs0, abs1)                 # ... of the same modulus (same powers per mode)


def test_reference_arm_only_rank0_prints():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "1",
                        "--steps", "1", "--warmup", "0"], capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""
    env["RANK"] = "0"
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "1",
                        "--steps", "1", "--warmup", "0"], capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0, r.stderr
    d = json.loads(r.stdout.strip().splitlines()[-1])
    assert d["impl"] == "reference" and d["value"] > 0 and d["unit"] == "z-steps/s"
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0


def test_bench_gpus_flag_starts_its_own_ranks():
    """`python bench.py --gpus 2` outside torchrun re-launches itself as 2 ranks (one per GPU on the box; here on CPU
    over gloo with the measurement stubbed to 10 ms x (1 + rank)): one JSON line, from rank 0, n_gpus = 2, the time the
    slowest rank's, the value the whole job's."""
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_PORT")}
    env["GMMNLSE_BENCH_STUB_MS"] = "10.0"
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "4", "--config", "5"],
                       capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["n_gpus"] == 2 and d["scaling"] == "weak"
    assert d["ms_per_step"] == pytest.approx(20.0 / 4)                 # max over ranks: rank 1 took 20 ms
    assert d["value"] == pytest.approx(2 * 4 * 20 / 20e-3)             # 2 ranks x 4 steps x 20 z-steps in 20 ms
