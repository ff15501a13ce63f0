"""Plane-axis sharding: the driver loop of paper_1708_05324_b200/sharded.py.

CPU: two gloo ranks run the loop with a numpy stand-in for the plan (the shard pieces restated with oracle functions),
and the result must be the oracle's plain MPA -- partition, block sums, exclusive prefix, max-reduce and stopping rule
are the host logic under test.  GPU: two shards of the real library as two threads of one process on one device (host
threads meet at a barrier; no kernel waits on another) against the unsharded gmmnlse_propagate.
"""
import os
import sys
import threading

import numpy as np
import pytest

from oracle import gmmnlse_oracle as O
from paper_1708_05324_b200 import sharded
from paper_1708_05324_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def rel(a, b):
    return np.linalg.norm(np.ravel(a) - np.ravel(b)) / np.linalg.norm(np.ravel(b))


def test_plane_ranges_cover_every_plane_once():
    for Mc in (1, 2, 7, 10, 20):
        for n in (1, 2, 3, 8):
            r = sharded.plane_ranges(Mc, n)
            assert len(r) == n and r[0][0] == 0 and r[-1][1] == Mc
            assert all(a[1] == b[0] for a, b in zip(r, r[1:]))
            sizes = [hi - lo for lo, hi in r]
            assert max(sizes) - min(sizes) <= 1 and sizes[0] >= 1      # shard 0 always has a plane (it forms G_0)


class NumpyShardPlan:
    """The gmmnlse_shard_* pieces written out with oracle functions on [P][N][2] float64 tensors (test only)."""

    def __init__(self, w):
        self.w = w
        self.omega = O.omega_grid(w.N, w.dt)
        self.D = O.dispersion_operator(w.beta, self.omega)
        self.K = 1j * w.kappa * (1.0 + self.omega / w.omega0 if w.shock else np.ones_like(self.omega))
        self.nlt = lambda A: O.nonlinear_term(A, w.S, w.f_R, w.h_R, w.dt)

    @staticmethod
    def _c(t):
        return t.numpy().view(np.complex128)[..., 0]

    def _g(self, psi, j):
        Af = psi * np.exp(self.D * (j * self.w.dz))
        return np.exp(-self.D * (j * self.w.dz)) * (self.K * O.to_freq(self.nlt(O.to_time(Af))))

    def shard_begin(self, A_in):
        self.psi0 = O.to_freq(self._c(A_in))
        self.psi, self.G = {}, {}

    def shard_iterate(self, j_lo, j_hi, Mc, first, block):
        if first:
            self.psi = {j: self.psi0 for j in range(j_lo + 1, j_hi + 1)}
            if j_lo == 0:
                self.G[0] = self._g(self.psi0, 0)
        acc = 0.5 * self.G[0] if j_lo == 0 else 0.0
        for j in range(j_lo + 1, j_hi + 1):
            self.G[j] = self._g(self.psi[j], j)
            acc = acc + (0.5 if j == Mc else 1.0) * self.G[j]
        self._c(block)[...] = acc

    def shard_update(self, j_lo, j_hi, Mc, first, all_sums, shard, n_shards):
        sums = self._c(all_sums)
        acc = 0.5 * self.G[0] if shard == 0 else sums[:shard].sum(axis=0)
        err = 0.0
        for j in range(j_lo + 1, j_hi + 1):
            new = self.psi0 + self.w.dz * (acc + 0.5 * self.G[j])
            acc = acc + self.G[j]
            err = max(err, np.linalg.norm(new - self.psi[j]) / np.linalg.norm(new))
            self.psi[j] = new
        return err

    def shard_advance(self, Mc, all_sums, n_shards):
        self.psi0 = (self.psi0 + self.w.dz * self._c(all_sums).sum(axis=0)) * np.exp(self.D * (Mc * self.w.dz))

    def shard_end(self, A_out):
        self._c(A_out)[...] = O.to_time(self.psi0)


def _gloo_worker(rank, world, port, M, n_small, out, stop_rule=0):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = W.make_config(2, N=256, max_group=1)
    A0 = np.ascontiguousarray(w.A0.astype(np.complex128))
    A_in = torch.from_numpy(A0.view(np.float64).reshape(w.P, w.N, 2).copy())
    A_out = torch.empty_like(A_in)
    st = {}
    status = sharded.propagate_sharded(NumpyShardPlan(w), sharded.TorchComm(), A_in, n_small * w.dz, A_out, M=M,
                                       dz=w.dz, tol=w.tol, stats=st, stop_rule=stop_rule)
    out.put((rank, status, st, A_out.numpy().view(np.complex128)[..., 0].copy()))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("M,n_small,stop_rule", [
    (10, 25, 0), (3, 6, 0), (1, 2, 0),          # ragged tail; uneven split; more ranks than planes
    (10, 30, 1),                                # the a-posteriori stopping rule (reading S25)
])
def test_sharded_loop_world2_gloo_equals_oracle_mpa(M, n_small, stop_rule):
    pytest.importorskip("torch")
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 29700 + (os.getpid() + 7 * M + 3 * stop_rule) % 2000
    procs = [ctx.Process(target=_gloo_worker, args=(r, 2, port, M, n_small, out, stop_rule)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted((out.get(timeout=240) for _ in procs), key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    w = W.make_config(2, N=256, max_group=1)
    ost = {}
    ref = O.mpa_propagate(w.A0, n_small * w.dz, w.dz, M, w.beta, w.S, w.kappa, w.omega0, w.f_R, w.h_R, w.dt,
                          shock=w.shock, tol=w.tol, stats=ost, stop_rule=stop_rule)
    for rank, status, st, field in res:
        assert status == 0
        assert st["large_steps"] == ost["large_steps"] and st["iterations"] == ost["iterations"]
        assert rel(field, ref) < 1e-12                                   # same arithmetic, another summation order
    assert np.array_equal(res[0][3], res[1][3])                           # every rank ends with the same field


class _ThreadComm:
    """n shards as n host threads of one process: blocks meet in a shared buffer between two barrier crossings."""

    def __init__(self, rank, world, shared, barrier, errs):
        self.rank, self.world, self._sh, self._bar, self._errs = rank, world, shared, barrier, errs

    def all_gather(self, out, block):
        self._sh[self.rank].copy_(block)
        self._bar.wait()
        out.copy_(self._sh)
        self._bar.wait()

    def all_reduce_max(self, x):
        self._errs[self.rank] = x
        self._bar.wait()
        m = max(self._errs)
        self._bar.wait()
        return m


@pytest.mark.gpu
@pytest.mark.parametrize("cfg,kw,n_shards", [
    (2, dict(N=1024, L=37 * 50e-6), 2),          # CUDA-core path, ragged last step (7 planes)
    (4, dict(N=1024, L=40 * 50e-6), 2),          # kind::f16 tensor-core contraction, M = 20: 10 planes per shard
    (3, dict(N=1024, L=20 * 100e-6), 3),         # 3xTF32 contraction, 10 planes over 3 shards (4 + 3 + 3)
])
def test_sharded_gpu_two_threads_equal_unsharded(cfg, kw, n_shards):
    torch = pytest.importorskip("torch")
    from paper_1708_05324_b200 import binding as B
    B.load_library()
    w = W.make_config(cfg, **kw)
    A = torch.from_numpy(w.A0.astype(np.complex64)).cuda()
    ref_out = torch.empty_like(A)
    with B.plan_from_workload(w, graph=1) as plan:
        plan.propagate(A, w.L, ref_out)
        torch.cuda.synchronize()
        ref_stats = plan.stats()
    shared = torch.empty((n_shards,) + tuple(A.shape), dtype=A.dtype, device=A.device)
    barrier, errs = threading.Barrier(n_shards), [0.0] * n_shards
    outs, stats, fails = [None] * n_shards, [dict() for _ in range(n_shards)], []

    def run(rank):
        try:
            torch.cuda.set_device(0)
            with B.plan_from_workload(w, graph=1) as plan:
                o = torch.empty_like(A)
                sharded.propagate_sharded(plan, _ThreadComm(rank, n_shards, shared, barrier, errs), A, w.L, o, M=w.M,
                                          dz=w.dz, tol=w.tol, stats=stats[rank])
                torch.cuda.synchronize()
                outs[rank] = o.cpu().numpy()
        except Exception as exc:                                       # release the others instead of deadlocking
            fails.append(exc)
            barrier.abort()

    threads = [threading.Thread(target=run, args=(r,)) for r in range(n_shards)]
    for t in threads:
        t.start()
    for t in threads:
        t.join(timeout=300)
    assert not fails, fails
    ref = ref_out.cpu().numpy()
    for r in range(n_shards):
        assert stats[r]["large_steps"] == ref_stats["large_steps"]
        assert abs(stats[r]["iterations"] - ref_stats["iterations"]) <= 1
        assert rel(outs[r], ref) <= 5e-6                               # fp32 rounding of another summation order
        assert np.array_equal(outs[r], outs[0])                        # every shard ends with the same field
    A_in = A.cpu().numpy().astype(np.complex128)
    omp = O.mpa_propagate(A_in, w.L, w.dz, w.M, w.beta, w.S, w.kappa, w.omega0, w.f_R, w.h_R, w.dt, shock=w.shock,
                          tol=w.tol)
    assert rel(outs[0], omp) <= 1e-4


@pytest.mark.gpu
def test_sharded_driver_over_a_real_nccl_group_of_one():
    """The NCCL path of TorchComm (all_gather_into_tensor on the real view of complex blocks, max all-reduce on a
    device scalar) on the one GPU this pool gives: a process group of world size 1, against the unsharded call."""
    torch = pytest.importorskip("torch")
    import torch.distributed as dist
    from paper_1708_05324_b200 import binding as B
    B.load_library()
    if dist.is_initialized():
        pytest.skip("a process group already exists in this process")
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(29900 + os.getpid() % 90), RANK="0", WORLD_SIZE="1")
    torch.cuda.set_device(0)
    dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device("cuda", 0))
    try:
        w = W.make_config(2, N=1024, L=25 * 50e-6)
        A = torch.from_numpy(w.A0.astype(np.complex64)).cuda()
        ref_out, out = torch.empty_like(A), torch.empty_like(A)
        st = {}
        with B.plan_from_workload(w, graph=1) as plan:
            plan.propagate(A, w.L, ref_out)
            torch.cuda.synchronize()
            ref_stats = plan.stats()
        with B.plan_from_workload(w, graph=1) as plan:
            sharded.propagate_sharded(plan, sharded.TorchComm(), A, w.L, out, M=w.M, dz=w.dz, tol=w.tol, stats=st)
            torch.cuda.synchronize()
        assert st["large_steps"] == ref_stats["large_steps"] and st["iterations"] == ref_stats["iterations"]
        assert rel(out.cpu().numpy(), ref_out.cpu().numpy()) <= 5e-6
    finally:
        dist.destroy_process_group()
