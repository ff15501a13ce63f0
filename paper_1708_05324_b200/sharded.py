"""Plane-axis sharding of the MPA over several GPUs (the M planes of a large
step are the parallel axis).

One process per GPU.  Every rank builds a plan of the SAME arguments on its own device and owns a contiguous range
of the planes; per iteration the path has exactly one exchange step, an all-gather of the ranks' block sums of the
trapezoid rule (P x N complex each: 2.9 MB at config 5) plus a scalar max all-reduce for the convergence test.  The
kernels are the library's (``gmmnlse_shard_*`` in include/gmmnlse.h); this module holds only the loop of
PAPER.md:218 and the two collectives, through an object with ``all_gather`` / ``all_reduce_max`` so that the same
loop runs over NCCL (:class:`TorchComm`), over gloo on CPU tensors in the tests, or in one process
(:class:`LocalComm`, a single shard).  The time axis is never split (every FFT would become an all-to-all).
"""
from __future__ import annotations

OK, WARN_NOCONV = 0, 1


def plane_ranges(Mc: int, n_shards: int):
    """[(j_lo, j_hi)] per shard: shard g owns planes j_lo+1 .. j_hi of 1..Mc, sizes differing by at most one;
    (j, j) = no planes (more shards than planes)."""
    base, extra = divmod(Mc, n_shards)
    out, lo = [], 0
    for g in range(n_shards):
        hi = lo + base + (1 if g < extra else 0)
        out.append((lo, hi))
        lo = hi
    return out


class LocalComm:
    """A single shard in one process: the collectives are identities."""
    rank, world = 0, 1

    def all_gather(self, out, block):
        out[0].copy_(block)

    def all_reduce_max(self, x: float) -> float:
        return x


class TorchComm:
    """The two collectives over a torch.distributed process group (NCCL on GPUs; gloo in the CPU tests)."""

    def __init__(self, group=None):
        import torch.distributed as dist
        self._dist, self._group = dist, group
        self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)

    def all_gather(self, out, block):
        import torch
        if out.is_complex():                       # NCCL has no complex types: gather the (re, im) views
            out, block = torch.view_as_real(out), torch.view_as_real(block)
        if out.is_cuda:
            self._dist.all_gather_into_tensor(out, block.contiguous(), group=self._group)
        else:
            self._dist.all_gather(list(out.unbind(0)), block, group=self._group)

    def all_reduce_max(self, x: float) -> float:
        import torch
        dev = "cuda" if self._dist.get_backend(self._group) == "nccl" else "cpu"
        t = torch.tensor([x], dtype=torch.float64, device=dev)
        self._dist.all_reduce(t, op=self._dist.ReduceOp.MAX, group=self._group)
        return float(t.item())


def converged(err, tol, stop_rule, it, err_prev, rho_prev):
    """The convergence decision of the library's loops (csrc/kernels.cuh mpa_converged): err < tol, or with
    stop_rule 1 (reading S25) and it >= 3 the a-posteriori bound err rho / (1 - rho) < tol, rho the larger
    of the last two error ratios.  Returns (decision, this iteration's ratio)."""
    rho_now = err / err_prev if err_prev > 0 else 0.0
    if err < tol:
        return True, rho_now
    if stop_rule == 1 and it >= 3:
        rho = max(rho_now, rho_prev)
        if rho < 1.0 and err * rho / (1.0 - rho) < tol:
            return True, rho_now
    return False, rho_now


def propagate_sharded(plan, comm, A_in, L, A_out, *, M, dz, tol=1e-6, max_iter=0, fixed_iter=0, stop_rule=0,
                      empty_like=None, stats=None):
    """Integrate over L with the MPA, this rank running its share of the planes of every large step.

    ``plan``: an object with the ``shard_*`` methods of :class:`binding.Plan` (same plan arguments on every rank);
    ``A_in`` / ``A_out``: this rank's device buffers [P][N] (every rank passes the same input and receives the same
    output).  ``empty_like(A, n)`` allocates an [n][P][N] buffer like A (default: torch).  Returns OK or WARN_NOCONV.
    """
    n_small = int(round(L / dz))
    if abs(n_small * dz - L) > 1e-9 * max(L, dz):
        raise ValueError("L must be an integer multiple of dz")
    if empty_like is None:
        import torch
        empty_like = lambda A, n: torch.empty((n,) + tuple(A.shape), dtype=A.dtype, device=A.device)
    cap = fixed_iter if fixed_iter > 0 else (max_iter if max_iter > 0 else 2 * M + 4)
    world, rank = comm.world, comm.rank
    all_sums = empty_like(A_in, world)
    block = empty_like(A_in, 1)[0]
    plan.shard_begin(A_in)
    done, status, n_large, n_iter, n_noconv, err = 0, OK, 0, 0, 0, 0.0
    while done < n_small:
        Mc = min(M, n_small - done)
        j_lo, j_hi = plane_ranges(Mc, world)[rank]
        it, err_prev, rho_prev = 0, 1e300, 1e300
        while True:
            first = it == 0
            if j_hi > j_lo:
                plan.shard_iterate(j_lo, j_hi, Mc, first, block)
            else:                                   # more ranks than planes: this rank contributes nothing
                block.zero_()
            comm.all_gather(all_sums, block)         # the path's one exchange step
            e_loc = plan.shard_update(j_lo, j_hi, Mc, first, all_sums, rank, world) if j_hi > j_lo else 0.0
            err = comm.all_reduce_max(e_loc)
            it += 1
            conv, rho = converged(err, tol, stop_rule, it, err_prev, rho_prev)   # every rank takes the same decision
            err_prev, rho_prev = err, (1e300 if it == 1 else rho)
            if fixed_iter > 0:
                if it >= cap:
                    break
            elif conv:
                break
            elif it >= cap:
                n_noconv += 1
                status = WARN_NOCONV
                break
        plan.shard_advance(Mc, all_sums, world)
        n_iter += it
        n_large += 1
        done += Mc
    plan.shard_end(A_out)
    if stats is not None:
        stats.update(large_steps=n_large, iterations=n_iter, last_err=err, not_converged=n_noconv)
    return status
