"""Row-sharded LSQR over several GPUs: the driver loop around the phase calls of include/gsr.h (gsr_shard_*).

SURVEY.md section 8(f2); PAPER.md:72 (rows of A split over the processes, the astrometric part distributed, the
attitude / instrumental / global parts replicated) and PAPER.md:74 (the reduces after the products).

Plumbing only.  Every number is computed by the library's kernels on each rank's rows; this module (i) cuts the rows
at star boundaries, (ii) calls the phases in lock step and (iii) sums the exchange buffer over the ranks where the
library says so -- one `allreduce(sum)` per exchange, NCCL over NVLink when the ranks are processes with one GPU
each.  It knows nothing of the algorithm: which phase comes next and how many doubles travel is the library's answer.

Two communicators:
  DistComm  -- one shard per process, `torch.distributed` (nccl on GPUs; gloo in the CPU tests of the host logic);
  LocalComm -- several shards driven by ONE process (each its own gsr_system, on one GPU or several): the sum is a
               plain tensor sum.  No rank ever waits on another one's kernels; this is how the phase calls are checked
               on a single GPU, and it is not a way to measure scaling.
"""
from dataclasses import dataclass

import numpy as np

SHARD_MORE, SHARD_INIT_DONE, SHARD_ITER_DONE = 0, 1, 2


# ------------------------------------------------------------------------------------------- the row partition
@dataclass(frozen=True)
class RowRange:
    star_lo: int    # first star of the rank
    star_hi: int    # one past its last star
    row_lo: int     # first row (= first observation of star_lo)
    row_hi: int     # one past the last row


def partition_stars(obs_per_star, world: int):
    """Cut the rows (sorted by star) into `world` contiguous ranges at star boundaries, as equal in rows as the
    boundaries allow: rank k ends at the star boundary nearest to row (k+1) * M / world.  `obs_per_star`: the number
    of rows of every star (length S; an int array or a (S, obs) pair meaning S stars of obs rows each).
    Ranges may be empty when there are fewer stars than ranks."""
    if world < 1:
        raise ValueError("world must be >= 1")
    if isinstance(obs_per_star, tuple):
        n_stars, obs = obs_per_star
        ptr = np.arange(n_stars + 1, dtype=np.int64) * int(obs)
    else:
        c = np.asarray(obs_per_star, dtype=np.int64)
        if c.ndim != 1 or (c < 0).any():
            raise ValueError("obs_per_star: a 1-D array of non-negative counts")
        ptr = np.concatenate([[0], np.cumsum(c)])
    m, n_stars = int(ptr[-1]), len(ptr) - 1
    cuts = [0]
    for k in range(1, world):
        target = k * m / world
        j = int(np.searchsorted(ptr, target, side="left"))          # first boundary >= target
        if j > 0 and (j > n_stars or target - ptr[j - 1] <= ptr[j] - target):
            j -= 1                                                   # the boundary below is nearer
        cuts.append(min(max(j, cuts[-1]), n_stars))
    cuts.append(n_stars)
    return [RowRange(cuts[k], cuts[k + 1], int(ptr[cuts[k]]), int(ptr[cuts[k + 1]])) for k in range(world)]


# ------------------------------------------------------------------------------------------- communicators
class DistComm:
    """One shard per process; the sum over ranks is torch.distributed.all_reduce on the caller's process group."""

    def __init__(self, group=None):
        import torch.distributed as dist
        if not (dist.is_available() and dist.is_initialized()):
            raise RuntimeError("DistComm needs an initialised torch.distributed process group")
        self.dist, self.group = dist, group
        self.rank = dist.get_rank(group)
        self.world = dist.get_world_size(group)
        self.n_local = 1

    def counts_shared(self, local_index: int) -> bool:
        return self.rank == 0

    def allreduce(self, bufs):
        (t,) = bufs
        if self.world > 1 and t.numel() > 0:
            self.dist.all_reduce(t, op=self.dist.ReduceOp.SUM, group=self.group)


class LocalComm:
    """All shards in this process: the 'collective' is the sum of the shards' buffers, written back to each."""

    def __init__(self, n_local: int):
        self.rank, self.world, self.n_local = 0, n_local, n_local

    def counts_shared(self, local_index: int) -> bool:
        return local_index == 0

    def allreduce(self, bufs):
        if len(bufs) < 2 or bufs[0].numel() == 0:
            return
        total = bufs[0].clone()
        for t in bufs[1:]:
            total += t.to(total.device)
        for t in bufs:
            t.copy_(total)


# ------------------------------------------------------------------------------------------- the driver loop
class ShardedLsqr:
    """shards: the local shard objects (GsrSystem, or anything with the same shard_* methods), one per rank held by
    this process (exactly one with DistComm).  Each was created over its RowRange of the rows with the GLOBAL
    n_stars / n_knots / n_instr / n_glob."""

    def __init__(self, shards, comm, check_every: int = 16):
        shards = list(shards)
        if len(shards) != comm.n_local:
            raise ValueError(f"{comm.n_local} local shard(s) expected, got {len(shards)}")
        if check_every < 1:
            raise ValueError("check_every >= 1")
        self.shards, self.comm, self.check_every = shards, comm, int(check_every)
        self.xbufs = [sh.exchange_buffer() for sh in shards]
        self.exchanges = 0          # allreduce calls issued (all shards together count once)
        self.exchanged_doubles = 0  # doubles per rank that travelled
        self.iterations = 0

    def _exchange(self, counts):
        cnt = counts[0]
        if any(c != cnt for c in counts):
            raise RuntimeError(f"shards disagree on the exchange size: {counts}")
        if cnt:
            self.comm.allreduce([xb[:cnt] for xb in self.xbufs])
            self.exchanges += 1
            self.exchanged_doubles += cnt

    def _phase(self):
        out = [sh.shard_phase() for sh in self.shards]
        status = out[0][1]
        if any(o[1] != status for o in out):
            raise RuntimeError(f"shards disagree on the phase: {[o[1] for o in out]}")
        self._exchange([o[0] for o in out])
        return status

    def _poll(self):
        polls = [sh.shard_poll() for sh in self.shards]
        stopped = polls[0][0]
        if any(p[0] != stopped for p in polls):
            raise RuntimeError("shards disagree on the stop flag")
        return stopped, polls[0][1]

    def begin(self, bs, itnlim, atol=0.0, btol=0.0, conlim=0.0):
        """Start a solve: bs = this process's right-hand sides, one per local shard (each the shard's own rows of b).
        Runs the initialisation phases with their exchanges; returns (stopped, LsqrResult) of the first poll
        (stopped already when b = 0 or A^T b = 0: x = 0 is the solution)."""
        bs = list(bs)
        if len(bs) != len(self.shards):
            raise ValueError("one right-hand side per local shard")
        self.exchanges = self.exchanged_doubles = self.iterations = 0
        self.itnlim = int(itnlim)
        counts = [sh.shard_begin(b, xb, self.comm.counts_shared(i), itnlim, atol, btol, conlim)
                  for i, (sh, b, xb) in enumerate(zip(self.shards, bs, self.xbufs))]
        self._exchange(counts)
        while self._phase() != SHARD_INIT_DONE:
            pass
        return self._poll()

    def iterate(self, n_iters: int):
        """n_iters more LSQR iterations on every rank, in lock step, without looking at the stop flag (iterations after a
        stop are no-ops on the device, as in gsr_lsqr_iterate).  Asynchronous apart from the exchanges."""
        for _ in range(int(n_iters)):
            while self._phase() != SHARD_ITER_DONE:
                pass
            self.iterations += 1

    def poll(self):
        """(stopped, LsqrResult): the device-side stop flag and scalars, identical on every rank.  Synchronises."""
        return self._poll()

    def solve(self, bs, itnlim, atol=0.0, btol=0.0, conlim=0.0):
        """The whole solve; returns the LsqrResult every rank agrees on.  The stop flag is polled every check_every iterations."""
        stopped, res = self.begin(bs, itnlim, atol, btol, conlim)
        while not stopped and self.iterations < itnlim:
            self.iterate(min(self.check_every - self.iterations % self.check_every, itnlim - self.iterations))
            stopped, res = self._poll()
        if not stopped:                                # itnlim = 0
            stopped, res = self._poll()
        return res

    def solution(self, xs, gather_astro: bool = True):
        """Write the solution into xs (one n-vector per local shard, the ABI's column order).  The replicated blocks
        are identical on every rank; each astrometric entry is non-zero on its owner only, so with gather_astro the
        sum over ranks of the astrometric block (5 * n_stars doubles, once per solve) gives every rank the whole x."""
        xs = list(xs)
        for sh, x in zip(self.shards, xs):
            sh.lsqr_result(x)
        if gather_astro:
            n_astro = int(self.shards[0].n_unknowns - (self.shards[0].shard_exchange_len() - 2))
            self.comm.allreduce([x[:n_astro] for x in xs])
        return xs
