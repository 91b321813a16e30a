"""Multi-GPU form of the hot path: one process per GPU, the (v, c) pairs sharded over ranks by conduction band.

PAPER.md:104-108 eq. 9 distributes the conduction bands over ranks and PAPER.md:127-129 sums the per-rank
contributions to chi0.  On NVLink/NVSwitch that sum is ONE all-reduce per pass (chi~0(0): 2 N_G^2 doubles, chi_s:
2 N_w N_eig^2 doubles): every rank runs a1/a2 on its own conduction slice, the partial chi~0(0) are summed, rank 0's
subspace basis is broadcast (the basis must be bit-identical on all ranks: a3's split-K sums meet in an order that is
not fixed, so it is computed once), every rank runs a1/a4 on its slice, the partial chi_s are summed, and a5 runs
replicated.  All arithmetic AND the valence-block loop are in the C-ABI library (its pass-level calls);
`torch.distributed` is the plumbing for the two collectives.  With world size 1 (or no process group) the collectives
are no-ops.
"""
from __future__ import annotations


def shard_range(n: int, world: int, rank: int):
    """Contiguous, balanced split of n items: ranks < n % world get one more.  Returns (start, stop)."""
    if world < 1 or not (0 <= rank < world):
        raise ValueError(f"bad rank {rank} of {world}")
    base, extra = divmod(n, world)
    start = rank * base + min(rank, extra)
    return start, start + base + (1 if rank < extra else 0)


class Comm:
    """The two collectives of the sharded path on complex128 / float64 tensors (CUDA with nccl, CPU with gloo)."""

    def __init__(self, group=None):
        import torch.distributed as dist
        self.dist = dist if dist.is_available() and dist.is_initialized() else None
        self.group = group
        self.world = self.dist.get_world_size(group) if self.dist else 1
        self.rank = self.dist.get_rank(group) if self.dist else 0

    @staticmethod
    def _real_view(t):
        import torch
        return torch.view_as_real(t) if t.is_complex() else t

    def allreduce_sum_(self, t):
        if self.dist and self.world > 1:
            self.dist.all_reduce(self._real_view(t), op=self.dist.ReduceOp.SUM, group=self.group)
        return t

    def broadcast_(self, t, src=0):
        if self.dist and self.world > 1:
            self.dist.broadcast(self._real_view(t), src=src, group=self.group)
        return t


def rpa_energy_sharded(ctx, psi_v, psi_c_local, e_v, e_c_local, nvb, n_eig, tol, omega, weight, comm=None, keep_m=True,
                       backend=None):
    """E_c with this rank's conduction slice (`psi_c_local` [nc_local][n_pw], `e_c_local`), all valence bands on every rank.

    Runs the library's pass-level calls (rpa_b200.h): the valence-block loop, the resident M blocks and the cached
    real-space conduction functions are the single-GPU driver's own -- nothing is allocated per block here.  The partial
    chi~0(0) and chi_s live in the workspace and are reduced in place.  The context's workspace must hold
    rpa_energy_workspace_bytes(ctx, nv, nc_local, nvb, n_eig, n_w) (more lets the library keep M and u_c resident).
    Returns the same dict as rpa_energy_device; stage_ms has an extra 'allreduce' entry (both reductions and the
    broadcast, CUDA events on the current stream).  With one rank it is the very sequence rpa_energy_device runs.
    `backend` (default: the ctypes binding) supplies the six rpa_pass_* calls; the CPU tests of the host logic pass a
    stand-in, the product never does."""
    import torch
    if backend is None:
        from . import binding as backend
    rpa = backend

    comm = comm or Comm()
    marks = []

    def exchange(fn):
        if not psi_v.is_cuda:        # host-logic tests on CPU tensors: no device timers
            return fn()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        fn()
        b.record()
        marks.append((a, b))

    rpa.rpa_pass_begin(ctx, psi_v, psi_c_local, e_v, e_c_local, nvb, n_eig, omega, keep_m=keep_m, timing=True)
    try:
        chi0 = rpa.rpa_pass1_chi0(ctx)                                  # pass 1 on this rank's pairs (eq. 15)
        exchange(lambda: comm.allreduce_sum_(chi0))                     # sum over ranks (eq. 13)
        Cmat, lam = rpa.rpa_pass_basis(ctx, tol, compute=comm.rank == 0)
        exchange(lambda: (comm.broadcast_(Cmat), comm.broadcast_(lam)))  # one basis, bit-identical on every rank
        chi_s = rpa.rpa_pass2_chis(ctx)                                 # pass 2
        exchange(lambda: comm.allreduce_sum_(chi_s))
        out = rpa.rpa_pass_energy(ctx, weight)                          # replicated; synchronises
    finally:
        rpa.rpa_pass_end(ctx)
    out["stage_ms"]["allreduce"] = sum(a.elapsed_time(b) for a, b in marks)
    return out


def ctx_n_g(ctx, like):
    """N_G of a context (kept by the binding at creation)."""
    n = getattr(ctx, "n_g", None)
    if n is None:
        raise ValueError("context lacks n_g (create it with paper_2405_20258_b200.rpa_create)")
    return int(n)
