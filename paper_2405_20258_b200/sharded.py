"""Multi-GPU form of the hot path: one process per GPU, the (v, c) pairs sharded over ranks by conduction band.

PAPER.md:104-108 eq. 9 distributes the conduction bands over ranks and PAPER.md:127-129 sums the per-rank
contributions to chi0.  On NVLink/NVSwitch that sum is ONE all-reduce per pass (chi~0(0): 2 N_G^2 doubles, chi_s:
2 N_w N_eig^2 doubles): every rank runs a1/a2 on its own conduction slice, the partial chi~0(0) are summed, rank 0's
subspace basis is broadcast (the basis must be bit-identical on all ranks), every rank runs a1/a4 on its slice, the
partial chi_s are summed, and a5 runs replicated.  All arithmetic is in the C-ABI kernels; `torch.distributed` is the
plumbing for the two collectives.  With world size 1 (or no process group) the collectives are no-ops.
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


def rpa_energy_sharded(ctx, psi_v, psi_c_local, e_v, e_c_local, nvb, n_eig, tol, omega, weight, comm=None, keep_m=True):
    """E_c with this rank's conduction slice (`psi_c_local` [nc_local][n_pw], `e_c_local`), all valence bands on every rank.

    The context's workspace must hold rpa_workspace_bytes(ctx, nvb, nc_local, n_eig, n_w).  Returns the same dict as
    rpa_energy_device (stage_ms from CUDA events on the current stream, plus 'allreduce')."""
    import torch
    from . import binding as rpa

    comm = comm or Comm()
    dev = psi_v.device
    nv, nc, ng, n_w = psi_v.shape[0], psi_c_local.shape[0], ctx_n_g(ctx, psi_v), omega.shape[0]
    blocks = [(s, min(nv, s + nvb)) for s in range(0, nv, nvb)]
    ms = {k: 0.0 for k in ("mtxel", "chi0_static", "basis", "chi_freq", "energy", "allreduce")}
    marks = []

    def timed(stage, fn):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        out = fn()
        b.record()
        marks.append((stage, a, b))
        return out

    chi0 = torch.zeros((ng, ng), dtype=torch.complex128, device=dev)
    kept = []
    for i, (s, e) in enumerate(blocks):                                   # pass 1 (eq. 15)
        M = torch.empty((e - s, nc, ng), dtype=torch.complex128, device=dev)
        timed("mtxel", lambda: rpa.rpa_mtxel(ctx, psi_v[s:e].contiguous(), psi_c_local, M))
        timed("chi0_static", lambda: rpa.rpa_chi0_static(ctx, M, e_v[s:e].contiguous(), e_c_local, i > 0, chi0))
        if keep_m:
            kept.append(M)
    timed("allreduce", lambda: comm.allreduce_sum_(chi0))                 # sum over ranks (eq. 13)
    Cmat = torch.empty((n_eig, ng), dtype=torch.complex128, device=dev)
    lam = torch.empty(n_eig, dtype=torch.float64, device=dev)
    if comm.rank == 0:
        timed("basis", lambda: rpa.rpa_subspace_basis(ctx, chi0, n_eig, tol, Cmat, lam))
    timed("allreduce", lambda: (comm.broadcast_(Cmat), comm.broadcast_(lam)))
    chi_s = torch.zeros((n_w, n_eig, n_eig), dtype=torch.complex128, device=dev)
    for i, (s, e) in enumerate(blocks):                                   # pass 2
        if keep_m:
            M = kept[i]
        else:
            M = torch.empty((e - s, nc, ng), dtype=torch.complex128, device=dev)
            timed("mtxel", lambda: rpa.rpa_mtxel(ctx, psi_v[s:e].contiguous(), psi_c_local, M))
        timed("chi_freq", lambda: rpa.rpa_chi_subspace_freq(ctx, M, e_v[s:e].contiguous(), e_c_local, Cmat, n_eig, omega, i > 0, chi_s))
    timed("allreduce", lambda: comm.allreduce_sum_(chi_s))
    e_c, t = timed("energy", lambda: rpa.rpa_correlation_energy(ctx, chi_s, n_eig, weight))
    torch.cuda.synchronize(dev)
    for stage, a, b in marks:
        ms[stage] += a.elapsed_time(b)
    return dict(E_c=e_c, t=t, lam=lam.cpu().numpy(), stage_ms=ms)


def ctx_n_g(ctx, like):
    """N_G of a context (kept by the binding at creation)."""
    n = getattr(ctx, "n_g", None)
    if n is None:
        raise ValueError("context lacks n_g (create it with paper_2405_20258_b200.rpa_create)")
    return int(n)
