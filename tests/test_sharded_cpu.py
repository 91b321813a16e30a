"""Host logic of the multi-GPU path (paper_2405_20258_b200/sharded.py) on CPU: the conduction-band partition and the two
collectives, run as two gloo processes.  Each rank computes the partial chi~0(0) / chi_s of its conduction slice with the
ORACLE (tests may call it; there is no GPU here), the partials meet through Comm.allreduce_sum_, rank 0's basis is
broadcast, and every rank must end with the single-process oracle E_c (PAPER.md:104-108 eq. 9, :127 eq. 13)."""
import os
import socket

import numpy as np
import pytest

from paper_2405_20258_b200.sharded import shard_range


def test_shard_range_is_a_balanced_partition():
    for n in (0, 1, 7, 200, 12000):
        for world in (1, 2, 3, 8):
            parts = [shard_range(n, world, r) for r in range(world)]
            assert parts[0][0] == 0 and parts[-1][1] == n
            assert all(parts[i][1] == parts[i + 1][0] for i in range(world - 1))
            sizes = [b - a for a, b in parts]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard_range(5, 2, 2)


def _worker(rank, world, port, out):
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from oracle import rpa_oracle as orc
        from rpa_inputs import make_inputs
        from paper_2405_20258_b200.sharded import Comm
        inp = make_inputs(0, n_v=3, n_c=41)
        comm = Comm()
        assert (comm.world, comm.rank) == (world, rank)
        c0, c1 = shard_range(41, world, rank)
        M = orc.mtxel(inp.psi_v, inp.psi_c[c0:c1], inp.g_wfn, inp.g_eps, inp.fft)
        chi0 = torch.from_numpy(orc.chi0(M, inp.e_v, inp.e_c[c0:c1], inp.vcoul))
        comm.allreduce_sum_(chi0)
        n_eig = 20
        if rank == 0:
            lam, C = orc.subspace_basis(chi0.numpy(), n_eig)
            lam, C = torch.from_numpy(lam), torch.from_numpy(C)
        else:
            lam, C = torch.zeros(n_eig, dtype=torch.float64), torch.zeros((n_eig, inp.n_g), dtype=torch.complex128)
        comm.broadcast_(C)
        comm.broadcast_(lam)
        chis = torch.from_numpy(orc.chi_subspace_freq(M, inp.e_v, inp.e_c[c0:c1], inp.vcoul, C.numpy(), inp.omega))
        comm.allreduce_sum_(chis)
        e, _ = orc.correlation_energy(chis.numpy(), inp.weight)
        out.put((rank, e, float(lam[0])))
    finally:
        dist.destroy_process_group()


class OraclePassBackend:
    """Stand-in for the six rpa_pass_* calls of the binding, computing with the ORACLE on CPU tensors, so that the host
    logic of rpa_energy_sharded itself (call order, in-place reductions, which rank computes the basis, the broadcast)
    runs under two gloo ranks without a GPU.  Test code only."""

    def __init__(self, inp):
        self.inp, self.calls = inp, []

    def rpa_pass_begin(self, ctx, psi_v, psi_c, e_v, e_c, nvb, n_eig, omega, keep_m=True, timing=True):
        self.calls.append("begin")
        self.a = dict(psi_v=psi_v.numpy(), psi_c=psi_c.numpy(), e_v=e_v.numpy(), e_c=e_c.numpy(), n_eig=n_eig, omega=omega.numpy())

    def rpa_pass1_chi0(self, ctx):
        import torch
        from oracle import rpa_oracle as orc
        self.calls.append("pass1")
        a, inp = self.a, self.inp
        self.M = orc.mtxel(a["psi_v"], a["psi_c"], inp.g_wfn, inp.g_eps, inp.fft)
        self.chi0 = torch.from_numpy(orc.chi0(self.M, a["e_v"], a["e_c"], inp.vcoul))
        return self.chi0

    def rpa_pass_basis(self, ctx, tol=0.0, compute=True):
        import torch
        from oracle import rpa_oracle as orc
        self.calls.append("basis" if compute else "basis-skip")
        n_eig = self.a["n_eig"]
        if compute:
            lam, C = orc.subspace_basis(self.chi0.numpy(), n_eig)
            self.C, self.lam = torch.from_numpy(np.ascontiguousarray(C)), torch.from_numpy(lam)
        else:
            self.C = torch.full((n_eig, self.inp.n_g), float("nan"), dtype=torch.complex128)
            self.lam = torch.full((n_eig,), float("nan"), dtype=torch.float64)
        return self.C, self.lam

    def rpa_pass2_chis(self, ctx):
        import torch
        from oracle import rpa_oracle as orc
        self.calls.append("pass2")
        a = self.a
        self.chis = torch.from_numpy(orc.chi_subspace_freq(self.M, a["e_v"], a["e_c"], self.inp.vcoul, self.C.numpy(), a["omega"]))
        return self.chis

    def rpa_pass_energy(self, ctx, weight):
        from oracle import rpa_oracle as orc
        self.calls.append("energy")
        e, t = orc.correlation_energy(self.chis.numpy(), weight.numpy())
        return dict(E_c=e, t=t, lam=self.lam.numpy().copy(), stage_ms={})

    def rpa_pass_end(self, ctx):
        self.calls.append("end")


def _driver_worker(rank, world, port, out):
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from rpa_inputs import make_inputs
        from paper_2405_20258_b200.sharded import Comm, rpa_energy_sharded
        inp = make_inputs(0, n_v=3, n_c=41)
        c0, c1 = shard_range(41, world, rank)
        t = lambda a: torch.from_numpy(np.ascontiguousarray(a))
        be = OraclePassBackend(inp)
        r = rpa_energy_sharded(None, t(inp.psi_v), t(inp.psi_c[c0:c1]), t(inp.e_v), t(inp.e_c[c0:c1]), 2, 20, 0.0, t(inp.omega),
                               t(inp.weight), comm=Comm(), backend=be)
        out.put((rank, r["E_c"], float(r["lam"][0]), be.calls))
    finally:
        dist.destroy_process_group()


def test_sharded_driver_host_logic_two_gloo_ranks():
    """rpa_energy_sharded ITSELF under two gloo ranks (the oracle stands in for the library's pass-level calls): the
    partial sums are reduced in place, only rank 0 computes the basis, both ranks end with the single-process E_c."""
    import torch.multiprocessing as mp
    from oracle import rpa_oracle as orc
    from rpa_inputs import make_inputs
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_driver_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=300) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    ref = orc.rpa_energy(make_inputs(0, n_v=3, n_c=41), n_eig=20)
    for rank, e, lam0, calls in res:
        assert abs(e - ref["E_c"]) <= 1e-12 * abs(ref["E_c"])
        assert abs(lam0 - ref["lam"][0]) <= 1e-12 * abs(ref["lam"][0])
        assert calls == ["begin", "pass1", "basis" if rank == 0 else "basis-skip", "pass2", "energy", "end"]
    assert res[0][1] == res[1][1]


def test_two_rank_gloo_sum_matches_single_process():
    import torch.multiprocessing as mp
    from oracle import rpa_oracle as orc
    from rpa_inputs import make_inputs
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=300) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    ref = orc.rpa_energy(make_inputs(0, n_v=3, n_c=41), n_eig=20)
    for _, e, lam0 in res:
        assert abs(e - ref["E_c"]) <= 1e-12 * abs(ref["E_c"])
        assert abs(lam0 - ref["lam"][0]) <= 1e-12 * abs(ref["lam"][0])
    assert res[0][1] == res[1][1]          # both ranks hold the same sums and the same (broadcast) basis
