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
