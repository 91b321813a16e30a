"""N_eig accuracy / cost sweep (BASELINE.json configs[4]; cost of the frequency part ~ (N_G/N_b)^2).

    python -m paper_2405_20258_b200.sweep --config 2        # medium system (readings R2, R16 of DESIGN.md)
    python -m paper_2405_20258_b200.sweep --config 3        # large system

For N_eig/N_G in {5, 10, 20, 40 %} the whole hot path runs through rpa_energy_device (valence blocks of the config) and
its stage times are reported; the 100 % point is the full-basis chi~0(i omega) (C = identity, P8: equal to the subspace
result at N_eig = N_G), accumulated through the stage calls.  Prints one JSON object: per point E_c, the error of the
subspace approximation against the full basis (the method's own approximation on this workload, not a parity item) and
the time split MTXEL / static chi0 / basis / chi_s(i omega) / Tr ln.  `run_sweep` is the same as a function (the GPU
test of configs[4] calls it on a twin)."""
from __future__ import annotations

import argparse
import json
import os
import sys
import time

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))


def run_sweep(inp, fractions=None, nvb=None, device=0, log=None):
    """The five points on the inputs `inp` (an rpa_inputs.RpaInputs).  Returns {"workload", "points"}; a point holds
    fraction, n_eig, E_c, wall_s, stage_ms (MTXEL / static chi0 / basis / chi_s(i omega) / Tr ln) and, when the 100 % point
    is among them, rel_error_vs_full_basis."""
    import torch
    from . import binding as rpa
    from rpa_inputs import sweep_n_eig, SWEEP_FRACTIONS
    cfg = inp.cfg
    fr = list(fractions or SWEEP_FRACTIONS)
    dev = f"cuda:{device}"
    nv, nc, ng, n_w = inp.psi_v.shape[0], inp.psi_c.shape[0], inp.n_g, len(inp.omega)
    nvb = min(nvb or cfg.nvb or nv, nv)
    n_eigs = sweep_n_eig(ng, fr)
    ctx = rpa.rpa_create(inp.cell, inp.fft, inp.g_eps, inp.vcoul, inp.g_wfn, device=device)
    d = {k: torch.from_numpy(getattr(inp, k)).to(dev) for k in ("psi_v", "psi_c", "e_v", "e_c", "omega", "weight")}
    free_b, _ = torch.cuda.mem_get_info(device)
    # one workspace for every point (the context keeps the tensor it was lent alive)
    extra = nv * nc * ng * 16 + nc * int(np.prod(inp.fft)) * 16 + 8192          # all of M + the real-space conduction functions
    full_extra = n_w * ng * ng * 16 + nvb * nc * ng * 16                           # tensors of the full-basis point
    need = max([rpa.rpa_energy_workspace_bytes(ctx, nv, nc, nvb, k, n_w) for k in n_eigs if k < ng] +
               [rpa.rpa_workspace_bytes(ctx, nvb, nc, ng, n_w)])
    keep = need + extra + (full_extra if ng in n_eigs else 0) <= 0.85 * free_b
    ws = torch.empty(need + (extra if keep else 0), dtype=torch.uint8, device=dev)
    rpa.rpa_set_workspace(ctx, ws)
    points = []
    for f, n_eig in zip(fr, n_eigs):
        torch.cuda.synchronize(device)
        t0 = time.perf_counter()
        if n_eig < ng:
            r = rpa.rpa_energy_device(ctx, d["psi_v"], d["psi_c"], d["e_v"], d["e_c"], nvb, n_eig, 0.0, d["omega"], d["weight"], keep_m=keep)
            e_c, ms = r["E_c"], r["stage_ms"]
        else:   # full basis: chi~0(i w_k) itself (C = identity), no basis stage -- P8: equals the subspace result at N_eig = N_G
            chi = torch.zeros((n_w, ng, ng), dtype=torch.complex128, device=dev)
            M = torch.empty((nvb, nc, ng), dtype=torch.complex128, device=dev)
            ev = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
            ms = {"mtxel": 0.0, "chi0_static": 0.0, "basis": 0.0, "chi_freq": 0.0, "energy": 0.0}
            for b in range(0, nv, nvb):
                e = min(nv, b + nvb)
                ev[0].record()
                rpa.rpa_mtxel(ctx, d["psi_v"][b:e].contiguous(), d["psi_c"], M[: e - b])
                ev[1].record()
                rpa.rpa_chi_subspace_freq(ctx, M[: e - b], d["e_v"][b:e].contiguous(), d["e_c"], None, ng, d["omega"], b > 0, chi)
                ev[2].record()
                torch.cuda.synchronize(device)
                ms["mtxel"] += ev[0].elapsed_time(ev[1])
                ms["chi_freq"] += ev[1].elapsed_time(ev[2])
            ev[2].record()
            e_c, _ = rpa.rpa_correlation_energy(ctx, chi, ng, d["weight"])
            ev[3].record()
            torch.cuda.synchronize(device)
            ms["energy"] = ev[2].elapsed_time(ev[3])
            del chi, M
        torch.cuda.synchronize(device)
        points.append({"fraction": f, "n_eig": n_eig, "E_c": e_c, "wall_s": time.perf_counter() - t0, "stage_ms": ms})
        if log:
            print(f"# N_eig = {n_eig:5d} ({100 * f:5.1f} %)  E_c = {e_c:.12f}  {points[-1]['wall_s']:.1f} s", file=log)
    rpa.rpa_destroy(ctx)
    full = next((p["E_c"] for p in points if p["n_eig"] == ng), None)
    for p in points:
        p["rel_error_vs_full_basis"] = None if full is None else (p["E_c"] - full) / abs(full)
    return {"workload": f"configs[{getattr(cfg, 'seed', '?')}] '{cfg.name}' seed {cfg.seed}: N_G={ng}, N_v={nv}, N_c={nc}, N_w={n_w}, "
                        f"valence blocks of {nvb}", "points": points}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=2)
    ap.add_argument("--n-v", type=int, default=None)
    ap.add_argument("--n-c", type=int, default=None)
    ap.add_argument("--fractions", default="0.05,0.10,0.20,0.40,1.00")
    args = ap.parse_args()
    from rpa_inputs import make_inputs
    inp = make_inputs(args.config, n_v=args.n_v, n_c=args.n_c, qr_device="cuda")
    out = run_sweep(inp, [float(x) for x in args.fractions.split(",")], log=sys.stderr)
    out["workload"] = f"configs[{args.config}] " + out["workload"].split("] ", 1)[1]
    print(json.dumps(out))


if __name__ == "__main__":
    main()
