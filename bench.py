#!/usr/bin/env python
"""bench.py -- RPA E_c wall time on the B200 (BASELINE.json metric), one JSON line on stdout.

A step = one whole hot path (a1 MTXEL -> a2 CHI_SUM(0) -> a3 basis -> a1 again unless M is kept -> a4 chi_s(iw) ->
a5 E_c) on one synthetic config.  Default workload: configs[2] (the medium slab), the largest config for which both
arms of the driver's command (ours, then `--impl reference`) finish inside its per-arm limit; DESIGN.md section 7 has the
arithmetic.  `value` = seconds per E_c with inputs resident in HBM; `e2e` = the same through rpa_energy_host with pinned
HOST inputs (H2D of all inputs and D2H of the result inside the timed region).  Every fraction in the line follows from
SURVEY.md 8(d)'s per-unit work and the line's own times:

  MTXEL            16 (N_r + N_G) B per (v,c) pair and pass       (stage, and the plane kernel alone on ITS time)
  CHI_SUM(0)       4 N_G^2 FLOP per pair                           (lower triangle, 8 FLOP per complex MAC)
  projection       8 N_eig N_G FLOP per pair
  chi_s(i omega)   4 N_w N_eig^2 FLOP per pair

`--impl reference` times the CPU oracle (oracle/), as it stands, on bounded samples of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "rpa_ec_wall_time"
UNIT = "s"
DEFAULT_CONFIG = 2


def algorithmic_work(inp, n_eig, passes_mtxel):
    """Algorithmic FLOPs / bytes per stage for one E_c."""
    nv, nc, ng, n_w = inp.psi_v.shape[0], inp.psi_c.shape[0], inp.n_g, len(inp.omega)
    P = nv * nc
    n_r = int(np.prod(inp.fft))
    return {
        "pairs": P,
        "mtxel_bytes_per_pair_pass": 16.0 * (n_r + ng),                # read one real-space function + write one M row
        "mtxel_bytes": passes_mtxel * P * 16.0 * (n_r + ng),
        "chi0_flops": 4.0 * ng * ng * P,                               # Hermitian rank-P update, lower triangle, 8 flop / cMAC
        "proj_flops": 8.0 * n_eig * ng * P,
        "chis_flops": n_w * 4.0 * n_eig * n_eig * P,
    }


class ClockSampler:
    QUERY = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.QUERY}",
                                          "--format=csv,noheader,nounits", "-lms", "250"], stdout=subprocess.PIPE, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.3)
        self.proc.terminate()
        sm = [float(r[0]) for r in self.rows if r and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) > 1 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(len(r) > 3 + i and r[3 + i].lower().startswith("active") for r in self.rows)]
        pw = [float(r[2]) for r in self.rows if len(r) > 2 and r[2].replace(".", "").isdigit()]
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_min_mhz": min(sm) if sm else None,
                "sm_max_mhz": max(mx) if mx else None, "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": reasons}


# ------------------------------------------------------------------------------------------------------------------
# The oracle, as it stands, on a bounded sample of the workload.  The pair-proportional stages (a1, a2, a4) run on
# `sv` valence x `sc` conduction bands of the config; the dense stages do not depend on the number of pairs (a3 is an
# N_G x N_G eigenproblem and a5 N_w eigenproblems of size N_eig whatever the sample) and run at FULL size.
def oracle_pair_sample(inp, C, budget_pairs):
    from oracle import rpa_oracle as orc
    nv, nc = inp.psi_v.shape[0], inp.psi_c.shape[0]
    sv = max(1, min(nv, 2))
    sc = max(1, min(nc, budget_pairs // sv))
    t0 = time.perf_counter()
    orc.wfn_to_realspace(inp.psi_c[:min(sc, 32)], inp.g_wfn, inp.fft)           # cost of one band's transform, timed alone
    t_band = (time.perf_counter() - t0) / min(sc, 32)
    t0 = time.perf_counter()
    M = orc.mtxel(inp.psi_v[:sv], inp.psi_c[:sc], inp.g_wfn, inp.g_eps, inp.fft)
    t1 = time.perf_counter()
    chi = orc.chi0(M, inp.e_v[:sv], inp.e_c[:sc], inp.vcoul)
    t2 = time.perf_counter()
    chis = orc.chi_subspace_freq(M, inp.e_v[:sv], inp.e_c[:sc], inp.vcoul, C, inp.omega) if C is not None else None
    t3 = time.perf_counter()
    return {"sv": sv, "sc": sc, "t_band": t_band, "t_mtxel": t1 - t0, "t_chi0": t2 - t1, "t_chi_freq": t3 - t2, "chi0": chi, "chi_s": chis}


def oracle_dense(inp, chi0_sample, n_eig, chi_s_sample=None):
    """a3 on an N_G x N_G matrix and a5 on N_w matrices of size N_eig: their cost is that of the full workload."""
    from oracle import rpa_oracle as orc
    t0 = time.perf_counter()
    lam, C = orc.subspace_basis(chi0_sample, n_eig)
    t1 = time.perf_counter()
    if chi_s_sample is None:
        chi_s_sample = -np.tile(np.eye(n_eig, dtype=np.complex128) * 0.1, (len(inp.omega), 1, 1))
    orc.correlation_energy(chi_s_sample, inp.weight)
    t2 = time.perf_counter()
    return C, t1 - t0, t2 - t1


def oracle_estimate(inp, s, t_basis, t_energy, nvb):
    """Time of oracle.rpa_energy(inp, nvb=nvb) on the full workload from a sample: per valence block and pass the oracle
    transforms the block's valence bands and ALL conduction bands to real space (t_band each) and forms nvb x nc pair
    rows (t_pair each); a2 and a4 scale with the number of pairs; a3 and a5 were run at full size."""
    nv, nc = inp.psi_v.shape[0], inp.psi_c.shape[0]
    pairs_s = s["sv"] * s["sc"]
    t_pair = max(0.0, s["t_mtxel"] - (s["sv"] + s["sc"]) * s["t_band"]) / pairs_s
    nblocks = (nv + nvb - 1) // nvb
    t_mtxel = 2 * (nblocks * nc + nv) * s["t_band"] + 2 * nv * nc * t_pair          # two passes
    scale = nv * nc / float(pairs_s)
    est = t_mtxel + scale * (s["t_chi0"] + s["t_chi_freq"]) + t_basis + t_energy
    return est, {"mtxel": t_mtxel, "chi0_static": scale * s["t_chi0"], "basis": t_basis, "chi_freq": scale * s["t_chi_freq"], "energy": t_energy}


def sample_text(s, inp, nvb):
    nv, nc = inp.psi_v.shape[0], inp.psi_c.shape[0]
    return (f"{s['sv']} valence x {s['sc']} conduction bands of the config ({s['sv'] * s['sc']} of {nv * nc} pairs) through a1/a2/a4, "
            f"scaled to the full workload (pair rows by pairs, band transforms by bands x {2 * ((nv + nvb - 1) // nvb)} block passes); "
            f"a3 (N_G x N_G) and a5 (N_w x N_eig^2) at full size")


def cpu_threads():
    try:
        from threadpoolctl import threadpool_info
        n = [p.get("num_threads", 0) for p in threadpool_info()]
        if n:
            return int(max(n))
    except Exception:
        pass
    return os.cpu_count() or 1


def run_reference(args, n_eig):
    """--impl reference: the oracle on the host cores.  Inputs are generated once (QR on the CPU); the dense stages
    (a3, a5: independent of the sample) are timed once, before the warm-up; every step is one bounded pair sample."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    from rpa_inputs import make_inputs, CONFIGS
    cfg = CONFIGS[args.config]
    inp = make_inputs(args.config, n_v=args.n_v, n_c=args.n_c)
    nv, nc = inp.psi_v.shape[0], inp.psi_c.shape[0]
    nvb = cfg.nvb or nv
    workload = workload_text(args, cfg, inp, n_eig, nvb)
    first = oracle_pair_sample(inp, None, max(2, args.ref_pairs // 4))
    C, t_basis, t_energy = oracle_dense(inp, first["chi0"], n_eig)
    for _ in range(args.warmup):
        oracle_pair_sample(inp, C, max(2, args.ref_pairs // 4))
    ests, last, stages = [], None, None
    t0 = time.perf_counter()
    for _ in range(args.steps):
        last = oracle_pair_sample(inp, C, args.ref_pairs)
        est, stages = oracle_estimate(inp, last, t_basis, t_energy, nvb)
        ests.append(est)
    wall = time.perf_counter() - t0
    val = float(np.mean(ests))
    cores = cpu_threads()
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * wall / max(1, args.steps), "higher_is_better": False,
            "scaling": "strong", "vs_baseline": None, "dtype": "c128 (f64)", "data": "synthetic",
            "config": {"workload": workload, "note": "value = oracle time per E_c ESTIMATED from bounded samples; ms_per_step = one sample"},
            "stages_est_s": stages,
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle (estimated from a pair sample)",
                             "sample": sample_text(last, inp, nvb), "t_dense_once_s": t_basis + t_energy},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def workload_text(args, cfg, inp, n_eig, nvb):
    nv, nc = inp.psi_v.shape[0], inp.psi_c.shape[0]
    return (f"configs[{args.config}] '{cfg.name}' seed {cfg.seed}: cell {cfg.cell} bohr, FFT {tuple(cfg.fft)}, N_pw={inp.n_pw}, "
            f"N_G={inp.n_g}, N_v={nv}, N_c={nc}, N_eig={n_eig}, N_w={len(inp.omega)}, valence blocks of {nvb}")


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=DEFAULT_CONFIG,
                    help="index into BASELINE.json configs (default 2 = the medium slab; 0, 1 are the small cases, 3 the large one)")
    ap.add_argument("--n-v", type=int, default=None, help="override the number of valence bands (scaled-down twin)")
    ap.add_argument("--n-c", type=int, default=None)
    ap.add_argument("--n-eig", type=int, default=None)
    ap.add_argument("--keep-m", type=int, default=1,
                    help="1 (default): keep all M blocks resident in HBM and skip the second MTXEL pass when they fit in 85 %% of the "
                         "free device memory (the single-block case of PAPER.md:158); 0: always recompute")
    ap.add_argument("--ref-pairs", type=int, default=512, help="pairs in one bounded sample of the oracle")
    ap.add_argument("--e2e-steps", type=int, default=0, help="timed steps of the end-to-end leg (0 = min(steps, 5))")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    args = ap.parse_args()

    from rpa_inputs import make_inputs, CONFIGS
    cfg = CONFIGS[args.config]
    n_eig = args.n_eig or cfg.n_eig
    if args.impl == "reference":
        return run_reference(args, n_eig)

    import torch
    import paper_2405_20258_b200 as rpa
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl")
    dev = f"cuda:{local}"
    inp = make_inputs(args.config, n_v=args.n_v, n_c=args.n_c, qr_device=dev if args.config >= 2 else None)
    nv, nc, ng, n_w = inp.psi_v.shape[0], inp.psi_c.shape[0], inp.n_g, len(inp.omega)
    nc_all = nc
    nvb = cfg.nvb or nv
    workload = workload_text(args, cfg, inp, n_eig, nvb)
    comm = None
    if world > 1:
        # strong scaling: the conduction bands (hence the (v,c) pairs) are sharded over the ranks, one all-reduce per pass
        c0, c1 = rpa.shard_range(nc, world, rank)
        inp.psi_c, inp.e_c = np.ascontiguousarray(inp.psi_c[c0:c1]), np.ascontiguousarray(inp.e_c[c0:c1])
        nc = c1 - c0
        comm = rpa.Comm()
    ctx = rpa.rpa_create(inp.cell, inp.fft, inp.g_eps, inp.vcoul, inp.g_wfn, device=local)
    torch.cuda.empty_cache()
    need = rpa.rpa_energy_workspace_bytes(ctx, nv, nc, nvb, n_eig, n_w)       # inputs (host leg) + persistent + stage scratch
    m_all = nv * nc * ng * 16
    free_b, _ = torch.cuda.mem_get_info(local)
    inputs_b = sum(getattr(inp, k).nbytes for k in ("psi_v", "psi_c"))
    keep_m = bool(args.keep_m) and nvb < nv and need + m_all + inputs_b <= 0.85 * free_b
    if keep_m:
        need += m_all
    uc_all = nc * int(np.prod(inp.fft)) * 16 + 4096     # real-space conduction functions kept across valence blocks ...
    if args.keep_m and nvb < nv:                         # ... as many of them as fit in 85 % of the free memory
        need += max(0, min(uc_all, int(0.85 * free_b) - need - inputs_b))
    ws = torch.empty(need, dtype=torch.uint8, device=dev)
    rpa.rpa_set_workspace(ctx, ws)
    names_in = ("psi_v", "psi_c", "e_v", "e_c", "omega", "weight")
    d = {k: torch.from_numpy(getattr(inp, k)).to(dev) for k in names_in}
    h = {k: torch.from_numpy(getattr(inp, k)).pin_memory() for k in names_in}

    def step_dev():
        if world > 1:
            return rpa.rpa_energy_sharded(ctx, d["psi_v"], d["psi_c"], d["e_v"], d["e_c"], nvb, n_eig, 0.0, d["omega"], d["weight"],
                                          comm=comm, keep_m=bool(args.keep_m))
        return rpa.rpa_energy_device(ctx, d["psi_v"], d["psi_c"], d["e_v"], d["e_c"], nvb, n_eig, 0.0, d["omega"], d["weight"],
                                     keep_m=bool(args.keep_m))   # the library keeps what fits in the workspace it was lent

    def step_host():
        if world > 1:   # this rank's inputs from pinned host memory, then the sharded path; E_c read back inside
            t = {k: h[k].to(dev, non_blocking=True) for k in h}
            return rpa.rpa_energy_sharded(ctx, t["psi_v"], t["psi_c"], t["e_v"], t["e_c"], nvb, n_eig, 0.0, t["omega"], t["weight"],
                                          comm=comm, keep_m=bool(args.keep_m))
        return rpa.rpa_energy_host(ctx, h["psi_v"], h["psi_c"], h["e_v"], h["e_c"], nvb, n_eig, 0.0, h["omega"], h["weight"],
                                   keep_m=bool(args.keep_m))

    def barrier():
        if world > 1:
            import torch.distributed as dist
            dist.barrier()
        torch.cuda.synchronize()

    # FP64 peaks measured live (MEASURED_PEAKS.json has no FP64 entry)
    dmma_peak = rpa.rpa_fp64_peak(ctx, 0, 10)
    dfma_peak = rpa.rpa_fp64_peak(ctx, 1, 10)
    dmma_mix = rpa.rpa_fp64_peak(ctx, 2, 10)      # DMMA rate with 14 DADDs per 24 DMMAs: plain FP64 shares the pipe

    n_warm = max(args.warmup, 3) if args.config <= 2 else max(args.warmup, 1)   # configs[3]: a step runs for minutes, one warm-up is plenty
    for _ in range(n_warm):
        res = step_dev()
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    l0 = rpa.rpa_launch_count(ctx)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    stage_acc = {}
    rpa.rpa_profile_begin(ctx)          # event pairs around every launch of the hot kernel classes (device time per class)
    e0.record()
    for _ in range(args.steps):
        res = step_dev()
        for k, v in res["stage_ms"].items():
            stage_acc[k] = stage_acc.get(k, 0.0) + v
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    launches = rpa.rpa_launch_count(ctx) - l0
    kprof = rpa.rpa_profile_end(ctx)
    clocks = sampler.stop()
    if world > 1:
        import torch.distributed as dist
        t = torch.tensor([ms], device=dev, dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
    ms_per_step = ms / args.steps
    stage_ms = {k: v / args.steps for k, v in stage_acc.items()}

    e2e = None
    if not args.no_e2e:
        n_e2e = args.e2e_steps or min(args.steps, 5)
        step_host()
        barrier()
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            step_host()
        barrier()
        e2e_s = (time.perf_counter() - t0) / n_e2e
        h2d = sum(h[k].numel() * h[k].element_size() for k in h)
        e2e = {"value": e2e_s, "unit": UNIT, "steps": n_e2e, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(8 * (1 + n_eig + n_w))}

    if rank != 0:
        return
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
    hbm_src = "measured (MEASURED_PEAKS.json hbm_gbs)" if "hbm_gbs" in peaks else "fallback 6650 GB/s (B200_PROFILING.md)"
    passes = 1 if (keep_m or nvb >= nv) else 2
    work = algorithmic_work(inp, n_eig, passes)          # this rank's pairs (all of them on one GPU)
    P = nv * nc
    n_r, n3 = int(np.prod(inp.fft)), int(inp.fft[2])
    nk = [len(np.unique(inp.g_eps[:, a])) for a in range(3)]

    def rate(w, ms_):
        return w / (ms_ * 1e-3) if ms_ > 0 else 0.0

    stages = {
        "mtxel": {"ms": stage_ms["mtxel"], "GBps": rate(work["mtxel_bytes"], stage_ms["mtxel"]) / 1e9,
                  "frac_of_hbm": rate(work["mtxel_bytes"], stage_ms["mtxel"]) / 1e9 / hbm_peak, "passes": passes,
                  "bytes_model": "16 (N_r + N_G) B per (v,c) pair and pass (SURVEY 8d)"},
        "chi0_static": {"ms": stage_ms["chi0_static"], "TFLOPs": rate(work["chi0_flops"], stage_ms["chi0_static"]) / 1e12,
                        "frac_of_dmma_peak": rate(work["chi0_flops"], stage_ms["chi0_static"]) / 1e12 / dmma_peak},
        "basis": {"ms": stage_ms["basis"]},
        "chi_freq": {"ms": stage_ms["chi_freq"],
                     "TFLOPs": rate(work["proj_flops"] + work["chis_flops"], stage_ms["chi_freq"]) / 1e12,
                     "frac_of_dmma_peak": rate(work["proj_flops"] + work["chis_flops"], stage_ms["chi_freq"]) / 1e12 / dmma_peak},
        "energy": {"ms": stage_ms["energy"]},
    }
    if "allreduce" in stage_ms:
        stages["allreduce"] = {"ms": stage_ms["allreduce"]}
    # per-kernel-class device time (CUDA events around each launch, inside the timed region) against 8(d) work
    kwork = {   # class -> (unit, algorithmic work per E_c)
        "mtxel_plane": ("B", work["mtxel_bytes"]),       # the stage's 8(d) bytes on the plane kernel's own time
        "chi0": ("FLOP", work["chi0_flops"]), "proj": ("FLOP", work["proj_flops"]), "chis": ("FLOP", work["chis_flops"]),
    }
    jn, jsweeps, jkind = rpa.rpa_basis_info(ctx)
    if jn > 0:   # last dense eigen-decomposition of the basis stage
        if jkind == 1:
            kwork["basis"] = ("FLOP", jsweeps * 32.0 * jn ** 3)
        elif jkind == 2:   # tridiagonalisation (16/3 n^3 real FLOP for a complex Hermitian matrix) + back-transformation (8 n^2 n_eig)
            kwork["basis"] = ("ALU", 16.0 / 3.0 * jn ** 3 + 8.0 * jn * jn * n_eig)
        else:
            kwork["basis"] = ("ALU", jsweeps * 0.5 * jn * (jn - 1) * 44.0 * jn)
    kernels = {}
    for k, (kms, kn) in kprof.items():
        ent = {"ms_per_step": kms / args.steps, "launches_per_step": kn / args.steps, "share_of_step": kms / args.steps / ms_per_step}
        if k in kwork and kms > 0:
            unit, w = kwork[k]
            r = rate(w, kms / args.steps)
            ent.update({"GBps": r / 1e9, "frac_of_hbm": r / 1e9 / hbm_peak} if unit == "B" else
                       {"TFLOPs": r / 1e12, "frac_of_dfma_peak": r / 1e12 / dfma_peak} if unit == "ALU" else
                       {"TFLOPs": r / 1e12, "frac_of_dmma_peak": r / 1e12 / dmma_peak})
        kernels[k] = ent
    if kprof.get("mtxel_z", (0, 0))[0] > 0:
        # the z stage has no 8(d) figure of its own: its own input + output (the intermediate T it reads is the plane
        # kernel's product, not algorithmic traffic) -- reported as kernel I/O, labelled as such
        io = passes * P * 16.0 * (nk[0] * nk[1] * n3 + ng)
        kernels["mtxel_z"].update({"kernel_io_GBps": rate(io, kprof["mtxel_z"][0] / args.steps) / 1e9,
                                   "kernel_io_frac_of_hbm": rate(io, kprof["mtxel_z"][0] / args.steps) / 1e9 / hbm_peak,
                                   "kernel_io_model": "16 (nk_x nk_y N_z + N_G) B per pair: reads the intermediate T, writes M (not an 8(d) figure)"})
    prof_tab = {}
    try:
        prof_tab = json.load(open(os.path.join(ROOT, "profiles", "ncu_traffic.json")))
    except Exception:
        pass
    ptab = prof_tab.get("entries", {})

    def ncu_entry(cls):
        e = ptab.get(f"{cls}:cfg{args.config}")
        return e if isinstance(e, dict) and args.n_v is None and args.n_c is None and world == 1 else None

    names = {"mtxel_plane": "pair_plane_fft8_kernel (MTXEL a1: pair product + pruned xy transforms)",
             "chi0": "zherk_tma_kernel (CHI_SUM a2: Hermitian rank-P update on DMMA, TMA-staged)",
             "proj": "zgemm_dmma_kernel<0,0,1,2,0> (projection a4)",
             "chis": "zherk_tma_kernel batched over omega (chi_s a4: Hermitian rank-P update on DMMA, TMA-staged)",
             "basis": "jacobi_persistent_kernel (a3: one-sided Jacobi of chi~0(0), all sweeps in one cooperative launch)" if jkind == 0
             else "hetrd_fused_kernel + bisect/invit/backtransform kernels (a3: tridiagonalisation route for the lowest N_eig eigenpairs)" if jkind == 2
             else "block Jacobi of chi~0(0) (a3: batched zgemm_dmma Gram + pair_rotations_kernel + batched zgemm_dmma update)"}

    def roofline_of(cls):
        kd, (unit, w) = kernels[cls], kwork[cls]
        nl = max(1.0, kd["launches_per_step"])
        per_launch, avg_s = w / nl, kd["ms_per_step"] * 1e-3 / nl
        ne = ncu_entry(cls)
        out = {"kernel": names[cls], "share_of_step": kd["share_of_step"], "avg_launch_ms": avg_s * 1e3, "launches_per_step": nl}
        if unit == "B":
            out.update({"bound": "hbm", "achieved": per_launch / avg_s / 1e9, "peak": hbm_peak, "unit": "GB/s",
                        "frac": per_launch / avg_s / 1e9 / hbm_peak, "peak_source": hbm_src,
                        "algorithmic_bytes_per_launch": per_launch,
                        "bytes_model": "16 (N_r + N_G) B per (v,c) pair of the launch (SURVEY 8d), over the plane kernel's own time"})
        elif unit == "ALU":
            out.update({"bound": "alu", "achieved": w / (kd["ms_per_step"] * 1e-3) / 1e12, "peak": dfma_peak, "unit": "TFLOP/s",
                        "frac": w / (kd["ms_per_step"] * 1e-3) / 1e12 / dfma_peak,
                        "peak_source": "FP64 FMA register-only microbenchmark measured in this run (rpa_fp64_peak kind 1)",
                        "algorithmic_flops_per_launch": w})
        else:
            out.update({"bound": "tensor", "achieved": per_launch / avg_s / 1e12, "peak": dmma_peak, "unit": "TFLOP/s",
                        "frac": per_launch / avg_s / 1e12 / dmma_peak,
                        "peak_source": "FP64 mma.sync m8n8k4 register-only microbenchmark measured in this run (rpa_fp64_peak kind 0); "
                                       "MEASURED_PEAKS.json has no FP64 entry",
                        "algorithmic_flops_per_launch": per_launch,
                        "flops_model": "8 FLOP per complex MAC, Hermitian updates count the lower triangle only (SURVEY 8d)"})
        out["traffic"] = None
        if ne:   # dram__bytes_read + write of ONE launch from the ncu --set full capture named in profiles/ncu_traffic.json
            out["traffic"] = ne.get("dram_bytes_per_launch")
            out["traffic_source"] = f"{ne.get('source')} (commit {prof_tab.get('commit')})"
            if unit == "B" and out["traffic"]:
                out["traffic_over_algorithmic"] = out["traffic"] / per_launch
            if "units" in ne:          # pipe utilisation of that launch as ncu measured it
                out["ncu_units"] = ne["units"]
            if "binding_unit" in ne:   # where DRAM traffic is far below the algorithmic bytes the roof is elsewhere: say which unit
                out["binding_unit"] = ne["binding_unit"]
        return out

    dom = max(kwork, key=lambda k: kernels[k]["ms_per_step"])
    roofline = roofline_of(dom)
    roofline_mtxel = roofline_of("mtxel_plane") if dom != "mtxel_plane" and kernels["mtxel_plane"]["ms_per_step"] > 0 else None

    cpu_baseline = None
    if not args.no_cpu_baseline and world == 1:
        s = oracle_pair_sample(inp, None, args.ref_pairs)
        C, t_basis, t_energy = oracle_dense(inp, s["chi0"], n_eig)
        s2 = oracle_pair_sample(inp, C, args.ref_pairs)
        est, st = oracle_estimate(inp, s2, t_basis, t_energy, nvb)
        cpu_baseline = {"value": est, "unit": UNIT, "cores": cpu_threads(), "kind": "oracle (estimated from a pair sample)",
                        "sample": sample_text(s2, inp, nvb), "stages_est_s": st,
                        "t_sample_s": s2["t_mtxel"] + s2["t_chi0"] + s2["t_chi_freq"] + t_basis + t_energy}
    line = {"metric": METRIC, "value": ms_per_step * 1e-3, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": n_warm, "ms_per_step": ms_per_step, "higher_is_better": False, "scaling": "strong",
            "vs_baseline": None, "dtype": "c128 (f64)", "data": "synthetic",
            "config": {"workload": workload, "keep_m": keep_m, "mtxel_passes": passes,
                       "parallelism": f"conduction bands sharded over {world} ranks ({nc} of {nc_all} on rank 0), one all-reduce per pass" if world > 1 else "1 GPU",
                       "l2": "no flush needed: every step streams M blocks / real-space boxes far larger than the 126 MB L2"},
            "E_c": res["E_c"], "stages": stages, "kernels": kernels, "roofline": roofline, "roofline_mtxel": roofline_mtxel,
            "fp64_peaks_measured": {"dmma_tflops": dmma_peak, "dfma_tflops": dfma_peak, "dmma_tflops_with_14_dadd_per_24_dmma": dmma_mix},
            "cpu_baseline": cpu_baseline, "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks}
    print(json.dumps(line))


if __name__ == "__main__":
    main()
