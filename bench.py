#!/usr/bin/env python
"""bench.py -- RPA E_c wall time on the B200 (BASELINE.json metric), one JSON line on stdout.

A step = one whole hot path (a1 MTXEL -> a2 CHI_SUM(0) -> a3 basis -> a1 again unless M is kept -> a4 chi_s(iw) ->
a5 E_c) on one synthetic config.  `value` = seconds per E_c with inputs resident in HBM; `e2e` = the same through
rpa_energy_host with pinned HOST inputs (H2D of all inputs and D2H of the result inside the timed region).
`--impl reference` times the CPU oracle (oracle/), as it stands, on a bounded sample of the same workload.
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


def algorithmic_work(inp, n_eig, passes_mtxel):
    """Algorithmic FLOPs / bytes per stage for one E_c."""
    nv, nc, ng, n_w = inp.psi_v.shape[0], inp.psi_c.shape[0], inp.n_g, len(inp.omega)
    P = nv * nc
    n_r = int(np.prod(inp.fft))
    return {
        "mtxel_bytes": passes_mtxel * P * 16.0 * (n_r + ng),          # read one real-space function + write M row, per pair
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
                                          "--format=csv,noheader,nounits", "-lms", "100"], stdout=subprocess.PIPE, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm = [float(r[0]) for r in self.rows if r and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) > 1 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(len(r) > 3 + i and r[3 + i].lower().startswith("active") for r in self.rows)]
        pw = [float(r[2]) for r in self.rows if len(r) > 2 and r[2].replace(".", "").isdigit()]
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": reasons}


def oracle_sample(inp, n_eig, budget_pairs):
    """The oracle, as it stands, on a bounded sample of the workload: the pair-proportional stages (a1, a2, a4) on a
    subset of valence bands / conduction bands, the dense stages (a3, a5) in full.  Returns timings and the estimate
    of the full-workload time (pair stages scaled by pairs_full / pairs_sample, two MTXEL passes)."""
    from oracle import rpa_oracle as orc
    nv, nc = inp.psi_v.shape[0], inp.psi_c.shape[0]
    sv = max(1, min(nv, max(2, budget_pairs // nc)))
    sc = max(1, min(nc, budget_pairs // sv))
    t0 = time.perf_counter()
    M = orc.mtxel(inp.psi_v[:sv], inp.psi_c[:sc], inp.g_wfn, inp.g_eps, inp.fft)
    t1 = time.perf_counter()
    chi = orc.chi0(M, inp.e_v[:sv], inp.e_c[:sc], inp.vcoul)
    t2 = time.perf_counter()
    lam, Cm = orc.subspace_basis(chi, n_eig)
    t3 = time.perf_counter()
    chis = orc.chi_subspace_freq(M, inp.e_v[:sv], inp.e_c[:sc], inp.vcoul, Cm, inp.omega)
    t4 = time.perf_counter()
    e, _ = orc.correlation_energy(chis, inp.weight)
    t5 = time.perf_counter()
    scale = (nv * nc) / float(sv * sc)
    est = scale * (2 * (t1 - t0) + (t2 - t1) + (t4 - t3)) + (t3 - t2) + (t5 - t4)
    return {"sample_pairs": sv * sc, "pairs": nv * nc, "t_sample_s": t5 - t0, "t_full_est_s": est,
            "stages_s": {"mtxel": t1 - t0, "chi0_static": t2 - t1, "basis": t3 - t2, "chi_freq": t4 - t3, "energy": t5 - t4},
            "sample": f"{sv} valence x {sc} conduction bands of the config ({sv * sc} of {nv * nc} pairs) for a1/a2/a4 "
                      f"(scaled by pairs, MTXEL counted twice), a3/a5 at full size"}


def cpu_threads():
    try:
        from threadpoolctl import threadpool_info
        n = [p.get("num_threads", 0) for p in threadpool_info()]
        if n:
            return int(max(n))
    except Exception:
        pass
    return os.cpu_count() or 1


def run_reference(args, inp, n_eig, workload):
    """--impl reference: the oracle on host cores; every step is one bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    budget = args.ref_pairs
    for _ in range(args.warmup):
        oracle_sample(inp, n_eig, max(1, budget // 4))
    ests, last = [], None
    t0 = time.perf_counter()
    for _ in range(args.steps):
        last = oracle_sample(inp, n_eig, budget)
        ests.append(last["t_full_est_s"])
    wall = time.perf_counter() - t0
    val = float(np.mean(ests))
    cores = cpu_threads()
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * wall / max(1, args.steps), "higher_is_better": False,
            "scaling": "strong", "vs_baseline": None, "dtype": "c128 (f64)", "data": "synthetic",
            "config": {"workload": workload, "note": "value = oracle time per E_c estimated from a bounded sample"},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": last["sample"]},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=1, help="index into BASELINE.json configs (default 1 = small)")
    ap.add_argument("--n-v", type=int, default=None, help="override the number of valence bands (scaled-down twin)")
    ap.add_argument("--n-c", type=int, default=None)
    ap.add_argument("--n-eig", type=int, default=None)
    ap.add_argument("--keep-m", type=int, default=1,
                    help="1 (default): keep all M blocks resident in HBM and skip the second MTXEL pass when they fit in 85 %% of the "
                         "free device memory (the single-block case of PAPER.md:158); 0: always recompute")
    ap.add_argument("--ref-pairs", type=int, default=6000, help="pairs in the oracle's bounded sample (about 10 s of CPU)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    args = ap.parse_args()

    from rpa_inputs import make_inputs, CONFIGS
    cfg = CONFIGS[args.config]
    big = args.config >= 2 and args.impl == "ours"
    inp = make_inputs(args.config, n_v=args.n_v, n_c=args.n_c, qr_device="cuda" if big else None)
    n_eig = args.n_eig or cfg.n_eig
    nv, nc, ng, n_w = inp.psi_v.shape[0], inp.psi_c.shape[0], inp.n_g, len(inp.omega)
    nvb = cfg.nvb or nv
    workload = (f"configs[{args.config}] '{cfg.name}' seed {cfg.seed}: cell {cfg.cell} bohr, FFT {tuple(cfg.fft)}, N_pw={inp.n_pw}, "
                f"N_G={ng}, N_v={nv}, N_c={nc}, N_eig={n_eig}, N_w={n_w}, valence blocks of {nvb}")
    if args.impl == "reference":
        return run_reference(args, inp, n_eig, workload)

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
    if world > 1:
        # strong scaling: the conduction bands (hence the (v,c) pairs) are sharded over the ranks, one all-reduce per pass
        c0, c1 = rpa.shard_range(nc, world, rank)
        inp.psi_c, inp.e_c = np.ascontiguousarray(inp.psi_c[c0:c1]), np.ascontiguousarray(inp.e_c[c0:c1])
        nc = c1 - c0
        comm = rpa.Comm()
    ctx = rpa.rpa_create(inp.cell, inp.fft, inp.g_eps, inp.vcoul, inp.g_wfn, device=local)
    need = rpa.rpa_energy_workspace_bytes(ctx, nv, nc, nvb, n_eig, n_w)
    m_all = nv * nc * ng * 16
    free_b, _ = torch.cuda.mem_get_info(local)
    inputs_b = sum(getattr(inp, k).nbytes for k in ("psi_v", "psi_c"))
    keep_m = bool(args.keep_m) and nvb < nv and need + m_all + inputs_b <= 0.85 * free_b
    if world > 1:   # the sharded driver keeps its M blocks in torch tensors: the workspace is stage scratch only
        keep_m = bool(args.keep_m) and need + m_all + inputs_b <= 0.85 * free_b
        need = rpa.rpa_workspace_bytes(ctx, nvb, nc, n_eig, n_w)
    elif keep_m:
        need += m_all
    uc_all = nc * int(np.prod(inp.fft)) * 16 + 4096     # real-space conduction functions kept across valence blocks
    if world == 1 and args.keep_m and nvb < nv:           # ... as many of them as fit in 85 % of the free memory
        need += max(0, min(uc_all, int(0.85 * free_b) - need - inputs_b))
    ws = torch.empty(need, dtype=torch.uint8, device=dev)
    rpa.rpa_set_workspace(ctx, ws)
    d = {k: torch.from_numpy(getattr(inp, k)).to(dev) for k in ("psi_v", "psi_c", "e_v", "e_c", "omega", "weight")}
    h = {k: torch.from_numpy(getattr(inp, k)).pin_memory() for k in ("psi_v", "psi_c", "e_v", "e_c", "omega", "weight")}

    def step_dev():
        if world > 1:
            return rpa.rpa_energy_sharded(ctx, d["psi_v"], d["psi_c"], d["e_v"], d["e_c"], nvb, n_eig, 0.0, d["omega"], d["weight"],
                                          comm=comm, keep_m=keep_m)
        return rpa.rpa_energy_device(ctx, d["psi_v"], d["psi_c"], d["e_v"], d["e_c"], nvb, n_eig, 0.0, d["omega"], d["weight"],
                                     keep_m=bool(args.keep_m))   # the library keeps what fits in the workspace it was lent

    def step_host():
        if world > 1:   # this rank's inputs from pinned host memory, then the sharded path; E_c read back inside
            t = {k: h[k].to(dev, non_blocking=True) for k in h}
            return rpa.rpa_energy_sharded(ctx, t["psi_v"], t["psi_c"], t["e_v"], t["e_c"], nvb, n_eig, 0.0, t["omega"], t["weight"],
                                          comm=comm, keep_m=keep_m)
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

    n_warm = max(args.warmup, 3) if args.config <= 1 else max(args.warmup, 1)   # big configs: one step already runs for seconds
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
        step_host()
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            step_host()
        barrier()
        e2e_s = (time.perf_counter() - t0) / args.steps
        h2d = sum(h[k].numel() * h[k].element_size() for k in h)
        e2e = {"value": e2e_s, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(8 * (1 + n_eig + n_w))}

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
    work = algorithmic_work(inp, n_eig, passes)
    stages = {
        "mtxel": {"ms": stage_ms["mtxel"], "GBps": work["mtxel_bytes"] / (stage_ms["mtxel"] * 1e-3) / 1e9,
                  "frac_of_hbm": work["mtxel_bytes"] / (stage_ms["mtxel"] * 1e-3) / 1e9 / hbm_peak, "passes": passes},
        "chi0_static": {"ms": stage_ms["chi0_static"], "TFLOPs": work["chi0_flops"] / (stage_ms["chi0_static"] * 1e-3) / 1e12,
                        "frac_of_dmma_peak": work["chi0_flops"] / (stage_ms["chi0_static"] * 1e-3) / 1e12 / dmma_peak},
        "basis": {"ms": stage_ms["basis"]},
        "chi_freq": {"ms": stage_ms["chi_freq"],
                     "TFLOPs": (work["proj_flops"] + work["chis_flops"]) / (stage_ms["chi_freq"] * 1e-3) / 1e12,
                     "frac_of_dmma_peak": (work["proj_flops"] + work["chis_flops"]) / (stage_ms["chi_freq"] * 1e-3) / 1e12 / dmma_peak},
        "energy": {"ms": stage_ms["energy"]},
    }
    # per-kernel-class device time (CUDA events around each launch, inside the timed region) and algorithmic work
    n_r, n3 = int(np.prod(inp.fft)), int(inp.fft[2])
    nk = [len(np.unique(inp.g_eps[:, a])) for a in range(3)]
    P = nv * nc
    kwork = {   # (unit, algorithmic work per E_c)
        "mtxel_plane": ("B", passes * P * 16.0 * (n_r + nk[0] * nk[1] * n3)),   # read one real-space function, write its kept plane frequencies
        "mtxel_z": ("B", passes * P * 16.0 * (nk[0] * nk[1] * n3 + ng)),
        "chi0": ("FLOP", work["chi0_flops"]), "proj": ("FLOP", work["proj_flops"]), "chis": ("FLOP", work["chis_flops"]),
    }
    jn, jsweeps, jkind = rpa.rpa_basis_info(ctx)
    if jn > 0:   # direct Jacobi of chi~0(0): vector form = FP64 ALU work, block form = DMMA GEMM work
        if jkind == 1:
            kwork["basis"] = ("FLOP", jsweeps * 32.0 * jn ** 3)
        elif jkind == 2:   # tridiagonalisation (16/3 n^3 real FLOP for a complex Hermitian matrix) + back-transformation (8 n^2 n_eig)
            kwork["basis"] = ("ALU", 16.0 / 3.0 * jn ** 3 + 8.0 * jn * jn * n_eig)
        else:
            kwork["basis"] = ("ALU", jsweeps * 0.5 * jn * (jn - 1) * 44.0 * jn)
    kernels = {}
    for k, (kms, kn) in kprof.items():
        ent = {"ms_per_step": kms / args.steps, "launches_per_step": kn / args.steps}
        if k in kwork and kms > 0:
            unit, w = kwork[k]
            rate = w / (kms / args.steps * 1e-3)
            ent.update({"GBps": rate / 1e9, "frac_of_hbm": rate / 1e9 / hbm_peak} if unit == "B" else
                       {"TFLOPs": rate / 1e12, "frac_of_dfma_peak": rate / 1e12 / dfma_peak} if unit == "ALU" else
                       {"TFLOPs": rate / 1e12, "frac_of_dmma_peak": rate / 1e12 / dmma_peak})
        kernels[k] = ent
    traffic_tab = {}
    try:
        traffic_tab = json.load(open(os.path.join(ROOT, "profiles", "ncu_traffic.json")))
    except Exception:
        pass
    dom = max(kwork, key=lambda k: kernels[k]["ms_per_step"])
    kd = kernels[dom]
    names = {"mtxel_plane": "pair_plane_fft8_kernel (MTXEL a1: pair product + pruned xy transforms)",
             "mtxel_z": "fft_axis_kernel<false,1> (MTXEL a1: z transform + sphere gather)",
             "chi0": "zgemm_dmma_kernel<1,1,1,3,1> (CHI_SUM a2)", "proj": "zgemm_dmma_kernel<0,0,1,2,0> (projection a4)",
             "chis": "zgemm_dmma_kernel<1,1,1,3,1> batched over omega (chi_s a4)",
             "basis": "jacobi_persistent_kernel (a3: one-sided Jacobi of chi~0(0), all sweeps in one cooperative launch)" if jkind == 0
             else "hetrd_fused_kernel + bisect/invit/backtransform kernels (a3: tridiagonalisation route for the lowest N_eig eigenpairs)" if jkind == 2
             else "block Jacobi of chi~0(0) (a3: batched zgemm_dmma Gram + pair_rotations_kernel + batched zgemm_dmma update)"}
    tr = traffic_tab.get(f"{dom}:cfg{args.config}")
    if kwork[dom][0] == "B":
        per_launch = kwork[dom][1] / max(1.0, kd["launches_per_step"])
        avg_s = kd["ms_per_step"] * 1e-3 / max(1.0, kd["launches_per_step"])
        roofline = {"kernel": names[dom], "bound": "hbm", "achieved": per_launch / avg_s / 1e9, "peak": hbm_peak, "unit": "GB/s",
                    "frac": per_launch / avg_s / 1e9 / hbm_peak, "traffic": tr, "peak_source": hbm_src,
                    "algorithmic_bytes_per_launch": per_launch, "avg_launch_ms": avg_s * 1e3,
                    "bytes_model": "16 B x (N_r + nk_x nk_y N_z) per (v,c) pair in the launch (DESIGN.md 5.2)",
                    "share_of_step": kd["ms_per_step"] / ms_per_step}
    elif kwork[dom][0] == "ALU":
        avg_s = kd["ms_per_step"] * 1e-3
        roofline = {"kernel": names[dom], "bound": "alu", "achieved": kwork[dom][1] / avg_s / 1e12, "peak": dfma_peak, "unit": "TFLOP/s",
                    "frac": kwork[dom][1] / avg_s / 1e12 / dfma_peak, "traffic": tr,
                    "peak_source": "FP64 FMA register-only microbenchmark measured in this run (rpa_fp64_peak kind 1)",
                    "algorithmic_flops_per_launch": kwork[dom][1], "avg_launch_ms": avg_s * 1e3,
                    "flops_model": (f"16/3 n^3 + 8 n^2 N_eig FLOP, n = {jn}; bound by the two grid-wide barriers per Householder step"
                                    if jkind == 2 else
                                    f"{jsweeps} sweeps x n(n-1)/2 pairs x 44 n FLOP (16 n for the three dot products, 28 n for the "
                                    f"rotation), n = {jn}; the kernel is bound by the grid-wide barrier per round, not by the ALUs"),
                    "share_of_step": kd["ms_per_step"] / ms_per_step}
    else:
        per_launch = kwork[dom][1] / max(1.0, kd["launches_per_step"])
        avg_s = kd["ms_per_step"] * 1e-3 / max(1.0, kd["launches_per_step"])
        roofline = {"kernel": names[dom], "bound": "tensor", "achieved": per_launch / avg_s / 1e12, "peak": dmma_peak,
                    "unit": "TFLOP/s", "frac": per_launch / avg_s / 1e12 / dmma_peak, "traffic": tr,
                    "peak_source": "FP64 mma.sync m8n8k4 register-only microbenchmark measured in this run (rpa_fp64_peak); "
                                   "MEASURED_PEAKS.json has no FP64 entry",
                    "algorithmic_flops_per_launch": per_launch, "avg_launch_ms": avg_s * 1e3,
                    "flops_model": "8 flop per complex MAC; Hermitian updates count the lower triangle only (DESIGN.md 5.1)",
                    "share_of_step": kd["ms_per_step"] / ms_per_step}
    cpu_baseline = None
    if not args.no_cpu_baseline and world == 1:
        s = oracle_sample(inp, n_eig, args.ref_pairs)
        cpu_baseline = {"value": s["t_full_est_s"], "unit": UNIT, "cores": cpu_threads(), "kind": "oracle", "sample": s["sample"],
                        "t_sample_s": s["t_sample_s"]}
    line = {"metric": METRIC, "value": ms_per_step * 1e-3, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": n_warm, "ms_per_step": ms_per_step, "higher_is_better": False, "scaling": "strong",
            "vs_baseline": None, "dtype": "c128 (f64)", "data": "synthetic",
            "config": {"workload": workload, "keep_m": keep_m, "mtxel_passes": passes,
                       "parallelism": f"conduction bands sharded over {world} ranks, one all-reduce per pass" if world > 1 else "1 GPU",
                       "l2": "no flush needed: every step streams M blocks / real-space boxes far larger than the 126 MB L2"},
            "E_c": res["E_c"], "stages": stages, "kernels": kernels, "roofline": roofline,
            "fp64_peaks_measured": {"dmma_tflops": dmma_peak, "dfma_tflops": dfma_peak},
            "cpu_baseline": cpu_baseline, "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks}
    print(json.dumps(line))


if __name__ == "__main__":
    main()
