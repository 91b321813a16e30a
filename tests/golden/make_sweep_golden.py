"""Writes tests/golden/<name>_twin_sweep_seed<seed>.json: oracle-only values of the N_eig accuracy sweep (BASELINE.json
configs[4]) on a scaled-down twin of a config (same cell, grids, spheres, N_G; fewer bands).
Calls ONLY oracle/ and the seeded input generator.

    python tests/golden/make_sweep_golden.py 2 --n-v 16 --n-c 375       # medium system twin
    python tests/golden/make_sweep_golden.py 4 --n-v 32 --n-c 750 --no-p8   # the sweep config itself (large system, seed 4)

--no-p8 skips the subspace evaluation of the 100 % point (N_eig = N_G, hours of CPU at N_G = 7665) and stores the
full-basis value for it: their equality (pin P8) is already stored by the medium twin.

For N_eig = floor(f N_G + 0.5), f in {5, 10, 20, 40, 100 %} (reading R16): E_c from the subspace chi_s of the leading
N_eig eigenvectors of chi~0(0) (oracle steps a3-a5), and E_c_full from chi~0(i w_k) in the whole G basis.  M and the
eigen-decomposition are computed once and shared by the five points (the oracle's functions, called in the order of
rpa_energy)."""
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import rpa_oracle as orc  # noqa: E402
from rpa_inputs import make_inputs, CONFIGS, SWEEP_FRACTIONS, sweep_n_eig  # noqa: E402


def main():
    idx = int(sys.argv[1])

    def opt(name, default=None):
        return int(sys.argv[sys.argv.index(name) + 1]) if name in sys.argv else default

    n_v, n_c = opt("--n-v"), opt("--n-c")
    cfg = CONFIGS[idx]
    inp = make_inputs(idx, n_v=n_v, n_c=n_c)
    ng = inp.n_g
    t0 = time.time()
    M = orc.mtxel(inp.psi_v, inp.psi_c, inp.g_wfn, inp.g_eps, inp.fft)
    chi_static = orc.chi0(M, inp.e_v, inp.e_c, inp.vcoul, 0.0)
    lam_all, C_all = orc.subspace_basis(chi_static, ng)                 # all eigenpairs, ascending (most negative first)
    print("M, chi0, eigh done", time.time() - t0, flush=True)
    points = []
    no_p8 = "--no-p8" in sys.argv
    for f, n_eig in zip(SWEEP_FRACTIONS, sweep_n_eig(ng)):
        if no_p8 and n_eig == ng:
            continue
        chi_s = orc.chi_subspace_freq(M, inp.e_v, inp.e_c, inp.vcoul, C_all[:n_eig], inp.omega)
        e_c, t = orc.correlation_energy(chi_s, inp.weight)
        points.append({"fraction": f, "n_eig": n_eig, "E_c": e_c, "t": t.tolist()})
        del chi_s
        print(f, n_eig, e_c, time.time() - t0, flush=True)
    t_full = np.array([orc.trace_log_term(orc.chi0(M, inp.e_v, inp.e_c, inp.vcoul, float(w))) for w in inp.omega])
    e_full = float(np.dot(inp.weight, t_full) / orc.TWO_PI)
    if no_p8:
        points.append({"fraction": 1.0, "n_eig": ng, "E_c": e_full, "t": t_full.tolist(), "note": "full-basis value (P8 not re-evaluated)"})
    out = {
        "source": "oracle/rpa_oracle.py (mtxel, chi0, subspace_basis, chi_subspace_freq, correlation_energy, trace_log_term), "
                  "written by tests/golden/make_sweep_golden.py",
        "config": idx, "name": cfg.name, "seed": cfg.seed, "n_g": ng, "n_pw": inp.n_pw, "n_v": inp.psi_v.shape[0], "n_c": inp.psi_c.shape[0],
        "points": points, "E_c_full": e_full, "t_full": t_full.tolist(), "lam_first": lam_all[:8].tolist(),
        "oracle_seconds": time.time() - t0,
    }
    path = os.path.join(ROOT, "tests", "golden", f"{cfg.name}_twin_sweep_seed{cfg.seed}.json")
    with open(path, "w") as fh:
        json.dump(out, fh, indent=1)
    print("wrote", path, "in", out["oracle_seconds"], "s")


if __name__ == "__main__":
    main()
