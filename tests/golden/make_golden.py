"""Writes tests/golden/<name>.json: oracle-only reference values for a whole config (calls ONLY oracle/ and the
seeded input generator).  Usage: python tests/golden/make_golden.py <config index> [--nvb N]

Stored: E_c, t_k, the n_eig eigenvalues, E_c_full (optional) and a few sampled chi0 / M elements, so that GPU parity at
the full config size needs no multi-minute oracle run inside the test suite."""
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import rpa_oracle as orc  # noqa: E402
from rpa_inputs import make_inputs, CONFIGS  # noqa: E402


def main():
    idx = int(sys.argv[1])
    full = "--full-basis" in sys.argv

    def opt(name, default=None):
        return int(sys.argv[sys.argv.index(name) + 1]) if name in sys.argv else default

    n_v, n_c, n_eig = opt("--n-v"), opt("--n-c"), opt("--n-eig")      # scaled-down twin: same cell / grids, fewer bands
    cfg = CONFIGS[idx]
    inp = make_inputs(idx, n_v=n_v, n_c=n_c)
    twin = n_v is not None or n_c is not None
    t0 = time.time()
    r = orc.rpa_energy(inp, n_eig=n_eig, nvb=cfg.nvb or 8, full_basis=full)
    rng = np.random.default_rng(99)
    ng = inp.n_g
    samp = rng.integers(0, ng, size=(64, 2))
    out = {
        "source": "oracle/rpa_oracle.py rpa_energy (PAPER.md eq. 1, 3, 6-8), written by tests/golden/make_golden.py",
        "config": idx, "name": cfg.name, "seed": cfg.seed, "n_g": ng, "n_pw": inp.n_pw, "n_eig": n_eig or cfg.n_eig,
        "n_v": inp.psi_v.shape[0], "n_c": inp.psi_c.shape[0],
        "E_c": r["E_c"], "t": r["t"].tolist(), "lam": r["lam"].tolist(),
        "chi0_samples": [[int(i), int(j), float(r["chi0"][i, j].real), float(r["chi0"][i, j].imag)] for i, j in samp],
        "chi0_maxabs": float(np.abs(r["chi0"]).max()),
        "chi_s_eigs_first_freq": np.linalg.eigvalsh(r["chi_s"][0]).tolist(),
        "oracle_seconds": None,
    }
    if full:
        out["E_c_full"] = r["E_c_full"]
    out["oracle_seconds"] = time.time() - t0
    path = os.path.join(ROOT, "tests", "golden", f"{cfg.name}{'_twin' if twin else ''}_seed{cfg.seed}.json")
    with open(path, "w") as f:
        json.dump(out, f, indent=1)
    print("wrote", path, "in", out["oracle_seconds"], "s")


if __name__ == "__main__":
    main()
