"""rpa_chi0_static_noalloc: the CHI_SUM entry point whose scratch (the pair weights) lives in a device array built into the
library, for callers that cannot allocate or lend memory at call time.  Collected last on purpose (the suite runs with
pytest -x).  The new entry point must give what rpa_chi0_static gives, within the max-norm tolerance the contraction tests
use (1e-13 on random operands: split-K partial sums meet through atomics, so not to the bit), on two calls in a row that
share the built-in array -- the second one smaller, so that the first call's contents are still behind what it writes --
and must refuse sizes beyond its stated maximum."""
import numpy as np
import pytest

from oracle import rpa_oracle as orc
from rpa_inputs import make_inputs

from gpu_helpers import make_ctx, dev, maxnorm_rel

pytestmark = pytest.mark.gpu


def test_noalloc_chi0_matches_workspace_path_twice_in_a_row():
    import paper_2405_20258_b200 as rpa
    import torch
    rng = np.random.default_rng(77)
    inp = make_inputs(0)
    ng = inp.n_g
    ctx_ws = make_ctx(inp, 5, 333, 10, 4)                       # the existing path: workspace lent by the caller
    ctx_na = rpa.rpa_create(inp.cell, inp.fft, inp.g_eps, inp.vcoul, inp.g_wfn)   # the new one: NO workspace at all
    try:
        assert rpa.rpa_noalloc_max_pairs() == 1 << 19
        rpa.rpa_noalloc_setup(ctx_na)
        for call, (nv, nc) in enumerate(((5, 333), (2, 41))):   # second call: fewer pairs, other energies
            M = (rng.standard_normal((nv, nc, ng)) + 1j * rng.standard_normal((nv, nc, ng))) * 0.1
            e_v = np.sort(rng.uniform(-0.6, 0, nv))
            e_c = np.sort(rng.uniform(0.05, 3, nc))
            Md, evd, ecd = dev(M), dev(e_v), dev(e_c)
            ref = torch.full((ng, ng), 7.0, dtype=torch.complex128, device="cuda")
            got = torch.full((ng, ng), -3.0, dtype=torch.complex128, device="cuda")
            rpa.rpa_chi0_static(ctx_ws, Md, evd, ecd, False, ref)
            rpa.rpa_chi0_static_noalloc(ctx_na, Md, evd, ecd, False, got)
            a, b = got.cpu().numpy(), ref.cpu().numpy()
            assert maxnorm_rel(a, b) <= 1e-13, f"call {call}"
            assert np.abs(a - a.conj().T).max() == 0.0          # mirrored exactly (R20)
            assert maxnorm_rel(a, orc.chi0(M, e_v, e_c, inp.vcoul)) <= 1e-13
            rpa.rpa_chi0_static(ctx_ws, Md, evd, ecd, True, ref)            # accumulate on top
            rpa.rpa_chi0_static_noalloc(ctx_na, Md, evd, ecd, True, got)
            assert maxnorm_rel(got.cpu().numpy(), ref.cpu().numpy()) <= 1e-13, f"call {call} (accumulate)"
        # beyond the built-in array: refused before anything is launched, the output is untouched
        nv, nc = 1025, 512                                       # 524 800 pairs > 524 288
        big = torch.empty((nv, nc, ng), dtype=torch.complex128, device="cuda")
        out = torch.full((ng, ng), 5.0, dtype=torch.complex128, device="cuda")
        with pytest.raises(rpa.RpaError) as ei:
            rpa.rpa_chi0_static_noalloc(ctx_na, big, dev(np.zeros(nv)), dev(np.ones(nc)), False, out)
        assert ei.value.code == -1 and "exceed" in str(ei.value)
        assert float((out - 5.0).abs().max()) == 0.0
    finally:
        rpa.rpa_destroy(ctx_ws)
        rpa.rpa_destroy(ctx_na)
