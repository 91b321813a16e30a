"""Helpers shared by the GPU parity tests: build a context from seeded inputs, run the stages through the C-ABI."""
import numpy as np


def torch_mod():
    import torch
    return torch


def make_ctx(inp, nvb, nc, n_eig, n_w, extra_bytes=0):
    import torch
    import paper_2405_20258_b200 as rpa
    ctx = rpa.rpa_create(inp.cell, inp.fft, inp.g_eps, inp.vcoul, inp.g_wfn, device=0)
    need = max(rpa.rpa_workspace_bytes(ctx, nvb, nc, n_eig, n_w), 1 << 20) + extra_bytes
    ws = torch.empty(need, dtype=torch.uint8, device="cuda")
    rpa.rpa_set_workspace(ctx, ws)
    return ctx


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def run_stages(ctx, inp, n_eig, nvb=None, tol=0.0, full_basis=False):
    """a1..a5 through the stage calls, looping over valence blocks in Python (the caller's loop of SURVEY 8b)."""
    import torch
    import paper_2405_20258_b200 as rpa
    nv, nc, ng = inp.psi_v.shape[0], inp.psi_c.shape[0], inp.n_g
    nvb = nv if not nvb else nvb
    psi_v, psi_c = dev(inp.psi_v), dev(inp.psi_c)
    e_v, e_c = dev(inp.e_v), dev(inp.e_c)
    omega, weight = dev(inp.omega), dev(inp.weight)
    n_w = omega.shape[0]
    chi0 = torch.zeros((ng, ng), dtype=torch.complex128, device="cuda")
    M = torch.empty((nvb, nc, ng), dtype=torch.complex128, device="cuda")
    chi_full = torch.zeros((n_w, ng, ng), dtype=torch.complex128, device="cuda") if full_basis else None
    blocks = [(s, min(nv, s + nvb)) for s in range(0, nv, nvb)]
    Ms = []
    for i, (s, e) in enumerate(blocks):
        Mb = M[: e - s]
        rpa.rpa_mtxel(ctx, psi_v[s:e].contiguous(), psi_c, Mb)
        rpa.rpa_chi0_static(ctx, Mb, e_v[s:e].contiguous(), e_c, i > 0, chi0)
        if full_basis:
            rpa.rpa_chi_subspace_freq(ctx, Mb, e_v[s:e].contiguous(), e_c, None, ng, omega, i > 0, chi_full)
        Ms.append(Mb.cpu().numpy().copy())
    Cmat = torch.empty((n_eig, ng), dtype=torch.complex128, device="cuda")
    lam = torch.empty(n_eig, dtype=torch.float64, device="cuda")
    iters = rpa.rpa_subspace_basis(ctx, chi0, n_eig, tol, Cmat, lam)
    chi_s = torch.zeros((n_w, n_eig, n_eig), dtype=torch.complex128, device="cuda")
    for i, (s, e) in enumerate(blocks):
        Mb = M[: e - s]
        rpa.rpa_mtxel(ctx, psi_v[s:e].contiguous(), psi_c, Mb)
        rpa.rpa_chi_subspace_freq(ctx, Mb, e_v[s:e].contiguous(), e_c, Cmat, n_eig, omega, i > 0, chi_s)
    e, t = rpa.rpa_correlation_energy(ctx, chi_s, n_eig, weight)
    out = dict(E_c=e, t=t, lam=lam.cpu().numpy(), C=Cmat.cpu().numpy(), chi0=chi0.cpu().numpy(),
               chi_s=chi_s.cpu().numpy(), M=np.concatenate(Ms, axis=0), iters=iters)
    if full_basis:
        out["E_c_full"], out["t_full"] = rpa.rpa_correlation_energy(ctx, chi_full, ng, weight)
    return out


def maxnorm_rel(a, b):
    """Reading R15: max|a - b| / max|b|."""
    return float(np.abs(a - b).max() / np.abs(b).max())


def eig_rel(lam, ref):
    """Reading R15: |d lambda_i| / max(|lambda_i|, 1e-6 |lambda_1|)."""
    den = np.maximum(np.abs(ref), 1e-6 * np.abs(ref).max())
    return float((np.abs(lam - ref) / den).max())


def projector_err(C, Cref):
    """|| C^H C - Cref^H Cref ||_F for row-eigenvector matrices [n_eig, n_g]."""
    p = C.conj().T @ C
    q = Cref.conj().T @ Cref
    return float(np.linalg.norm(p - q))
