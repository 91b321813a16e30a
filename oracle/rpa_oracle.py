"""CPU oracle for the static-subspace RPA correlation-energy hot path.

TEST INFRASTRUCTURE ONLY.  Only `tests/`, `__graft_entry__.smoke()` and the
`cpu_baseline` / `--impl reference` legs of `bench.py` may import this module.
The product path (paper_2405_20258_b200) never imports it and shares no code
with it.  Plain, slow, FP64 (complex128) numpy; each function states the
passage of /root/reference/PAPER.md (and the BASELINE.json `north_star`
reading listed in DESIGN.md) that it follows.  Library primitives used as
single steps: `@` (matrix product), `numpy.linalg.eigh` / `eigvalsh`.

Conventions: R5 chi = -v^1/2 M D M^H v^1/2;
R6 D(iw) = 2 Delta/(Delta^2 + w^2), Delta = e_c - e_v; R7 M_vc(G) =
(1/N_r) sum_r conj(u_v(r)) u_c(r) e^{-iG.r}; R8 sum_G |c_n(G)|^2 = 1, u has no
1/sqrt(Omega); R9 the basis diagonalises the Coulomb-symmetrised chi~0(0).

Parity pins: every function here is pinned by tests/test_oracle_pins.py
(closed forms, brute force, invariants); none is "parity unpinned".
"""
from __future__ import annotations

import numpy as np

TWO_PI = 2.0 * np.pi


# --------------------------------------------------------------------------
# Step a1 -- MTXEL (PAPER.md:52 eq. 3; :96; north_star "M_vc(G) = FFT[psi_v* psi_c]")
# --------------------------------------------------------------------------
def dft_matrix(n: int, freqs: np.ndarray, sign: int) -> np.ndarray:
    """F[k, r] = exp(sign * 2 pi i * freqs[k] * r / n), r = 0..n-1.

    The angle is reduced with the integer (freq * r mod n) before cos/sin are
    called, so the matrix is accurate to an ulp for any n."""
    freqs = np.asarray(freqs, dtype=np.int64)
    r = np.arange(n, dtype=np.int64)
    m = np.mod(np.outer(freqs, r), n).astype(np.float64)
    ang = TWO_PI * m / n
    return np.cos(ang) + 1j * float(sign) * np.sin(ang)


def wfn_to_realspace(psi: np.ndarray, g_wfn: np.ndarray, fft) -> np.ndarray:
    """u_n(r) = sum_G c_n(G) exp(+2 pi i (n1 r1/N1 + n2 r2/N2 + n3 r3/N3)) by a naive DFT.

    psi [nb, n_pw] -> u [nb, N1, N2, N3].  Coefficients are scattered into a
    zero box at (n mod N) and each axis is transformed with the full N x N DFT
    matrix (a separable naive DFT is still the naive DFT).  PAPER.md:52 eq. 3
    needs psi(r); normalisation per reading R8 (no 1/sqrt(Omega))."""
    n1, n2, n3 = (int(x) for x in fft)
    nb = psi.shape[0]
    box = np.zeros((nb, n1, n2, n3), dtype=np.complex128)
    i1 = np.mod(g_wfn[:, 0], n1)
    i2 = np.mod(g_wfn[:, 1], n2)
    i3 = np.mod(g_wfn[:, 2], n3)
    box[:, i1, i2, i3] = psi
    f1 = dft_matrix(n1, np.arange(n1), +1)   # [r1, k1] symmetric
    f2 = dft_matrix(n2, np.arange(n2), +1)
    f3 = dft_matrix(n3, np.arange(n3), +1)
    u = np.einsum("ra,nabc->nrbc", f1, box, optimize=True)
    u = f2 @ u                                                  # sum_b f2[s, b] u[n, r, b, c]
    u = u @ f3.T                                                # sum_c u[n, r, s, c] f3[t, c]
    return u


def mtxel(psi_v: np.ndarray, psi_c: np.ndarray, g_wfn: np.ndarray, g_eps: np.ndarray, fft) -> np.ndarray:
    """M[v, c, G] = (1/N_r) sum_r conj(u_v(r)) u_c(r) exp(-2 pi i G.r/N), G on the epsilon sphere.

    PAPER.md:52 eq. 3 with reading R7.  The forward sum is evaluated only at
    the epsilon-sphere Miller indices: per axis the DFT matrix has one row per
    distinct index on that axis, then the sphere points are picked out."""
    n1, n2, n3 = (int(x) for x in fft)
    n_r = n1 * n2 * n3
    u_v = wfn_to_realspace(psi_v, g_wfn, fft)
    u_c = wfn_to_realspace(psi_c, g_wfn, fft)
    k1 = np.unique(g_eps[:, 0])
    k2 = np.unique(g_eps[:, 1])
    k3 = np.unique(g_eps[:, 2])
    f1 = dft_matrix(n1, k1, -1)
    f2 = dft_matrix(n2, k2, -1)
    f3 = dft_matrix(n3, k3, -1)
    p1 = np.searchsorted(k1, g_eps[:, 0])
    p2 = np.searchsorted(k2, g_eps[:, 1])
    p3 = np.searchsorted(k3, g_eps[:, 2])
    nv, nc = psi_v.shape[0], psi_c.shape[0]
    out = np.empty((nv, nc, g_eps.shape[0]), dtype=np.complex128)
    for v in range(nv):
        for c0 in range(0, nc, 128):                            # chunked over c only to bound memory
            prod = np.conj(u_v[v])[None] * u_c[c0:c0 + 128]     # [<=128, N1, N2, N3]
            t = prod @ f3.T                                     # axis 3: sum_t prod[..., t] f3[k, t]
            t = f2 @ t                                          # axis 2: sum_s f2[j, s] t[n, r, s, k]
            t = np.einsum("ir,nrjk->nijk", f1, t, optimize=True)  # axis 1
            out[v, c0:c0 + 128] = t[:, p1, p2, p3] / n_r
    return out


def mtxel_convolution(psi_v, psi_c, g_wfn, g_eps) -> np.ndarray:
    """Pin P3 helper: M_vc(G) = sum_G' conj(c_v(G')) c_c(G'+G), exact when the grid is alias-free.

    Independent route (no transform at all): used by the pin tests only."""
    lut = {tuple(g): i for i, g in enumerate(g_wfn.tolist())}
    nv, nc = psi_v.shape[0], psi_c.shape[0]
    out = np.zeros((nv, nc, g_eps.shape[0]), dtype=np.complex128)
    for ig, g in enumerate(g_eps.tolist()):
        src, dst = [], []
        for i, gp in enumerate(g_wfn.tolist()):
            j = lut.get((gp[0] + g[0], gp[1] + g[1], gp[2] + g[2]))
            if j is not None:
                src.append(i)
                dst.append(j)
        out[:, :, ig] = np.conj(psi_v[:, src]) @ psi_c[:, dst].T
    return out


# --------------------------------------------------------------------------
# Step a2 -- CHI_SUM (eq. 6 with :71 eq. 5; north_star step 2)
# --------------------------------------------------------------------------
def pair_weights(e_v: np.ndarray, e_c: np.ndarray, omega: float, f_v=None, f_c=None) -> np.ndarray:
    """D_vc(i omega) = 2 Delta/(Delta^2 + omega^2), Delta = e_c - e_v (reading R6), shape [nv, nc].

    With occupations (eq. 4-5, reading R21): times max(f_v - f_c, 0), so that a partially occupied band,
    which sits in both band sets, meets every other band once and itself with weight 0; a pair with Delta = omega = 0
    has weight 0."""
    delta = e_c[None, :] - e_v[:, None]
    den = delta * delta + omega * omega
    d = np.where(den > 0.0, 2.0 * delta / np.where(den > 0.0, den, 1.0), 0.0)
    if f_v is not None:
        d = d * np.maximum(np.asarray(f_v)[:, None] - np.asarray(f_c)[None, :], 0.0)
    return d


def chi0(M: np.ndarray, e_v, e_c, vcoul, omega: float = 0.0, f_v=None, f_c=None) -> np.ndarray:
    """chi~0(i omega)[G,G'] = - sum_vc a_vc(G) D_vc(i omega) conj(a_vc(G')), a = v^1/2 M.

    PAPER.md:75 eq. 6 (sum over valence / conduction pairs), :71 eq. 5 with
    integer occupations (f_c - f_v = -1: the minus sign, reading R5), Coulomb
    symmetrised as in north_star step 2.  The pair sum is one matrix product."""
    nv, nc, ng = M.shape
    a = (M * np.sqrt(vcoul)[None, None, :]).reshape(nv * nc, ng)
    d = pair_weights(np.asarray(e_v), np.asarray(e_c), omega, f_v, f_c).reshape(nv * nc)
    return -(a.T * d[None, :]) @ np.conj(a)


def chi0_loops(M, e_v, e_c, vcoul, omega: float = 0.0) -> np.ndarray:
    """The same as `chi0`, as explicit triple loops (tiny inputs; pin P14)."""
    nv, nc, ng = M.shape
    out = np.zeros((ng, ng), dtype=np.complex128)
    for g in range(ng):
        for gp in range(ng):
            acc = 0.0 + 0.0j
            for v in range(nv):
                for c in range(nc):
                    delta = e_c[c] - e_v[v]
                    d = 2.0 * delta / (delta * delta + omega * omega)
                    acc += (np.sqrt(vcoul[g]) * M[v, c, g]) * d * np.conj(np.sqrt(vcoul[gp]) * M[v, c, gp])
            out[g, gp] = -acc
    return out


# --------------------------------------------------------------------------
# Step a3 -- static subspace basis (north_star step 3)
# --------------------------------------------------------------------------
def subspace_basis(chi0_static: np.ndarray, n_eig: int):
    """The n_eig eigenpairs of chi~0(0) with the greatest |lambda| (= most negative).

    PAPER.md:82.  Dense Hermitian eigensolver; ascending order puts the most
    negative first.  Returns (lam [n_eig], C [n_eig, N_G]) with row i = eigenvector i
    (the C-ABI's layout)."""
    h = 0.5 * (chi0_static + chi0_static.conj().T)
    lam, vec = np.linalg.eigh(h)
    return lam[:n_eig].copy(), np.ascontiguousarray(vec[:, :n_eig].T)


# --------------------------------------------------------------------------
# Step a4 -- projected chi_s(i omega) (PAPER.md:84 eq. 7, :88 eq. 8; north_star step 4)
# --------------------------------------------------------------------------
def chi_subspace_freq(M, e_v, e_c, vcoul, C: np.ndarray, omegas, f_v=None, f_c=None) -> np.ndarray:
    """chi_s(i w_k) = - sum_vc B_vc D_vc(i w_k) B_vc^H,  B_vc = C^H v^1/2 M_vc.

    PAPER.md:84 eq. 7 (M_s = M C_s) and :88 eq. 8 (chi_s = M_s^dagger Delta M_s).
    C is [n_eig, N_G] with eigenvectors as rows, so B[p, i] = sum_G conj(C[i, G]) a_p(G).
    Returns [n_w, n_eig, n_eig]."""
    nv, nc, ng = M.shape
    a = (M * np.sqrt(vcoul)[None, None, :]).reshape(nv * nc, ng)
    b = a @ np.conj(C).T                                          # [P, n_eig]
    out = np.empty((len(omegas), C.shape[0], C.shape[0]), dtype=np.complex128)
    for k, w in enumerate(omegas):
        d = pair_weights(np.asarray(e_v), np.asarray(e_c), float(w), f_v, f_c).reshape(nv * nc)
        out[k] = -(b.T * d[None, :]) @ np.conj(b)
    return out


# --------------------------------------------------------------------------
# Step a5 -- E_c (PAPER.md:35 eq. 1; :160; north_star step 5)
# --------------------------------------------------------------------------
def trace_log_term(chi: np.ndarray) -> float:
    """Tr[ln(1 - chi) + chi] = sum_i [log1p(-mu_i) + mu_i] over the eigenvalues mu of Hermitian chi.

    PAPER.md:35 eq. 1 integrand in the symmetrised form (chi v -> chi~), evaluated by
    the eigenvalue sum north_star prescribes for the oracle."""
    mu = np.linalg.eigvalsh(0.5 * (chi + chi.conj().T))
    return float(np.sum(np.log1p(-mu) + mu))


def correlation_energy(chis: np.ndarray, weight: np.ndarray):
    """E_c = (1/2 pi) sum_k W_k Tr[ln(1 - chi(i w_k)) + chi(i w_k)].  Returns (E_c, t_k[n_w])."""
    t = np.array([trace_log_term(c) for c in chis])
    return float(np.dot(weight, t) / TWO_PI), t


def cholesky_trace_log_term(chi: np.ndarray) -> float:
    """Pin P10 helper: the same integrand via L L^H = 1 - chi: 2 sum ln L_ii + Re Tr chi."""
    n = chi.shape[0]
    a = np.eye(n) - 0.5 * (chi + chi.conj().T)
    L = np.zeros_like(a)
    for j in range(n):                       # textbook Cholesky-Crout, column by column
        s = a[j, j].real - np.sum(np.abs(L[j, :j]) ** 2)
        L[j, j] = np.sqrt(s)
        for i in range(j + 1, n):
            L[i, j] = (a[i, j] - np.sum(L[i, :j] * np.conj(L[j, :j]))) / L[j, j]
    return float(2.0 * np.sum(np.log(np.diag(L).real)) + np.trace(chi).real)


def epsilon_inverse(chis: np.ndarray) -> np.ndarray:
    """eps_s^-1(i w_k) = (1 - chi_s(i w_k))^-1 for every frequency (the factorisation of eps "also gives
    eps^-1"), by the library's general inverse.  [n_w, n, n] -> [n_w, n, n]."""
    n = chis.shape[-1]
    return np.array([np.linalg.inv(np.eye(n) - 0.5 * (c + c.conj().T)) for c in chis])


# --------------------------------------------------------------------------
# Whole path (SURVEY 3.4 / PAPER.md:158 two-pass structure), for tests and timing
# --------------------------------------------------------------------------
def rpa_energy(inp, n_eig: int | None = None, nvb: int | None = None, full_basis: bool = False):
    """Run a1..a5 on an `RpaInputs`.  Valence blocks of `nvb` bands are accumulated
    (eq. 15); M is recomputed in the second pass.

    Returns a dict with E_c, t_k, lam, C, chi0 (static), chi_s and, if
    `full_basis`, E_c_full from chi~0(i w_k) in the whole G basis."""
    n_eig = inp.cfg.n_eig if n_eig is None else n_eig
    nv = inp.psi_v.shape[0]
    nvb = nv if not nvb else nvb
    blocks = [(s, min(nv, s + nvb)) for s in range(0, nv, nvb)]
    ng = inp.g_eps.shape[0]
    chi_static = np.zeros((ng, ng), dtype=np.complex128)
    chi_full = np.zeros((len(inp.omega), ng, ng), dtype=np.complex128) if full_basis else None
    for s, e in blocks:                                           # pass 1
        M = mtxel(inp.psi_v[s:e], inp.psi_c, inp.g_wfn, inp.g_eps, inp.fft)
        chi_static += chi0(M, inp.e_v[s:e], inp.e_c, inp.vcoul, 0.0)
        if full_basis:
            for k, w in enumerate(inp.omega):
                chi_full[k] += chi0(M, inp.e_v[s:e], inp.e_c, inp.vcoul, float(w))
    lam, C = subspace_basis(chi_static, n_eig)
    chi_s = np.zeros((len(inp.omega), n_eig, n_eig), dtype=np.complex128)
    for s, e in blocks:                                           # pass 2
        M = mtxel(inp.psi_v[s:e], inp.psi_c, inp.g_wfn, inp.g_eps, inp.fft)
        chi_s += chi_subspace_freq(M, inp.e_v[s:e], inp.e_c, inp.vcoul, C, inp.omega)
    e_c, t = correlation_energy(chi_s, inp.weight)
    out = dict(E_c=e_c, t=t, lam=lam, C=C, chi0=chi_static, chi_s=chi_s)
    if full_basis:
        out["E_c_full"], out["t_full"] = correlation_energy(chi_full, inp.weight)
    return out
