"""Pins for the CPU oracle: the oracle is checked against
closed forms, brute force, invariants and independent library routines --
never against itself and never against the CUDA path.  CPU only."""
import math

import numpy as np
import pytest

from oracle import rpa_oracle as orc
from rpa_inputs import make_inputs, quadrature, sphere, coulomb, RpaConfig

RNG = np.random.default_rng(1234)


def closed_form_pair(delta, b):
    """P1: single pair, E_c = 1/2 (sqrt(D^2+b) - D - b/(2D)), stable form.

    Derivation (north_star): chi(iw) has the single eigenvalue -s D(iw), b = 2 D s;
    int_0^inf ln((w^2+A^2)/(w^2+B^2)) dw = pi (A - B)."""
    root = math.sqrt(delta * delta + b)
    return -b * b / (4.0 * delta * (root + delta) ** 2)


def tiny_cfg(**kw):
    base = dict(name="pin", seed=11, cell=(7.0, 7.0, 9.0), fft=(12, 12, 15), ecut_wfn=1.6, ecut_eps=0.9,
                n_v=3, n_c=10, ev_range=(-0.6, 0.0), ec_range=(0.05, 3.0), n_eig=5, n_w=8)
    base.update(kw)
    return RpaConfig(**base)


# ------------------------------------------------------------------ P1 / P15
@pytest.mark.parametrize("delta,s", [(0.5, 0.1), (0.05, 0.1), (3.6, 0.1), (1.0, 5.0), (0.07, 0.01)])
def test_p1_single_pair_closed_form(delta, s):
    ng = 6
    m = RNG.standard_normal(ng) + 1j * RNG.standard_normal(ng)
    v = RNG.uniform(0.5, 2.0, ng)
    m *= math.sqrt(s / np.sum(v * np.abs(m) ** 2))           # s = sum_G v |M|^2
    M = m.reshape(1, 1, ng)
    e_v, e_c = np.array([-delta]), np.array([0.0])
    omega, weight = quadrature(200, 0.5)
    chis = np.array([orc.chi0(M, e_v, e_c, v, w) for w in omega])
    e, _ = orc.correlation_energy(chis, weight)
    ref = closed_form_pair(delta, 2.0 * delta * s)
    assert ref < 0
    assert abs(e - ref) <= 2e-11 * abs(ref)


def test_p15_scalar_case_by_hand():
    # N_G = 1, one pair: chi = -v |M|^2 2/Delta at w=0; t = ln(1-chi)+chi
    M = np.array([[[0.3 - 0.4j]]])
    chi = orc.chi0(M, np.array([-0.2]), np.array([0.3]), np.array([2.0]), 0.0)
    assert chi.shape == (1, 1)
    assert chi[0, 0] == pytest.approx(-2.0 * 0.25 * 2 / 0.5)
    w = 0.7
    chiw = orc.chi0(M, np.array([-0.2]), np.array([0.3]), np.array([2.0]), w)[0, 0]
    assert chiw.real == pytest.approx(-2.0 * 0.25 * 2 * 0.5 / (0.25 + 0.49))
    assert orc.trace_log_term(chi) == pytest.approx(math.log(1 + 2.0) - 2.0)
    e, t = orc.correlation_energy(np.array([chi, chi]), np.array([0.5, 1.5]))
    assert e == pytest.approx((math.log(3.0) - 2.0) * 2.0 / (2 * math.pi))


# ------------------------------------------------------------------ P2
def test_p2_diagonal_multi_pair_through_whole_chain():
    ng = 7
    e_v = np.array([-0.5, -0.1])
    e_c = np.array([0.2, 0.9, 1.7, 2.2])
    v = RNG.uniform(0.3, 3.0, ng)
    M = np.zeros((2, 4, ng), dtype=np.complex128)
    pairs = [(0, 0), (0, 1), (0, 2), (0, 3), (1, 0), (1, 1), (1, 2)]        # pair p -> unit vector e_p
    amp = RNG.uniform(0.2, 0.9, ng) * np.exp(1j * RNG.uniform(0, 6, ng))
    for g, (iv, ic) in enumerate(pairs):
        M[iv, ic, g] = amp[g]
    omega, weight = quadrature(160, 0.5)
    chi_static = orc.chi0(M, e_v, e_c, v)
    assert np.allclose(chi_static, np.diag(np.diag(chi_static)))
    lam, C = orc.subspace_basis(chi_static, ng)
    chi_s = orc.chi_subspace_freq(M, e_v, e_c, v, C, omega)
    e, _ = orc.correlation_energy(chi_s, weight)
    ref = 0.0
    for g, (iv, ic) in enumerate(pairs):
        d = e_c[ic] - e_v[iv]
        ref += closed_form_pair(d, 2.0 * d * v[g] * abs(amp[g]) ** 2)
    assert abs(e - ref) <= 1e-10 * abs(ref)
    # eigenvalues are the diagonal, most negative first
    assert np.allclose(lam, np.sort(np.diag(chi_static).real))


# ------------------------------------------------------------------ P3 / P4 / P5 / P14
def test_p5_dft_matrix_against_library_fft_and_textbook_cases():
    for n in (24, 40, 48, 120, 64, 160, 15):
        f = orc.dft_matrix(n, np.arange(n), -1)
        x = RNG.standard_normal(n) + 1j * RNG.standard_normal(n)
        assert np.allclose(f @ x, np.fft.fft(x), atol=1e-12)
        imp = np.zeros(n)
        imp[0] = 1
        assert np.allclose(f @ imp, 1.0)                       # impulse -> constant
        sh = np.roll(x, 3)                                       # shift theorem
        assert np.allclose(f @ sh, (f @ x) * np.exp(-2j * np.pi * 3 * np.arange(n) / n), atol=1e-12)
        fi = orc.dft_matrix(n, np.arange(n), +1)
        assert np.allclose(fi @ (f @ x) / n, x, atol=1e-13)
    # negative frequencies are reduced mod n
    assert np.allclose(orc.dft_matrix(12, [-3], -1), orc.dft_matrix(12, [9], -1))


def test_p5_wfn_to_realspace_against_library_ifft():
    inp = make_inputs(tiny_cfg())
    u = orc.wfn_to_realspace(inp.psi_c[:3], inp.g_wfn, inp.fft)
    n1, n2, n3 = inp.fft
    for b in range(3):
        box = np.zeros((n1, n2, n3), dtype=complex)
        for c, g in zip(inp.psi_c[b], inp.g_wfn):
            box[g[0] % n1, g[1] % n2, g[2] % n3] = c
        assert np.allclose(u[b], np.fft.ifftn(box) * (n1 * n2 * n3), atol=1e-12)
    # grid Parseval (R8 normalisation): (1/N_r) sum_r |u|^2 = sum_G |c|^2 = 1
    assert np.allclose(np.sum(np.abs(u) ** 2, axis=(1, 2, 3)) / (n1 * n2 * n3), 1.0)


def test_p3_fft_route_equals_gspace_convolution():
    inp = make_inputs(tiny_cfg())
    M = orc.mtxel(inp.psi_v, inp.psi_c, inp.g_wfn, inp.g_eps, inp.fft)
    Mc = orc.mtxel_convolution(inp.psi_v, inp.psi_c, inp.g_wfn, inp.g_eps)
    assert M.shape == (3, 10, inp.n_g)
    assert np.abs(M - Mc).max() < 1e-15
    # and on the real tiny config, a few pairs
    inp = make_inputs(0)
    M = orc.mtxel(inp.psi_v[:2], inp.psi_c[:3], inp.g_wfn, inp.g_eps, inp.fft)
    Mc = orc.mtxel_convolution(inp.psi_v[:2], inp.psi_c[:3], inp.g_wfn, inp.g_eps)
    assert np.abs(M - Mc).max() < 1e-15


def test_p4_orthogonality_and_bounds():
    inp = make_inputs(tiny_cfg())
    g0 = int(np.where((inp.g_eps == 0).all(axis=1))[0][0])
    M = orc.mtxel(inp.psi_v, inp.psi_c, inp.g_wfn, inp.g_eps, inp.fft)
    assert np.abs(M[:, :, g0]).max() < 1e-15                    # <v|c> = 0
    Mvv = orc.mtxel(inp.psi_v, inp.psi_v, inp.g_wfn, inp.g_eps, inp.fft)
    assert np.allclose(Mvv[:, :, g0], np.eye(3), atol=1e-14)    # <v|v'> = delta
    assert np.abs(M).max() <= 1.0 + 1e-14


def test_p14_brute_force_tiny_grid():
    cfg = tiny_cfg(cell=(5.0, 5.0, 6.0), fft=(6, 6, 8), ecut_wfn=0.9, ecut_eps=0.8, n_v=2, n_c=3)
    inp = make_inputs(cfg)
    n1, n2, n3 = (int(x) for x in inp.fft)
    psi = np.concatenate([inp.psi_v, inp.psi_c])

    def u_of(c):                                                # fully naive 3-D sums, python loops
        u = np.zeros((n1, n2, n3), dtype=complex)
        for r1 in range(n1):
            for r2 in range(n2):
                for r3 in range(n3):
                    acc = 0j
                    for coef, g in zip(c, inp.g_wfn):
                        ph = (int(g[0]) * r1 / n1 + int(g[1]) * r2 / n2 + int(g[2]) * r3 / n3)
                        acc += coef * np.exp(2j * np.pi * ph)
                    u[r1, r2, r3] = acc
        return u

    us = [u_of(c) for c in psi]
    r1, r2, r3 = np.meshgrid(np.arange(n1), np.arange(n2), np.arange(n3), indexing="ij")
    Mref = np.zeros((2, 3, inp.n_g), dtype=complex)
    for v in range(2):
        for c in range(3):
            p = np.conj(us[v]) * us[2 + c]
            for ig, g in enumerate(inp.g_eps):
                ph = g[0] * r1 / n1 + g[1] * r2 / n2 + g[2] * r3 / n3
                Mref[v, c, ig] = np.sum(p * np.exp(-2j * np.pi * ph)) / (n1 * n2 * n3)
    M = orc.mtxel(inp.psi_v, inp.psi_c, inp.g_wfn, inp.g_eps, inp.fft)
    assert np.abs(M - Mref).max() < 1e-14
    for w in (0.0, 0.8):
        assert np.abs(orc.chi0(M, inp.e_v, inp.e_c, inp.vcoul, w)
                      - orc.chi0_loops(Mref, inp.e_v, inp.e_c, inp.vcoul, w)).max() < 1e-12 * np.abs(inp.vcoul).max()


# ------------------------------------------------------------------ P6
def test_p6_chi_hermitian_negative_monotone_and_tail():
    inp = make_inputs(tiny_cfg())
    M = orc.mtxel(inp.psi_v, inp.psi_c, inp.g_wfn, inp.g_eps, inp.fft)
    prev = None
    for w in (0.0, 0.3, 1.0, 4.0):
        chi = orc.chi0(M, inp.e_v, inp.e_c, inp.vcoul, w)
        scale = np.abs(chi).max()
        assert np.abs(chi - chi.conj().T).max() <= 1e-14 * scale
        ev = np.linalg.eigvalsh(chi)
        assert ev.max() <= 1e-12 * scale
        if prev is not None:                                   # chi(iw) - chi(iw') >= 0 for w > w'
            assert np.linalg.eigvalsh(chi - prev).min() >= -1e-12 * scale
        prev = chi
    w = 1e4
    a = (M * np.sqrt(inp.vcoul)).reshape(-1, inp.n_g)
    delta = (inp.e_c[None, :] - inp.e_v[:, None]).reshape(-1)
    tail = -(a.T * (2 * delta)) @ a.conj()
    assert np.allclose(w * w * orc.chi0(M, inp.e_v, inp.e_c, inp.vcoul, w), tail, rtol=1e-6, atol=1e-9 * np.abs(tail).max())


# ------------------------------------------------------------------ P7 / P13 / P16
def test_p7_p13_basis_residuals_and_static_projection_is_diagonal():
    inp = make_inputs(tiny_cfg())
    M = orc.mtxel(inp.psi_v, inp.psi_c, inp.g_wfn, inp.g_eps, inp.fft)
    chi = orc.chi0(M, inp.e_v, inp.e_c, inp.vcoul)
    n_eig = 6
    lam, C = orc.subspace_basis(chi, n_eig)
    assert C.shape == (n_eig, inp.n_g)
    assert np.all(np.diff(lam) >= 0) and lam[0] < 0
    all_ev = np.linalg.eigvalsh(chi)
    assert np.allclose(lam, all_ev[:n_eig])                      # most negative = greatest |lambda| (chi <= 0)
    assert np.all(np.abs(lam) >= np.abs(all_ev[n_eig:]).max() - 1e-15)
    assert np.allclose(C.conj() @ C.T, np.eye(n_eig), atol=1e-13)
    res = chi @ C.T - C.T * lam[None, :]
    assert np.abs(res).max() <= 1e-13 * abs(lam[0])
    chi_s0 = orc.chi_subspace_freq(M, inp.e_v, inp.e_c, inp.vcoul, C, [0.0])[0]
    assert np.abs(chi_s0 - np.diag(lam)).max() <= 1e-13 * abs(lam[0])


# ------------------------------------------------------------------ P8 / P9 / P11 / P12
def test_p8_full_subspace_equals_full_basis_and_p9_interlacing():
    inp = make_inputs(tiny_cfg())
    ng = inp.n_g
    full = orc.rpa_energy(inp, n_eig=ng, full_basis=True)
    assert full["E_c_full"] < 0
    assert abs(full["E_c"] - full["E_c_full"]) <= 1e-11 * abs(full["E_c_full"])
    prev = 0.0
    for n in (1, 3, ng // 2, ng - 1, ng):                       # E_full <= E(N') <= E(N) <= 0 for N' >= N
        e = orc.rpa_energy(inp, n_eig=n)["E_c"]
        assert e <= prev + 1e-15
        assert e >= full["E_c_full"] - 1e-13
        prev = e


def test_p11_block_size_and_p12_phase_invariance():
    inp = make_inputs(tiny_cfg())
    ref = orc.rpa_energy(inp)["E_c"]
    for nvb in (1, 2):
        assert abs(orc.rpa_energy(inp, nvb=nvb)["E_c"] - ref) <= 1e-12 * abs(ref)
    ph_v = np.exp(1j * RNG.uniform(0, 6.28, inp.psi_v.shape[0]))[:, None]
    ph_c = np.exp(1j * RNG.uniform(0, 6.28, inp.psi_c.shape[0]))[:, None]
    import dataclasses
    inp2 = dataclasses.replace(inp, psi_v=inp.psi_v * ph_v, psi_c=inp.psi_c * ph_c)
    r2 = orc.rpa_energy(inp2)
    assert abs(r2["E_c"] - ref) <= 1e-12 * abs(ref)
    chi_ref = orc.rpa_energy(inp)["chi0"]
    assert np.abs(r2["chi0"] - chi_ref).max() <= 1e-13 * np.abs(chi_ref).max()


# ------------------------------------------------------------------ P10
def test_p10_cholesky_logdet_equals_eigenvalue_sum():
    for n in (1, 2, 5, 17):
        a = RNG.standard_normal((n, 3 * n)) + 1j * RNG.standard_normal((n, 3 * n))
        chi = -(a @ a.conj().T) * 0.3
        assert orc.cholesky_trace_log_term(chi) == pytest.approx(orc.trace_log_term(chi), rel=1e-12, abs=1e-13)


# ------------------------------------------------------------------ inputs / golden
def test_input_recipe_sizes_match_survey_table():
    sizes = {0: (739, 147), 1: (4139, 691), 2: (20359, 3877), 3: (49993, 7665)}
    from rpa_inputs import CONFIGS
    for i, (npw, ng) in sizes.items():
        c = CONFIGS[i]
        cell = np.diag(c.cell)
        assert len(sphere(cell, c.ecut_wfn)) == npw
        assert len(sphere(cell, c.ecut_eps)) == ng
    inp = make_inputs(0)
    allb = np.concatenate([inp.psi_v, inp.psi_c])
    assert np.allclose(allb.conj() @ allb.T, np.eye(208), atol=1e-12)
    assert np.all(np.diff(inp.e_v) >= 0) and inp.e_c.min() - inp.e_v.max() >= 0.05
    assert np.allclose(inp.vcoul, coulomb(inp.cell, inp.g_eps, inp.cfg.q))
    # the mapped rule integrates 1/(1+w^2) over (0, inf) to pi/2
    om, wt = quadrature(64, 0.5)
    assert np.dot(wt, 1.0 / (1.0 + om * om)) == pytest.approx(math.pi / 2, rel=1e-12)


def test_tiny_config_subspace_error_is_the_methods_own_approximation():
    """The tiny config end to end; stores nothing, checks the sanity bounds of SURVEY's appendix:
    subspace E_c is above the full-basis E_c by a few percent (method's approximation, P9)."""
    inp = make_inputs(0)
    r = orc.rpa_energy(inp, full_basis=True)
    assert r["E_c_full"] < r["E_c"] < 0
    rel = (r["E_c"] - r["E_c_full"]) / abs(r["E_c_full"])
    assert 0.03 < rel < 0.10


# ------------------------------------------------------------------ partial occupations (NEXT-4, reading R21)
def test_partial_occupations_closed_form_reduction_and_single_counting():
    """Pins for the occupation-weighted pair weight (eq. 4-5): (a) the single-pair closed form with
    b = 2 Delta (f_v - f_c) |v^1/2 M|^2; (b) f_v = 1, f_c = 0 is the integer-occupation result; (c) a partially occupied
    band listed in both band sets meets itself with weight 0 and every other band once (by hand on a 3-band case)."""
    ng = 5
    m = RNG.standard_normal(ng) + 1j * RNG.standard_normal(ng)
    v = RNG.uniform(0.5, 2.0, ng)
    s = float(np.sum(v * np.abs(m) ** 2))
    delta, fv, fc = 0.4, 0.85, 0.25
    omega, weight = quadrature(200, 0.5)
    M = m.reshape(1, 1, ng)
    chis = np.array([orc.chi0(M, np.array([-delta]), np.array([0.0]), v, w, np.array([fv]), np.array([fc])) for w in omega])
    e, _ = orc.correlation_energy(chis, weight)
    ref = closed_form_pair(delta, 2.0 * delta * (fv - fc) * s)
    assert abs(e - ref) <= 2e-11 * abs(ref)
    # (b)
    Mr = RNG.standard_normal((2, 3, ng)) + 1j * RNG.standard_normal((2, 3, ng))
    e_v, e_c = np.array([-0.5, -0.2]), np.array([0.1, 0.6, 1.5])
    a = orc.chi0(Mr, e_v, e_c, v, 0.3)
    b = orc.chi0(Mr, e_v, e_c, v, 0.3, np.ones(2), np.zeros(3))
    assert np.array_equal(a, b)
    # (c) bands: 0 occupied (f = 1), 1 partial (f = 0.4), 2 empty (f = 0); valence set {0, 1}, conduction set {1, 2}
    e = np.array([-0.5, 0.0, 0.7])
    f = np.array([1.0, 0.4, 0.0])
    d = orc.pair_weights(e[[0, 1]], e[[1, 2]], 0.2, f[[0, 1]], f[[1, 2]])
    by_hand = np.array([[0.6 * 2 * 0.5 / (0.25 + 0.04), 1.0 * 2 * 1.2 / (1.44 + 0.04)],
                        [0.0, 0.4 * 2 * 0.7 / (0.49 + 0.04)]])
    assert np.allclose(d, by_hand, rtol=1e-15, atol=0)
    assert orc.pair_weights(e[[1]], e[[1]], 0.0, f[[1]], f[[1]])[0, 0] == 0.0      # Delta = omega = 0


def test_epsilon_inverse_pins():
    """eps^-1 (NEXT-3): defining identity (1 - chi) eps^-1 = 1, the diagonal case 1/(1 - mu), and Hermiticity."""
    n = 9
    a = RNG.standard_normal((n, 4)) + 1j * RNG.standard_normal((n, 4))
    chi = -(a @ a.conj().T)                                   # Hermitian negative-semidefinite like chi_s
    mu = -RNG.uniform(0.0, 2.0, n)
    chis = np.array([chi, np.diag(mu).astype(complex)])
    inv = orc.epsilon_inverse(chis)
    assert np.abs((np.eye(n) - chi) @ inv[0] - np.eye(n)).max() <= 1e-13
    assert np.abs(inv[0] - inv[0].conj().T).max() <= 1e-14
    assert np.allclose(np.diag(inv[1]).real, 1.0 / (1.0 - mu), rtol=1e-15)
    assert np.abs(inv[1] - np.diag(np.diag(inv[1]))).max() == 0.0
