"""Pins for the oracle's H apply, Chebyshev filter, Hartree solve and split-operator step (CPU only).

The pins are the ones SURVEY.md section 8(c) lists: closed forms (plane waves, constant V, erf
potential of a Gaussian charge), invariants (Hermiticity, unitarity, reversibility, order 2) and
brute force (a dense H built here with numpy, independent of the oracle, diagonalised with eigh).
"""
import math

import numpy as np
import pytest
from scipy.linalg import expm
from scipy.special import erf

from paper_2601_21005_b200 import workloads as W


def kgrid(g):
    def k1(n, h):
        return 2 * np.pi * np.fft.fftfreq(n, d=h)       # library's ordering: m in [-n/2, n/2)
    kz, ky, kx = np.meshgrid(k1(g.nz, g.hz), k1(g.ny, g.hy), k1(g.nx, g.hx), indexing="ij")
    return kx, ky, kz


def dense_H(g, vloc, kb, ecut=0.0):
    """H as a dense matrix, built with numpy.fft and outer products (independent of the oracle)."""
    ng = g.ng
    kx, ky, kz = kgrid(g)
    k2 = 0.5 * (kx ** 2 + ky ** 2 + kz ** 2)
    if ecut > 0:
        k2 = np.minimum(k2, ecut)
    eye = np.eye(ng, dtype=np.complex128).reshape((ng,) + g.shape)
    T = np.fft.ifftn(k2[None] * np.fft.fftn(eye, axes=(1, 2, 3)), axes=(1, 2, 3)).reshape(ng, ng).T
    H = T + np.diag(vloc.ravel())
    if kb is not None:
        for s in range(kb.nsphere):
            sl = slice(kb.sph_ptr[s], kb.sph_ptr[s + 1])
            idx = kb.sph_idx[sl]
            for p in range(kb.nproj):
                b = np.zeros(ng)
                b[idx] = kb.beta[sl, p]
                H += g.dV * kb.D[s, p] * np.outer(b, b)
    return H


def small_problem(n=8, h=0.7, with_kb=True, seed=3):
    g = W.Grid(n, n, n, h, h, h)
    rng = np.random.default_rng(seed)
    centers = rng.uniform(0, n * h, size=(3, 3))
    vloc = W.gaussian_vloc(g, centers, [1.0, 2.0, 1.5], [0.9, 1.2, 0.8])
    kb = W.kb_projectors(g, centers[:2], radius=1.8, sigma=0.7) if with_kb else None
    return g, vloc, kb, rng


def rvec(rng, g, nvec=1):
    return rng.standard_normal((nvec,) + g.shape) + 1j * rng.standard_normal((nvec,) + g.shape)


# ------------------------------------------------------------------ kinetic / local V pins
@pytest.mark.parametrize("ld", [False, True])
def test_plane_waves_are_kinetic_eigenvectors_including_nyquist(oracle, ld):
    g = W.Grid(8, 6, 12, 0.5, 0.6, 0.45)
    z, y, x = np.meshgrid(np.arange(g.nz), np.arange(g.ny), np.arange(g.nx), indexing="ij")
    zero = np.zeros(g.shape)
    for mx, my, mz in [(0, 0, 0), (1, 0, 0), (0, -2, 0), (0, 0, 5), (-4, 3, -6), (3, -3, 2), (-4, -3, -6)]:
        pw = np.exp(2j * np.pi * (mx * x / g.nx + my * y / g.ny + mz * z / g.nz))[None]
        k2 = (2 * np.pi * mx / (g.nx * g.hx)) ** 2 + (2 * np.pi * my / (g.ny * g.hy)) ** 2 + \
             (2 * np.pi * mz / (g.nz * g.hz)) ** 2
        out = oracle.apply_H(g, zero, None, pw, ld)
        assert np.abs(out - 0.5 * k2 * pw).max() < 1e-12 * max(1.0, k2)
        out = oracle.apply_H(g, zero + 0.37, None, pw, ld)           # V = const c: eigenvalue k^2/2 + c
        assert np.abs(out - (0.5 * k2 + 0.37) * pw).max() < 1e-12 * max(1.0, k2)


def test_dense_matrix_and_hermiticity(oracle):
    g, vloc, kb, rng = small_problem(8)
    H = dense_H(g, vloc, kb)
    assert np.abs(H - H.conj().T).max() < 1e-12
    v = rvec(rng, g, 3)
    out = oracle.apply_H(g, vloc, kb, v)
    want = (H @ v.reshape(3, -1).T).T.reshape(v.shape)
    assert np.abs(out - want).max() < 1e-11
    out_ld = oracle.apply_H(g, vloc, kb, v, ld=True)
    assert np.linalg.norm(out_ld - out) / np.linalg.norm(out) < 1e-14
    # Hermiticity of the oracle's own operator on a non-cubic grid: <u|Hv> = conj <v|Hu>
    g2 = W.Grid(12, 10, 6, 0.5, 0.55, 0.7)
    c2 = np.array([[2.0, 2.2, 2.1], [3.4, 3.0, 1.0]])
    v2 = W.gaussian_vloc(g2, c2, [1.0, 2.0], [0.8, 1.0])
    kb2 = W.kb_projectors(g2, c2, radius=1.9, sigma=0.7)
    u, w = rvec(rng, g2), rvec(rng, g2)
    a = np.vdot(u, oracle.apply_H(g2, v2, kb2, w))
    b = np.vdot(w, oracle.apply_H(g2, v2, kb2, u))
    assert abs(a - np.conj(b)) < 1e-11 * abs(a)


def test_kb_single_projector_is_eigenvector_of_vnl(oracle):
    g = W.Grid(12, 12, 12, 0.5, 0.5, 0.5)
    kb = W.kb_projectors(g, np.array([[3.0, 3.0, 3.0]]), radius=2.0, sigma=0.7)   # on a grid point
    zero = np.zeros(g.shape)
    for p in range(4):
        b = np.zeros(g.ng, dtype=np.complex128)
        b[kb.sph_idx] = kb.beta[:, p]
        b = b.reshape((1,) + g.shape)
        vnl = oracle.apply_H(g, zero, kb, b) - oracle.apply_H(g, zero, None, b)
        assert np.abs(vnl - kb.D[0, p] * b).max() < 1e-13


# ------------------------------------------------------------------ Chebyshev pins
def test_cheb_polynomial_vs_dense_diagonalisation(oracle):
    g, vloc, kb, rng = small_problem(8)
    H = dense_H(g, vloc, kb)
    ev, U = np.linalg.eigh(H)
    emin, emax = W.spectral_bounds(g, vloc, True)
    assert emin < ev[0] and ev[-1] < emax                           # spectrum inside analytic bounds
    eb, de = 0.5 * (emax + emin), 0.5 * (emax - emin)
    nterms = 40
    coeffs = rng.standard_normal(nterms)                            # ANY coefficients
    v = rvec(rng, g, 2)
    got = oracle.cheb_filter(g, vloc, kb, v, coeffs, emin, emax)
    x = (ev - eb) / de
    p = sum(coeffs[n] * np.cos(n * np.arccos(x)) for n in range(nterms))
    want = ((U * p[None, :]) @ (U.conj().T @ v.reshape(2, -1).T)).T.reshape(v.shape)
    assert np.linalg.norm(got - want) / np.linalg.norm(want) < 1e-12
    got_ld = oracle.cheb_filter(g, vloc, kb, v, coeffs, emin, emax, ld=True)
    assert np.linalg.norm(got_ld - want) / np.linalg.norm(want) < 1e-12


def test_cheb_unit_coefficient_gives_Tn_closed_form(oracle):
    g = W.Grid(8, 8, 8, 0.6, 0.6, 0.6)
    z, y, x = np.meshgrid(np.arange(8), np.arange(8), np.arange(8), indexing="ij")
    pw = np.exp(2j * np.pi * (2 * x - 3 * y + z) / 8)[None]
    eps = 0.5 * (2 * np.pi / (8 * 0.6)) ** 2 * (4 + 9 + 1) + 0.25
    vloc = np.full(g.shape, 0.25)
    emin, emax = -1.0, 45.0
    xt = (eps - 0.5 * (emax + emin)) / (0.5 * (emax - emin))
    for n in (0, 1, 2, 7, 30):
        c = np.zeros(n + 1)
        c[n] = 1.0
        got = oracle.cheb_filter(g, vloc, None, pw, c, emin, emax)
        assert np.abs(got - math.cos(n * math.acos(xt)) * pw).max() < 1e-11


def test_cheb_converged_filter_equals_f_of_H(oracle):
    g, vloc, kb, rng = small_problem(8, h=1.0)
    H = dense_H(g, vloc, kb)
    ev, U = np.linalg.eigh(H)
    emin, emax = W.spectral_bounds(g, vloc, True)

    def f(e):
        return W.sqrt_fermi(e, mu=-0.2, beta=4.0)
    coeffs = W.cheb_coeffs(f, emin, emax, 300)
    assert abs(coeffs[-1]) < 1e-13
    v = rvec(rng, g, 1)
    got = oracle.cheb_filter(g, vloc, kb, v, coeffs, emin, emax)
    want = ((U * f(ev)[None, :]) @ (U.conj().T @ v.reshape(1, -1).T)).T.reshape(v.shape)
    assert np.linalg.norm(got - want) / np.linalg.norm(want) < 1e-11


# ------------------------------------------------------------------ Hartree pins
def test_hartree_gaussian_charge_matches_erf_closed_form(oracle):
    n, h, sigma, Q = 48, 0.5, 1.0, 1.7
    g = W.Grid(n, n, n, h, h, h)
    c = np.array([12.13, 11.9, 12.31])                              # off-grid centre
    ax = np.arange(n) * h
    z, y, x = np.meshgrid(ax, ax, ax, indexing="ij")
    d = np.sqrt((x - c[0]) ** 2 + (y - c[1]) ** 2 + (z - c[2]) ** 2)
    rho = Q * (2 * np.pi * sigma ** 2) ** -1.5 * np.exp(-d ** 2 / (2 * sigma ** 2))
    vh = oracle.poisson(g, rho)
    with np.errstate(divide="ignore", invalid="ignore"):
        want = np.where(d > 0, Q * erf(d / (math.sqrt(2) * sigma)) / d, Q * math.sqrt(2 / np.pi) / sigma)
    Rc = n * h / 2
    m = d < Rc - 6 * sigma
    assert m.sum() > 5000
    assert (np.abs(vh - want)[m] / np.abs(want[m])).max() < 1e-9
    m7 = d < Rc - 7 * sigma
    assert (np.abs(vh - want)[m7] / np.abs(want[m7])).max() < 1e-11


def test_hartree_density_and_linearity(oracle):
    g = W.Grid(10, 8, 6, 0.5, 0.6, 0.7)
    rng = np.random.default_rng(5)
    psi = rvec(rng, g, 3)
    vh, rho = oracle.hartree(g, psi, 0.37)
    assert np.abs(rho - 0.37 * np.sum(np.abs(psi) ** 2, axis=0)).max() < 1e-13
    vh2, _ = oracle.hartree(g, psi, 0.74)
    assert np.abs(vh2 - 2 * vh).max() < 1e-12 * np.abs(vh).max()
    # against numpy.fft with the same kernel, written out independently
    kx, ky, kz = kgrid(g)
    k = np.sqrt(kx ** 2 + ky ** 2 + kz ** 2)
    Rc = min(g.box) / 2
    with np.errstate(divide="ignore", invalid="ignore"):
        vk = np.where(k > 0, 4 * np.pi * (1 - np.cos(k * Rc)) / k ** 2, 2 * np.pi * Rc ** 2)
    want = np.fft.ifftn(vk * np.fft.fftn(rho)).real
    assert np.abs(vh - want).max() < 1e-12 * np.abs(want).max()


# ------------------------------------------------------------------ TD pins
def test_td_local_only_is_unitary_and_const_V_is_a_phase(oracle):
    g, vloc, _, rng = small_problem(8, with_kb=False)
    psi = rvec(rng, g, 2)
    out = oracle.td_propagate(g, vloc, None, psi, 0.05, 20)
    assert np.abs(oracle.norms(out) / oracle.norms(psi) - 1).max() < 1e-13
    # V = const, single plane wave: exact phase e^{-i (k^2/2 + c) t}
    z, y, x = np.meshgrid(np.arange(8), np.arange(8), np.arange(8), indexing="ij")
    pw = np.exp(2j * np.pi * (x - 2 * y + 3 * z) / 8)[None]
    eps = 0.5 * (2 * np.pi / (8 * g.hx)) ** 2 * 14
    for c in (0.0, 0.4):
        out = oracle.td_propagate(g, np.full(g.shape, c), None, pw, 0.05, 7)
        assert np.abs(out - np.exp(-1j * (eps + c) * 0.35) * pw).max() < 1e-12


def test_td_frozen_V_is_second_order_and_reversible(oracle):
    g = W.Grid(6, 6, 6, 0.8, 0.8, 0.8)
    rng = np.random.default_rng(11)
    centers = rng.uniform(0, 4.8, size=(2, 3))
    vloc = W.gaussian_vloc(g, centers, [1.0, 2.0], [0.9, 1.1])
    H = dense_H(g, vloc, None)
    psi = rvec(rng, g, 1)
    t = 0.4
    exact = (expm(-1j * H * t) @ psi.reshape(-1)).reshape(psi.shape)
    errs = []
    for nst in (4, 8, 16):
        out = oracle.td_propagate(g, vloc, None, psi, t / nst, nst)
        errs.append(np.linalg.norm(out - exact))
    assert 3.5 < errs[0] / errs[1] < 4.5 and 3.5 < errs[1] / errs[2] < 4.5
    fwd = oracle.td_propagate(g, vloc, None, psi, 0.05, 5)
    back = oracle.td_propagate(g, vloc, None, fwd, -0.05, 5)
    assert np.linalg.norm(back - psi) / np.linalg.norm(psi) < 1e-13


def test_td_kb_orthonormal_projectors_exact_and_unitary(oracle):
    """With ONE sphere centred on a grid point the 4 projectors are orthonormal, so NL(tau) is
    exactly exp(-i V_NL tau); with T = V = 0 removed we check the factor through a full step against
    the dense split-operator product."""
    g = W.Grid(8, 8, 8, 0.6, 0.6, 0.6)
    rng = np.random.default_rng(2)
    kb = W.kb_projectors(g, np.array([[2.4, 2.4, 2.4]]), radius=1.7, sigma=0.6)
    vloc = W.gaussian_vloc(g, np.array([[2.0, 2.5, 2.2]]), [1.5], [1.0])
    psi = rvec(rng, g, 1)
    dt = 0.05
    out = oracle.td_propagate(g, vloc, kb, psi, dt, 1)
    zero = np.zeros(g.shape)
    T = dense_H(g, zero, None)
    VNL = dense_H(g, zero, kb) - T
    Uv = np.exp(-0.5j * dt * vloc.ravel())
    Unl = expm(-0.5j * dt * VNL)
    x = Uv * psi.reshape(-1)
    x = Unl @ x
    x = expm(-1j * dt * T) @ x
    x = Unl @ x
    x = Uv * x
    assert np.linalg.norm(out.reshape(-1) - x) / np.linalg.norm(x) < 1e-12
    out = oracle.td_propagate(g, vloc, kb, psi, dt, 10)
    assert abs(oracle.norms(out)[0] / oracle.norms(psi)[0] - 1) < 1e-12


def test_td_hartree_mode_uses_start_of_step_density(oracle):
    """One step with hartree_mode=1 equals one frozen-V step with V = V_loc + V_H[rho(psi_0)]."""
    g, vloc, _, rng = small_problem(8, with_kb=False)
    psi = rvec(rng, g, 3)
    rs = 2.0 / (3 * g.dV) * 0.01
    vh, _ = oracle.hartree(g, psi, rs)
    a = oracle.td_propagate(g, vloc, None, psi, 0.05, 1, hartree_mode=1, rho_scale=rs)
    b = oracle.td_propagate(g, vloc + vh, None, psi, 0.05, 1)
    assert np.linalg.norm(a - b) / np.linalg.norm(b) < 1e-14
    # and it stays unitary over several steps (V real at every step)
    c = oracle.td_propagate(g, vloc, None, psi, 0.05, 6, hartree_mode=1, rho_scale=rs)
    assert np.abs(oracle.norms(c) / oracle.norms(psi) - 1).max() < 1e-13


def test_td_hartree_trajectory_conserves_energy_to_first_order_in_dt(oracle):
    """Pin for the multi-step TD-Hartree trajectory (R-8): the exact flow of
    i d/dt psi_v = (T + V_loc + V_H[rho(t)]) psi_v, rho = rho_scale sum_v |psi_v|^2, conserves
    E = rho_scale sum_v <psi_v|T + V_loc|psi_v> dV + 1/2 int rho V_H.  The split-operator step with the start-of-step
    density is first-order consistent with that flow, so the drift over a fixed time halves with dt; a potential that
    is not rebuilt every step, or enters with the wrong sign or scale, leaves a drift that does not shrink.  The
    energy is evaluated here with numpy.fft for T and the (erf-pinned) oracle Hartree potential."""
    n, h = 12, 0.7
    g = W.Grid(n, n, n, h, h, h)
    L = n * h
    rng = np.random.default_rng(4)
    vloc = W.gaussian_vloc(g, rng.uniform(0, L, size=(2, 3)), [1.0, 1.5], [1.0, 1.2])
    z, y, x = np.meshgrid(*(np.arange(n) * h,) * 3, indexing="ij")

    def packet(c, s, k):
        d2 = sum(np.minimum(np.abs(a - ci), L - np.abs(a - ci)) ** 2 for a, ci in zip((x, y, z), c))
        return np.exp(-d2 / (2 * s * s)) * np.exp(1j * (k[0] * x + k[1] * y + k[2] * z))

    kk = 2 * np.pi / L
    psi = np.stack([packet((3.0, 4.0, 4.5), 1.3, (kk, 0, 0)), packet((5.0, 3.5, 4.0), 1.5, (0, -kk, kk))])
    psi /= np.sqrt((np.abs(psi) ** 2).sum(axis=(1, 2, 3), keepdims=True) * g.dV)
    rs = 4.0                                                     # 4 electrons per orbital: max V_H ~ 5 Ha
    kx = 2 * np.pi * np.fft.fftfreq(n, h)
    k2 = kx[:, None, None] ** 2 + kx[None, :, None] ** 2 + kx[None, None, :] ** 2

    def energy(p):
        e = 0.0
        for v in p:
            e += rs * (0.5 * (k2 * np.abs(np.fft.fftn(v)) ** 2).sum() / v.size + (vloc * np.abs(v) ** 2).sum()) * g.dV
        vh, rho = oracle.hartree(g, p, rs)
        return e + 0.5 * (rho * vh).sum() * g.dV

    e0 = energy(psi)
    drift = []
    for dt in (0.1, 0.05, 0.025):
        out = oracle.td_propagate(g, vloc, None, psi, dt, int(round(1.0 / dt)), hartree_mode=1, rho_scale=rs)
        drift.append(abs(energy(out) - e0))
    assert 1.8 < drift[0] / drift[1] < 2.2 and 1.8 < drift[1] / drift[2] < 2.2
    assert drift[2] < 0.004 * abs(e0)
    vh0, _ = oracle.hartree(g, psi, rs)
    frozen = oracle.td_propagate(g, vloc + vh0, None, psi, 0.025, 40)     # same start, V_H never rebuilt
    assert abs(energy(frozen) - e0) > 20 * drift[2]


def test_td_overlapping_kb_spheres_converge_to_the_dense_propagator(oracle):
    """Pin for the KB factor NL(tau) with overlapping, off-grid (non-orthonormal) projectors (R-11): NL(tau) agrees with
    exp(-i V_NL tau) to first order in tau, so the split-operator product converges to the dense exp(-i H t) at
    least linearly; a wrong sign, a missing dV or a wrong D would leave an error that does not shrink."""
    g = W.Grid(6, 6, 6, 0.8, 0.8, 0.8)
    rng = np.random.default_rng(5)
    centers = np.array([[1.9, 2.3, 2.1], [2.9, 2.6, 2.4]])      # 1.1 bohr apart, radius 1.7: 23 shared points
    kb = W.kb_projectors(g, centers, radius=1.7, sigma=0.6)
    a, b = (set(kb.sph_idx[kb.sph_ptr[i]:kb.sph_ptr[i + 1]].tolist()) for i in (0, 1))
    assert len(a & b) > 10
    vloc = W.gaussian_vloc(g, centers, [1.0, 2.0], [0.9, 1.1])
    H = dense_H(g, vloc, kb)
    psi = rvec(rng, g, 1)
    t = 0.4
    exact = (expm(-1j * H * t) @ psi.reshape(-1)).reshape(psi.shape)
    errs = []
    for nst in (8, 16, 32, 64):
        out = oracle.td_propagate(g, vloc, kb, psi, t / nst, nst)
        errs.append(np.linalg.norm(out - exact) / np.linalg.norm(exact))
    assert all(errs[i] / errs[i + 1] > 2.0 for i in range(3))
    assert errs[-1] < 5e-5


# ------------------------------------------------------------------ spectral bounds (NEXT-1)
def test_power_iteration_bounds_converge_to_dense_extreme_eigenvalues(oracle):
    """Shifted power iteration (R-20) against numpy's eigvalsh of the independently built dense H:
    Rayleigh quotients always lie inside the spectrum, tighten with the iteration count, and reach both ends
    to ~1e-12 of the spectral range after 1600 iterations."""
    for n, h, with_kb in [(8, 0.7, True), (10, 0.6, False)]:
        g, vloc, kb, _ = small_problem(n, h, with_kb)
        H = dense_H(g, vloc, kb)
        ev = np.linalg.eigvalsh(0.5 * (H + H.conj().T))
        rng_ = ev[-1] - ev[0]
        prev = None
        for niter in (20, 100, 400, 1600):
            emin, emax = oracle.spectral_bounds(g, vloc, kb, niter, 1234)
            assert ev[0] - 1e-10 * rng_ <= emin <= emax <= ev[-1] + 1e-10 * rng_
            if prev is not None:
                assert emin <= prev[0] + 1e-12 * rng_ and emax >= prev[1] - 1e-12 * rng_
            prev = (emin, emax)
        assert abs(prev[0] - ev[0]) < 1e-11 * rng_ and abs(prev[1] - ev[-1]) < 1e-11 * rng_
        # the analytic bounds the configs use (R-3) enclose the true spectrum
        lo, hi = W.spectral_bounds(g, vloc, with_kb)
        assert lo <= ev[0] and ev[-1] <= hi
    # V = 0: the top of the spectrum is the Nyquist corner, 1/2 sum (pi/h_i)^2, and the bottom is 0
    g = W.Grid(8, 8, 8, 0.5, 0.6, 0.7)
    emin, emax = oracle.spectral_bounds(g, np.zeros(g.shape), None, 300, 7)
    top = 0.5 * sum((math.pi / hh) ** 2 for hh in (0.5, 0.6, 0.7))
    assert abs(emax - top) < 1e-12 * top and -1e-12 * top <= emin < 1e-4 * top
    # the long double instantiation agrees
    g, vloc, kb, _ = small_problem(8, 0.7, True)
    a = oracle.spectral_bounds(g, vloc, kb, 50, 99)
    b = oracle.spectral_bounds(g, vloc, kb, 50, 99, ld=True)
    assert np.allclose(a, b, rtol=1e-12, atol=1e-12)


# ------------------------------------------------------------------ NEXT-3: kinetic-energy cutoff
def test_kinetic_cutoff_plane_waves_dense_matrix_spectrum_and_propagator(oracle):
    """With the cutoff the kinetic operator is min(1/2 k^2, E_cut), diagonal in k ("an energy cutoff ... to the
    kinetic energy operator"): closed-form eigenvalues for plane waves below and above the cutoff, a dense matrix built
    here with numpy, the spectrum bounded by E_cut + max V (the point of the cutoff), and the V = 0 propagator
    exp(-i min(1/2 k^2, E_cut) t) in closed form."""
    ecut = 6.0
    g = W.Grid(8, 6, 12, 0.5, 0.6, 0.45)
    z, y, x = np.meshgrid(np.arange(g.nz), np.arange(g.ny), np.arange(g.nx), indexing="ij")
    try:
        oracle.set_kinetic_cutoff(ecut)
        seen_above = seen_below = False
        for (mx, my, mz) in [(0, 0, 0), (1, 0, 0), (1, -2, 3), (-4, 3, -6), (3, 2, 5), (0, -3, 0)]:
            k = 2 * np.pi * np.array([mx / (g.nx * g.hx), my / (g.ny * g.hy), mz / (g.nz * g.hz)])
            e = min(0.5 * float(k @ k), ecut)
            seen_above |= 0.5 * float(k @ k) > ecut
            seen_below |= 0.5 * float(k @ k) < ecut
            pw = np.exp(2j * np.pi * (mx * x / g.nx + my * y / g.ny + mz * z / g.nz))[None]
            for ld in (False, True):
                out = oracle.apply_H(g, np.full(g.shape, 0.3), None, pw, ld=ld)
                assert np.max(np.abs(out - (e + 0.3) * pw)) < 1e-11
            t = 0.7
            prop = oracle.td_propagate(g, None, None, pw, t / 7, 7, 0, 0.0, ld=True)
            assert np.max(np.abs(prop - np.exp(-1j * e * t) * pw)) < 1e-11
        assert seen_above and seen_below
        g2, vloc, kb, rng = small_problem(8, 0.7, True)
        H = dense_H(g2, vloc, kb, ecut=ecut)
        psi = rvec(rng, g2, 2)
        want = (H @ psi.reshape(2, -1).T).T.reshape(psi.shape)
        assert np.max(np.abs(oracle.apply_H(g2, vloc, kb, psi, ld=True) - want)) < 1e-11
        ev = np.linalg.eigvalsh(H)
        assert ev[-1] <= ecut + vloc.max() + np.abs(kb.D).max() * 1.01 + 1e-9
        assert np.linalg.eigvalsh(dense_H(g2, vloc, kb))[-1] > ev[-1] + 5.0      # the cutoff did shrink the spectrum
        # a filter on the narrower window: polynomial of the cut-off H by dense diagonalisation
        emin, emax = ev[0] - 0.5, ev[-1] + 0.5
        co = rng.standard_normal(12)
        w_, U = np.linalg.eigh(H)
        xs = (w_ - 0.5 * (emax + emin)) / (0.5 * (emax - emin))
        pol = np.polynomial.chebyshev.chebval(xs, co)
        want = ((U * pol) @ (U.conj().T @ psi.reshape(2, -1).T)).T.reshape(psi.shape)
        got = oracle.cheb_filter(g2, vloc, kb, psi, co, emin, emax, ld=True)
        assert np.max(np.abs(got - want)) < 1e-10
    finally:
        oracle.set_kinetic_cutoff(0.0)
    # and off again: the plain operator
    pw = np.exp(2j * np.pi * (3 * x / g.nx))[None]
    k = 2 * np.pi * 3 / (g.nx * g.hx)
    assert np.max(np.abs(oracle.apply_H(g, None, None, pw, ld=True) - 0.5 * k * k * pw)) < 1e-11


# ------------------------------------------------------------------ NEXT-2: pair propagation and xi projection
def _xi_dense(g, seed, nxi, nfrag):
    """xi_m as dense +-1 / 0 arrays from a big-int restatement of the keyed hash (workloads._sm64): R-23."""
    L = 32
    xi = np.zeros((nxi, g.ng))
    for m in range(nxi):
        for f in range(nfrag):
            kb_ = W._sm64(W._sm64(seed) ^ (2 * m))
            b = W._sm64(kb_ ^ f) % (g.ng // L)
            ks = W._sm64(W._sm64(seed) ^ (2 * m + 1))
            for j in range(L):
                sg = -1.0 if (W._sm64(ks ^ (f * L + j)) >> 63) else 1.0
                xi[m, b * L + j] += sg                    # overlapping fragments add up, as in the oracle's loop
    return xi


def test_pair_propagation_and_xi_projection(oracle):
    """(i) the xi projections are those of a brute-force dense xi built here from the hash definition; (ii) both copies
    follow td_propagate applied to each separately; (iii) a pure phase kick leaves the density unchanged, so the
    projections of the two copies agree at t = 0; (iv) lambda = 0 gives identical copies at every step; (v) the u^R
    coefficients (difference / lambda) are linear in lambda to first order; (vi) at short times they are those of the
    continuity equation: rho^lambda - rho = lambda t div(rho grad v_pert) + O(t^2) for real start orbitals, i.e.
    u^R(t) = t V_H[div(rho grad v)] with the Hartree solve of the erf pin -- sign and scale of the response."""
    g = W.Grid(16, 16, 16, 0.6, 0.6, 0.6)
    rng = np.random.default_rng(17)
    L = np.array(g.box)
    z, y, x = np.meshgrid(np.arange(g.nz) * g.hz, np.arange(g.ny) * g.hy, np.arange(g.nx) * g.hx, indexing="ij")

    def gauss(c, s):
        d = [np.minimum(np.abs(a - ci), Li - np.abs(a - ci)) for a, ci, Li in zip((x, y, z), c, L)]
        return np.exp(-(d[0] ** 2 + d[1] ** 2 + d[2] ** 2) / (2 * s * s))
    vloc = -1.0 * gauss(L / 2, 1.5)
    psi = np.stack([gauss(L / 2 + [0.7, 0, 0], 1.6), gauss(L / 2 - [0, 0.9, 0.3], 1.9)]).astype(np.complex128)   # real orbitals
    vpert = 0.3 * np.cos(2 * np.pi * x / L[0]) + 0.2 * np.sin(2 * np.pi * (y / L[1] + z / L[2]))                 # smooth, periodic
    rs = 2.0 / (2 * g.dV) * 0.05
    seed, nxi, nfrag, dt, nsteps = 99, 6, 5, 0.01, 4
    lam = 1e-3
    kick = oracle.apply_kick(psi, vpert, lam)
    assert np.max(np.abs(kick - np.exp(-1j * lam * vpert)[None] * psi)) < 1e-15
    a, b, out = oracle.td_pair(g, vloc, None, psi, kick, dt, nsteps, rs, seed, nxi, nfrag, ld=True)
    # (i) brute-force projection at step 0 and (ii) trajectories
    xi = _xi_dense(g, seed, nxi, nfrag)
    vh0, _ = oracle.hartree(g, psi, rs, ld=True)
    assert np.max(np.abs(out[0, :, 0] - g.dV * xi @ vh0.ravel())) < 1e-12 * np.max(np.abs(out[0]))
    assert np.max(np.abs(a - oracle.td_propagate(g, vloc, None, psi, dt, nsteps, 1, rs, ld=True))) < 1e-13
    assert np.max(np.abs(b - oracle.td_propagate(g, vloc, None, kick, dt, nsteps, 1, rs, ld=True))) < 1e-13
    # (iii) no response at t = 0
    assert np.max(np.abs(out[0, :, 1] - out[0, :, 0])) < 1e-13 * np.max(np.abs(out[0]))
    # (iv) lambda = 0
    _, _, out0 = oracle.td_pair(g, vloc, None, psi, psi, dt, nsteps, rs, seed, nxi, nfrag, ld=True)
    assert np.array_equal(out0[:, :, 0], out0[:, :, 1])
    # (v) linear in lambda
    ur = (out[:, :, 1] - out[:, :, 0]) / lam
    kick2 = oracle.apply_kick(psi, vpert, lam / 2)
    _, _, outh = oracle.td_pair(g, vloc, None, psi, kick2, dt, nsteps, rs, seed, nxi, nfrag, ld=True)
    urh = (outh[:, :, 1] - outh[:, :, 0]) / (lam / 2)
    assert np.max(np.abs(ur[1:] - urh[1:])) < 2e-3 * np.max(np.abs(ur[1:]))
    # (vi) continuity equation at first order in t, spectral derivatives with numpy
    kx, ky, kz = kgrid(g)
    rho = rs * np.sum(np.abs(psi) ** 2, axis=0)

    def grad(f):
        F = np.fft.fftn(f)
        return [np.fft.ifftn(1j * k * F).real for k in (kx, ky, kz)]
    gv = grad(vpert)
    div = sum(np.fft.ifftn(1j * k * np.fft.fftn(rho * gi)).real for k, gi in zip((kx, ky, kz), gv))
    resp = oracle.poisson(g, div, ld=True)                  # V_H[div(rho grad v)]
    want1 = g.dV * xi @ resp.ravel()                        # d u^R / dt at t = 0, projected
    for n in (1, 2):
        t = n * dt
        assert np.max(np.abs(ur[n] - t * want1)) < 0.08 * np.max(np.abs(t * want1)), (n, ur[n], t * want1)


# ------------------------------------------------------------------ NEXT-4: time-ordering, zeta pair, Sigma(t)
def test_time_ordering_and_zeta_pair_projections(oracle):
    """(i) time-ordering equals the definition written with numpy.fft on the zero-padded causal series (FFT, conjugate
    the negative frequencies, inverse FFT: P:104); (ii) a real causal series gives Re c^T(t) = c^R(t)/2 for t > 0 and
    c^R(0) at t = 0 (the even part of the causal function), and a weakly damped oscillation 2 sin(W t) e^{-g t} gives
    approximately i e^{-i W t} e^{-g t}: only the e^{-i W |t|} branch survives, as in a time-ordered propagator (error O(g/W)); (iii) the zeta pair follows
    td_propagate with -dt / +dt under the frozen potential and its projections are those of a dense xi built here;
    (iv) with enough xi the contraction of R-26 reproduces the grid integral of Eq. 5."""
    rng = np.random.default_rng(5)
    nt, nxi, dt = 48, 3, 0.1
    cr = rng.standard_normal((nt, nxi))
    ct = oracle.time_order(cr, ld=True)
    M = 2 * nt
    pad = np.zeros((M, nxi)); pad[:nt] = cr
    Cw = np.fft.ifft(pad, axis=0) * M                       # sum_n c e^{+i 2 pi k n / M}
    k = np.fft.fftfreq(M, 1.0 / M)
    CT = np.where((k < 0)[:, None], np.conj(Cw), Cw)
    want = np.fft.fft(CT, axis=0)[:nt] / M                  # (1/M) sum_k C^T e^{-i 2 pi k n / M}
    assert np.max(np.abs(ct - want)) < 1e-13 * np.max(np.abs(want)) * M
    assert np.max(np.abs(ct.real[1:] - 0.5 * cr[1:])) < 1e-12 and np.max(np.abs(ct.real[0] - cr[0])) < 1e-12
    nt2, Wf, gam = 400, 1.3, 0.02
    t = np.arange(nt2) * dt
    osc = (2 * np.sin(Wf * t) * np.exp(-gam * t))[:, None]
    cto = oracle.time_order(osc, ld=False)[:, 0]
    ref = 1j * np.exp(-1j * Wf * t) * np.exp(-gam * t)
    assert np.max(np.abs(cto[5:nt2 // 2] - ref[5:nt2 // 2])) < 0.06
    # zeta pair
    g, vloc, kb, rng2 = small_problem(8, 0.7, True)
    zbar = rvec(rng2, g, 1)[0]
    occ = 0.6 * zbar + 0.1 * rvec(rng2, g, 1)[0]
    pair = np.stack([occ, zbar - occ])
    phi = rng2.standard_normal(g.shape)
    seed, nxi2, nfrag, nsteps = 31, 5, 3, 3
    out_pair, p = oracle.td_zeta(g, vloc, kb, pair, phi, 0.05, nsteps, seed, nxi2, nfrag, ld=True)
    assert np.max(np.abs(out_pair[0] - oracle.td_propagate(g, vloc, kb, pair[:1], -0.05, nsteps, 0, 0.0, ld=True)[0])) < 1e-13
    assert np.max(np.abs(out_pair[1] - oracle.td_propagate(g, vloc, kb, pair[1:], 0.05, nsteps, 0, 0.0, ld=True)[0])) < 1e-13
    xi = _xi_dense(g, seed, nxi2, nfrag)
    assert np.max(np.abs(p[0, :, 0] - g.dV * xi @ (phi.ravel() * pair[0].ravel()))) < 1e-12
    mid = oracle.td_propagate(g, vloc, kb, pair[1:], 0.05, 2, 0, 0.0, ld=True)[0]
    assert np.max(np.abs(p[2, :, 1] - g.dV * xi @ (phi.ravel() * mid.ravel()))) < 1e-12
    # resolution of the identity in the xi basis (R-26): many xi reproduce dV sum phi zeta u
    nbig, nf = 4000, 4
    u = rng2.standard_normal(g.shape)
    xib = _xi_dense(g, 7, nbig, nf)
    lhs = g.dV * np.sum(phi * pair[0] * u)
    cm, pm = g.dV * xib @ u.ravel(), g.dV * xib @ (phi.ravel() * pair[0].ravel())
    rhs = g.ng / (nbig * nf * 32 * g.dV) * np.sum(cm * pm)
    assert abs(rhs - lhs) < 0.25 * np.sqrt(np.sum(np.abs(phi * pair[0]) ** 2) * np.sum(u ** 2)) * g.dV * np.sqrt(g.ng / (nbig * nf * 32)) * 3
