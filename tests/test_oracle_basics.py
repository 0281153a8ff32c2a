"""Pins for the oracle's RNG, FFT and the workload generators (CPU only).

Each test checks the oracle against something other than itself: published values, an O(N^2)
direct DFT, numpy.fft (a library), closed forms, the paper's Table 1.
"""
import os

import numpy as np
import pytest

from paper_2601_21005_b200 import workloads as W

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _rows(name):
    with open(os.path.join(GOLD, name)) as f:
        return [ln.split() for ln in f if ln.strip() and not ln.startswith("#")]


# ------------------------------------------------------------------ RNG (SURVEY 8(c) pin "RNG")
def test_splitmix64_published_stream(oracle):
    want = [int(r[0], 16) for r in _rows("splitmix64_state0.txt")]
    assert oracle.splitmix64_stream(0, 3) == want


def test_keyed_hash_golden_and_python_ints(oracle):
    M = (1 << 64) - 1

    def sm(x):                      # independent restatement on Python ints
        x = (x + 0x9E3779B97F4A7C15) & M
        x = ((x ^ (x >> 30)) * 0xBF58476D1CE4E5B9) & M
        x = ((x ^ (x >> 27)) * 0x94D049BB133111EB) & M
        return x ^ (x >> 31)

    for s, v, g, h in _rows("keyed_hash.txt"):
        s, v, g, h = int(s), int(v), int(g), int(h, 16)
        assert oracle.keyed_hash(s, v, g) == h
        assert sm(sm(sm(s) ^ v) ^ g) == h
    # the workload generator's own uniform uses the same hash: top 53 bits
    assert W.hash_uniform(1, 2, 3) == (0xD0734750FDE362B3 >> 11) * 2.0 ** -53


def test_random_vectors_sign_rule_and_statistics(oracle):
    g = W.Grid(32, 32, 32, 0.5, 0.5, 0.5)
    v = oracle.random_vectors(g, 20260121, 0, 4)
    assert v.shape == (4, 32, 32, 32) and np.all(v.imag == 0) and np.all(np.abs(v.real) == 1.0)
    # sign = top bit; golden rows fix individual entries: (1,0,0) -> -1, (0,0,0) -> +1, (1,2,3) -> -1
    assert oracle.random_vectors(g, 0, 0, 1).ravel()[0] == 1.0
    assert oracle.random_vectors(g, 1, 0, 1).ravel()[0] == -1.0
    assert oracle.random_vectors(g, 1, 2, 1).ravel()[3] == -1.0
    # first_vec makes output independent of batching
    assert np.array_equal(oracle.random_vectors(g, 20260121, 2, 2), v[2:4])
    ng = g.ng
    gram = (v.reshape(4, -1).real @ v.reshape(4, -1).real.T) / ng
    assert np.allclose(np.diag(gram), 1.0)
    assert np.abs(gram - np.eye(4)).max() < 5 / np.sqrt(ng)
    assert abs(v.real.mean()) < 5 / np.sqrt(4 * ng)


# ------------------------------------------------------------------ FFT (SURVEY 8(c) pin "FFT")
@pytest.mark.parametrize("n", [32, 96, 128, 256, 384, 45, 14])
@pytest.mark.parametrize("ld", [False, True])
def test_fft1d_vs_direct_dft(oracle, n, ld):
    rng = np.random.default_rng(n)
    x = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    j = np.arange(n)
    F = np.exp(-2j * np.pi * np.outer(j, j) / n)          # O(N^2) definition, e^{-ikr} forward
    assert np.abs(oracle.fft1d(x, -1, ld) - F @ x).max() < 1e-11
    assert np.abs(oracle.fft1d(x, +1, ld) - F.conj() @ x).max() < 1e-11
    assert np.abs(oracle.fft1d(x, -1, ld) - np.fft.fft(x)).max() < 1e-12 * n


def test_fft3_library_parseval_roundtrip_planewave(oracle):
    rng = np.random.default_rng(1)
    nz, ny, nx = 6, 8, 12
    a = rng.standard_normal((nz, ny, nx)) + 1j * rng.standard_normal((nz, ny, nx))
    f = oracle.fft3(a, -1)
    assert np.abs(f - np.fft.fftn(a)).max() < 1e-12
    assert abs(np.sum(np.abs(f) ** 2) / a.size - np.sum(np.abs(a) ** 2)) < 1e-10     # Parseval
    assert np.abs(oracle.fft3(f, +1) / a.size - a).max() < 1e-14                      # inverse
    # single plane wave e^{+i 2 pi (mx x/nx + my y/ny + mz z/nz)} -> single bin (mz,my,mx)
    mz, my, mx = 5, 3, 7
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    pw = np.exp(2j * np.pi * (mx * x / nx + my * y / ny + mz * z / nz))
    f = oracle.fft3(pw, -1)
    want = np.zeros_like(f)
    want[mz, my, mx] = a.size
    assert np.abs(f - want).max() < 1e-10


# ------------------------------------------------------------------ generators
def test_cluster_stoichiometry_matches_paper_table1():
    for nsi, nh, ne, r2 in _rows("paper_clusters.txt"):
        si, hy = W.diamond_cluster(int(r2))
        assert (len(si), len(hy)) == (int(nsi), int(nh))
        assert 4 * len(si) + len(hy) == int(ne)
    for r2, nsi, nh in [(64, 35, 36), (108, 87, 76)]:          # BASELINE.json configs[1], [2]
        si, hy = W.diamond_cluster(r2)
        assert (len(si), len(hy)) == (nsi, nh)


def test_cluster_geometry_bond_lengths():
    si, hy = W.diamond_cluster(64)
    d = np.linalg.norm(si[:, None, :] - si[None, :, :], axis=-1)
    np.fill_diagonal(d, 99)
    assert np.allclose(d.min(axis=1), W.A_SI * np.sqrt(3) / 4)     # Si-Si bond 4.44 bohr
    dh = np.linalg.norm(hy[:, None, :] - si[None, :, :], axis=-1).min(axis=1)
    assert np.allclose(dh, W.H_BOND)
    # every Si is 4-coordinated (Si + H neighbours)
    bond = W.A_SI * np.sqrt(3) / 4
    nsi = (np.abs(d - bond) < 1e-9).sum(axis=1)
    nh = (np.abs(np.linalg.norm(si[:, None, :] - hy[None, :, :], axis=-1) - W.H_BOND) < 1e-9).sum(axis=1)
    assert np.all(nsi + nh == 4)


def test_box_fit_and_paper_arithmetic():
    # SURVEY 8 box fit: cluster radius + 2.8 + 8 <= L/2
    for name, r2 in [("cfg1", 64), ("cfg2", 108), ("cfg3", 480), ("cfg4", 2540)]:
        n, h = W._CFG[name][0], W._CFG[name][1]
        R = np.sqrt(r2) * W.A_SI / 8
        assert R + 2.8 + 8.0 <= n * h / 2 + 1e-9
    assert round(3 / (0.06 * 0.05)) == 1000                      # PAPER.md:155, N_tau


def test_vloc_matches_bruteforce_minimum_image():
    g = W.Grid(12, 10, 8, 0.5, 0.6, 0.7)
    centers = np.array([[0.3, 5.8, 2.0], [5.9, 0.1, 5.5]])
    v = W.gaussian_vloc(g, centers, [1.0, 2.0], [0.5, 0.4])
    z, y, x = np.meshgrid(np.arange(8) * 0.7, np.arange(10) * 0.6, np.arange(12) * 0.5, indexing="ij")
    want = np.zeros_like(v)
    L = g.box
    for c, dep, sg in zip(centers, [1.0, 2.0], [0.5, 0.4]):
        d = [x - c[0], y - c[1], z - c[2]]
        d = [di - Li * np.round(di / Li) for di, Li in zip(d, L)]
        want -= dep * np.exp(-(d[0] ** 2 + d[1] ** 2 + d[2] ** 2) / (2 * sg * sg))
    assert np.abs(v - want).max() < 1e-14


def test_kb_lists_normalised_sorted_in_sphere():
    g = W.Grid(16, 16, 16, 0.5, 0.5, 0.5)
    centers = np.array([[4.0, 4.0, 4.0], [0.2, 7.9, 3.3]])
    kb = W.kb_projectors(g, centers)
    assert kb.nsphere == 2 and kb.nproj == 4 and kb.sph_ptr[-1] == len(kb.sph_idx)
    for s in range(2):
        sl = slice(kb.sph_ptr[s], kb.sph_ptr[s + 1])
        idx, b = kb.sph_idx[sl].astype(np.int64), kb.beta[sl]
        assert np.all(np.diff(idx) > 0)
        assert np.allclose(g.dV * np.sum(b * b, axis=0), 1.0)
        ix, iy, iz = idx % 16, (idx // 16) % 16, idx // 256
        d = np.stack([ix * 0.5 - centers[s][0], iy * 0.5 - centers[s][1], iz * 0.5 - centers[s][2]], 1)
        d -= 8.0 * np.round(d / 8.0)
        assert np.all(np.sum(d * d, axis=1) <= 2.5 ** 2 + 1e-12)
        assert abs(len(idx) - 4 / 3 * np.pi * 2.5 ** 3 / g.dV) < 40      # ~524 points at h = 0.5
        assert kb.D[s, 1] == kb.D[s, 2] == kb.D[s, 3] and np.all(np.abs(kb.D[s]) <= 1)
    # centre on a grid point: s and p projectors are exactly orthogonal by parity
    b = kb.beta[kb.sph_ptr[0]:kb.sph_ptr[1]]
    gram = g.dV * b.T @ b
    assert np.abs(gram - np.eye(4)).max() < 1e-13


def test_cheb_coeffs_interpolate_at_nodes_and_decay():
    emin, emax, nt = -1.0, 59.2, 64
    a = W.cheb_coeffs(W.sqrt_fermi, emin, emax, nt, oversample=1)
    theta = np.pi * (np.arange(nt) + 0.5) / nt
    x = np.cos(theta)
    series = sum(a[n] * np.cos(n * theta) for n in range(nt))
    assert np.abs(series - W.sqrt_fermi(0.5 * (emax + emin) + 0.5 * (emax - emin) * x)).max() < 1e-13
    a8 = W.cheb_coeffs(W.sqrt_fermi, emin, emax, 128)
    direct = np.array([(2 - (n == 0)) / 1024 * np.sum(
        W.sqrt_fermi(29.1 + 30.1 * np.cos(np.pi * (np.arange(1024) + 0.5) / 1024)) *
        np.cos(n * np.pi * (np.arange(1024) + 0.5) / 1024)) for n in range(128)])
    assert np.abs(a8 - direct).max() < 1e-14
    assert 1e-3 < abs(a8[127]) < 1e-2                              # |a_127| ~ 3e-3


def test_workload_cfg0_matches_baseline_config():
    w = W.make_workload("cfg0")
    assert w.grid.shape == (32, 32, 32) and w.nvec == 4 and w.nterms == 128 and w.kb.nsphere == 0
    assert -8.0 < w.emin < -0.9 and abs(w.emax - (1.5 * (np.pi / 0.5) ** 2 + w.vloc.max())) < 1e-12
