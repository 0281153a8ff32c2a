"""GPU parity at the sizes of BASELINE.json's configs, in the launch configuration bench.py times.

Full-size oracle runs are only feasible for a few applications, so ("Oracle cost and
parity coverage"): every config shape gets a single H apply compared element by element on a declared
subset of vectors; cfg1 (the bench workload) also gets a filter prefix on two vectors taken from the
64-vector batch that bench.py filters; cfg2 gets a TD-Hartree prefix on all 16 vectors (the Hartree
term couples them).  What was compared at full length and what at a prefix is stated in each test.
"""
import numpy as np
import pytest

from paper_2601_21005_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL_H = 1e-11
TOL_FULL = 1e-8


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch


@pytest.fixture(scope="module")
def api(torch_cuda):
    from paper_2601_21005_b200 import api as a
    a.load()
    return a


def relerr(got, want):
    got = got.reshape(got.shape[0], -1)
    want = want.reshape(want.shape[0], -1)
    return float(np.max(np.linalg.norm(got - want, axis=1) / np.linalg.norm(want, axis=1)))


def test_cfg1_bench_configuration_sampled_vectors(api, torch_cuda, oracle, monkeypatch):
    """cfg1 exactly as bench.py runs it (96^3, 64 vectors in one call, max_nvec = 64): the first 33 terms of
    the 512-term coefficient list.  Vectors 0, 37 and 63 of the batch are compared with the oracle."""
    torch = torch_cuda
    w = W.make_workload("cfg1")
    coeffs = w.coeffs[:33]
    ctx = api.context_for(w)
    psi = ctx.sgw_random_vectors(W.SEED_VEC, 0, w.nvec)
    ref0 = oracle.random_vectors(w.grid, W.SEED_VEC, 0, w.nvec)
    assert np.array_equal(psi.cpu().numpy().view(np.uint64), ref0.view(np.uint64))
    h = ctx.sgw_apply_H(psi)
    pick = [0, 37, 63]
    assert relerr(h[pick].cpu().numpy(), oracle.apply_H(w.grid, w.vloc, None, ref0[pick], ld=True)) < TOL_H
    ctx.sgw_cheb_filter(psi, coeffs, w.emin, w.emax)
    want = oracle.cheb_filter(w.grid, w.vloc, None, ref0[pick], coeffs, w.emin, w.emax, ld=True)
    assert relerr(psi[pick].cpu().numpy(), want) < TOL_FULL
    assert ctx.sgw_sync_check() == 0
    ctx.close()


def test_cfg2_td_hartree_prefix_all_vectors(api, torch_cuda, oracle, monkeypatch):
    """cfg2 (128^3, 16 vectors): a 9-term filter, then 3 split-operator steps with the Hartree potential
    rebuilt every step from all 16 vectors (prefix of the 2000 steps), every vector compared."""
    torch = torch_cuda
    w = W.make_workload("cfg2", nterms=9)
    ctx = api.context_for(w)
    psi = ctx.sgw_random_vectors(W.SEED_VEC, 0, w.nvec)
    ref = oracle.random_vectors(w.grid, W.SEED_VEC, 0, w.nvec)
    ctx.sgw_cheb_filter(psi, w.coeffs, w.emin, w.emax)
    ref = oracle.cheb_filter(w.grid, w.vloc, None, ref, w.coeffs, w.emin, w.emax, ld=True)
    assert relerr(psi.cpu().numpy(), ref) < TOL_FULL
    ctx.sgw_set_td(1, w.rho_scale)
    n0 = ctx.sgw_norms(psi).cpu().numpy()
    ctx.sgw_td_propagate(psi, w.dt, 3)
    ref = oracle.td_propagate(w.grid, w.vloc, None, ref, w.dt, 3, 1, w.rho_scale, ld=True)
    assert relerr(psi.cpu().numpy(), ref) < TOL_FULL
    # local-only propagation is unitary: norms conserved (property that holds at any length)
    n1 = ctx.sgw_norms(psi).cpu().numpy()
    assert np.max(np.abs(n1 / n0 - 1.0)) < 1e-12
    assert ctx.sgw_sync_check() == 0
    ctx.close()


def test_cfg3_shape_apply_H_and_terms_with_kb(api, torch_cuda, oracle, monkeypatch):
    """cfg3 shape (256^3, Si705H300 local + KB projectors): 2 vectors out of the 256; one H apply and a
    4-term filter (3 applications) compared element by element."""
    torch = torch_cuda
    w = W.make_workload("cfg3", nvec=2, nterms=4)
    assert w.atoms == "Si705H300" and w.kb.nsphere == 705
    ctx = api.context_for(w)
    psi = ctx.sgw_random_vectors(W.SEED_VEC, 100, 2)          # vectors 100, 101 of the batch
    ref = oracle.random_vectors(w.grid, W.SEED_VEC, 100, 2)
    h = ctx.sgw_apply_H(psi)
    assert relerr(h.cpu().numpy(), oracle.apply_H(w.grid, w.vloc, w.kb, ref, ld=True)) < TOL_H
    ctx.sgw_cheb_filter(psi, w.coeffs, w.emin, w.emax)
    want = oracle.cheb_filter(w.grid, w.vloc, w.kb, ref, w.coeffs, w.emin, w.emax, ld=True)
    assert relerr(psi.cpu().numpy(), want) < TOL_FULL
    assert ctx.sgw_sync_check() == 0
    ctx.close()


@pytest.mark.slow
def test_cfg4_shape_apply_H_and_td_step_with_kb(api, torch_cuda, oracle):
    """cfg4 shape (384^3, Si8381H1620 = 10001 atoms, local + KB): one vector; one H apply and one
    TD-Hartree step compared element by element (the largest supported axis length, radix-3 factor)."""
    torch = torch_cuda
    w = W.make_workload("cfg4", nvec=1, nterms=2)
    assert w.atoms == "Si8381H1620"
    ctx = api.context_for(w)
    psi = ctx.sgw_random_vectors(W.SEED_VEC, 31, 1)
    ref = oracle.random_vectors(w.grid, W.SEED_VEC, 31, 1)
    h = ctx.sgw_apply_H(psi)
    assert relerr(h.cpu().numpy(), oracle.apply_H(w.grid, w.vloc, w.kb, ref, ld=True)) < TOL_H
    del h
    ctx.sgw_set_td(1, w.rho_scale)
    ctx.sgw_td_propagate(psi, w.dt, 1)
    want = oracle.td_propagate(w.grid, w.vloc, w.kb, ref, w.dt, 1, 1, w.rho_scale, ld=True)
    assert relerr(psi.cpu().numpy(), want) < TOL_FULL
    ctx.close()


@pytest.mark.parametrize("n,nz,nvec,use_kb", [(32, 32, 4, False), (48, 48, 3, True), (64, 24, 2, True), (24, 12, 5, True),
                                              (12, 12, 2, False)])
def test_lean_passes_small_grids(api, torch_cuda, oracle, monkeypatch, n, nz, nvec, use_kb):
    """The lean passes on cubic grids, non-cubic grids (three axis launches) and an axis length that is not a
    multiple of 8 (4 pencils per tile): H apply, odd and even term counts, TD with and without the Hartree rebuild."""
    torch = torch_cuda
    g = W.Grid(n, n, nz, 0.5, 0.5, 0.55)
    rng = np.random.default_rng(7 * n + nz)
    L = np.array(g.box)
    centers = rng.uniform(0, 1, size=(3, 3)) * L
    vloc = W.gaussian_vloc(g, centers, [1.0, 2.0, 1.5], [0.9, 1.2, 0.8])
    kb = W.kb_projectors(g, centers[:2], radius=min(1.8, 0.45 * L.min()), sigma=0.7) if use_kb else W.KB.empty()
    psi = rng.standard_normal((nvec,) + g.shape) + 1j * rng.standard_normal((nvec,) + g.shape)
    ctx = api.Context(g.nx, g.ny, g.nz, g.hx, g.hy, g.hz, nvec)
    ctx.sgw_set_vloc(torch.from_numpy(vloc).cuda())
    if kb.nsphere:
        ctx.sgw_set_nonlocal(torch.from_numpy(kb.sph_ptr).cuda(), torch.from_numpy(kb.sph_idx).cuda(),
                             torch.from_numpy(kb.beta).cuda(), torch.from_numpy(kb.D).cuda())
    kbo = kb if kb.nsphere else None
    got = ctx.sgw_apply_H(torch.from_numpy(psi).cuda()).cpu().numpy()
    assert relerr(got, oracle.apply_H(g, vloc, kbo, psi, ld=True)) < TOL_H
    emin, emax = W.spectral_bounds(g, vloc, True)
    for nterms in (2, 3, 8, 9):
        coeffs = rng.standard_normal(nterms)
        t = torch.from_numpy(psi).cuda()
        ctx.sgw_cheb_filter(t, coeffs, emin, emax)
        assert relerr(t.cpu().numpy(), oracle.cheb_filter(g, vloc, kbo, psi, coeffs, emin, emax, ld=True)) < TOL_FULL
    rs = 2.0 / (nvec * g.dV) * 0.01
    for mode in (0, 1):
        ctx.sgw_set_td(mode, rs)
        t = torch.from_numpy(psi).cuda()
        ctx.sgw_td_propagate(t, 0.05, 3)
        assert relerr(t.cpu().numpy(), oracle.td_propagate(g, vloc, kbo, psi, 0.05, 3, mode, rs, ld=True)) < TOL_FULL
    assert ctx.sgw_sync_check() == 0
    ctx.close()


@pytest.mark.parametrize("n,nvec", [(32, 80), (48, 40)])
def test_many_planes_per_cta(api, torch_cuda, oracle, monkeypatch, n, nvec):
    """Enough xy planes (2560 / 1920) that every persistent CTA owns several plane groups and every warp group
    many tiles: the regime of the bench workload, at a size the oracle finishes in seconds."""
    torch = torch_cuda
    g = W.Grid(n, n, n, 0.5, 0.5, 0.5)
    rng = np.random.default_rng(n + nvec)
    centers = rng.uniform(0, 1, size=(3, 3)) * np.array(g.box)
    vloc = W.gaussian_vloc(g, centers, [1.0, 2.0, 1.5], [0.9, 1.2, 0.8])
    psi = rng.standard_normal((nvec,) + g.shape) + 1j * rng.standard_normal((nvec,) + g.shape)
    ctx = api.Context(g.nx, g.ny, g.nz, g.hx, g.hy, g.hz, nvec)
    ctx.sgw_set_vloc(torch.from_numpy(vloc).cuda())
    emin, emax = W.spectral_bounds(g, vloc, False)
    coeffs = rng.standard_normal(12)
    t = torch.from_numpy(psi).cuda()
    ctx.sgw_cheb_filter(t, coeffs, emin, emax)
    assert relerr(t.cpu().numpy(), oracle.cheb_filter(g, vloc, None, psi, coeffs, emin, emax, ld=True)) < TOL_FULL
    rs = 2.0 / (nvec * g.dV) * 0.01
    ctx.sgw_set_td(1, rs)
    t = torch.from_numpy(psi).cuda()
    ctx.sgw_td_propagate(t, 0.05, 4)
    assert relerr(t.cpu().numpy(), oracle.td_propagate(g, vloc, None, psi, 0.05, 4, 1, rs, ld=True)) < TOL_FULL
    assert ctx.sgw_sync_check() == 0
    ctx.close()


def test_spectral_bounds_vs_oracle_and_enclosure(api, torch_cuda, oracle):
    """NEXT-1: shifted power iteration on the GPU against the oracle's (same algorithm, same start
    vectors), with and without KB projectors, and the enclosure by the analytic bounds the configs use."""
    torch = torch_cuda
    for n, use_kb in [(24, True), (32, False)]:
        g = W.Grid(n, n, n, 0.5, 0.5, 0.5)
        rng = np.random.default_rng(n)
        centers = rng.uniform(0, 1, size=(3, 3)) * np.array(g.box)
        vloc = W.gaussian_vloc(g, centers, [1.0, 2.0, 1.5], [0.9, 1.2, 0.8])
        kb = W.kb_projectors(g, centers[:2], radius=1.8, sigma=0.7) if use_kb else W.KB.empty()
        ctx = api.Context(g.nx, g.ny, g.nz, g.hx, g.hy, g.hz, 1)
        ctx.sgw_set_vloc(torch.from_numpy(vloc).cuda())
        if kb.nsphere:
            ctx.sgw_set_nonlocal(torch.from_numpy(kb.sph_ptr).cuda(), torch.from_numpy(kb.sph_idx).cuda(),
                                 torch.from_numpy(kb.beta).cuda(), torch.from_numpy(kb.D).cuda())
        for niter in (5, 60):
            emin, emax = ctx.sgw_spectral_bounds(niter, 4242)
            omin, omax = oracle.spectral_bounds(g, vloc, kb if kb.nsphere else None, niter, 4242, ld=True)
            span = omax - omin
            assert abs(emin - omin) < 1e-9 * span and abs(emax - omax) < 1e-9 * span
        lo, hi = W.spectral_bounds(g, vloc, bool(kb.nsphere))
        assert lo <= emin <= emax <= hi
        ctx.close()


@pytest.mark.parametrize("G,ctas", [("2", "2"), ("3", "1"), ("1", "1")])
def test_lean_plane_kernel_group_and_cta_variants(api, torch_cuda, oracle, monkeypatch, G, ctas):
    """The lean plane kernel with several planes per CTA-owned group (ragged last group: 5 * 32 planes is not a
    multiple of 3) and with the one-CTA-per-SM (16-warp) variant, against the oracle."""
    torch = torch_cuda
    monkeypatch.setenv("SGW_LEAN_G", G)
    monkeypatch.setenv("SGW_LEAN_CTAS", ctas)
    n, nvec = 32, 5
    g = W.Grid(n, n, n, 0.5, 0.5, 0.5)
    rng = np.random.default_rng(11)
    centers = rng.uniform(0, 1, size=(3, 3)) * np.array(g.box)
    vloc = W.gaussian_vloc(g, centers, [1.0, 2.0, 1.5], [0.9, 1.2, 0.8])
    psi = rng.standard_normal((nvec,) + g.shape) + 1j * rng.standard_normal((nvec,) + g.shape)
    ctx = api.Context(g.nx, g.ny, g.nz, g.hx, g.hy, g.hz, nvec)
    ctx.sgw_set_vloc(torch.from_numpy(vloc).cuda())
    emin, emax = W.spectral_bounds(g, vloc, False)
    coeffs = rng.standard_normal(7)
    t = torch.from_numpy(psi).cuda()
    ctx.sgw_cheb_filter(t, coeffs, emin, emax)
    assert relerr(t.cpu().numpy(), oracle.cheb_filter(g, vloc, None, psi, coeffs, emin, emax, ld=True)) < TOL_FULL
    ctx.sgw_set_td(1, 2.0 / (nvec * g.dV) * 0.01)
    t = torch.from_numpy(psi).cuda()
    ctx.sgw_td_propagate(t, 0.05, 3)
    want = oracle.td_propagate(g, vloc, None, psi, 0.05, 3, 1, 2.0 / (nvec * g.dV) * 0.01, ld=True)
    assert relerr(t.cpu().numpy(), want) < TOL_FULL
    ctx.close()


@pytest.mark.parametrize("n,nz,nvec", [(64, 48, 4), (96, 24, 5), (128, 24, 4), (256, 12, 4)])
def test_lean_plane_cluster_kernel(api, torch_cuda, oracle, monkeypatch, n, nz, nvec):
    """The cluster-owned plane kernel (clusters of 2 / 3 / 4 / 8 CTAs for 64^2 / 96^2 / 128^2 / 256^2 planes), forced
    on for both families, against the oracle; nvec * nz planes exceed the resident clusters (at most 2 * 148 / size),
    so the plane loop runs a ragged second round."""
    torch = torch_cuda
    monkeypatch.setenv("SGW_LEAN_CLUSTER", "1")
    g = W.Grid(n, n, nz, 0.5, 0.5, 0.5)
    rng = np.random.default_rng(23)
    centers = rng.uniform(0, 1, size=(3, 3)) * np.array(g.box)
    vloc = W.gaussian_vloc(g, centers, [1.0, 2.0, 1.5], [0.9, 1.2, 0.8])
    psi = rng.standard_normal((nvec,) + g.shape) + 1j * rng.standard_normal((nvec,) + g.shape)
    ctx = api.Context(g.nx, g.ny, g.nz, g.hx, g.hy, g.hz, nvec)
    ctx.sgw_set_vloc(torch.from_numpy(vloc).cuda())
    emin, emax = W.spectral_bounds(g, vloc, False)
    coeffs = rng.standard_normal(6)
    t = torch.from_numpy(psi).cuda()
    ctx.sgw_cheb_filter(t, coeffs, emin, emax)
    assert relerr(t.cpu().numpy(), oracle.cheb_filter(g, vloc, None, psi, coeffs, emin, emax, ld=True)) < TOL_FULL
    ctx.sgw_set_td(1, 2.0 / (nvec * g.dV) * 0.01)
    t = torch.from_numpy(psi).cuda()
    ctx.sgw_td_propagate(t, 0.05, 2)
    want = oracle.td_propagate(g, vloc, None, psi, 0.05, 2, 1, 2.0 / (nvec * g.dV) * 0.01, ld=True)
    assert relerr(t.cpu().numpy(), want) < TOL_FULL
    ctx.close()


@pytest.mark.parametrize("n,nz,nvec,vminor", [(32, 24, 7, "1"), (64, 16, 5, "0"), (96, 8, 6, "1"), (256, 8, 3, "1")])
def test_lean_plane_team_kernel_and_vector_minor_order(api, torch_cuda, oracle, monkeypatch, n, nz, nvec, vminor):
    """The team-owned plane kernel (N/8 warp groups per plane, arrival counter per plane, software-pipelined row and
    column tiles; default for 256^2 and 384^2 planes), forced on for small planes so that many teams run several
    rounds with a ragged last round, with the tile order running over the vectors first (vminor) or last; both
    operator families, against the oracle."""
    torch = torch_cuda
    monkeypatch.setenv("SGW_LEAN_TEAM", "1")
    monkeypatch.setenv("SGW_LEAN_VMINOR", vminor)
    g = W.Grid(n, n, nz, 0.5, 0.5, 0.5)
    rng = np.random.default_rng(29 + n)
    centers = rng.uniform(0, 1, size=(3, 3)) * np.array(g.box)
    vloc = W.gaussian_vloc(g, centers, [1.0, 2.0, 1.5], [0.9, 1.2, 0.8])
    psi = rng.standard_normal((nvec,) + g.shape) + 1j * rng.standard_normal((nvec,) + g.shape)
    ctx = api.Context(g.nx, g.ny, g.nz, g.hx, g.hy, g.hz, nvec)
    ctx.sgw_set_vloc(torch.from_numpy(vloc).cuda())
    got = ctx.sgw_apply_H(torch.from_numpy(psi).cuda()).cpu().numpy()
    assert relerr(got, oracle.apply_H(g, vloc, None, psi, ld=True)) < TOL_H
    emin, emax = W.spectral_bounds(g, vloc, False)
    coeffs = rng.standard_normal(6)
    t = torch.from_numpy(psi).cuda()
    ctx.sgw_cheb_filter(t, coeffs, emin, emax)
    assert relerr(t.cpu().numpy(), oracle.cheb_filter(g, vloc, None, psi, coeffs, emin, emax, ld=True)) < TOL_FULL
    rs = 2.0 / (nvec * g.dV) * 0.01
    ctx.sgw_set_td(1, rs)
    t = torch.from_numpy(psi).cuda()
    ctx.sgw_td_propagate(t, 0.05, 3)
    assert relerr(t.cpu().numpy(), oracle.td_propagate(g, vloc, None, psi, 0.05, 3, 1, rs, ld=True)) < TOL_FULL
    assert ctx.sgw_sync_check() == 0
    ctx.close()


@pytest.mark.parametrize("shape", [(32, 48, 24), (64, 32, 16)])
def test_vector_minor_order_on_axis_passes(api, torch_cuda, oracle, monkeypatch, shape):
    """Non-square planes take three axis passes; with the tile order running over the vectors first (the order used
    when the potential / phase table does not fit L2) the results are those of the oracle, with KB projectors."""
    torch = torch_cuda
    monkeypatch.setenv("SGW_LEAN_VMINOR", "1")
    nx, ny, nz = shape
    nvec = 5
    g = W.Grid(nx, ny, nz, 0.5, 0.45, 0.55)
    rng = np.random.default_rng(nx + ny)
    centers = rng.uniform(0, 1, size=(3, 3)) * np.array(g.box)
    vloc = W.gaussian_vloc(g, centers, [1.0, 2.0, 1.5], [0.9, 1.2, 0.8])
    kb = W.kb_projectors(g, centers[:2], radius=1.8, sigma=0.7)
    psi = rng.standard_normal((nvec,) + g.shape) + 1j * rng.standard_normal((nvec,) + g.shape)
    ctx = api.Context(g.nx, g.ny, g.nz, g.hx, g.hy, g.hz, nvec)
    ctx.sgw_set_vloc(torch.from_numpy(vloc).cuda())
    ctx.sgw_set_nonlocal(torch.from_numpy(kb.sph_ptr).cuda(), torch.from_numpy(kb.sph_idx).cuda(),
                         torch.from_numpy(kb.beta).cuda(), torch.from_numpy(kb.D).cuda())
    emin, emax = W.spectral_bounds(g, vloc, True)
    coeffs = rng.standard_normal(7)
    t = torch.from_numpy(psi).cuda()
    ctx.sgw_cheb_filter(t, coeffs, emin, emax)
    assert relerr(t.cpu().numpy(), oracle.cheb_filter(g, vloc, kb, psi, coeffs, emin, emax, ld=True)) < TOL_FULL
    rs = 2.0 / (nvec * g.dV) * 0.01
    ctx.sgw_set_td(1, rs)
    t = torch.from_numpy(psi).cuda()
    ctx.sgw_td_propagate(t, 0.05, 3)
    assert relerr(t.cpu().numpy(), oracle.td_propagate(g, vloc, kb, psi, 0.05, 3, 1, rs, ld=True)) < TOL_FULL
    ctx.close()


@pytest.mark.parametrize("n,nvec,use_kb,l2mb", [(32, 5, True, None), (48, 3, False, "0"), (64, 4, True, "0"), (96, 3, False, None),
                                                 (128, 2, True, None), (96, 5, True, "0")])
def test_tma_accumulate_kernel_apply_H_and_clenshaw_filter(api, torch_cuda, oracle, monkeypatch, n, nvec, use_kb, l2mb):
    """The TMA accumulate kernel (sgw_acc.cuh: bulk / tensor-map loads into a shared-memory ring, in-place round trip,
    bulk reduce-add into the accumulator) forced on for every cubic size it is built for: H apply and the Clenshaw
    form of the Chebyshev series for 1..10 coefficients against the oracle's forward recurrence, in the one-launch
    (vector-major) order and, with SGW_ACC_L2_MB=0, in the two-launch (planes, then z columns) order."""
    torch = torch_cuda
    monkeypatch.setenv("SGW_ACC", "1")
    if l2mb is not None:
        monkeypatch.setenv("SGW_ACC_L2_MB", l2mb)
    g = W.Grid(n, n, n, 0.5, 0.45, 0.55)
    rng = np.random.default_rng(41 + n)
    centers = rng.uniform(0, 1, size=(3, 3)) * np.array(g.box)
    vloc = W.gaussian_vloc(g, centers, [1.0, 2.0, 1.5], [0.9, 1.2, 0.8])
    kb = W.kb_projectors(g, centers[:2], radius=1.8, sigma=0.7) if use_kb else W.KB.empty()
    kbo = kb if kb.nsphere else None
    psi = rng.standard_normal((nvec,) + g.shape) + 1j * rng.standard_normal((nvec,) + g.shape)
    ctx = api.Context(g.nx, g.ny, g.nz, g.hx, g.hy, g.hz, nvec)
    ctx.sgw_set_vloc(torch.from_numpy(vloc).cuda())
    if kb.nsphere:
        ctx.sgw_set_nonlocal(torch.from_numpy(kb.sph_ptr).cuda(), torch.from_numpy(kb.sph_idx).cuda(),
                             torch.from_numpy(kb.beta).cuda(), torch.from_numpy(kb.D).cuda())
    got = ctx.sgw_apply_H(torch.from_numpy(psi).cuda()).cpu().numpy()
    assert relerr(got, oracle.apply_H(g, vloc, kbo, psi, ld=True)) < TOL_H
    emin, emax = W.spectral_bounds(g, vloc, True)
    for nterms in (1, 2, 3, 4, 5, 10):
        coeffs = rng.standard_normal(nterms)
        t = torch.from_numpy(psi).cuda()
        ctx.sgw_cheb_filter(t, coeffs, emin, emax)
        assert relerr(t.cpu().numpy(), oracle.cheb_filter(g, vloc, kbo, psi, coeffs, emin, emax, ld=True)) < TOL_FULL, nterms
    assert ctx.sgw_sync_check() == 0
    ctx.close()


@pytest.mark.parametrize("shape,nvec,use_kb", [((32, 32, 32), 3, True), ((24, 32, 16), 2, False), ((64, 64, 64), 2, True)])
def test_kinetic_cutoff_five_pass_route(api, torch_cuda, oracle, shape, nvec, use_kb):
    """NEXT-3: with sgw_set_kinetic_cutoff the kinetic operator is min(1/2 k^2, E_cut), which is not
    separable; H apply, the Chebyshev filter and the split-operator step then take the five-pass full-3D-transform route.
    Against the oracle with the same cutoff (cubic and non-cubic grids, with and without KB and the Hartree rebuild),
    and back to the separable operator after sgw_set_kinetic_cutoff(0)."""
    torch = torch_cuda
    nx, ny, nz = shape
    ecut = 9.0
    g = W.Grid(nx, ny, nz, 0.5, 0.45, 0.55)
    rng = np.random.default_rng(nx + nz)
    centers = rng.uniform(0, 1, size=(3, 3)) * np.array(g.box)
    vloc = W.gaussian_vloc(g, centers, [1.0, 2.0, 1.5], [0.9, 1.2, 0.8])
    kb = W.kb_projectors(g, centers[:2], radius=1.8, sigma=0.7) if use_kb else W.KB.empty()
    kbo = kb if kb.nsphere else None
    psi = rng.standard_normal((nvec,) + g.shape) + 1j * rng.standard_normal((nvec,) + g.shape)
    ctx = api.Context(g.nx, g.ny, g.nz, g.hx, g.hy, g.hz, nvec)
    ctx.sgw_set_vloc(torch.from_numpy(vloc).cuda())
    if kb.nsphere:
        ctx.sgw_set_nonlocal(torch.from_numpy(kb.sph_ptr).cuda(), torch.from_numpy(kb.sph_idx).cuda(),
                             torch.from_numpy(kb.beta).cuda(), torch.from_numpy(kb.D).cuda())
    plain = ctx.sgw_apply_H(torch.from_numpy(psi).cuda()).cpu().numpy()
    ctx.sgw_set_kinetic_cutoff(ecut)
    try:
        oracle.set_kinetic_cutoff(ecut)
        got = ctx.sgw_apply_H(torch.from_numpy(psi).cuda()).cpu().numpy()
        want = oracle.apply_H(g, vloc, kbo, psi, ld=True)
        assert relerr(got, want) < TOL_H
        assert relerr(plain, want) > 1e-3                     # the cutoff changes the operator on this grid
        emin, emax = float(vloc.min()) - 2.0, ecut + float(vloc.max()) + 2.0      # the narrower window the cutoff buys
        for nterms in (2, 5, 8):
            coeffs = rng.standard_normal(nterms)
            t = torch.from_numpy(psi).cuda()
            ctx.sgw_cheb_filter(t, coeffs, emin, emax)
            assert relerr(t.cpu().numpy(), oracle.cheb_filter(g, vloc, kbo, psi, coeffs, emin, emax, ld=True)) < TOL_FULL
        rs = 2.0 / (nvec * g.dV) * 0.01
        for mode in (0, 1):
            ctx.sgw_set_td(mode, rs)
            t = torch.from_numpy(psi).cuda()
            ctx.sgw_td_propagate(t, 0.05, 3)
            assert relerr(t.cpu().numpy(), oracle.td_propagate(g, vloc, kbo, psi, 0.05, 3, mode, rs, ld=True)) < TOL_FULL
    finally:
        oracle.set_kinetic_cutoff(0.0)
    ctx.sgw_set_kinetic_cutoff(0.0)
    again = ctx.sgw_apply_H(torch.from_numpy(psi).cuda()).cpu().numpy()
    assert relerr(again, plain) < 1e-14
    assert ctx.sgw_sync_check() == 0
    ctx.close()


@pytest.mark.parametrize("n,nvec,use_kb", [(32, 3, False), (48, 2, True), (64, 2, False)])
def test_pair_propagation_with_xi_projection(api, torch_cuda, oracle, n, nvec, use_kb):
    """NEXT-2: perturbed copy exp(-i lambda v) eta, both copies propagated under their own
    Hartree potentials, and the xi projections of both potentials at every step, against the oracle: the kick bit for
    bit up to rounding, both trajectories to 1e-8, the projections to 1e-10 of their scale, and the u^R coefficients
    (difference / lambda) to 1e-6 of theirs (they are a small difference of the projections)."""
    torch = torch_cuda
    g = W.Grid(n, n, n, 0.5, 0.5, 0.5)
    rng = np.random.default_rng(3 * n)
    centers = rng.uniform(0, 1, size=(3, 3)) * np.array(g.box)
    vloc = W.gaussian_vloc(g, centers, [1.0, 2.0, 1.5], [0.9, 1.2, 0.8])
    kb = W.kb_projectors(g, centers[:2], radius=1.8, sigma=0.7) if use_kb else W.KB.empty()
    kbo = kb if kb.nsphere else None
    vpert = W.gaussian_vloc(g, centers[1:2], [0.7], [1.5]) + 0.1
    psi = rng.standard_normal((nvec,) + g.shape) + 1j * rng.standard_normal((nvec,) + g.shape)
    lam, dt, nsteps, seed, nxi, nfrag = 1e-2, 0.05, 4, 77, 9, 6
    rs = 2.0 / (nvec * g.dV) * 0.01
    ctx = api.Context(g.nx, g.ny, g.nz, g.hx, g.hy, g.hz, nvec)
    ctx.sgw_set_vloc(torch.from_numpy(vloc).cuda())
    if kb.nsphere:
        ctx.sgw_set_nonlocal(torch.from_numpy(kb.sph_ptr).cuda(), torch.from_numpy(kb.sph_idx).cuda(),
                             torch.from_numpy(kb.beta).cuda(), torch.from_numpy(kb.D).cuda())
    ctx.sgw_set_td(1, rs)
    a = torch.from_numpy(psi).cuda()
    b = a.clone()
    ctx.sgw_apply_kick(b, torch.from_numpy(vpert).cuda(), lam)
    kick = oracle.apply_kick(psi, vpert, lam)
    assert relerr(b.cpu().numpy(), kick) < 1e-14
    out = ctx.sgw_td_propagate_pair(a, b, dt, nsteps, seed, nxi, nfrag).cpu().numpy()
    ra, rb, rout = oracle.td_pair(g, vloc, kbo, psi, kick, dt, nsteps, rs, seed, nxi, nfrag, ld=True)
    assert relerr(a.cpu().numpy(), ra) < TOL_FULL and relerr(b.cpu().numpy(), rb) < TOL_FULL
    scale = np.max(np.abs(rout))
    assert np.max(np.abs(out - rout)) < 1e-10 * scale
    ur, rur = (out[:, :, 1] - out[:, :, 0]) / lam, (rout[:, :, 1] - rout[:, :, 0]) / lam
    assert np.max(np.abs(ur[0])) < 1e-9 * scale / lam                    # no response at t = 0 (a pure phase kick)
    assert np.max(np.abs(ur - rur)) < 1e-6 * np.max(np.abs(rur))
    assert ctx.sgw_sync_check() == 0
    ctx.close()


@pytest.mark.parametrize("n,nvec,use_kb", [(32, 5, False), (48, 3, True), (64, 3, False), (96, 2, True)])
def test_tma_split_operator_kernel(api, torch_cuda, oracle, monkeypatch, n, nvec, use_kb):
    """The TMA split-operator kernel (sgw_acc.cuh: td_tma_kernel, one launch per axis: tile load, in-place round trip with
    the complex k table, bulk store; default from 256 points per axis) forced on for small cubic grids: frozen potential,
    Hartree rebuild with the density accumulated in the z launch, reverse time, and KB factors, against the oracle."""
    torch = torch_cuda
    monkeypatch.setenv("SGW_ACC_TD", "1")
    g = W.Grid(n, n, n, 0.5, 0.45, 0.55)
    rng = np.random.default_rng(5 * n)
    centers = rng.uniform(0, 1, size=(3, 3)) * np.array(g.box)
    vloc = W.gaussian_vloc(g, centers, [1.0, 2.0, 1.5], [0.9, 1.2, 0.8])
    kb = W.kb_projectors(g, centers[:2], radius=1.8, sigma=0.7) if use_kb else W.KB.empty()
    kbo = kb if kb.nsphere else None
    psi = rng.standard_normal((nvec,) + g.shape) + 1j * rng.standard_normal((nvec,) + g.shape)
    ctx = api.Context(g.nx, g.ny, g.nz, g.hx, g.hy, g.hz, nvec)
    ctx.sgw_set_vloc(torch.from_numpy(vloc).cuda())
    if kb.nsphere:
        ctx.sgw_set_nonlocal(torch.from_numpy(kb.sph_ptr).cuda(), torch.from_numpy(kb.sph_idx).cuda(),
                             torch.from_numpy(kb.beta).cuda(), torch.from_numpy(kb.D).cuda())
    rs = 2.0 / (nvec * g.dV) * 0.01
    for mode, dt, nsteps in ((0, 0.05, 1), (0, -0.05, 3), (1, 0.05, 4)):
        ctx.sgw_set_td(mode, rs)
        t = torch.from_numpy(psi).cuda()
        ctx.sgw_td_propagate(t, dt, nsteps)
        assert relerr(t.cpu().numpy(), oracle.td_propagate(g, vloc, kbo, psi, dt, nsteps, mode, rs, ld=True)) < TOL_FULL, (mode, dt)
    assert ctx.sgw_sync_check() == 0
    ctx.close()


@pytest.mark.parametrize("n", [256, 384])
def test_tma_kernels_at_256_and_384_agree_with_the_register_operand_passes(api, torch_cuda, monkeypatch, n):
    """256 and 384 points per axis are where the TMA kernels run in their warp-specialised layout (setmaxnreg: 16 warps,
    consumer warpgroups at 152 registers; three / two consumer groups), where the split-operator kernel is the default
    and, at 384, where the strided launches move tile pairs; the oracle reaches these sizes only on the golden samples
    (tests/test_gpu_golden.py: 2 vectors / 1 vector in the TD part).  Here 5 vectors -- not a multiple of the groups nor
    of the 4 vectors a KB block takes -- with KB spheres, 3 TD-Hartree steps (density summed per block in the z launch,
    sphere-point correction) and 3 filter applications are compared with the register-operand passes (SGW_ACC=0 /
    SGW_ACC_TD=0), which the oracle pins on the small grids and on every golden config."""
    torch = torch_cuda
    nvec = 5
    g = W.Grid(n, n, n, 0.5, 0.5, 0.5)
    rng = np.random.default_rng(77)
    centers = rng.uniform(0.2, 0.8, size=(6, 3)) * np.array(g.box)
    vloc = W.gaussian_vloc(g, centers, [1.0, 2.0, 1.5, 0.7, 1.1, 1.9], [0.9, 1.2, 0.8, 1.0, 1.4, 0.7])
    kb = W.kb_projectors(g, centers[:4], radius=2.4, sigma=0.8)
    coeffs = np.array([0.3, -0.2, 0.15, 0.1])
    rs = 2.0 / (nvec * g.dV) * 0.01
    out = {}
    for tag, acc in (("tma", "1"), ("lean", "0")):
        monkeypatch.setenv("SGW_ACC", acc)
        monkeypatch.setenv("SGW_ACC_TD", acc)
        ctx = api.Context(g.nx, g.ny, g.nz, g.hx, g.hy, g.hz, nvec)
        ctx.sgw_set_vloc(torch.from_numpy(vloc).cuda())
        ctx.sgw_set_nonlocal(torch.from_numpy(kb.sph_ptr).cuda(), torch.from_numpy(kb.sph_idx).cuda(),
                             torch.from_numpy(kb.beta).cuda(), torch.from_numpy(kb.D).cuda())
        psi = ctx.sgw_random_vectors(W.SEED_VEC, 3, nvec)
        ctx.sgw_cheb_filter(psi, coeffs, -1.0, 45.0)
        filt = psi.clone()
        ctx.sgw_set_td(1, rs)
        ctx.sgw_td_propagate(psi, 0.05, 3)
        assert ctx.sgw_sync_check() == 0
        out[tag] = (filt.cpu().numpy(), psi.cpu().numpy())
        ctx.close()
        del psi, filt
        torch.cuda.empty_cache()
    assert relerr(out["tma"][0], out["lean"][0]) < 1e-11
    assert relerr(out["tma"][1], out["lean"][1]) < 1e-10


def test_zeta_pair_time_ordering_and_sigma(api, torch_cuda, oracle):
    """NEXT-4: the zeta pair (backward / forward under the frozen potential) with its
    phi-weighted xi projections, the time-ordering of retarded coefficient series (a length that is no FFT length: 50),
    and the Sigma(t) contraction of Eq. 5 in the xi basis, against the oracle and numpy."""
    torch = torch_cuda
    n = 32
    g = W.Grid(n, n, n, 0.5, 0.5, 0.5)
    rng = np.random.default_rng(8)
    centers = rng.uniform(0, 1, size=(3, 3)) * np.array(g.box)
    vloc = W.gaussian_vloc(g, centers, [1.0, 2.0, 1.5], [0.9, 1.2, 0.8])
    kb = W.kb_projectors(g, centers[:2], radius=1.8, sigma=0.7)
    zbar = rng.standard_normal(g.shape) + 0j
    occ = 0.5 * zbar + 0.2 * (rng.standard_normal(g.shape) + 1j * rng.standard_normal(g.shape))
    pair = np.stack([occ, zbar - occ])
    phi = rng.standard_normal(g.shape)
    dt, nsteps, seed, nxi, nfrag = 0.05, 5, 123, 11, 4
    ctx = api.Context(g.nx, g.ny, g.nz, g.hx, g.hy, g.hz, 2)
    ctx.sgw_set_vloc(torch.from_numpy(vloc).cuda())
    ctx.sgw_set_nonlocal(torch.from_numpy(kb.sph_ptr).cuda(), torch.from_numpy(kb.sph_idx).cuda(),
                         torch.from_numpy(kb.beta).cuda(), torch.from_numpy(kb.D).cuda())
    ctx.sgw_set_td(1, 0.3)                                  # the zeta call must ignore the Hartree mode (frozen potential)
    t = torch.from_numpy(pair).cuda()
    p = ctx.sgw_td_propagate_zeta(t, torch.from_numpy(phi).cuda(), dt, nsteps, seed, nxi, nfrag)
    rpair, rp = oracle.td_zeta(g, vloc, kb, pair, phi, dt, nsteps, seed, nxi, nfrag, ld=True)
    assert relerr(t.cpu().numpy(), rpair) < TOL_FULL
    assert np.max(np.abs(p.cpu().numpy() - rp)) < 1e-10 * np.max(np.abs(rp))
    nt = 50
    cr = rng.standard_normal((nt, nxi, 2))
    crd = torch.from_numpy(cr).cuda()
    ur = crd[:, :, 1]                                       # strided view, as the pair call's output is used
    ct = ctx.sgw_time_order(ur)
    want = oracle.time_order(cr[:, :, 1], ld=True)
    assert np.max(np.abs(ct.cpu().numpy() - want)) < 1e-12 * np.max(np.abs(want)) * nt
    ctn = torch.from_numpy(want[:nsteps].copy()).cuda()
    sig = ctx.sgw_sigma_t(ctn, p, nfrag).cpu().numpy()
    ref = g.ng / (nxi * nfrag * 32 * g.dV) * np.einsum("nm,nmk->nk", want[:nsteps], rp)
    assert np.max(np.abs(sig - ref)) < 1e-10 * np.max(np.abs(ref))
    assert ctx.sgw_sync_check() == 0
    ctx.close()


def test_cfg2_full_length_propagation_invariants(api, torch_cuda):
    """cfg2 at full size and full length (16 vectors, 2000 steps, dt = 0.05): properties that hold at any length.
    With the Hartree term rebuilt every step the propagator stays unitary (norms conserved); with a frozen potential
    it is also exactly reversible (2000 steps forward, 2000 steps back)."""
    torch = torch_cuda
    w = W.make_workload("cfg2", nterms=17)
    ctx = api.context_for(w)
    psi = ctx.sgw_random_vectors(W.SEED_VEC, 0, w.nvec)
    ctx.sgw_cheb_filter(psi, w.coeffs, w.emin, w.emax)
    start = psi.clone()
    n0 = ctx.sgw_norms(psi)
    ctx.sgw_set_td(1, w.rho_scale)
    ctx.sgw_td_propagate(psi, w.dt, w.td_steps)
    assert w.td_steps == 2000
    drift = (ctx.sgw_norms(psi) / n0 - 1.0).abs().max()
    assert float(drift) < 1e-10
    assert float((psi - start).abs().max()) > 1e-3          # it did move
    psi.copy_(start)
    ctx.sgw_set_td(0, 0.0)
    ctx.sgw_td_propagate(psi, w.dt, 2000)
    ctx.sgw_td_propagate(psi, -w.dt, 2000)
    err = torch.linalg.vector_norm((psi - start).reshape(w.nvec, -1), dim=1) / torch.linalg.vector_norm(start.reshape(w.nvec, -1), dim=1)
    assert float(err.max()) < 1e-9
    assert ctx.sgw_sync_check() == 0
    ctx.close()
