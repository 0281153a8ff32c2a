"""Config-scale parity against the oracle's committed golden samples (tests/golden/cfg*_*.txt).

The golden files are written by tests/golden/make_config_golden.py from the long-double oracle alone.  Each test
runs the library in the launch configuration bench.py uses for that config (full vector batch, default kernels, no
environment overrides) and compares, element by element, the sampled grid points of the declared vectors:
relative L2 error over the samples <= 1e-8 per vector (BASELINE.json north_star: "at most 1e-8 after a full filter
or propagation"), plus the full-grid sum |psi|^2 of each compared vector (a property of every element).

  cfg1  64-vector batch, ALL 512 terms; vectors 0 / 37 / 63
  cfg2  all 16 vectors, 9-term filter, then 200 of the 2000 TD-Hartree steps
  cfg3  64-vector sub-batch [64, 128), first 65 of the 2048 coefficients with KB; vectors 100 / 101; then 20
        TD-Hartree steps of those two vectors (complex family at 256^2 in its default launch configuration)
  cfg4  all 32 vectors in flight, first 17 of the 2048 coefficients with KB; vector 31; then 5 TD-Hartree steps of it
"""
import os

import numpy as np
import pytest

from paper_2601_21005_b200 import workloads as W

pytestmark = pytest.mark.gpu

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
TOL = 1e-8


def load_golden(name):
    path = os.path.join(GOLD, name)
    norms, meta = {}, {}
    with open(path) as f:
        for ln in f:
            if not ln.startswith("#"):
                break
            t = ln[1:].split()
            if t and t[0] == "norm2":
                norms[int(t[1])] = float(t[2])
            if t and t[0] == "grid":
                meta = {"grid": (int(t[1]), int(t[2]), int(t[3])), "stride": int(t[5]), "count": int(t[7])}
    rows = np.loadtxt(path, comments="#")
    vec = rows[:, 0].astype(np.int64)
    out = {}
    for v in np.unique(vec):
        m = vec == v
        out[int(v)] = (rows[m, 1].astype(np.int64), rows[m, 2] + 1j * rows[m, 3])
    assert all(len(ix) == meta["count"] for ix, _ in out.values())
    return out, norms, meta


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


def check(torch, ctx, psi, slot_of, golden, norms):
    """psi: device batch; slot_of[v] = index of global vector v inside psi."""
    n2 = ctx.sgw_norms(psi).cpu().numpy()
    for v, (idx, want) in golden.items():
        j = slot_of[v]
        got = psi[j].reshape(-1)[torch.from_numpy(idx).to(psi.device)].cpu().numpy()
        err = np.linalg.norm(got - want) / np.linalg.norm(want)
        assert err < TOL, (v, err)
        assert np.max(np.abs(got - want)) < TOL * np.max(np.abs(want)), v
        assert abs(n2[j] / norms[v] - 1.0) < 2 * TOL, (v, n2[j], norms[v])


def test_cfg1_full_length_filter_vs_golden(api, torch_cuda):
    torch = torch_cuda
    gold, norms, meta = load_golden("cfg1_filter512.txt")
    w = W.make_workload("cfg1")
    assert (w.grid.nx, w.grid.ny, w.grid.nz) == meta["grid"] and w.nterms == 512 and w.nvec == 64
    ctx = api.context_for(w)
    psi = ctx.sgw_random_vectors(W.SEED_VEC, 0, w.nvec)
    ctx.sgw_cheb_filter(psi, w.coeffs, w.emin, w.emax)
    check(torch, ctx, psi, {v: v for v in gold}, gold, norms)
    assert ctx.sgw_sync_check() == 0
    ctx.close()


def test_cfg2_filter_then_200_td_hartree_steps_vs_golden(api, torch_cuda):
    torch = torch_cuda
    gold_f, norms_f, meta = load_golden("cfg2_filter9.txt")
    gold_t, norms_t, _ = load_golden("cfg2_td200.txt")
    w = W.make_workload("cfg2", nterms=9)
    assert (w.grid.nx, w.grid.ny, w.grid.nz) == meta["grid"] and w.nvec == 16 and len(gold_t) == 16
    ctx = api.context_for(w)
    psi = ctx.sgw_random_vectors(W.SEED_VEC, 0, w.nvec)
    ctx.sgw_cheb_filter(psi, w.coeffs, w.emin, w.emax)
    check(torch, ctx, psi, {v: v for v in gold_f}, gold_f, norms_f)
    ctx.sgw_set_td(1, w.rho_scale)
    ctx.sgw_td_propagate(psi, w.dt, 120)
    ctx.sgw_td_propagate(psi, w.dt, 80)                     # two calls: the step sequence does not depend on the split
    check(torch, ctx, psi, {v: v for v in gold_t}, gold_t, norms_t)
    assert ctx.sgw_sync_check() == 0
    ctx.close()


def test_cfg3_filter_64_applications_and_20_td_steps_with_kb_vs_golden(api, torch_cuda):
    torch = torch_cuda
    gold_f, norms_f, meta = load_golden("cfg3_filter65.txt")
    gold_t, norms_t, _ = load_golden("cfg3_td20.txt")
    w = W.make_workload("cfg3")
    assert (w.grid.nx, w.grid.ny, w.grid.nz) == meta["grid"] and w.kb.nsphere == 705 and w.nterms == 2048
    ctx = api.context_for(w, max_nvec=64)                   # bench.py's sub-batch size for cfg3
    psi = ctx.sgw_random_vectors(W.SEED_VEC, 64, 64)        # global vectors 64..127
    ctx.sgw_cheb_filter(psi, w.coeffs[:65], w.emin, w.emax)
    check(torch, ctx, psi, {100: 36, 101: 37}, gold_f, norms_f)
    pair = psi[36:38].clone()
    del psi
    torch.cuda.empty_cache()
    ctx.sgw_set_td(1, 2.0 / (2 * w.grid.dV))
    ctx.sgw_td_propagate(pair, w.dt, 20)
    check(torch, ctx, pair, {100: 0, 101: 1}, gold_t, norms_t)
    assert ctx.sgw_sync_check() == 0
    ctx.close()


@pytest.mark.slow
def test_cfg4_filter_16_applications_and_5_td_steps_with_kb_vs_golden(api, torch_cuda):
    torch = torch_cuda
    gold_f, norms_f, meta = load_golden("cfg4_filter17.txt")
    gold_t, norms_t, _ = load_golden("cfg4_td5.txt")
    w = W.make_workload("cfg4")
    assert (w.grid.nx, w.grid.ny, w.grid.nz) == meta["grid"] and w.atoms == "Si8381H1620" and w.nvec == 32
    ctx = api.context_for(w)                                # all 32 vectors in flight
    psi = ctx.sgw_random_vectors(W.SEED_VEC, 0, w.nvec)
    ctx.sgw_cheb_filter(psi, w.coeffs[:17], w.emin, w.emax)
    check(torch, ctx, psi, {31: 31}, gold_f, norms_f)
    one = psi[31:32].clone()
    del psi
    torch.cuda.empty_cache()
    ctx.sgw_set_td(1, 2.0 / (1 * w.grid.dV))
    ctx.sgw_td_propagate(one, w.dt, 5)
    check(torch, ctx, one, {31: 0}, gold_t, norms_t)
    assert ctx.sgw_sync_check() == 0
    ctx.close()
