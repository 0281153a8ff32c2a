"""Writes the config-scale golden samples tests/golden/cfg*_*.txt from the ORACLE ALONE.

    python tests/golden/make_config_golden.py cfg1 | cfg2 | cfg3 | cfg4 | all

Imports only `oracle/` (long-double instantiation, reading R-17) and the shared input generators
`paper_2601_21005_b200/workloads.py`; nothing here touches the CUDA path.  Each file holds, for a declared set of
vectors of a BASELINE.json config, the oracle's result at a strided sample of grid points (flat index g = k * stride,
stride prime, so every x, y and z residue is visited) plus the full-grid sum |psi|^2 of every compared vector, after

  cfg1  all 512 Chebyshev terms (511 H applications), vectors 0 / 37 / 63 of the 64-vector batch       (Eq. 3)
  cfg2  the 9-term filter, then 200 split-operator steps with the Hartree rebuild, all 16 vectors
  cfg3  the first 65 of the 2048 coefficients (64 H applications) with KB projectors, vectors 100 / 101; then 20
        TD-Hartree steps of those two vectors (rho_scale for a 2-vector batch)
  cfg4  the first 17 of the 2048 coefficients (16 H applications) with KB projectors, vector 31; then 5 TD-Hartree
        steps of that vector (rho_scale for a 1-vector batch)

File format: '#' header lines (what, citation, stride, count, norms), then one row per sample:
    <vector id> <flat grid index> <re> <im>        (%.17e: exact round trip of the doubles the oracle returns)
"""
from __future__ import annotations

import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))
from oracle import sgw_oracle as o  # noqa: E402
from paper_2601_21005_b200 import workloads as W  # noqa: E402

TARGET_SAMPLES = 2048


def _is_prime(n):
    if n < 2:
        return False
    i = 2
    while i * i <= n:
        if n % i == 0:
            return False
        i += 1
    return True


def sample_stride(ng: int) -> int:
    """smallest prime >= ng / TARGET_SAMPLES"""
    s = max(2, ng // TARGET_SAMPLES)
    while not _is_prime(s):
        s += 1
    return s


def write_golden(name, what, grid, vec_ids, psi):
    ng = grid.ng
    stride = sample_stride(ng)
    idx = np.arange(0, ng, stride)
    flat = psi.reshape(psi.shape[0], -1)
    path = os.path.join(HERE, name)
    with open(path, "w") as f:
        f.write(f"# {what}\n")
        f.write("# written by tests/golden/make_config_golden.py from oracle/ (long double) only\n")
        f.write(f"# grid {grid.nx} {grid.ny} {grid.nz} stride {stride} count {len(idx)}\n")
        for j, v in enumerate(vec_ids):
            n2 = float(np.sum(flat[j].real.astype(np.longdouble) ** 2 + flat[j].imag.astype(np.longdouble) ** 2))
            f.write(f"# norm2 {v} {n2:.17e}\n")
        for j, v in enumerate(vec_ids):
            for g in idx:
                z = flat[j, g]
                f.write(f"{v} {g} {z.real:.17e} {z.imag:.17e}\n")
    print(f"wrote {path}: {len(vec_ids)} vectors x {len(idx)} samples", flush=True)


def cfg1():
    w = W.make_workload("cfg1")
    pick = [0, 37, 63]
    psi = np.concatenate([o.random_vectors(w.grid, W.SEED_VEC, v, 1) for v in pick])
    out = o.cheb_filter(w.grid, w.vloc, None, psi, w.coeffs, w.emin, w.emax, ld=True)
    write_golden("cfg1_filter512.txt",
                 "cfg1 (BASELINE.json configs[1]): 96^3 h=0.45 Si35H36 V_loc, all 512 Chebyshev terms (P:49-53 Eq. 3; R-1), "
                 "vectors 0/37/63 (seed 20260121)", w.grid, pick, out)


def cfg2():
    w = W.make_workload("cfg2", nterms=9)
    ids = list(range(w.nvec))
    psi = o.random_vectors(w.grid, W.SEED_VEC, 0, w.nvec)
    psi = o.cheb_filter(w.grid, w.vloc, None, psi, w.coeffs, w.emin, w.emax, ld=True)
    write_golden("cfg2_filter9.txt",
                 "cfg2 (BASELINE.json configs[2]): 128^3 h=0.5 Si87H76 V_loc, 16 vectors after the 9-term filter "
                 "(workloads.make_workload('cfg2', nterms=9))", w.grid, ids, psi)
    psi = o.td_propagate(w.grid, w.vloc, None, psi, w.dt, 200, 1, w.rho_scale, ld=True)
    write_golden("cfg2_td200.txt",
                 "cfg2: the same 16 vectors after 200 split-operator steps dt=0.05 with the Hartree potential rebuilt every "
                 "step from all 16 vectors (P:57, P:84, P:155; R-8, R-9, R-10), rho_scale = 2/(16 dV)", w.grid, ids, psi)


def cfg3():
    w = W.make_workload("cfg3")
    pick = [100, 101]
    psi = o.random_vectors(w.grid, W.SEED_VEC, 100, 2)
    coeffs = np.ascontiguousarray(w.coeffs[:65])
    psi = o.cheb_filter(w.grid, w.vloc, w.kb, psi, coeffs, w.emin, w.emax, ld=True)
    write_golden("cfg3_filter65.txt",
                 "cfg3 (BASELINE.json configs[3]): 256^3 h=0.5 Si705H300 V_loc + 705 KB spheres (P:177; R-12), first 65 of the "
                 "2048 coefficients (64 H applications), vectors 100/101", w.grid, pick, psi)
    rho_scale = 2.0 / (2 * w.grid.dV)
    psi = o.td_propagate(w.grid, w.vloc, w.kb, psi, w.dt, 20, 1, rho_scale, ld=True)
    write_golden("cfg3_td20.txt",
                 "cfg3: the two filtered vectors after 20 split-operator steps dt=0.05 with KB factors (R-11) and the Hartree "
                 "rebuild from these 2 vectors, rho_scale = 2/(2 dV)", w.grid, pick, psi)


def cfg4():
    w = W.make_workload("cfg4")
    pick = [31]
    psi = o.random_vectors(w.grid, W.SEED_VEC, 31, 1)
    coeffs = np.ascontiguousarray(w.coeffs[:17])
    psi = o.cheb_filter(w.grid, w.vloc, w.kb, psi, coeffs, w.emin, w.emax, ld=True)
    write_golden("cfg4_filter17.txt",
                 "cfg4 (BASELINE.json configs[4]): 384^3 h=0.6 Si8381H1620 V_loc + 8381 KB spheres, first 17 of the 2048 "
                 "coefficients (16 H applications), vector 31", w.grid, pick, psi)
    rho_scale = 2.0 / (1 * w.grid.dV)
    psi = o.td_propagate(w.grid, w.vloc, w.kb, psi, w.dt, 5, 1, rho_scale, ld=True)
    write_golden("cfg4_td5.txt",
                 "cfg4: the filtered vector after 5 split-operator steps dt=0.05 with KB factors and the Hartree rebuild from "
                 "this 1 vector, rho_scale = 2/(1 dV)", w.grid, pick, psi)


if __name__ == "__main__":
    which = sys.argv[1] if len(sys.argv) > 1 else "all"
    o.build()
    for name, fn in (("cfg1", cfg1), ("cfg2", cfg2), ("cfg3", cfg3), ("cfg4", cfg4)):
        if which in (name, "all"):
            t0 = time.time()
            fn()
            print(f"{name}: {time.time() - t0:.0f} s", flush=True)
