"""ctypes loader for the CPU oracle (oracle/sgw_oracle.cpp).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this module.  It imports nothing from the CUDA package.  All arrays are NumPy, host memory;
complex vectors are complex128 with shape [nvec, nz, ny, nx].
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sgw_oracle.cpp")
_LIB = os.path.join(_HERE, "libsgw_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (no fast-math, no FMA contraction: DESIGN.md reading R-17)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off", "-fcx-limited-range",
               "-o", _LIB, _SRC]
        subprocess.check_call(cmd)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.sgwo_hash.restype = C.c_uint64
        _lib.sgwo_hash.argtypes = [C.c_uint64] * 3
        _lib.sgwo_splitmix64_next.restype = C.c_uint64
        _lib.sgwo_splitmix64_next.argtypes = [C.POINTER(C.c_uint64)]
        _lib.sgwo_max_threads.restype = C.c_int
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _grid_args(grid):
    return [C.c_int(grid.nx), C.c_int(grid.ny), C.c_int(grid.nz),
            C.c_double(grid.hx), C.c_double(grid.hy), C.c_double(grid.hz)]


def _kb_args(kb):
    if kb is None or kb.nsphere == 0:
        return [C.c_int(0), None, None, C.c_int(4), None, None], ()
    keep = (np.ascontiguousarray(kb.sph_ptr, np.int64), np.ascontiguousarray(kb.sph_idx, np.int32),
            np.ascontiguousarray(kb.beta, np.float64), np.ascontiguousarray(kb.D, np.float64))
    return [C.c_int(kb.nsphere), _p(keep[0]), _p(keep[1]), C.c_int(kb.nproj), _p(keep[2]), _p(keep[3])], keep


def _vec(a):
    return np.ascontiguousarray(a, dtype=np.complex128)


def set_kinetic_cutoff(ecut: float):
    """Kinetic operator min(1/2 k^2, ecut) in H and the propagator (0 = off, the default)."""
    lib().sgwo_set_kinetic_cutoff(C.c_double(ecut))


def set_threads(n: int):
    lib().sgwo_set_threads(C.c_int(n))


def max_threads() -> int:
    return lib().sgwo_max_threads()


def splitmix64_stream(state0: int, n: int):
    st = C.c_uint64(state0)
    return [lib().sgwo_splitmix64_next(C.byref(st)) for _ in range(n)]


def keyed_hash(seed: int, vec: int, g: int) -> int:
    return lib().sgwo_hash(seed, vec, g)


def random_vectors(grid, seed: int, first_vec: int, nvec: int):
    out = np.empty((nvec,) + grid.shape, np.complex128)
    lib().sgwo_random_vectors(C.c_uint64(seed), C.c_int(first_vec), C.c_int(nvec), C.c_int64(grid.ng), _p(out))
    return out


def fft1d(x, sign: int, ld: bool = False):
    x = _vec(x)
    out = np.empty_like(x)
    lib().sgwo_fft1d(C.c_int(x.size), C.c_int(sign), _p(x), _p(out), C.c_int(int(ld)))
    return out


def fft3(a, sign: int, ld: bool = False):
    """Unnormalised 3D DFT of a[nz,ny,nx]; sign=-1 forward, +1 inverse (no 1/N)."""
    a = _vec(a).copy()
    nz, ny, nx = a.shape
    lib().sgwo_fft3(C.c_int(nx), C.c_int(ny), C.c_int(nz), C.c_int(sign), _p(a), C.c_int(int(ld)))
    return a


def apply_H(grid, vloc, kb, psi, ld: bool = False):
    psi = _vec(psi)
    out = np.empty_like(psi)
    kba, keep = _kb_args(kb)
    v = None if vloc is None else np.ascontiguousarray(vloc, np.float64)
    lib().sgwo_apply_H(*_grid_args(grid), _p(v), *kba, C.c_int(psi.shape[0]), _p(psi), _p(out), C.c_int(int(ld)))
    return out


def cheb_filter(grid, vloc, kb, psi, coeffs, emin, emax, ld: bool = False):
    psi = _vec(psi).copy()
    kba, keep = _kb_args(kb)
    v = None if vloc is None else np.ascontiguousarray(vloc, np.float64)
    co = np.ascontiguousarray(coeffs, np.float64)
    lib().sgwo_cheb_filter(*_grid_args(grid), _p(v), *kba, C.c_int(psi.shape[0]), _p(psi), _p(co),
                           C.c_double(emin), C.c_double(emax), C.c_int(len(co)), C.c_int(int(ld)))
    return psi


def hartree(grid, psi, rho_scale, ld: bool = False):
    psi = _vec(psi)
    vh = np.empty(grid.shape, np.float64)
    rho = np.empty(grid.shape, np.float64)
    lib().sgwo_hartree(*_grid_args(grid), C.c_int(psi.shape[0]), _p(psi), C.c_double(rho_scale), _p(vh), _p(rho),
                       C.c_int(int(ld)))
    return vh, rho


def poisson(grid, rho, ld: bool = False):
    rho = np.ascontiguousarray(rho, np.float64)
    vh = np.empty(grid.shape, np.float64)
    lib().sgwo_poisson(*_grid_args(grid), _p(rho), _p(vh), C.c_int(int(ld)))
    return vh


def td_propagate(grid, vloc, kb, psi, dt, nsteps, hartree_mode=0, rho_scale=0.0, ld: bool = False):
    psi = _vec(psi).copy()
    kba, keep = _kb_args(kb)
    v = None if vloc is None else np.ascontiguousarray(vloc, np.float64)
    lib().sgwo_td_propagate(*_grid_args(grid), _p(v), *kba, C.c_int(psi.shape[0]), _p(psi), C.c_double(dt),
                            C.c_int(nsteps), C.c_int(hartree_mode), C.c_double(rho_scale), C.c_int(int(ld)))
    return psi


def spectral_bounds(grid, vloc, kb, niter, seed, ld: bool = False):
    """Shifted power iteration (R-20): returns (E_min, E_max) estimates."""
    kba, keep = _kb_args(kb)
    v = None if vloc is None else np.ascontiguousarray(vloc, np.float64)
    emin, emax = C.c_double(), C.c_double()
    lib().sgwo_spectral_bounds(*_grid_args(grid), _p(v), *kba, C.c_int(niter), C.c_uint64(seed), C.byref(emin),
                               C.byref(emax), C.c_int(int(ld)))
    return emin.value, emax.value


def norms(psi):
    psi = _vec(psi)
    out = np.empty(psi.shape[0], np.float64)
    ng = psi[0].size
    lib().sgwo_norms(C.c_int64(ng), C.c_int(psi.shape[0]), _p(psi), _p(out))
    return out


def apply_kick(psi, vpert, lam):
    """Perturbed copy exp(-i lam v_pert) psi (R-21)."""
    psi = _vec(psi).copy()
    vp = np.ascontiguousarray(vpert, np.float64)
    lib().sgwo_apply_kick(C.c_int64(psi[0].size), C.c_int(psi.shape[0]), _p(psi), _p(vp), C.c_double(lam))
    return psi


def td_pair(grid, vloc, kb, psi, psi_lam, dt, nsteps, rho_scale, xi_seed, nxi, nfrag, ld: bool = False):
    """Pair propagation with the xi projections of both Hartree potentials at the start of every step
    (R-21..R-23).  Returns (psi, psi_lam, out[nsteps, nxi, 2])."""
    a, b = _vec(psi).copy(), _vec(psi_lam).copy()
    kba, keep = _kb_args(kb)
    v = None if vloc is None else np.ascontiguousarray(vloc, np.float64)
    out = np.zeros((nsteps, nxi, 2), np.float64)
    lib().sgwo_td_pair(*_grid_args(grid), _p(v), *kba, C.c_int(a.shape[0]), _p(a), _p(b), C.c_double(dt), C.c_int(nsteps),
                       C.c_double(rho_scale), C.c_uint64(xi_seed), C.c_int(nxi), C.c_int(nfrag), _p(out), C.c_int(int(ld)))
    return a, b, out


def time_order(cr, ld: bool = False):
    """Time-ordering of retarded coefficient series cr[nt, nxi] (real) -> ct[nt, nxi] (complex); R-24."""
    cr = np.ascontiguousarray(cr, np.float64)
    nt, nxi = cr.shape
    ct = np.zeros((nt, nxi), np.complex128)
    lib().sgwo_time_order(C.c_int(nxi), C.c_int(nt), _p(cr), C.c_int(nxi), C.c_int(1), _p(ct), C.c_int(int(ld)))
    return ct


def td_zeta(grid, vloc, kb, pair, phi, dt, nsteps, xi_seed, nxi, nfrag, ld: bool = False):
    """zeta pair (pair[0] backwards, pair[1] forwards, frozen V_loc) with the phi-weighted xi projections at the start of
    every step (Eq. 5; R-25).  Returns (pair, p[nsteps, nxi, 2] complex)."""
    pair = _vec(pair).copy()
    assert pair.shape[0] == 2
    kba, keep = _kb_args(kb)
    v = None if vloc is None else np.ascontiguousarray(vloc, np.float64)
    ph = np.ascontiguousarray(phi, np.float64)
    out = np.zeros((nsteps, nxi, 2), np.complex128)
    lib().sgwo_td_zeta(*_grid_args(grid), _p(v), *kba, _p(pair), _p(ph), C.c_double(dt), C.c_int(nsteps), C.c_uint64(xi_seed),
                       C.c_int(nxi), C.c_int(nfrag), _p(out), C.c_int(int(ld)))
    return pair, out
