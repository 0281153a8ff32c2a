"""Thin Python binding of libsgw (include/sgw.h): argument marshalling only.

Every step of the path runs in the library's CUDA kernels.  PyTorch supplies device memory and the
stream.  The function names are the C ABI's.  There is no fallback: if libsgw.so is missing or
there is no CUDA device the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("SGW_LIB", os.path.join(_HERE, "libsgw.so"))
_lib = None

ERRORS = {-1: "SGW_EINVAL", -2: "SGW_ESIZE", -3: "SGW_ENOMEM", -4: "SGW_ECUDA"}
EXPORTS = ["sgw_init_grid", "sgw_destroy", "sgw_set_vloc", "sgw_set_nonlocal", "sgw_random_vectors",
           "sgw_apply_H", "sgw_cheb_filter", "sgw_hartree", "sgw_set_td", "sgw_td_propagate", "sgw_norms",
           "sgw_launch_count", "sgw_last_error", "sgw_sync_check", "sgw_spectral_bounds", "sgw_profile_enable", "sgw_profile_reset", "sgw_profile_get",
           "sgw_probe_fp64", "sgw_set_kinetic_cutoff", "sgw_apply_kick",
           "sgw_td_propagate_pair", "sgw_td_propagate_zeta", "sgw_time_order", "sgw_sigma_t",
           "sgw_hartree_static", "sgw_static_setup", "sgw_static_max_grid_points"]


class SGWError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"{ERRORS.get(code, code)}: {msg}")
        self.code = code


def load():
    """dlopen libsgw.so (built by paper_2601_21005_b200.build); fails loudly if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise FileNotFoundError(f"{LIB_PATH} not built: run python -m paper_2601_21005_b200.build")
        lib = C.CDLL(LIB_PATH)
        vp, i, d, u64, i64 = C.c_void_p, C.c_int, C.c_double, C.c_uint64, C.c_int64
        lib.sgw_init_grid.argtypes = [C.POINTER(vp), i, i, i, d, d, d, i, vp]
        lib.sgw_destroy.argtypes = [vp]
        lib.sgw_set_vloc.argtypes = [vp, vp]
        lib.sgw_set_nonlocal.argtypes = [vp, i, vp, vp, i, vp, vp]
        lib.sgw_random_vectors.argtypes = [vp, u64, i, i, vp]
        lib.sgw_apply_H.argtypes = [vp, i, vp, vp]
        lib.sgw_cheb_filter.argtypes = [vp, i, vp, C.POINTER(d), d, d, i]
        lib.sgw_hartree.argtypes = [vp, i, vp, d, vp, vp]
        lib.sgw_hartree_static.argtypes = [vp, i, vp, d, vp, vp]
        lib.sgw_static_setup.argtypes = [vp]
        lib.sgw_static_max_grid_points.argtypes = []
        lib.sgw_static_max_grid_points.restype = i64
        lib.sgw_set_td.argtypes = [vp, i, d]
        lib.sgw_td_propagate.argtypes = [vp, i, vp, d, i]
        lib.sgw_norms.argtypes = [vp, i, vp, vp]
        lib.sgw_launch_count.argtypes = [vp]
        lib.sgw_sync_check.argtypes = [vp]
        lib.sgw_spectral_bounds.argtypes = [vp, i, u64, C.POINTER(d), C.POINTER(d)]
        lib.sgw_launch_count.restype = i64
        lib.sgw_last_error.restype = C.c_char_p
        lib.sgw_profile_enable.argtypes = [vp, i]
        lib.sgw_profile_reset.argtypes = [vp]
        lib.sgw_profile_get.argtypes = [vp, i, i, C.POINTER(i64), C.POINTER(d)]
        lib.sgw_probe_fp64.argtypes = [vp, C.POINTER(d)]
        lib.sgw_set_kinetic_cutoff.argtypes = [vp, d]
        lib.sgw_apply_kick.argtypes = [vp, i, vp, vp, d]
        lib.sgw_td_propagate_pair.argtypes = [vp, i, vp, vp, d, i, u64, i, i, vp]
        lib.sgw_td_propagate_zeta.argtypes = [vp, vp, vp, d, i, u64, i, i, vp]
        lib.sgw_time_order.argtypes = [vp, i, i, vp, i64, i64, vp]
        lib.sgw_sigma_t.argtypes = [vp, i, i, i, vp, vp, vp]
        _lib = lib
    return _lib


def _check(rc):
    if rc != 0:
        raise SGWError(rc, load().sgw_last_error().decode())


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def _cvec(t, ng):
    if t.dtype != torch.complex128 or not t.is_cuda or not t.is_contiguous():
        raise TypeError("vectors must be contiguous CUDA complex128 tensors")
    if t.numel() % ng:
        raise ValueError("vector batch size is not a multiple of the grid size")
    return t.numel() // ng


def _real(t, n):
    if t.dtype != torch.float64 or not t.is_cuda or not t.is_contiguous() or t.numel() != n:
        raise TypeError("real fields must be contiguous CUDA float64 tensors of N_g elements")


class Context:
    """Owns one sgw_ctx.  Methods mirror the C entry points one to one."""

    def __init__(self, nx, ny, nz, hx, hy, hz, max_nvec, stream=None, device="cuda:0"):
        self.lib = load()
        self.device = torch.device(device)
        self.shape = (nz, ny, nx)
        self.ng = nx * ny * nz
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self._h = C.c_void_p()
        with torch.cuda.device(self.device):
            _check(self.lib.sgw_init_grid(C.byref(self._h), nx, ny, nz, hx, hy, hz, max_nvec,
                                          C.c_void_p(self.stream.cuda_stream)))

    def close(self):
        if self._h:
            self.lib.sgw_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def sgw_set_vloc(self, vloc):
        if vloc is not None:
            _real(vloc, self.ng)
        _check(self.lib.sgw_set_vloc(self._h, _ptr(vloc)))

    def sgw_set_nonlocal(self, sph_ptr, sph_idx, beta, D):
        if sph_ptr is None or sph_ptr.numel() <= 1:
            _check(self.lib.sgw_set_nonlocal(self._h, 0, None, None, 4, None, None))
            return
        assert sph_ptr.dtype == torch.int64 and sph_idx.dtype == torch.int32
        assert beta.dtype == torch.float64 and D.dtype == torch.float64
        assert all(t.is_cuda and t.is_contiguous() for t in (sph_ptr, sph_idx, beta, D))
        nsphere, nproj = D.shape
        _check(self.lib.sgw_set_nonlocal(self._h, nsphere, _ptr(sph_ptr), _ptr(sph_idx), nproj, _ptr(beta), _ptr(D)))

    def sgw_random_vectors(self, seed, first_vec, nvec, out=None):
        if out is None:
            out = torch.empty((nvec,) + self.shape, dtype=torch.complex128, device=self.device)
        assert _cvec(out, self.ng) >= nvec
        _check(self.lib.sgw_random_vectors(self._h, seed, first_vec, nvec, _ptr(out)))
        return out

    def sgw_apply_H(self, psi, out=None):
        nvec = _cvec(psi, self.ng)
        if out is None:
            out = torch.empty_like(psi)
        assert _cvec(out, self.ng) == nvec
        _check(self.lib.sgw_apply_H(self._h, nvec, _ptr(psi), _ptr(out)))
        return out

    def sgw_cheb_filter(self, psi, coeffs, emin, emax):
        nvec = _cvec(psi, self.ng)
        co = np.ascontiguousarray(coeffs, dtype=np.float64)
        _check(self.lib.sgw_cheb_filter(self._h, nvec, _ptr(psi), co.ctypes.data_as(C.POINTER(C.c_double)),
                                        float(emin), float(emax), int(co.size)))
        return psi

    def sgw_hartree(self, psi, rho_scale, want_rho=False):
        nvec = _cvec(psi, self.ng)
        vh = torch.empty(self.shape, dtype=torch.float64, device=self.device)
        rho = torch.empty(self.shape, dtype=torch.float64, device=self.device) if want_rho else None
        _check(self.lib.sgw_hartree(self._h, nvec, _ptr(psi), float(rho_scale), _ptr(vh), _ptr(rho)))
        return (vh, rho) if want_rho else vh

    def sgw_hartree_static(self, psi, rho_scale, vh, rho=None):
        """sgw_hartree with the solve's scratch in the library's static device array; the caller passes the outputs."""
        nvec = _cvec(psi, self.ng)
        _check(self.lib.sgw_hartree_static(self._h, nvec, _ptr(psi), float(rho_scale), _ptr(vh), _ptr(rho)))
        return vh

    def sgw_static_setup(self):
        _check(self.lib.sgw_static_setup(self._h))

    def sgw_static_max_grid_points(self):
        return int(self.lib.sgw_static_max_grid_points())

    def sgw_set_td(self, hartree_mode, rho_scale):
        _check(self.lib.sgw_set_td(self._h, int(hartree_mode), float(rho_scale)))

    def sgw_td_propagate(self, psi, dt, nsteps):
        nvec = _cvec(psi, self.ng)
        _check(self.lib.sgw_td_propagate(self._h, nvec, _ptr(psi), float(dt), int(nsteps)))
        return psi

    def sgw_norms(self, psi):
        nvec = _cvec(psi, self.ng)
        out = torch.empty(nvec, dtype=torch.float64, device=self.device)
        _check(self.lib.sgw_norms(self._h, nvec, _ptr(psi), _ptr(out)))
        return out

    def sgw_profile_enable(self, on):
        _check(self.lib.sgw_profile_enable(self._h, int(on)))

    def sgw_profile_reset(self):
        _check(self.lib.sgw_profile_reset(self._h))

    def sgw_profile_get(self, axis, kind):
        n, ms = C.c_int64(), C.c_double()
        _check(self.lib.sgw_profile_get(self._h, axis, kind, C.byref(n), C.byref(ms)))
        return n.value, ms.value

    def sgw_apply_kick(self, psi, vpert, lam):
        nvec = _cvec(psi, self.ng)
        _real(vpert, self.ng)
        _check(self.lib.sgw_apply_kick(self._h, nvec, _ptr(psi), _ptr(vpert), float(lam)))
        return psi

    def sgw_td_propagate_pair(self, psi, psi_lam, dt, nsteps, xi_seed, nxi, nfrag):
        nvec = _cvec(psi, self.ng)
        assert _cvec(psi_lam, self.ng) == nvec
        out = torch.empty((nsteps, nxi, 2), dtype=torch.float64, device=self.device)
        _check(self.lib.sgw_td_propagate_pair(self._h, nvec, _ptr(psi), _ptr(psi_lam), float(dt), int(nsteps), int(xi_seed),
                                              int(nxi), int(nfrag), _ptr(out)))
        return out

    def sgw_td_propagate_zeta(self, pair, phi, dt, nsteps, xi_seed, nxi, nfrag):
        assert _cvec(pair, self.ng) == 2
        _real(phi, self.ng)
        out = torch.empty((nsteps, nxi, 2), dtype=torch.complex128, device=self.device)
        _check(self.lib.sgw_td_propagate_zeta(self._h, _ptr(pair), _ptr(phi), float(dt), int(nsteps), int(xi_seed), int(nxi),
                                              int(nfrag), _ptr(out)))
        return out

    def sgw_time_order(self, cr):
        """cr: [nt, nxi] float64 CUDA tensor (any strides) -> [nt, nxi] complex128."""
        assert cr.dtype == torch.float64 and cr.is_cuda and cr.dim() == 2
        nt, nxi = cr.shape
        ct = torch.empty((nt, nxi), dtype=torch.complex128, device=self.device)
        _check(self.lib.sgw_time_order(self._h, nxi, nt, _ptr(cr), cr.stride(0), cr.stride(1), _ptr(ct)))
        return ct

    def sgw_sigma_t(self, ct, p, nfrag):
        nt, nxi = ct.shape
        assert p.shape == (nt, nxi, 2) and ct.is_contiguous() and p.is_contiguous()
        sig = torch.empty((nt, 2), dtype=torch.complex128, device=self.device)
        _check(self.lib.sgw_sigma_t(self._h, nt, nxi, int(nfrag), _ptr(ct), _ptr(p), _ptr(sig)))
        return sig

    def sgw_set_kinetic_cutoff(self, ecut):
        _check(self.lib.sgw_set_kinetic_cutoff(self._h, float(ecut)))

    def sgw_probe_fp64(self):
        r = C.c_double()
        _check(self.lib.sgw_probe_fp64(self._h, C.byref(r)))
        return r.value

    def sgw_spectral_bounds(self, niter, seed):
        emin, emax = C.c_double(), C.c_double()
        _check(self.lib.sgw_spectral_bounds(self._h, int(niter), int(seed), C.byref(emin), C.byref(emax)))
        return emin.value, emax.value

    def sgw_sync_check(self):
        _check(self.lib.sgw_sync_check(self._h))
        return 0

    def sgw_launch_count(self):
        return int(self.lib.sgw_launch_count(self._h))


def context_for(workload, max_nvec=None, stream=None, device="cuda:0") -> Context:
    """Context with the workload's potentials uploaded (workload: paper_2601_21005_b200.workloads.Workload)."""
    g = workload.grid
    ctx = Context(g.nx, g.ny, g.nz, g.hx, g.hy, g.hz, max_nvec or max(1, workload.nvec), stream, device)
    dev = ctx.device
    ctx.sgw_set_vloc(torch.from_numpy(workload.vloc).to(dev))
    kb = workload.kb
    if kb.nsphere:
        ctx.sgw_set_nonlocal(torch.from_numpy(kb.sph_ptr).to(dev), torch.from_numpy(kb.sph_idx).to(dev),
                             torch.from_numpy(kb.beta).to(dev), torch.from_numpy(kb.D).to(dev))
    return ctx
