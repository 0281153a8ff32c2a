"""Seeded synthetic input generators for the sGW hot path (NumPy only).

This module builds *data* -- cluster geometries, the local potential V_loc(r), the sparse
Kleinman-Bylander sphere lists, Chebyshev coefficients, analytic spectral bounds -- that is handed
unchanged to BOTH the CPU oracle (``oracle/``) and the CUDA library.  It holds none of the method's
arithmetic (no FFT, no Hamiltonian apply, no recurrence, no propagator) and imports neither side.

The inputs stand in for the paper's Si_xH_y workloads ("Numerical Experiments":
spherical cuts of a diamond superlattice, a = 10.26 bohr, H-passivated); the real relaxed
geometries, RMG densities and Troullier-Martins pseudopotentials are not available, so the shapes
are kept and the potentials are Gaussians (BASELINE.json configs[0..4]; SURVEY.md section 8(c,d)).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

A_SI = 10.26          # bohr, diamond cubic cell
H_BOND = 2.8          # bohr, Si-H cap distance (BASELINE.json configs[1])
SEED_VEC = 20260121   # stochastic vectors
SEED_WELL = 20260122  # config-0 well positions
SEED_D = 20260123     # KB coefficients
MU = -0.2             # Ha   (BASELINE.json configs[0])
BETA = 50.0           # 1/Ha (BASELINE.json configs[0])
KB_RADIUS = 2.5       # bohr (BASELINE.json configs[3])
KB_SIGMA = 0.8        # bohr
DELTA_NL = 2.0        # Ha, spectral-bound padding when KB is present

_M64 = (1 << 64) - 1


# --------------------------------------------------------------------------------------------
# counter-based uniform numbers for the generators (positions, KB coefficients)
# --------------------------------------------------------------------------------------------
def _sm64(x: int) -> int:
    """splitmix64 output function on a Python int (mod 2^64)."""
    x = (x + 0x9E3779B97F4A7C15) & _M64
    x = ((x ^ (x >> 30)) * 0xBF58476D1CE4E5B9) & _M64
    x = ((x ^ (x >> 27)) * 0x94D049BB133111EB) & _M64
    return x ^ (x >> 31)


def hash_uniform(seed: int, vec: int, g: int) -> float:
    """u in [0,1): top 53 bits of the keyed hash of (seed, vec, g) (SURVEY.md 8(c) 'uniform')."""
    key = _sm64(_sm64(seed) ^ vec)
    h = _sm64(key ^ g)
    return (h >> 11) * 2.0 ** -53


# --------------------------------------------------------------------------------------------
# geometry: atom-centred spherical cut of the ideal diamond lattice, H-passivated
# --------------------------------------------------------------------------------------------
_FCC = [(0, 0, 0), (0, 2, 2), (2, 0, 2), (2, 2, 0)]          # units of a/4
_BONDS_A = [(1, 1, 1), (1, -1, -1), (-1, 1, -1), (-1, -1, 1)]  # from sublattice A to B


def diamond_cluster(r2_units: int):
    """Si and H positions (bohr, relative to the central Si atom).

    ``r2_units`` is the squared cut radius in units of (a/8)^2: keep lattice
    sites with |r|^2 <= r2_units (a/8)^2, remove in ONE pass the Si atoms left with <= 1 Si
    neighbour, then put one H at 2.8 bohr along every missing tetrahedral bond
    (BASELINE.json configs[1]).
    """
    r2 = r2_units / 4.0                       # in (a/4)^2
    m = int(math.isqrt(int(r2))) + 5
    sites = {}
    rng = range(-(m // 4) - 2, m // 4 + 3)
    for cx in rng:
        for cy in rng:
            for cz in rng:
                for f in _FCC:
                    for sub in (0, 1):
                        p = (4 * cx + f[0] + sub, 4 * cy + f[1] + sub, 4 * cz + f[2] + sub)
                        if p[0] * p[0] + p[1] * p[1] + p[2] * p[2] <= r2:
                            sites[p] = sub

    def bonds(sub):
        return _BONDS_A if sub == 0 else [(-b[0], -b[1], -b[2]) for b in _BONDS_A]

    def nneigh(p, table):
        return sum(((p[0] + b[0], p[1] + b[1], p[2] + b[2]) in table) for b in bonds(table[p]))

    keep = {p: s for p, s in sites.items() if nneigh(p, sites) > 1}
    unit = A_SI / 4.0
    si, hy = [], []
    for p in sorted(keep):
        si.append((p[0] * unit, p[1] * unit, p[2] * unit))
        for b in bonds(keep[p]):
            q = (p[0] + b[0], p[1] + b[1], p[2] + b[2])
            if q not in keep:
                s = H_BOND / math.sqrt(3.0)
                hy.append((p[0] * unit + b[0] * s, p[1] * unit + b[1] * s, p[2] * unit + b[2] * s))
    return np.array(si, dtype=np.float64).reshape(-1, 3), np.array(hy, dtype=np.float64).reshape(-1, 3)


# --------------------------------------------------------------------------------------------
# grids and potentials
# --------------------------------------------------------------------------------------------
@dataclass
class Grid:
    nx: int
    ny: int
    nz: int
    hx: float
    hy: float
    hz: float

    @property
    def shape(self):            # array shape [nz][ny][nx], x fastest
        return (self.nz, self.ny, self.nx)

    @property
    def ng(self):
        return self.nx * self.ny * self.nz

    @property
    def dV(self):
        return self.hx * self.hy * self.hz

    @property
    def box(self):
        return (self.nx * self.hx, self.ny * self.hy, self.nz * self.hz)


def _axis_window(center, sigma_cut, n, h):
    """Grid indices (wrapped) and minimum-image displacements within +-sigma_cut of center."""
    lo = int(math.floor((center - sigma_cut) / h))
    hi = int(math.ceil((center + sigma_cut) / h))
    if hi - lo + 1 >= n:                       # window covers the axis: take every point once
        idx = np.arange(n)
        d = idx * h - center
        L = n * h
        d -= L * np.round(d / L)
        return idx, d
    i = np.arange(lo, hi + 1)
    return np.mod(i, n), i * h - center


def gaussian_vloc(grid: Grid, centers, depths, sigmas, cut_sigmas: float = 8.5):
    """V_loc(r) = -sum_a depth_a exp(-|r-R_a|^2_min-image / (2 sigma_a^2)), shape [nz][ny][nx].

    Each Gaussian is evaluated on the box |d_i| <= cut_sigmas*sigma (dropped tail < 3e-16 depth).
    """
    v = np.zeros(grid.shape, dtype=np.float64)
    for (cx, cy, cz), dep, sg in zip(centers, depths, sigmas):
        ix, dx = _axis_window(cx, cut_sigmas * sg, grid.nx, grid.hx)
        iy, dy = _axis_window(cy, cut_sigmas * sg, grid.ny, grid.hy)
        iz, dz = _axis_window(cz, cut_sigmas * sg, grid.nz, grid.hz)
        gx = np.exp(-dx * dx / (2 * sg * sg))
        gy = np.exp(-dy * dy / (2 * sg * sg))
        gz = np.exp(-dz * dz / (2 * sg * sg))
        v[np.ix_(iz, iy, ix)] -= dep * gz[:, None, None] * gy[None, :, None] * gx[None, None, :]
    return v


@dataclass
class KB:
    """Sparse Kleinman-Bylander projector lists (SURVEY.md 8(a) a6, 8(b) sgw_set_nonlocal)."""
    nsphere: int
    nproj: int
    sph_ptr: np.ndarray    # int64 [nsphere+1]
    sph_idx: np.ndarray    # int32 [npts]   flat grid index g = ix + nx*(iy + ny*iz)
    beta: np.ndarray       # float64 [npts][nproj]
    D: np.ndarray          # float64 [nsphere][nproj]

    @staticmethod
    def empty():
        return KB(0, 4, np.zeros(1, np.int64), np.zeros(0, np.int32),
                  np.zeros((0, 4)), np.zeros((0, 4)))


def kb_projectors(grid: Grid, centers, radius: float = KB_RADIUS, sigma: float = KB_SIGMA,
                  seed: int = SEED_D) -> KB:
    """One s and three p Gaussian projectors per centre on the grid points within ``radius``.

    beta_s ~ exp(-r^2/2 sigma^2), beta_{p_i} ~ r_i exp(-r^2/2 sigma^2), each normalised so that
    dV * sum_j beta_j^2 = 1; D_s, D_p = 2u-1 with u hash-uniform (one D_p shared by the three p).
    """
    ptr = [0]
    idxs, betas, Ds = [], [], []
    for a, (cx, cy, cz) in enumerate(centers):
        ix, dx = _axis_window(cx, radius, grid.nx, grid.hx)
        iy, dy = _axis_window(cy, radius, grid.ny, grid.hy)
        iz, dz = _axis_window(cz, radius, grid.nz, grid.hz)
        DZ, DY, DX = np.meshgrid(dz, dy, dx, indexing="ij")
        IZ, IY, IX = np.meshgrid(iz, iy, ix, indexing="ij")
        r2 = DX * DX + DY * DY + DZ * DZ
        m = r2 <= radius * radius
        g = (IX[m] + grid.nx * (IY[m] + grid.ny * IZ[m])).astype(np.int64)
        order = np.argsort(g, kind="stable")
        g = g[order]
        e = np.exp(-r2[m][order] / (2 * sigma * sigma))
        b = np.stack([e, DX[m][order] * e, DY[m][order] * e, DZ[m][order] * e], axis=1)
        b /= np.sqrt(grid.dV * np.sum(b * b, axis=0))[None, :]
        ds = 2.0 * hash_uniform(seed, a, 0) - 1.0
        dp = 2.0 * hash_uniform(seed, a, 1) - 1.0
        idxs.append(g.astype(np.int32))
        betas.append(b)
        Ds.append([ds, dp, dp, dp])
        ptr.append(ptr[-1] + len(g))
    if not idxs:
        return KB.empty()
    return KB(len(Ds), 4, np.array(ptr, np.int64), np.concatenate(idxs),
              np.ascontiguousarray(np.concatenate(betas, axis=0)), np.array(Ds, np.float64))


# --------------------------------------------------------------------------------------------
# Chebyshev coefficients and spectral bounds
# --------------------------------------------------------------------------------------------
def sqrt_fermi(e, mu: float = MU, beta: float = BETA):
    """f(E) = [1 + exp(beta (E - mu))]^(-1/2), overflow-safe."""
    t = np.clip(beta * (np.asarray(e, dtype=np.float64) - mu), -700.0, 700.0)
    return 1.0 / np.sqrt(1.0 + np.exp(t))


def cheb_coeffs(func, emin: float, emax: float, nterms: int, oversample: int = 8):
    """a_n = ((2-delta_n0)/M) sum_{j<M} f(x_j) cos(n theta_j), theta_j = pi (j+1/2)/M, M = 8 nterms.

    ``func`` takes energies E = Ebar + dE*x ('Inputs built by the harness').
    """
    from scipy.fft import dct
    M = oversample * nterms
    theta = math.pi * (np.arange(M) + 0.5) / M
    eb, de = 0.5 * (emax + emin), 0.5 * (emax - emin)
    fx = func(eb + de * np.cos(theta))
    a = dct(fx, type=2)[:nterms] / M          # DCT-II: 2 sum_j f_j cos(pi n (2j+1)/(2M))
    a[0] *= 0.5
    return np.ascontiguousarray(a)


def spectral_bounds(grid: Grid, vloc, has_kb: bool):
    """Analytic [E_min, E_max] = [min V - D, 1/2 sum (pi/h_i)^2 + max V + D] (BASELINE.json cfg 0)."""
    d = DELTA_NL if has_kb else 0.0
    tmax = 0.5 * ((math.pi / grid.hx) ** 2 + (math.pi / grid.hy) ** 2 + (math.pi / grid.hz) ** 2)
    return float(vloc.min()) - d, tmax + float(vloc.max()) + d


# --------------------------------------------------------------------------------------------
# the five BASELINE.json configs
# --------------------------------------------------------------------------------------------
@dataclass
class Workload:
    name: str
    grid: Grid
    nvec: int
    nterms: int            # Chebyshev terms (0 = none)
    td_steps: int          # TD steps (0 = none)
    dt: float
    vloc: np.ndarray
    kb: KB
    emin: float
    emax: float
    coeffs: np.ndarray
    rho_scale: float
    atoms: str
    extra: dict = field(default_factory=dict)


_CFG = {
    # name: (n, h, nvec, nterms, td_steps, r2_units or None, use_kb)
    "cfg0": (32, 0.5, 4, 128, 0, None, False),
    "cfg1": (96, 0.45, 64, 512, 0, 64, False),
    "cfg2": (128, 0.5, 16, 512, 2000, 108, False),
    "cfg3": (256, 0.5, 256, 2048, 0, 480, True),
    "cfg4": (384, 0.6, 32, 2048, 500, 2540, True),
}


def snap_center(grid: Grid):
    return np.array([(grid.nx // 2) * grid.hx, (grid.ny // 2) * grid.hy, (grid.nz // 2) * grid.hz])


def make_workload(name: str, *, n: int | None = None, nvec: int | None = None,
                  nterms: int | None = None, td_steps: int | None = None, subcell: bool = False) -> Workload:
    """Build config ``name`` ('cfg0'..'cfg4'); keyword overrides shrink it for tests.

    ``subcell=True`` with a smaller ``n``: the central n^3 sub-cell of the config (same spacing, only the atoms whose
    local Gaussians and KB spheres lie inside it, same spectral window as the full config) -- the bounded sample the
    CPU oracle is timed on in bench.py.
    """
    n0, h, nv0, nt0, td0, r2u, use_kb = _CFG[name]
    full_n = n0
    n = n or n0
    grid = Grid(n, n, n, h, h, h)
    nvec = nvec if nvec is not None else nv0
    nterms = nterms if nterms is not None else nt0
    td_steps = td_steps if td_steps is not None else td0
    c0 = snap_center(grid)
    if r2u is None:
        L = grid.box
        centers = np.array([[hash_uniform(SEED_WELL, a, d) * L[d] for d in range(3)] for a in range(8)])
        depths, sigmas = [1.0] * 8, [1.0] * 8
        si = np.zeros((0, 3))
        atoms = "8 Gaussian wells"
    else:
        si_rel, h_rel = diamond_cluster(r2u)
        if subcell and n < full_n:
            half = 0.5 * n * h - KB_RADIUS - h
            si_rel = si_rel[np.max(np.abs(si_rel), axis=1) <= half]
            h_rel = h_rel[np.max(np.abs(h_rel), axis=1) <= half]
        si, hy = si_rel + c0, h_rel + c0
        centers = np.concatenate([si, hy], axis=0)
        depths = [2.0] * len(si) + [1.0] * len(hy)
        sigmas = [1.2] * len(si) + [0.8] * len(hy)
        atoms = f"Si{len(si)}H{len(hy)}"
    vloc = gaussian_vloc(grid, centers, depths, sigmas)
    kb = kb_projectors(grid, si) if use_kb else KB.empty()
    emin, emax = spectral_bounds(grid, vloc, use_kb)
    coeffs = cheb_coeffs(sqrt_fermi, emin, emax, nterms) if nterms > 0 else np.zeros(0)
    rho_scale = 2.0 / (max(nvec, 1) * grid.dV)
    return Workload(name, grid, nvec, nterms, td_steps, 0.05, vloc, kb, emin, emax, coeffs,
                    rho_scale, atoms)
