// sgw_cut.cu -- the Hamiltonian with the paper's kinetic-energy cutoff ("apply an energy cutoff of 28 Hartrees
// to the kinetic energy operator"; the cutoff bounds the spectral width and with it N_chb; reading R-14).
//
// T_cut = F^-1 min(1/2 |k|^2, E_cut) F is diagonal in k but no longer a sum T_x + T_y + T_z, and exp(-i T_cut dt) no
// longer a product of 1D factors, so the separable passes of the default path (sgw_lean.cuh, sgw_acc.cuh) cannot
// represent it.  It takes the route the Poisson solve already uses: a full 3D transform in five passes (forward x,
// forward y, z round trip with a 3D table, inverse y, inverse x) with the pointwise work (potential, recurrence, phases)
// fused into the first and the last pass.  ~7 array sweeps per application instead of 2-3: the price of the paper's
// operator, measured in bench.py next to the separable one.
#include <cmath>
#include <cstring>

#include "sgw_ctx.h"
#include "sgw_kernels.cuh"

using namespace sgw;

namespace {

#define SGW_TRY(expr)             \
    do {                          \
        int rc_ = (expr);         \
        if (rc_ != 0) return rc_; \
    } while (0)

inline unsigned blocks_for(long long n, int t) { return (unsigned)((n + t - 1) / t); }

// table[g] = min(1/2 |k|^2, ecut) / N_g on the grid's k layout (natural DFT order on every axis)
__global__ void kin3d_kernel(double* tab, int nx, int ny, int nz, double hx, double hy, double hz, double ecut) {
    const long long ng = (long long)nx * ny * nz;
    const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= ng) return;
    const int ix = (int)(i % nx), iy = (int)((i / nx) % ny), iz = (int)(i / ((long long)nx * ny));
    const double pi = 3.14159265358979323846;
    const int mx = (2 * ix >= nx) ? ix - nx : ix, my = (2 * iy >= ny) ? iy - ny : iy, mz = (2 * iz >= nz) ? iz - nz : iz;
    const double kx = 2 * pi * mx / (nx * hx), ky = 2 * pi * my / (ny * hy), kz = 2 * pi * mz / (nz * hz);
    double t = 0.5 * (kx * kx + ky * ky + kz * kz);
    if (t > ecut) t = ecut;
    tab[i] = t / (double)ng;
}

// out[g] = exp(-i N_g tab[g] dt) / N_g
__global__ void td3d_kernel(const double* __restrict__ tab, double dt, cd* __restrict__ out, long long ng) {
    const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= ng) return;
    double s, c;
    sincos(tab[i] * (double)ng * dt, &s, &c);
    out[i] = make_double2(c / (double)ng, -s / (double)ng);
}

__global__ void axpy_kernel(cd* __restrict__ y, const cd* __restrict__ x, double a, int init, long long n) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const cd u = x[i];
    if (init) y[i] = cscale(u, a);
    else { cd v = y[i]; v.x += a * u.x; v.y += a * u.y; y[i] = v; }
}

OpParams zero_params() {
    OpParams p;
    memset(&p, 0, sizeof(p));
    return p;
}

// W <- F_y F_x src (two forward passes; the first may multiply by the phase table on load), then the z round trip with
// the 3D table, then the inverse y pass; the caller runs the last (inverse x) pass with its own epilogue
int cut_front(sgw_ctx* c, int nv, const cd* src, cd* W, const cd* phase_on_load, bool complex_table, double kscale) {
    OpParams p = zero_params();
    p.out = W;
    p.phase = phase_on_load;
    SGW_TRY(run_pass(c, 0, K_FWD, phase_on_load ? 3 : 0, src, p, nv));
    p.phase = nullptr;
    SGW_TRY(run_pass(c, 1, K_FWD, 0, W, p, nv));
    if (complex_table) { p.mul3c = c->td_kin3d; SGW_TRY(run_pass(c, 2, K_RT_MUL3D, 1, W, p, nv)); }
    else { p.mul3d = c->kin3d; p.kscale = kscale; SGW_TRY(run_pass(c, 2, K_RT_MUL3D, 2, W, p, nv)); }
    p.mul3c = nullptr; p.mul3d = nullptr;
    return run_pass(c, 1, K_INV, 0, W, p, nv);
}

}  // namespace

extern "C" int sgw_set_kinetic_cutoff(sgw_ctx* c, double ecut) {
    if (!c || !(ecut == ecut)) return set_error(SGW_EINVAL, "sgw_set_kinetic_cutoff: bad argument");
    cudaStreamSynchronize(c->stream);
    drop_filter_graph(c);
    c->td3d_valid = false;
    if (!(ecut > 0.0)) {
        cudaFree(c->kin3d); cudaFree(c->td_kin3d); cudaFree(c->wcut);
        c->kin3d = nullptr; c->td_kin3d = nullptr; c->wcut = nullptr; c->ecut = 0.0;
        return SGW_OK;
    }
    if (!c->kin3d) SGW_TRY(check_cuda(cudaMalloc((void**)&c->kin3d, c->ng * sizeof(double)), "kinetic table"));
    if (!c->td_kin3d) SGW_TRY(check_cuda(cudaMalloc((void**)&c->td_kin3d, c->ng * sizeof(cd)), "kinetic phase table"));
    if (!c->wcut) SGW_TRY(check_cuda(cudaMalloc((void**)&c->wcut, (size_t)c->max_nvec * c->ng * sizeof(cd)), "cutoff workspace"));
    kin3d_kernel<<<blocks_for(c->ng, 256), 256, 0, c->stream>>>(c->kin3d, c->nx, c->ny, c->nz, c->hx, c->hy, c->hz, ecut);
    c->launches++;
    SGW_TRY(check_cuda(cudaStreamSynchronize(c->stream), "kin3d_kernel"));
    c->ecut = ecut;
    return SGW_OK;
}

namespace sgw {

// out = F^-1 min(1/2 k^2, E_cut) F in + V_loc in   (the KB term is added by the caller)
int cut_apply_H(sgw_ctx* c, int nv, const cd* in, cd* out) {
    SGW_TRY(cut_front(c, nv, in, c->wcut, nullptr, false, 1.0));
    OpParams p = zero_params();
    p.out = out; p.src = in; p.vtab = c->vloc;
    return run_pass(c, 0, K_INV, 3, c->wcut, p, nv);
}

// forward three-term recurrence (Eq. 3; R-1) on the five-pass operator: term n takes cur = phi_{n-1},
// acc = phi_{n-2} and leaves acc = phi_n = hs (s T_cut + vtab) cur - acc (hs = 1/2 and no subtraction for n = 1);
// the series is updated after every term (and after the term's KB contribution)
int cut_cheb_filter(sgw_ctx* c, int nvec, cd* psi, const double* a, double s, int nterms) {
    const long long n = (long long)nvec * c->ng;
    SGW_TRY(ensure_ws(c, 2));
    cd *Pb = psi, *Qb = c->ws[0], *Ob = c->ws[1];
    const int L = nterms - 1;
    const unsigned nb = blocks_for(n, 256);
    axpy_kernel<<<nb, 256, 0, c->stream>>>(Ob, Pb, a[0], 1, n);
    c->launches++;
    for (int k = 1; k <= L; ++k) {
        const bool odd = k & 1;
        cd* cur = odd ? Pb : Qb;
        cd* acc = odd ? Qb : Pb;
        const double hs = (k == 1) ? 0.5 : 1.0;
        SGW_TRY(cut_front(c, nvec, cur, c->wcut, nullptr, false, s));
        OpParams p = zero_params();
        p.src = cur; p.acc = acc; p.vtab = c->vtab; p.hs = hs; p.alpha = (k == 1) ? 0.0 : -1.0;
        SGW_TRY(run_pass(c, 0, K_INV, 4, c->wcut, p, nvec));
        SGW_TRY(kb_apply(c, nvec, cur, acc, 0, s * hs));
        axpy_kernel<<<nb, 256, 0, c->stream>>>(Ob, acc, a[k], 0, n);
        c->launches++;
    }
    SGW_TRY(check_cuda(cudaGetLastError(), "cut_cheb_filter"));
    return check_cuda(cudaMemcpyAsync(psi, Ob, (size_t)n * sizeof(cd), cudaMemcpyDeviceToDevice, c->stream), "copy result");
}

// split-operator steps with exp(-i T_cut dt) as one 3D factor (R-8, R-11): potential half-step phases on
// load of the first and on store of the last pass, KB factors conjugated by the phase as in the separable path
int cut_td_propagate(sgw_ctx* c, int nvec, cd* psi, double dt, int nsteps) {
    const long long ng = c->ng;
    if (!c->td3d_valid || c->td3d_dt != dt) {
        td3d_kernel<<<blocks_for(ng, 256), 256, 0, c->stream>>>(c->kin3d, dt, c->td_kin3d, ng);
        c->launches++;
        c->td3d_dt = dt; c->td3d_valid = true;
    }
    const bool kb = c->nsphere > 0;
    const int chunk = nvec < c->max_nvec ? nvec : c->max_nvec;
    for (int step = 0; step < nsteps; ++step) {
        if (c->hartree_mode || step == 0) {
            const double* vh = nullptr;
            if (c->hartree_mode) {
                SGW_TRY(sgw_hartree(c, nvec, psi, c->rho_scale, c->vh, nullptr));
                vh = c->vh;
            }
            phase_kernel<<<blocks_for(ng, 256), 256, 0, c->stream>>>(c->vloc, vh, 0.5 * dt, c->phase, ng);
            c->launches++;
        }
        for (int cv = 0; cv < nvec; cv += chunk) {
            const int nc = (nvec - cv < chunk) ? nvec - cv : chunk;
            cd* ps = psi + (long long)cv * ng;
            if (kb) SGW_TRY(kb_apply(c, nc, ps, ps, 1, 0.5 * dt, c->phase, +1));
            SGW_TRY(cut_front(c, nc, ps, ps, c->phase, true, 1.0));
            OpParams p = zero_params();
            p.out = ps; p.phase = c->phase;
            SGW_TRY(run_pass(c, 0, K_INV, 5, ps, p, nc));
            if (kb) SGW_TRY(kb_apply(c, nc, ps, ps, 1, 0.5 * dt, c->phase, -1));
        }
    }
    return check_cuda(cudaGetLastError(), "cut_td_propagate");
}

}  // namespace sgw
