// sgw_solvers.cu -- the hot-path entry points of libsgw (include/sgw.h): random vectors, H apply,
// Chebyshev filter, Hartree, split-operator propagation, norms.
#include <cmath>
#include <cstring>
#include <vector>

#include "sgw_ctx.h"
#include "sgw_kernels.cuh"

using namespace sgw;

namespace {

inline unsigned blocks_for(long long n, int t) { return (unsigned)((n + t - 1) / t); }

#define SGW_TRY(expr)            \
    do {                         \
        int rc_ = (expr);        \
        if (rc_ != 0) return rc_; \
    } while (0)

int launched(sgw_ctx* c, const char* what) {
    c->launches++;
    return check_cuda(cudaGetLastError(), what);
}

}  // namespace
int sgw::ensure_ws(sgw_ctx* c, int n) {
    for (int a = 0; a < n; ++a)
        if (!c->ws[a])
            SGW_TRY(check_cuda(cudaMalloc((void**)&c->ws[a], (size_t)c->max_nvec * c->ng * sizeof(cd)), "workspace"));
    return 0;
}

namespace {
int ensure_kbc(sgw_ctx* c, int nvec) {
    const long long need = (long long)nvec * c->nsphere * c->nproj;
    if (need <= c->kbc_cap) return 0;
    SGW_TRY(check_cuda(cudaStreamSynchronize(c->stream), "sync"));
    cudaFree(c->kbc);
    c->kbc = nullptr; c->kbc_cap = 0;
    SGW_TRY(check_cuda(cudaMalloc((void**)&c->kbc, need * sizeof(cd)), "kb buffer"));
    c->kbc_cap = need;
    return 0;
}

template <int NP>
int kb_apply_np(sgw_ctx* c, int nvec, const cd* src, cd* dst, int mode, double scale_or_tau, const cd* phase, int fold) {
    dim3 grid(c->nsphere, nvec);
    const double dV = c->hx * c->hy * c->hz;
    // fold = +1: projections of phase*src, contribution times conj(phase)  (opening half step: the pass multiplies by phase on load)
    // fold = -1: projections of conj(phase)*src, contribution times phase  (closing half step: the pass multiplied by phase on store)
    kb_project_kernel<NP><<<grid, 128, 0, c->stream>>>(src, c->ng, c->sph_ptr, c->sph_idx, c->beta, dV, c->kbc, c->nsphere,
                                                       fold ? phase : nullptr, fold < 0 ? 1 : 0);
    SGW_TRY(launched(c, "kb_project"));
    kb_scatter_kernel<NP><<<grid, 128, 0, c->stream>>>(dst, c->ng, c->sph_ptr, c->sph_idx, c->beta, c->D, c->kbc,
                                                       c->nsphere, mode, scale_or_tau, fold ? phase : nullptr, fold > 0 ? 1 : 0);
    return launched(c, "kb_scatter");
}

// dst += sum beta f <beta|src>, all projections taken from src before any scatter (R-11)
}  // namespace
int sgw::kb_apply(sgw_ctx* c, int nvec, const cd* src, cd* dst, int mode, double scale_or_tau, const cd* phase, int fold) {
    if (c->nsphere == 0) return 0;
    SGW_TRY(ensure_kbc(c, nvec));
    switch (c->nproj) {
        case 1: return kb_apply_np<1>(c, nvec, src, dst, mode, scale_or_tau, phase, fold);
        case 2: return kb_apply_np<2>(c, nvec, src, dst, mode, scale_or_tau, phase, fold);
        case 3: return kb_apply_np<3>(c, nvec, src, dst, mode, scale_or_tau, phase, fold);
        case 4: return kb_apply_np<4>(c, nvec, src, dst, mode, scale_or_tau, phase, fold);
        case 5: return kb_apply_np<5>(c, nvec, src, dst, mode, scale_or_tau, phase, fold);
        case 6: return kb_apply_np<6>(c, nvec, src, dst, mode, scale_or_tau, phase, fold);
        case 7: return kb_apply_np<7>(c, nvec, src, dst, mode, scale_or_tau, phase, fold);
        case 8: return kb_apply_np<8>(c, nvec, src, dst, mode, scale_or_tau, phase, fold);
    }
    return set_error(SGW_EINVAL, "bad nproj");
}

namespace {
OpParams zero_params() {
    OpParams p;
    memset(&p, 0, sizeof(p));
    return p;
}

// rho = scale * sum |psi|^2 ; V_H by the cut-Coulomb Poisson solve (R-10).  Results in c->vh (and rho/rho2).
int hartree_into(sgw_ctx* c, int nvec, const cd* psi, double rho_scale, double* rho2, bool rho_ready = false,
                 bool keep_complex = false) {
    const long long ng = c->ng;
    if (!rho_ready) {          // otherwise c->rho was accumulated by the last pass of the previous step
        density_kernel<<<blocks_for(ng, 256), 256, 0, c->stream>>>(psi, nvec, ng, rho_scale, c->rho, rho2);
        SGW_TRY(launched(c, "density"));
    }
    real_to_complex_kernel<<<blocks_for(ng, 256), 256, 0, c->stream>>>(c->rho, c->pois, ng);
    SGW_TRY(launched(c, "r2c"));
    OpParams p = zero_params();
    p.out = c->pois;
    SGW_TRY(run_pass(c, 0, K_FWD, 1, c->pois, p));
    SGW_TRY(run_pass(c, 1, K_FWD, 1, c->pois, p));
    p.mul3d = c->vk3d;
    SGW_TRY(run_pass(c, 2, K_RT_MUL3D, 1, c->pois, p));
    p.mul3d = nullptr;
    SGW_TRY(run_pass(c, 1, K_INV, 1, c->pois, p));
    SGW_TRY(run_pass(c, 0, K_INV, 1, c->pois, p));
    if (keep_complex) return 0;      // the caller reads V_H as the real part of c->pois
    complex_to_real_kernel<<<blocks_for(ng, 256), 256, 0, c->stream>>>(c->pois, c->vh, ng);
    return launched(c, "c2r");
}

}  // namespace

extern "C" int sgw_random_vectors(sgw_ctx* c, uint64_t seed, int first_vec, int nvec, void* d_psi) {
    if (!c || nvec < 0 || first_vec < 0 || (nvec > 0 && !d_psi)) return set_error(SGW_EINVAL, "sgw_random_vectors: bad argument");
    if (nvec == 0) return SGW_OK;
    dim3 grid(blocks_for(c->ng, 1024), nvec);
    rng_kernel<<<grid, 256, 0, c->stream>>>((cd*)d_psi, sm64(seed), first_vec, c->ng);
    return launched(c, "rng_kernel");
}

extern "C" int sgw_norms(sgw_ctx* c, int nvec, const void* d_psi, double* d_out) {
    if (!c || nvec < 0 || (nvec > 0 && (!d_psi || !d_out))) return set_error(SGW_EINVAL, "sgw_norms: bad argument");
    if (nvec == 0) return SGW_OK;
    SGW_TRY(check_cuda(cudaMemsetAsync(d_out, 0, nvec * sizeof(double), c->stream), "memset"));
    const long long seg = 256LL * 256;          // segments of length L ~ 256 per thread block row
    dim3 grid((unsigned)((c->ng + seg - 1) / seg), nvec);
    norms_kernel<<<grid, 256, 0, c->stream>>>((const cd*)d_psi, c->ng, d_out);
    return launched(c, "norms_kernel");
}

static int power_iteration(sgw_ctx* c, double shift, int niter, uint64_t seed, int vec, double* d_red, double* lambda) {
    const long long ng = c->ng;
    cd *x = c->ws[0], *y = c->ws[1];
    SGW_TRY(sgw_random_vectors(c, seed, vec, 1, x));
    // |x0|^2 = N_g exactly for +-1 entries: normalise with that
    scale_kernel<<<blocks_for(ng, 256), 256, 0, c->stream>>>(x, 1.0 / sqrt((double)ng), ng);
    SGW_TRY(launched(c, "scale"));
    const unsigned nb = (unsigned)((ng + 256LL * 16 - 1) / (256LL * 16));      // segments of 16 elements per thread
    for (int it = 0; it < niter; ++it) {
        SGW_TRY(sgw_apply_H(c, 1, x, y));
        SGW_TRY(check_cuda(cudaMemsetAsync(d_red, 0, 2 * sizeof(double), c->stream), "memset"));
        power_reduce_kernel<<<nb, 256, 0, c->stream>>>(x, y, shift, ng, d_red);
        SGW_TRY(launched(c, "power_reduce"));
        power_scale_kernel<<<blocks_for(ng, 256), 256, 0, c->stream>>>(x, y, d_red, ng, d_red + 2);
        SGW_TRY(launched(c, "power_scale"));
    }
    double lam = 0.0;
    SGW_TRY(check_cuda(cudaMemcpyAsync(&lam, d_red + 2, sizeof(double), cudaMemcpyDeviceToHost, c->stream), "read lambda"));
    SGW_TRY(check_cuda(cudaStreamSynchronize(c->stream), "sync"));
    *lambda = lam + shift;
    return SGW_OK;
}

extern "C" int sgw_spectral_bounds(sgw_ctx* c, int niter, uint64_t seed, double* h_emin, double* h_emax) {
    if (!c || niter < 1 || !h_emin || !h_emax) return set_error(SGW_EINVAL, "sgw_spectral_bounds: bad argument");
    SGW_TRY(ensure_ws(c, 2));
    double* d_red = nullptr;
    SGW_TRY(check_cuda(cudaMalloc((void**)&d_red, 3 * sizeof(double)), "reduction buffer"));
    double la = 0.0, lb = 0.0;
    int rc = power_iteration(c, 0.0, niter, seed, 0, d_red, &la);
    if (!rc) rc = power_iteration(c, la, niter, seed, 1, d_red, &lb);
    cudaFree(d_red);
    if (rc) return rc;
    *h_emin = la < lb ? la : lb;
    *h_emax = la < lb ? lb : la;
    return SGW_OK;
}

extern "C" int sgw_apply_H(sgw_ctx* c, int nvec, const void* d_in, void* d_out) {
    if (!c || nvec < 0 || (nvec > 0 && (!d_in || !d_out)) || d_in == d_out) return set_error(SGW_EINVAL, "sgw_apply_H: bad argument");
    const cd* in = (const cd*)d_in;
    cd* out = (cd*)d_out;
    for (int v0 = 0; v0 < nvec; v0 += c->max_nvec) {
        const int nv = (nvec - v0 < c->max_nvec) ? nvec - v0 : c->max_nvec;
        const cd* i0 = in + (long long)v0 * c->ng;
        cd* o0 = out + (long long)v0 * c->ng;
        if (c->use_engine) {
            SGW_TRY(c->use_engine == 2 ? lean_apply_H(c, nv, i0, o0) : eng_apply_H(c, nv, i0, o0));
            SGW_TRY(kb_apply(c, nv, i0, o0, 0, 1.0));
            continue;
        }
        OpParams p = zero_params();
        p.out = o0;
        int rp = run_plane(c, PL_SUM, nv, i0, o0, nullptr, false);
        if (rp < 0) return rp;
        if (rp == 1) {
            p.mul_re = c->kin[0];
            SGW_TRY(run_pass(c, 0, K_RT_STORE, nv, i0, p));
            p.mul_re = c->kin[1]; p.acc = o0;
            SGW_TRY(run_pass(c, 1, K_RT_ACC, nv, i0, p));
        }
        p.acc = o0;
        SGW_TRY(kb_apply(c, nv, i0, o0, 0, 1.0));
        p.mul_re = c->kin[2]; p.vtab = c->vloc;
        SGW_TRY(run_pass(c, 2, K_RT_HFIN, nv, i0, p));
    }
    return SGW_OK;
}

extern "C" int sgw_hartree(sgw_ctx* c, int nvec, const void* d_psi, double rho_scale, double* d_vh, double* d_rho) {
    if (!c || nvec < 0 || (nvec > 0 && !d_psi) || !d_vh) return set_error(SGW_EINVAL, "sgw_hartree: bad argument");
    SGW_TRY(hartree_into(c, nvec, (const cd*)d_psi, rho_scale, d_rho));
    return check_cuda(cudaMemcpyAsync(d_vh, c->vh, c->ng * sizeof(double), cudaMemcpyDeviceToDevice, c->stream), "copy vh");
}

namespace {
// the launches of one filter call, in stream order on c->stream (arguments already checked)
int cheb_filter_body(sgw_ctx* c, int nvec, void* d_psi, const double* h_coeffs, double Emin, double Emax, int nterms) {
    const long long ng = c->ng;
    const double Eb = 0.5 * (Emax + Emin), dE = 0.5 * (Emax - Emin), s = 2.0 / dE;
    if (nterms == 1) {
        scale_kernel<<<blocks_for(ng * nvec, 256), 256, 0, c->stream>>>((cd*)d_psi, h_coeffs[0], ng * nvec);
        return launched(c, "scale");
    }
    SGW_TRY(ensure_ws(c, c->use_engine ? 2 : 3));
    // tables scaled by s = 2/dE so that one pass yields 2*Ht*phi directly (R-1; Eq. 3 mapping to [-1,1])
    for (int a = 0; a < 3; ++a) {
        scale_table_kernel<<<blocks_for(c->dims[a], 128), 128, 0, c->stream>>>(c->kin[a], s, c->cheb_kin[a], c->dims[a]);
        SGW_TRY(launched(c, "scale_table"));
    }
    vtab_kernel<<<blocks_for(ng, 256), 256, 0, c->stream>>>(c->vloc, s, Eb, c->vtab, ng);
    SGW_TRY(launched(c, "vtab"));
    for (int v0 = 0; v0 < nvec; v0 += c->max_nvec) {
        const int nv = (nvec - v0 < c->max_nvec) ? nvec - v0 : c->max_nvec;
        cd* X0 = (cd*)d_psi + (long long)v0 * ng;
        if (c->use_engine) {
            SGW_TRY(c->use_engine == 2 ? lean_cheb_filter(c, nv, X0, h_coeffs, s, nterms)
                                       : eng_cheb_filter(c, nv, X0, h_coeffs, s, nterms));
            continue;
        }
        cd *P1 = c->ws[0], *W = c->ws[1], *O = c->ws[2];
        cd* cur = X0;
        cd* other = P1;              // receives phi_n; holds phi_{n-2} for n >= 2
        // series terms not yet added to O: flags for degrees n-2 and n-1 (phi_{n-2}, phi_{n-1}, phi_n are
        // all in registers in the last pass of term n, so O is touched only every third term)
        bool pend_m2 = false, pend_m1 = true;  // before n = 1: degree 0 (= n-1) is pending
        bool series_started = false;
        for (int n = 1; n < nterms; ++n) {
            const bool last = (n == nterms - 1);
            const bool flush = last || pend_m2;
            const int chunk = (c->l2_chunk > 0 && c->l2_chunk < nv) ? c->l2_chunk : nv;
            for (int cv = 0; cv < nv; cv += chunk) {          // vector chunks sized so that W stays L2-resident
                const int nc = (nv - cv < chunk) ? nv - cv : chunk;
                const long long co = (long long)cv * ng;
                OpParams p = zero_params();
                p.out = W;
                int rp = run_plane(c, PL_SUM, nc, cur + co, W, nullptr, true);
                if (rp < 0) return rp;
                if (rp == 1) {
                    p.mul_re = c->cheb_kin[0];
                    SGW_TRY(run_pass(c, 0, K_RT_STORE, nc, cur + co, p));
                    p.mul_re = c->cheb_kin[1]; p.acc = W;
                    SGW_TRY(run_pass(c, 1, K_RT_ACC, nc, cur + co, p));
                }
                p.acc = W;
                SGW_TRY(kb_apply(c, nc, cur + co, W, 0, s));
                p.mul_re = c->cheb_kin[2]; p.vtab = c->vtab;
                p.out = other + co; p.prev = other + co; p.use_prev = (n >= 2);
                p.hs = (n == 1) ? 0.5 : 1.0;
                p.flush = flush; p.series = O + co; p.series_init = !series_started;
                p.c0 = pend_m2 ? h_coeffs[n - 2] : 0.0;
                p.c1 = pend_m1 ? h_coeffs[n - 1] : 0.0;
                p.c2 = h_coeffs[n];
                SGW_TRY(run_pass(c, 2, K_RT_CHEB, nc, cur + co, p));
            }
            if (flush) { series_started = true; pend_m2 = false; pend_m1 = false; }
            else { pend_m2 = pend_m1; pend_m1 = true; }
            cd* t = cur; cur = other; other = t;
        }
        SGW_TRY(check_cuda(cudaMemcpyAsync(X0, O, (size_t)nv * ng * sizeof(cd), cudaMemcpyDeviceToDevice, c->stream), "copy out"));
    }
    return SGW_OK;
}

// Small grids are launch-bound (cfg0: 2 MB per array, 256 launches of a few us each): when a call repeats with the
// same vector block, window and coefficients, its launches are captured on an internal stream, instantiated as a
// CUDA graph and replayed on the caller's stream from then on (the first call with a key launches plainly).  SGW_GRAPH=0 disables, SGW_GRAPH_BYTES moves
// the size limit (bytes of one vector block; default 16 MB).
bool filter_graph_wanted(const sgw_ctx* c, int nvec, int nterms) {
    if (c->use_engine != 2 || c->prof_on || c->nsphere > 0 || nvec > c->max_nvec || nterms < 3) return false;
    const char* e = getenv("SGW_GRAPH");
    if (e && atoi(e) == 0) return false;
    double limit = 16.0e6;
    const char* b = getenv("SGW_GRAPH_BYTES");
    if (b && atof(b) > 0) limit = atof(b);
    return (double)nvec * (double)c->ng * sizeof(cd) <= limit;
}
}  // namespace

extern "C" int sgw_cheb_filter(sgw_ctx* c, int nvec, void* d_psi, const double* h_coeffs, double Emin, double Emax,
                               int nterms) {
    if (!c || nvec < 0 || (nvec > 0 && !d_psi) || !h_coeffs || nterms < 1 || !(Emax > Emin))
        return set_error(SGW_EINVAL, "sgw_cheb_filter: bad argument");
    if (nvec == 0) return SGW_OK;
    if (!filter_graph_wanted(c, nvec, nterms)) return cheb_filter_body(c, nvec, d_psi, h_coeffs, Emin, Emax, nterms);
    const bool same = c->fg_psi == d_psi && c->fg_nvec == nvec && c->fg_nterms == nterms && c->fg_emin == Emin &&
                      c->fg_emax == Emax && (int)c->fg_coeffs.size() == nterms &&
                      memcmp(c->fg_coeffs.data(), h_coeffs, nterms * sizeof(double)) == 0;
    if (!same) {
        // first call with this key: plain launches (capture + instantiation cost more than they save on a single
        // call); the key is remembered and a repeat captures
        drop_filter_graph(c);
        c->fg_psi = d_psi; c->fg_nvec = nvec; c->fg_nterms = nterms; c->fg_emin = Emin; c->fg_emax = Emax;
        c->fg_coeffs.assign(h_coeffs, h_coeffs + nterms);
        return cheb_filter_body(c, nvec, d_psi, h_coeffs, Emin, Emax, nterms);
    }
    if (!c->fgraph) {
        SGW_TRY(ensure_ws(c, 2));                     // no allocation inside the capture
        if (!c->gstream) SGW_TRY(check_cuda(cudaStreamCreateWithFlags(&c->gstream, cudaStreamNonBlocking), "graph stream"));
        cudaStream_t user = c->stream;
        const int64_t before = c->launches;
        SGW_TRY(check_cuda(cudaStreamBeginCapture(c->gstream, cudaStreamCaptureModeRelaxed), "begin capture"));
        c->stream = c->gstream;
        const int rc = cheb_filter_body(c, nvec, d_psi, h_coeffs, Emin, Emax, nterms);
        c->stream = user;
        cudaGraph_t g = nullptr;
        const cudaError_t ce = cudaStreamEndCapture(c->gstream, &g);
        const int64_t nodes = c->launches - before;
        c->launches = before;
        if (rc != 0) { if (g) cudaGraphDestroy(g); return rc; }
        SGW_TRY(check_cuda(ce, "end capture"));
        const cudaError_t ie = cudaGraphInstantiate(&c->fgraph, g, 0);
        cudaGraphDestroy(g);
        if (ie != cudaSuccess) { c->fgraph = nullptr; return check_cuda(ie, "graph instantiate"); }
        c->fg_launches = nodes;
    }
    SGW_TRY(check_cuda(cudaGraphLaunch(c->fgraph, c->stream), "graph launch"));
    c->launches += c->fg_launches;
    return SGW_OK;
}

extern "C" int sgw_td_propagate(sgw_ctx* c, int nvec, void* d_psi, double dt, int nsteps) {
    if (!c || nvec < 0 || (nvec > 0 && !d_psi) || nsteps < 0) return set_error(SGW_EINVAL, "sgw_td_propagate: bad argument");
    if (nvec == 0 || nsteps == 0) return SGW_OK;
    const long long ng = c->ng;
    cd* psi = (cd*)d_psi;
    if (!c->td_kin_valid || c->td_dt != dt) {
        for (int a = 0; a < 3; ++a) {
            const int N = c->dims[a];
            std::vector<cd> t(N);
            for (int j = 0; j < N; ++j) {
                const long double ph = (long double)c->h_kin[a][j] * (long double)dt;
                t[j] = make_double2((double)(cosl(ph) / N), (double)(-sinl(ph) / N));
            }
            SGW_TRY(check_cuda(cudaMemcpyAsync(c->td_kin[a], t.data(), N * sizeof(cd), cudaMemcpyHostToDevice, c->stream), "td table"));
            SGW_TRY(check_cuda(cudaStreamSynchronize(c->stream), "td table sync"));
        }
        c->td_dt = dt; c->td_kin_valid = true;
    }
    const bool kb = c->nsphere > 0;
    // lean passes without KB: the last pass of a step accumulates the density of its result (atomics), so only
    // the first step of a call reads the vectors for the density
    const bool fuse_density = c->hartree_mode && c->use_engine == 2 && !kb;
    // lean passes without KB: consecutive half-step phases are merged into one table applied on load (R-8)
    const bool merged = c->use_engine == 2 && !kb;
    if (merged && !c->vprev) {
        SGW_TRY(check_cuda(cudaMalloc((void**)&c->vprev, ng * sizeof(double)), "vprev"));
        SGW_TRY(check_cuda(cudaMalloc((void**)&c->phase_last, ng * sizeof(cd)), "phase_last"));
    }
    for (int step = 0; step < nsteps; ++step) {
        if (c->hartree_mode || step == 0) {
            const double* vh = nullptr;
            if (c->hartree_mode) {
                SGW_TRY(hartree_into(c, nvec, psi, c->rho_scale, nullptr, fuse_density && step > 0, merged));
                vh = c->vh;
                if (fuse_density && step + 1 < nsteps)
                    SGW_TRY(check_cuda(cudaMemsetAsync(c->rho, 0, ng * sizeof(double), c->stream), "rho reset"));
            }
            if (!merged) {
                phase_kernel<<<blocks_for(ng, 256), 256, 0, c->stream>>>(c->vloc, vh, 0.5 * dt, c->phase, ng);
                SGW_TRY(launched(c, "phase"));
            }
        }
        const bool last = step + 1 == nsteps;
        if (merged && (c->hartree_mode || step <= 1 || last)) {
            // frozen V: the merged table is exp(-i V dt/2) in step 0 and exp(-i V dt) from step 1 on
            phase_merge_kernel<<<blocks_for(ng, 256), 256, 0, c->stream>>>(c->vloc, c->hartree_mode ? c->pois : nullptr, c->vprev,
                                                                            0.5 * dt, step == 0 ? 1 : 0, c->phase,
                                                                            last ? c->phase_last : nullptr, ng);
            SGW_TRY(launched(c, "phase_merge"));
        }
        const int chunk = (!kb && c->l2_chunk > 0 && c->l2_chunk < nvec) ? c->l2_chunk : nvec;
        for (int cv = 0; cv < nvec; cv += chunk) {            // chunks small enough to stay in L2 across the 3 passes
            const int nc = (nvec - cv < chunk) ? nvec - cv : chunk;
            cd* ps = psi + (long long)cv * ng;
            OpParams p = zero_params();
            p.out = ps;
            // lean passes with KB: the potential phases stay fused in the passes (on load in x, on store in z); the
            // KB factors, which sit between them, are conjugated by the phase at their sphere points instead:
            //   P (psi + conj(P) S[P psi]) = P psi + S[P psi]   and   P psi3 + P S[conj(P) (P psi3)] = P (psi3 + S[psi3])
            const bool kb_fold = kb && c->use_engine == 2;
            if (kb_fold) {
                SGW_TRY(kb_apply(c, nc, ps, ps, 1, 0.5 * dt, c->phase, +1));
            } else if (kb) {
                dim3 g2(blocks_for(ng, 256), nc);
                apply_phase_kernel<<<g2, 256, 0, c->stream>>>(ps, c->phase, ng);
                SGW_TRY(launched(c, "apply_phase"));
                SGW_TRY(kb_apply(c, nc, ps, ps, 1, 0.5 * dt));
            } else {
                p.pro_phase = c->phase;
            }
            int rp = 1;
            if (c->use_engine) {
                SGW_TRY(c->use_engine == 2 ? lean_td_step(c, nc, ps, kb && !kb_fold, fuse_density && step + 1 < nsteps, merged, last)
                                           : eng_td_step(c, nc, ps, kb));
                rp = 2;
            } else {
                rp = run_plane(c, PL_TD, nc, ps, ps, p.pro_phase, false);
            }
            if (rp < 0) return rp;
            if (rp == 1) {
                p.mul_c = c->td_kin[0];
                SGW_TRY(run_pass(c, 0, K_RT_TD, nc, ps, p));
                p.pro_phase = nullptr; p.mul_c = c->td_kin[1];
                SGW_TRY(run_pass(c, 1, K_RT_TD, nc, ps, p));
            }
            p.pro_phase = nullptr;
            p.mul_c = c->td_kin[2];
            if (!kb) p.epi_phase = c->phase;
            if (rp != 2) SGW_TRY(run_pass(c, 2, K_RT_TD, nc, ps, p));
            if (kb_fold) {
                SGW_TRY(kb_apply(c, nc, ps, ps, 1, 0.5 * dt, c->phase, -1));
            } else if (kb) {
                SGW_TRY(kb_apply(c, nc, ps, ps, 1, 0.5 * dt));
                dim3 g2(blocks_for(ng, 256), nc);
                apply_phase_kernel<<<g2, 256, 0, c->stream>>>(ps, c->phase, ng);
                SGW_TRY(launched(c, "apply_phase"));
            }
        }
    }
    return SGW_OK;
}
