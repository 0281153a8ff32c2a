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

// the real family (H apply, Chebyshev filter) runs through the TMA accumulate kernel where it is built (cubic grids,
// axis length a multiple of 8) and enabled (SGW_ACC=0/1; default: on from 64 points per axis; smaller grids are
// launch-bound and keep the register-operand passes with their cached graph)
bool acc_enabled(const sgw_ctx* c) {
    if (!c->acc) return false;
    if (c->use_acc >= 0) return c->use_acc != 0;
    return c->nx >= 64;
}

int launched(sgw_ctx* c, const char* what) {
    c->launches++;
    return check_cuda(cudaGetLastError(), what);
}

}  // namespace
int sgw::ensure_ws(sgw_ctx* c, int n) {
    for (int a = 0; a < n && a < 2; ++a)
        if (!c->ws[a])
            SGW_TRY(check_cuda(cudaMalloc((void**)&c->ws[a], (size_t)c->max_nvec * c->ng * sizeof(cd)), "workspace"));
    return 0;
}

namespace {
template <int NP>
int kb_apply_np(sgw_ctx* c, int nvec, const cd* src, cd* dst, int mode, double scale_or_tau, const cd* phase, int fold) {
    dim3 grid(c->nsphere, (nvec + KB_VB - 1) / KB_VB);
    const double dV = c->hx * c->hy * c->hz;
    // fold = +1: projections of phase*src, contribution times conj(phase)  (opening half step: the pass multiplies by phase on load)
    // fold = -1: projections of conj(phase)*src, contribution times phase  (closing half step: the pass multiplied by phase on store)
    cudaEvent_t e1 = prof_begin(c, K_KB_PROJECT);
    kb_project_kernel<NP><<<grid, 128, 0, c->stream>>>(src, c->ng, nvec, c->sph_ptr, c->sph_idx, c->beta, dV, c->kbc, c->nsphere,
                                                       fold ? phase : nullptr, fold < 0 ? 1 : 0);
    prof_end(c, e1);
    SGW_TRY(launched(c, "kb_project"));
    e1 = prof_begin(c, K_KB_SCATTER);
    kb_scatter_kernel<NP><<<grid, 128, 0, c->stream>>>(dst, c->ng, nvec, c->sph_ptr, c->sph_idx, c->beta, c->D, c->kbc,
                                                       c->nsphere, mode, scale_or_tau, fold ? phase : nullptr, fold > 0 ? 1 : 0);
    prof_end(c, e1);
    return launched(c, "kb_scatter");
}

// dst += sum beta f <beta|src>, all projections taken from src before any scatter (R-11)
}  // namespace
int sgw::kb_apply(sgw_ctx* c, int nvec, const cd* src, cd* dst, int mode, double scale_or_tau, const cd* phase, int fold) {
    if (c->nsphere == 0) return 0;
    if (nvec > c->max_nvec) return set_error(SGW_EINVAL, "kb_apply: more vectors than max_nvec");
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

// what the last inverse pass of the Poisson solve writes
struct HartreeOut {
    double* vh = nullptr;        // V_H itself (sgw_hartree), or
    bool merge = false;          // the merged half-step phase tables of the propagator (R-8): c->phase, c->vprev, ...
    int first = 0;
    double half_dt = 0.0;
    cd* last = nullptr;
    double* rho_reset = nullptr;
};

// rho = scale * sum |psi|^2 ; V_H by the cut-Coulomb Poisson solve (R-10): forward x (straight from the real density),
// forward y, z round trip with v(k)/N_g, inverse y, inverse x (which writes V_H or the phase tables): five launches.
int hartree_into(sgw_ctx* c, int nvec, const cd* psi, double rho_scale, double* rho2, bool rho_ready, const HartreeOut& o) {
    const long long ng = c->ng;
    if (!rho_ready) {          // otherwise c->rho was accumulated by the last pass of the previous step
        cudaEvent_t e1 = prof_begin(c, K_DENSITY);
        density_kernel<<<blocks_for(ng, 256), 256, 0, c->stream>>>(psi, nvec, ng, rho_scale, c->rho, rho2);
        prof_end(c, e1);
        SGW_TRY(launched(c, "density"));
    }
    OpParams p = zero_params();
    p.out = c->pois;
    p.rin = c->rho;
    SGW_TRY(run_pass(c, 0, K_FWD, 1, c->pois, p));
    p.rin = nullptr;
    SGW_TRY(run_pass(c, 1, K_FWD, 0, c->pois, p));
    p.mul3d = c->vk3d;
    SGW_TRY(run_pass(c, 2, K_RT_MUL3D, 0, c->pois, p));
    p.mul3d = nullptr;
    SGW_TRY(run_pass(c, 1, K_INV, 0, c->pois, p));
    if (o.merge) {
        p.vloc = c->vloc; p.vprev = c->vprev; p.table = c->phase; p.last = o.last; p.rho_reset = o.rho_reset;
        p.half_dt = o.half_dt; p.first = o.first;
        return run_pass(c, 0, K_INV, 1, c->pois, p);
    }
    p.vh_out = o.vh;
    return run_pass(c, 0, K_INV, 2, c->pois, p);
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
    double la = 0.0, lb = 0.0;
    SGW_TRY(power_iteration(c, 0.0, niter, seed, 0, c->red, &la));
    SGW_TRY(power_iteration(c, la, niter, seed, 1, c->red, &lb));
    *h_emin = la < lb ? la : lb;
    *h_emax = la < lb ? lb : la;
    return SGW_OK;
}

// dependent-free DFMA chains: 8 independent accumulators per thread, 32 warps per SM
static __global__ void __launch_bounds__(1024) fp64_probe_kernel(double* out, int iters, double a, double b) {
    double x[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) x[j] = 1.0 + 1e-3 * (threadIdx.x + j);
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int j = 0; j < 8; ++j) x[j] = fma(x[j], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int j = 0; j < 8; ++j) s += x[j];
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

extern "C" int sgw_probe_fp64(sgw_ctx* c, double* h_flops_per_s) {
    if (!c || !h_flops_per_s) return set_error(SGW_EINVAL, "sgw_probe_fp64: bad argument");
    const int blocks = 2 * c->num_sms, threads = 1024, iters = 1 << 15;
    double* buf = nullptr;
    SGW_TRY(check_cuda(cudaMalloc((void**)&buf, (size_t)blocks * threads * sizeof(double)), "probe buffer"));
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    double best = 0.0;
    for (int rep = 0; rep < 4; ++rep) {          // the first repetition warms up
        cudaEventRecord(e0, c->stream);
        fp64_probe_kernel<<<blocks, threads, 0, c->stream>>>(buf, iters, 0.999999, 1e-6);
        cudaEventRecord(e1, c->stream);
        c->launches++;
        cudaError_t e = cudaEventSynchronize(e1);
        float ms = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
        if (e != cudaSuccess) { cudaFree(buf); cudaEventDestroy(e0); cudaEventDestroy(e1); return check_cuda(e, "fp64 probe"); }
        const double rate = 2.0 * 8.0 * (double)iters * blocks * threads / (ms * 1e-3);
        if (rep > 0 && rate > best) best = rate;
    }
    cudaFree(buf); cudaEventDestroy(e0); cudaEventDestroy(e1);
    *h_flops_per_s = best;
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
        if (c->ecut > 0.0) SGW_TRY(cut_apply_H(c, nv, i0, o0));
        else SGW_TRY(acc_enabled(c) ? acc_apply_H(c, nv, i0, o0) : lean_apply_H(c, nv, i0, o0));
        SGW_TRY(kb_apply(c, nv, i0, o0, 0, 1.0));
    }
    return SGW_OK;
}

extern "C" int sgw_hartree(sgw_ctx* c, int nvec, const void* d_psi, double rho_scale, double* d_vh, double* d_rho) {
    if (!c || nvec < 0 || (nvec > 0 && !d_psi) || !d_vh) return set_error(SGW_EINVAL, "sgw_hartree: bad argument");
    HartreeOut o;
    o.vh = d_vh;
    return hartree_into(c, nvec, (const cd*)d_psi, rho_scale, d_rho, false, o);
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
    SGW_TRY(ensure_ws(c, 2));
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
        if (c->ecut > 0.0) SGW_TRY(cut_cheb_filter(c, nv, X0, h_coeffs, s, nterms));
        else SGW_TRY(acc_enabled(c) ? acc_cheb_filter(c, nv, X0, h_coeffs, s, nterms) : lean_cheb_filter(c, nv, X0, h_coeffs, s, nterms));
    }
    return SGW_OK;
}

// Small grids are launch-bound (cfg0: 2 MB per array, 256 launches of a few us each): when a call repeats with the
// same vector block, window and coefficients, its launches are captured on an internal stream, instantiated as a
// CUDA graph and replayed on the caller's stream from then on (the first call with a key launches plainly).  SGW_GRAPH=0 disables, SGW_GRAPH_BYTES moves
// the size limit (bytes of one vector block; default 16 MB); both are read when the context is created.
bool filter_graph_wanted(const sgw_ctx* c, int nvec, int nterms) {
    if (!c->graph_on || c->prof_on || c->nsphere > 0 || nvec > c->max_nvec || nterms < 3 || c->ecut > 0.0) return false;
    return (double)nvec * (double)c->ng * sizeof(cd) <= c->graph_bytes;
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
    if (c->ecut > 0.0) return cut_td_propagate(c, nvec, psi, dt, nsteps);
    if (!c->td_kin_valid || c->td_dt != dt) {
        // exp(-i 1/2 k^2 dt)/N per axis, built on the device from the 1/2 k^2 tables (no host synchronisation)
        for (int a = 0; a < 3; ++a) {
            td_table_kernel<<<blocks_for(c->dims[a], 128), 128, 0, c->stream>>>(c->kin_raw[a], dt, c->td_kin[a], c->dims[a]);
            SGW_TRY(launched(c, "td_table"));
        }
        c->td_dt = dt; c->td_kin_valid = true;
    }
    const bool kb = c->nsphere > 0;
    // The last pass of a step accumulates the density of its result (atomics), so only the first step of a call reads
    // the vectors for the density.  With KB the closing nonlocal factor changes the vectors at the sphere points after that pass: the accumulated
    // density is corrected there (minus the old values before the factor, plus the new ones after it) instead of
    // reading all vectors again.
    const bool fuse_density = c->hartree_mode != 0;
    // consecutive half-step potential factors are merged into one table applied on load (R-8).  With KB the closing
    // factor of step n and the opening one of step n+1 are adjacent as well (the KB factors sit inside them), so the
    // merged table serves both cases.
    const bool merged = true;
    int chunk = nvec < c->max_nvec ? nvec : c->max_nvec;
    if (!kb && c->l2_chunk > 0 && c->l2_chunk < chunk) chunk = c->l2_chunk;   // chunks small enough to stay in L2 across the passes
    for (int step = 0; step < nsteps; ++step) {
        const bool last = step + 1 == nsteps;
        if (c->hartree_mode) {
            HartreeOut o;
            o.merge = true; o.first = step == 0 ? 1 : 0; o.half_dt = 0.5 * dt; o.last = last ? c->phase_last : nullptr;
            o.rho_reset = (fuse_density && !last) ? c->rho : nullptr;
            SGW_TRY(hartree_into(c, nvec, psi, c->rho_scale, nullptr, fuse_density && step > 0, o));
        } else if (step <= 1 || last) {
            // frozen V: the merged table is exp(-i V dt/2) in step 0 and exp(-i V dt) from step 1 on
            phase_merge_kernel<<<blocks_for(ng, 256), 256, 0, c->stream>>>(c->vloc, c->vprev, 0.5 * dt, step == 0 ? 1 : 0,
                                                                            c->phase, last ? c->phase_last : nullptr, ng);
            SGW_TRY(launched(c, "phase_merge"));
        }
        for (int cv = 0; cv < nvec; cv += chunk) {
            const int nc = (nvec - cv < chunk) ? nvec - cv : chunk;
            cd* ps = psi + (long long)cv * ng;
            // with KB: the potential phases stay fused in the passes (on load in x, on store in z); the KB factors,
            // which sit between them, are conjugated by the phase at their sphere points instead:
            //   P (psi + conj(P) S[P psi]) = P psi + S[P psi]   and   P psi3 + P S[conj(P) (P psi3)] = P (psi3 + S[psi3])
            // opening KB factor: conjugated by the (merged) table the x pass multiplies by on load; closing KB factor:
            // plain, because the closing potential factor is deferred to the next step's load -- except in the last
            // step of the call, where the z pass multiplies by phase_last on store
            if (kb) SGW_TRY(kb_apply(c, nc, ps, ps, 1, 0.5 * dt, c->phase, +1));
            SGW_TRY(lean_td_step(c, nc, ps, false, fuse_density && !last, merged, last));
            const bool fix = kb && fuse_density && !last && c->nuniq > 0;
            if (fix) {
                cudaEvent_t e1 = prof_begin(c, 1 * K_NKINDS + K_DENSITY);     // booked under axis 1 of the density kind
                density_points_kernel<<<blocks_for(c->nuniq, 128), 128, 0, c->stream>>>(ps, nc, ng, c->sph_uniq, c->nuniq, -c->rho_scale, c->rho);
                prof_end(c, e1);
                SGW_TRY(launched(c, "density_points"));
            }
            if (kb) SGW_TRY(last ? kb_apply(c, nc, ps, ps, 1, 0.5 * dt, c->phase_last, -1) : kb_apply(c, nc, ps, ps, 1, 0.5 * dt));
            if (fix) {
                cudaEvent_t e1 = prof_begin(c, 1 * K_NKINDS + K_DENSITY);     // booked under axis 1 of the density kind
                density_points_kernel<<<blocks_for(c->nuniq, 128), 128, 0, c->stream>>>(ps, nc, ng, c->sph_uniq, c->nuniq, c->rho_scale, c->rho);
                prof_end(c, e1);
                SGW_TRY(launched(c, "density_points"));
            }
        }
    }
    return SGW_OK;
}

// =====================================================================================================
// NEXT-2: perturbed / unperturbed pair propagation with the xi projection of both Hartree potentials
// =====================================================================================================
extern "C" int sgw_apply_kick(sgw_ctx* c, int nvec, void* d_psi, const double* d_vpert, double lambda) {
    if (!c || nvec < 0 || (nvec > 0 && (!d_psi || !d_vpert))) return set_error(SGW_EINVAL, "sgw_apply_kick: bad argument");
    if (nvec == 0) return SGW_OK;
    dim3 grid(blocks_for(c->ng, 256), nvec);
    kick_kernel<<<grid, 256, 0, c->stream>>>((cd*)d_psi, d_vpert, lambda, c->ng);
    return launched(c, "kick_kernel");
}

namespace {
// one split-operator step of one copy with the Hartree potential already in c->vh (potential half steps on load in x and
// on store in z, KB factors conjugated by the phase: the same step as sgw_td_propagate, without the merged tables)
int pair_step(sgw_ctx* c, int nvec, cd* psi, double dt) {
    const long long ng = c->ng;
    const bool kb = c->nsphere > 0;
    phase_kernel<<<blocks_for(ng, 256), 256, 0, c->stream>>>(c->vloc, c->vh, 0.5 * dt, c->phase, ng);
    SGW_TRY(launched(c, "phase"));
    const int chunk = nvec < c->max_nvec ? nvec : c->max_nvec;
    for (int cv = 0; cv < nvec; cv += chunk) {
        const int nc = (nvec - cv < chunk) ? nvec - cv : chunk;
        cd* ps = psi + (long long)cv * ng;
        if (kb) SGW_TRY(kb_apply(c, nc, ps, ps, 1, 0.5 * dt, c->phase, +1));
        SGW_TRY(lean_td_step(c, nc, ps, false, false, false, false));     // phase on load in x, on store in z
        if (kb) SGW_TRY(kb_apply(c, nc, ps, ps, 1, 0.5 * dt, c->phase, -1));
    }
    return SGW_OK;
}
}  // namespace

extern "C" int sgw_td_propagate_pair(sgw_ctx* c, int nvec, void* d_psi, void* d_psi_lambda, double dt, int nsteps, uint64_t xi_seed,
                                     int nxi, int nfrag, double* d_out) {
    if (!c || nvec < 0 || nsteps < 0 || nxi < 0 || nfrag < 0 || (nvec > 0 && (!d_psi || !d_psi_lambda)) || d_psi == d_psi_lambda ||
        (nxi > 0 && nsteps > 0 && !d_out))
        return set_error(SGW_EINVAL, "sgw_td_propagate_pair: bad argument");
    if (c->ng % 32) return set_error(SGW_ESIZE, "sgw_td_propagate_pair: N_g must be a multiple of the segment length 32");
    if (c->ecut > 0.0) return set_error(SGW_EINVAL, "sgw_td_propagate_pair: not available with a kinetic-energy cutoff");
    if (nvec == 0 || nsteps == 0) return SGW_OK;
    if (!c->td_kin_valid || c->td_dt != dt) {
        for (int a = 0; a < 3; ++a) {
            td_table_kernel<<<blocks_for(c->dims[a], 128), 128, 0, c->stream>>>(c->kin_raw[a], dt, c->td_kin[a], c->dims[a]);
            SGW_TRY(launched(c, "td_table"));
        }
        c->td_dt = dt; c->td_kin_valid = true;
    }
    const double dV = c->hx * c->hy * c->hz;
    if (nxi > 0) SGW_TRY(check_cuda(cudaMemsetAsync(d_out, 0, (size_t)nsteps * nxi * 2 * sizeof(double), c->stream), "clear projections"));
    cd* copy[2] = {(cd*)d_psi, (cd*)d_psi_lambda};
    for (int n = 0; n < nsteps; ++n) {
        for (int k = 0; k < 2; ++k) {
            // V_H[rho_copy(t_n)] -> c->vh, its xi projections, then the step of this copy under V_loc + that potential
            HartreeOut o;
            o.vh = c->vh;
            SGW_TRY(hartree_into(c, nvec, copy[k], c->rho_scale, nullptr, false, o));
            if (nxi > 0) {
                xi_project_kernel<<<nxi, 256, 0, c->stream>>>(c->vh, c->ng, sm64(xi_seed), nfrag, dV, d_out + ((size_t)n * nxi) * 2 + k, 2);
                SGW_TRY(launched(c, "xi_project"));
            }
            SGW_TRY(pair_step(c, nvec, copy[k], dt));
        }
    }
    return SGW_OK;
}

// =====================================================================================================
// NEXT-4: zeta pair with its projections, time-ordering, Sigma(t)
// =====================================================================================================
extern "C" int sgw_td_propagate_zeta(sgw_ctx* c, void* d_pair, const double* d_phi, double dt, int nsteps, uint64_t xi_seed, int nxi,
                                     int nfrag, void* d_out) {
    if (!c || !d_pair || nsteps < 0 || nxi < 0 || nfrag < 0 || (nxi > 0 && nsteps > 0 && (!d_out || !d_phi)))
        return set_error(SGW_EINVAL, "sgw_td_propagate_zeta: bad argument");
    if (c->ng % 32) return set_error(SGW_ESIZE, "sgw_td_propagate_zeta: N_g must be a multiple of the segment length 32");
    if (nsteps == 0) return SGW_OK;
    const double dV = c->hx * c->hy * c->hz;
    const int saved_mode = c->hartree_mode;
    c->hartree_mode = 0;                                   // the pair moves under the frozen potential (R-25)
    cd* pair = (cd*)d_pair;
    cd* out = (cd*)d_out;
    int rc = SGW_OK;
    if (nxi > 0) rc = check_cuda(cudaMemsetAsync(d_out, 0, (size_t)nsteps * nxi * 2 * sizeof(cd), c->stream), "clear projections");
    for (int n = 0; n < nsteps && !rc; ++n) {
        for (int k = 0; k < 2 && !rc; ++k) {
            if (nxi > 0) {
                xi_project_weighted_kernel<<<nxi, 256, 0, c->stream>>>(pair + (long long)k * c->ng, d_phi, c->ng, sm64(xi_seed), nfrag, dV,
                                                                       out + ((size_t)n * nxi) * 2 + k, 2);
                rc = launched(c, "xi_project_weighted");
            }
            if (!rc) rc = sgw_td_propagate(c, 1, pair + (long long)k * c->ng, k == 0 ? -dt : dt, 1);
        }
    }
    c->hartree_mode = saved_mode;
    return rc;
}

extern "C" int sgw_time_order(sgw_ctx* c, int nxi, int nt, const double* d_cr, int64_t stride_n, int64_t stride_m, void* d_ct) {
    if (!c || nxi < 0 || nt < 0 || (nxi > 0 && nt > 0 && (!d_cr || !d_ct))) return set_error(SGW_EINVAL, "sgw_time_order: bad argument");
    if (nxi == 0 || nt == 0) return SGW_OK;
    const size_t smem = (size_t)(nt + (nt & 1)) * sizeof(double) + (size_t)2 * nt * sizeof(cd);
    if (smem > 200 * 1024) return set_error(SGW_ESIZE, "sgw_time_order: series too long (at most about 5000 samples)");
    if (smem > 48 * 1024)
        SGW_TRY(check_cuda(cudaFuncSetAttribute(time_order_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem), "time_order attribute"));
    time_order_kernel<<<nxi, 256, smem, c->stream>>>(d_cr, stride_n, stride_m, nt, nxi, (cd*)d_ct);
    return launched(c, "time_order");
}

extern "C" int sgw_sigma_t(sgw_ctx* c, int nt, int nxi, int nfrag, const void* d_ct, const void* d_p, void* d_sigma) {
    if (!c || nt < 0 || nxi <= 0 || nfrag <= 0 || (nt > 0 && (!d_ct || !d_p || !d_sigma))) return set_error(SGW_EINVAL, "sgw_sigma_t: bad argument");
    if (nt == 0) return SGW_OK;
    const double dV = c->hx * c->hy * c->hz;
    const double norm = (double)c->ng / ((double)nxi * (double)nfrag * 32.0 * dV);
    sigma_kernel<<<nt, 256, 0, c->stream>>>((const cd*)d_ct, (const cd*)d_p, nxi, norm, (cd*)d_sigma);
    return launched(c, "sigma");
}
