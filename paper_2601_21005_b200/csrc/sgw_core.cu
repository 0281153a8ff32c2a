// sgw_core.cu -- context, tables, pass geometry, setup entry points of libsgw (include/sgw.h).
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <algorithm>
#include <cstring>

#include "sgw_ctx.h"

#define SGW_DECL(N)                                             \
    extern "C" int sgw_pass_launch_##N(const sgw::PassCall*);   \
    extern "C" int sgw_lean_launch_##N(const sgw::LeanCall*, int);  \
    extern "C" int sgw_acc_launch_##N(const sgw::AccCall*);         \
    extern "C" int sgw_td_launch_##N(const sgw::TdCall*);
SGW_DECL(8) SGW_DECL(12) SGW_DECL(16) SGW_DECL(24) SGW_DECL(32) SGW_DECL(48) SGW_DECL(64) SGW_DECL(96)
SGW_DECL(128) SGW_DECL(192) SGW_DECL(256) SGW_DECL(384)
#undef SGW_DECL

namespace sgw {

static thread_local std::string g_err;

int set_error(int code, const std::string& msg) {
    g_err = msg;
    return code;
}
int check_cuda(cudaError_t e, const char* what) {
    if (e == cudaSuccess) return 0;
    return set_error(e == cudaErrorMemoryAllocation ? SGW_ENOMEM : SGW_ECUDA,
                     std::string(what) + ": " + cudaGetErrorString(e));
}

#define SGW_SIZES(X) X(8) X(12) X(16) X(24) X(32) X(48) X(64) X(96) X(128) X(192) X(256) X(384)
static pass_launch_fn launcher_for(int n) {
    switch (n) {
#define SGW_CASE(N) case N: return sgw_pass_launch_##N;
        SGW_SIZES(SGW_CASE)
#undef SGW_CASE
        default: return nullptr;
    }
}
static acc_launch_fn acc_launcher_for(int n) {
    switch (n) {
#define SGW_CASE(N) case N: return sgw_acc_launch_##N;
        SGW_SIZES(SGW_CASE)
#undef SGW_CASE
        default: return nullptr;
    }
}
static td_launch_fn td_launcher_for(int n) {
    switch (n) {
#define SGW_CASE(N) case N: return sgw_td_launch_##N;
        SGW_SIZES(SGW_CASE)
#undef SGW_CASE
        default: return nullptr;
    }
}
static lean_launch_fn lean_launcher_for(int n) {
    switch (n) {
#define SGW_CASE(N) case N: return sgw_lean_launch_##N;
        SGW_SIZES(SGW_CASE)
#undef SGW_CASE
        default: return nullptr;
    }
}

// event pair around a launch while profiling is on: returns the closing event (or nullptr)
cudaEvent_t prof_begin(sgw_ctx* c, int tag) {
    if (!c->prof_on || c->prof_used >= 60000) return nullptr;
    if (c->prof_ev.size() < 2 * (c->prof_used + 1)) {
        cudaEvent_t a, b;
        if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) return nullptr;
        c->prof_ev.push_back(a); c->prof_ev.push_back(b); c->prof_tag.push_back(0);
    }
    c->prof_tag[c->prof_used] = tag;
    cudaEventRecord(c->prof_ev[2 * c->prof_used], c->stream);
    return c->prof_ev[2 * c->prof_used + 1];
}
void prof_end(sgw_ctx* c, cudaEvent_t e1) {
    if (!e1) return;
    cudaEventRecord(e1, c->stream);
    c->prof_used++;
}

PassGeom geom_for_axis(const sgw_ctx* c, int axis, int nvec, long long* ntiles) {
    PassGeom g;
    g.ng = c->ng;
    const long long nxy = (long long)c->nx * c->ny;
    if (axis == 0) {                 // contiguous pencils: tile = Bx consecutive rows
        g.fastn = 1; g.B = c->Bx; g.sN = 1; g.sB = c->nx;
        g.TI = (int)((long long)c->ny * c->nz / c->Bx); g.SI = (long long)c->Bx * c->nx; g.SO = c->ng; g.GO = 1;
        *ntiles = (long long)g.TI * nvec;
    } else if (axis == 1) {          // tile = B consecutive x at fixed (z, vec)
        g.fastn = 0; g.B = c->B; g.sN = c->nx; g.sB = 1;
        g.TI = c->nx / c->B; g.SI = c->B; g.SO = nxy; g.GO = c->nz;
        *ntiles = (long long)g.TI * c->nz * nvec;
    } else {                         // tile = B consecutive xy points at fixed vec
        g.fastn = 0; g.B = c->B; g.sN = nxy; g.sB = 1;
        g.TI = (int)(nxy / c->B); g.SI = c->B; g.SO = c->ng; g.GO = 1;
        *ntiles = (long long)g.TI * nvec;
    }
    return g;
}

int run_pass(sgw_ctx* c, int axis, int kind, int variant, const cd* in, const OpParams& p, int nvec) {
    PassCall call;
    call.kind = kind;
    call.variant = variant;
    call.gm = geom_for_axis(c, axis, nvec, &call.ntiles);
    call.in = in;
    call.tw = c->tw[axis];
    call.p = p;
    call.stream = c->stream;
    if (call.ntiles <= 0) return 0;
    if (call.ntiles > 0x7fffffffLL) return set_error(SGW_EINVAL, "too many tiles for one launch");
    cudaEvent_t e1 = prof_begin(c, axis * K_NKINDS + kind);
    int rc = c->pass[axis](&call);
    if (rc != 0) return set_error(SGW_ECUDA, std::string("pass launch failed: ") + cudaGetErrorString(cudaGetLastError()));
    prof_end(c, e1);
    c->launches++;
    return 0;
}

static void prof_collect(sgw_ctx* c) {
    cudaStreamSynchronize(c->stream);
    for (size_t i = 0; i < c->prof_used; ++i) {
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, c->prof_ev[2 * i], c->prof_ev[2 * i + 1]) == cudaSuccess) {
            c->prof_ms[c->prof_tag[i]] += ms;
            c->prof_n[c->prof_tag[i]]++;
        }
    }
    c->prof_used = 0;
}

template <class T>
static int dev_alloc(T** p, size_t n) {
    *p = nullptr;
    if (n == 0) return 0;
    return check_cuda(cudaMalloc((void**)p, n * sizeof(T)), "cudaMalloc");
}
template <class T>
static int upload(T* d, const T* h, size_t n, cudaStream_t s) {
    int rc = check_cuda(cudaMemcpyAsync(d, h, n * sizeof(T), cudaMemcpyHostToDevice, s), "cudaMemcpyAsync");
    if (rc) return rc;
    return check_cuda(cudaStreamSynchronize(s), "cudaStreamSynchronize");
}

}  // namespace sgw

using namespace sgw;

// v(k)/N_g on the grid's k layout (R-10)
static __global__ void vk3d_kernel(double* vk, int nx, int ny, int nz, double hx, double hy, double hz, double Rc) {
    const long long ng = (long long)nx * ny * nz;
    const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= ng) return;
    const int ix = (int)(i % nx), iy = (int)((i / nx) % ny), iz = (int)(i / ((long long)nx * ny));
    const double pi = 3.14159265358979323846;
    const int mx = (2 * ix >= nx) ? ix - nx : ix, my = (2 * iy >= ny) ? iy - ny : iy, mz = (2 * iz >= nz) ? iz - nz : iz;
    const double kx = 2 * pi * mx / (nx * hx), ky = 2 * pi * my / (ny * hy), kz = 2 * pi * mz / (nz * hz);
    const double k2 = kx * kx + ky * ky + kz * kz;
    const double v = (k2 == 0.0) ? 2 * pi * Rc * Rc : 4 * pi * (1.0 - cos(sqrt(k2) * Rc)) / k2;
    vk[i] = v / (double)ng;
}

extern "C" const char* sgw_last_error(void) { return g_err.c_str(); }

extern "C" int64_t sgw_launch_count(const sgw_ctx* c) { return c ? c->launches : 0; }

extern "C" int sgw_profile_enable(sgw_ctx* c, int on) {
    if (!c) return set_error(SGW_EINVAL, "sgw_profile_enable: null context");
    if (c->prof_on) sgw::prof_collect(c);
    c->prof_on = on != 0;
    return SGW_OK;
}

extern "C" int sgw_profile_reset(sgw_ctx* c) {
    if (!c) return set_error(SGW_EINVAL, "sgw_profile_reset: null context");
    sgw::prof_collect(c);
    for (int i = 0; i < 3 * K_NKINDS; ++i) { c->prof_ms[i] = 0; c->prof_n[i] = 0; }
    return SGW_OK;
}

extern "C" int sgw_profile_get(sgw_ctx* c, int axis, int kind, int64_t* count, double* total_ms) {
    if (!c || axis < 0 || axis > 2 || kind < 0 || kind >= K_NKINDS || !count || !total_ms)
        return set_error(SGW_EINVAL, "sgw_profile_get: bad argument");
    sgw::prof_collect(c);
    *count = c->prof_n[axis * K_NKINDS + kind];
    *total_ms = c->prof_ms[axis * K_NKINDS + kind];
    return SGW_OK;
}

extern "C" int sgw_sync_check(sgw_ctx* c) {
    if (!c) return set_error(SGW_EINVAL, "sgw_sync_check: null context");
    int rc = check_cuda(cudaStreamSynchronize(c->stream), "sgw_sync_check");
    if (rc) return rc;
    return check_cuda(cudaGetLastError(), "sgw_sync_check");
}

void sgw::drop_filter_graph(sgw_ctx* c) {
    if (c->fgraph) { cudaGraphExecDestroy(c->fgraph); c->fgraph = nullptr; }
    c->fg_psi = nullptr;
}

extern "C" int sgw_destroy(sgw_ctx* c) {
    if (!c) return SGW_OK;
    cudaStreamSynchronize(c->stream);
    sgw::drop_filter_graph(c);
    if (c->gstream) cudaStreamDestroy(c->gstream);
    for (cudaEvent_t e : c->prof_ev) cudaEventDestroy(e);
    for (int a = 0; a < 3; ++a) {
        cudaFree(c->tw[a]); cudaFree(c->kin[a]); cudaFree(c->kin_raw[a]); cudaFree(c->cheb_kin[a]); cudaFree(c->td_kin[a]);
    }
    cudaFree(c->ws[0]); cudaFree(c->ws[1]);
    cudaFree(c->vloc); cudaFree(c->vtab); cudaFree(c->vk3d); cudaFree(c->sph_ptr); cudaFree(c->sph_idx); cudaFree(c->sph_uniq);
    cudaFree(c->beta); cudaFree(c->D); cudaFree(c->kbc); cudaFree(c->pois); cudaFree(c->rho); cudaFree(c->vh);
    cudaFree(c->phase); cudaFree(c->phase_last); cudaFree(c->vprev); cudaFree(c->red); cudaFree(c->team_cnt); cudaFree(c->kin3d); cudaFree(c->td_kin3d); cudaFree(c->wcut);
    delete c;
    return SGW_OK;
}

static int env_int(const char* name, int dflt) {
    const char* e = getenv(name);
    return e ? atoi(e) : dflt;
}

extern "C" int sgw_init_grid(sgw_ctx** out, int nx, int ny, int nz, double hx, double hy, double hz, int max_nvec,
                             void* cuda_stream) {
    if (!out || nx <= 0 || ny <= 0 || nz <= 0 || !(hx > 0) || !(hy > 0) || !(hz > 0) || max_nvec <= 0)
        return set_error(SGW_EINVAL, "sgw_init_grid: bad argument");
    const int dims[3] = {nx, ny, nz};
    for (int a = 0; a < 3; ++a)
        if (!launcher_for(dims[a]))
            return set_error(SGW_ESIZE, "sgw_init_grid: unsupported axis length " + std::to_string(dims[a]));
    if (nx % 4) return set_error(SGW_ESIZE, "sgw_init_grid: nx must be a multiple of 4");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0)
        return set_error(SGW_ECUDA, "sgw_init_grid: no CUDA device (there is no CPU fallback)");
    sgw_ctx* c = new sgw_ctx();      // value-initialised: every pointer NULL, every counter 0
    c->nx = nx; c->ny = ny; c->nz = nz; c->hx = hx; c->hy = hy; c->hz = hz;
    c->ng = (long long)nx * ny * nz;
    c->max_nvec = max_nvec;
    c->stream = (cudaStream_t)cuda_stream;
    int rc = check_cuda(cudaGetDevice(&c->device), "cudaGetDevice");
    if (!rc) rc = check_cuda(cudaDeviceGetAttribute(&c->num_sms, cudaDevAttrMultiProcessorCount, c->device), "SM count");
    c->B = (nx % 8 == 0) ? 8 : 4;
    c->Bx = ((long long)ny * nz) % 8 == 0 ? 8 : (((long long)ny * nz) % 4 == 0 ? 4 : 1);
    c->leanB = (nx % 8 == 0 && ny % 8 == 0) ? 8 : 4;
    // run-time switches (all read here, once per context; listed in include/sgw.h)
    c->lean_G = env_int("SGW_LEAN_G", 0);
    c->lean_ctas = env_int("SGW_LEAN_CTAS", 0);
    c->lean_cluster = env_int("SGW_LEAN_CLUSTER", -1);
    c->lean_team = env_int("SGW_LEAN_TEAM", -1);
    c->use_acc = env_int("SGW_ACC", -1);
    c->acc_pairz = (nx == 384 && ny == 384) ? env_int("SGW_ACC_PAIRZ", 1) : 0;
    c->acc_l2_bytes = 1.0e6 * env_int("SGW_ACC_L2_MB", 104);   // 128^3: 101 MB, one launch 0.61 ms against 0.76 ms in two
    c->acc = (nx == ny && ny == nz && nx >= 32 && nx % 8 == 0) ? acc_launcher_for(nx) : nullptr;
    {
        cudaDriverEntryPointQueryResult qr;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &c->tmap_encode, cudaEnableDefault, &qr) != cudaSuccess ||
            qr != cudaDriverEntryPointSuccess)
            c->tmap_encode = nullptr;
    }
    if (!c->tmap_encode) c->acc = nullptr;
    c->tdk = c->acc ? td_launcher_for(nx) : nullptr;
    c->use_acc_td = env_int("SGW_ACC_TD", -1);
    c->lean_vminor = env_int("SGW_LEAN_VMINOR", -1);
    c->lean_chunk = env_int("SGW_LEAN_CHUNK", 0);
    c->l2_chunk = env_int("SGW_L2_CHUNK", 0);
    c->pdl = env_int("SGW_PDL", 0) == 1;
    c->graph_on = env_int("SGW_GRAPH", 1) != 0;
    c->graph_bytes = 16.0e6;
    { const char* b = getenv("SGW_GRAPH_BYTES"); if (b && atof(b) > 0) c->graph_bytes = atof(b); }
    { const int b = env_int("SGW_LEAN_B", 0); if (b == 4 || (b == 8 && c->leanB == 8)) c->leanB = b; }
    const double hh[3] = {hx, hy, hz};
    for (int a = 0; a < 3 && !rc; ++a) {
        c->dims[a] = dims[a]; c->hs[a] = hh[a];
        c->pass[a] = launcher_for(dims[a]);
        c->lean[a] = lean_launcher_for(dims[a]);
        const int N = dims[a];
        std::vector<cd> tw(N);
        std::vector<double> kin(N), raw(N);
        for (int j = 0; j < N; ++j) {
            const long double ang = -2.0L * acosl(-1.0L) * (long double)j / (long double)N;
            tw[j] = make_double2((double)cosl(ang), (double)sinl(ang));
            const int m = (2 * j >= N) ? j - N : j;
            const long double k = 2.0L * acosl(-1.0L) * (long double)m / ((long double)N * (long double)hh[a]);
            raw[j] = (double)(0.5L * k * k);
            kin[j] = (double)(0.5L * k * k / (long double)N);
        }
        if (!rc) rc = dev_alloc(&c->tw[a], N);
        if (!rc) rc = dev_alloc(&c->kin[a], N);
        if (!rc) rc = dev_alloc(&c->kin_raw[a], N);
        if (!rc) rc = dev_alloc(&c->cheb_kin[a], N);
        if (!rc) rc = dev_alloc(&c->td_kin[a], N);
        if (!rc) rc = upload(c->tw[a], tw.data(), N, c->stream);
        if (!rc) rc = upload(c->kin[a], kin.data(), N, c->stream);
        if (!rc) rc = upload(c->kin_raw[a], raw.data(), N, c->stream);
    }
    if (!rc) rc = dev_alloc(&c->vtab, c->ng);
    if (!rc) rc = dev_alloc(&c->vk3d, c->ng);
    if (!rc) rc = dev_alloc(&c->pois, c->ng);
    if (!rc) rc = dev_alloc(&c->rho, c->ng);
    if (!rc) rc = dev_alloc(&c->vh, c->ng);
    if (!rc) rc = dev_alloc(&c->phase, c->ng);
    if (!rc) rc = dev_alloc(&c->phase_last, c->ng);
    if (!rc) rc = dev_alloc(&c->vprev, c->ng);
    if (!rc) rc = dev_alloc(&c->red, 4);
    if (!rc) rc = dev_alloc(&c->team_cnt, (size_t)max_nvec * nz);
    if (!rc) {
        const double Lx = nx * hx, Ly = ny * hy, Lz = nz * hz;
        const double Rc = 0.5 * fmin(Lx, fmin(Ly, Lz));
        vk3d_kernel<<<(unsigned)((c->ng + 255) / 256), 256, 0, c->stream>>>(c->vk3d, nx, ny, nz, hx, hy, hz, Rc);
        c->launches++;
        rc = check_cuda(cudaStreamSynchronize(c->stream), "vk3d_kernel");
    }
    if (rc) { sgw_destroy(c); return rc; }
    *out = c;
    return SGW_OK;
}

extern "C" int sgw_set_vloc(sgw_ctx* c, const double* d_vloc) {
    if (!c) return set_error(SGW_EINVAL, "sgw_set_vloc: null context");
    sgw::drop_filter_graph(c);
    if (!d_vloc) { cudaStreamSynchronize(c->stream); cudaFree(c->vloc); c->vloc = nullptr; return SGW_OK; }
    int rc = 0;
    if (!c->vloc) rc = dev_alloc(&c->vloc, c->ng);
    if (!rc) rc = check_cuda(cudaMemcpyAsync(c->vloc, d_vloc, c->ng * sizeof(double), cudaMemcpyDeviceToDevice, c->stream),
                             "sgw_set_vloc copy");
    if (!rc) rc = check_cuda(cudaStreamSynchronize(c->stream), "sgw_set_vloc");
    return rc;
}

extern "C" int sgw_set_nonlocal(sgw_ctx* c, int nsphere, const int64_t* d_ptr, const int32_t* d_idx, int nproj,
                                const double* d_beta, const double* d_D) {
    if (!c || nsphere < 0) return set_error(SGW_EINVAL, "sgw_set_nonlocal: bad argument");
    cudaStreamSynchronize(c->stream);
    sgw::drop_filter_graph(c);
    cudaFree(c->sph_ptr); cudaFree(c->sph_idx); cudaFree(c->beta); cudaFree(c->D); cudaFree(c->kbc); cudaFree(c->sph_uniq);
    c->sph_ptr = nullptr; c->sph_idx = nullptr; c->beta = nullptr; c->D = nullptr; c->kbc = nullptr; c->nsphere = 0;
    c->sph_uniq = nullptr; c->nuniq = 0;
    if (nsphere == 0) return SGW_OK;
    if (!d_ptr || !d_idx || !d_beta || !d_D || nproj < 1 || nproj > 8)
        return set_error(SGW_EINVAL, "sgw_set_nonlocal: bad argument");
    // every copy is ordered on the context's stream (the caller's arrays may have been produced on it, and a
    // non-blocking stream is not ordered against the legacy default stream), then one synchronisation
    cudaStream_t st = c->stream;
    int64_t npts = 0;
    int rc = check_cuda(cudaMemcpyAsync(&npts, d_ptr + nsphere, sizeof(int64_t), cudaMemcpyDeviceToHost, st), "read sph_ptr");
    if (!rc) rc = check_cuda(cudaStreamSynchronize(st), "read sph_ptr");
    if (rc) return rc;
    if (npts < 0) return set_error(SGW_EINVAL, "sgw_set_nonlocal: negative point count");
    if (!rc) rc = dev_alloc(&c->sph_ptr, (size_t)nsphere + 1);
    if (!rc) rc = dev_alloc(&c->sph_idx, (size_t)npts);
    if (!rc) rc = dev_alloc(&c->beta, (size_t)npts * nproj);
    if (!rc) rc = dev_alloc(&c->D, (size_t)nsphere * nproj);
    if (!rc) rc = dev_alloc(&c->kbc, (size_t)c->max_nvec * nsphere * nproj);      // no allocation inside the hot calls
    if (!rc) rc = check_cuda(cudaMemcpyAsync(c->sph_ptr, d_ptr, (nsphere + 1) * sizeof(int64_t), cudaMemcpyDeviceToDevice, st), "copy");
    if (!rc && npts) rc = check_cuda(cudaMemcpyAsync(c->sph_idx, d_idx, npts * sizeof(int32_t), cudaMemcpyDeviceToDevice, st), "copy");
    if (!rc && npts) rc = check_cuda(cudaMemcpyAsync(c->beta, d_beta, npts * nproj * sizeof(double), cudaMemcpyDeviceToDevice, st), "copy");
    if (!rc) rc = check_cuda(cudaMemcpyAsync(c->D, d_D, (size_t)nsphere * nproj * sizeof(double), cudaMemcpyDeviceToDevice, st), "copy");
    // the distinct sphere points (spheres overlap): where the closing nonlocal factor of a propagation step changes
    // the vectors after the last pass has accumulated their density (sgw_td_propagate)
    std::vector<int32_t> uniq((size_t)npts);
    if (!rc && npts) rc = check_cuda(cudaMemcpyAsync(uniq.data(), d_idx, npts * sizeof(int32_t), cudaMemcpyDeviceToHost, st), "read sph_idx");
    if (!rc) rc = check_cuda(cudaStreamSynchronize(st), "sgw_set_nonlocal");
    if (rc) return rc;
    std::sort(uniq.begin(), uniq.end());
    uniq.erase(std::unique(uniq.begin(), uniq.end()), uniq.end());
    if (!uniq.empty() && (uniq.front() < 0 || uniq.back() >= c->ng)) return set_error(SGW_EINVAL, "sgw_set_nonlocal: sphere point outside the grid");
    if (!uniq.empty()) {
        rc = dev_alloc(&c->sph_uniq, uniq.size());
        if (!rc) rc = check_cuda(cudaMemcpyAsync(c->sph_uniq, uniq.data(), uniq.size() * sizeof(int32_t), cudaMemcpyHostToDevice, st), "copy");
        if (!rc) rc = check_cuda(cudaStreamSynchronize(st), "sgw_set_nonlocal");
        if (rc) return rc;
    }
    c->nuniq = (int64_t)uniq.size();
    c->nsphere = nsphere; c->nproj = nproj;
    return SGW_OK;
}

extern "C" int sgw_set_td(sgw_ctx* c, int hartree_mode, double rho_scale) {
    if (!c || (hartree_mode != 0 && hartree_mode != 1)) return set_error(SGW_EINVAL, "sgw_set_td: bad argument");
    c->hartree_mode = hartree_mode;
    c->rho_scale = rho_scale;
    return SGW_OK;
}
