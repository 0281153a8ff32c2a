// sgw_core.cu -- context, tables, pass geometry, setup entry points of libsgw (include/sgw.h).
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>

#include "sgw_ctx.h"

#define SGW_DECL(N)                                             \
    extern "C" int sgw_pass_launch_##N(const sgw::PassCall*);   \
    extern "C" int sgw_plane_launch_##N(const sgw::PlaneCall*); \
    extern "C" int sgw_eng_launch_##N(const sgw::EngCall*, int); \
    extern "C" int sgw_lean_launch_##N(const sgw::LeanCall*, int);
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

static pass_launch_fn launcher_for(int n) {
    switch (n) {
#define SGW_CASE(N) case N: return sgw_pass_launch_##N;
        SGW_CASE(8) SGW_CASE(12) SGW_CASE(16) SGW_CASE(24) SGW_CASE(32) SGW_CASE(48) SGW_CASE(64) SGW_CASE(96)
        SGW_CASE(128) SGW_CASE(192) SGW_CASE(256) SGW_CASE(384)
#undef SGW_CASE
        default: return nullptr;
    }
}

static plane_launch_fn plane_launcher_for(int n) {
    switch (n) {
#define SGW_CASE(N) case N: return sgw_plane_launch_##N;
        SGW_CASE(8) SGW_CASE(12) SGW_CASE(16) SGW_CASE(24) SGW_CASE(32) SGW_CASE(48) SGW_CASE(64) SGW_CASE(96)
        SGW_CASE(128) SGW_CASE(192) SGW_CASE(256) SGW_CASE(384)
#undef SGW_CASE
        default: return nullptr;
    }
}

static eng_launch_fn eng_launcher_for(int n) {
    switch (n) {
#define SGW_CASE(N) case N: return sgw_eng_launch_##N;
        SGW_CASE(8) SGW_CASE(12) SGW_CASE(16) SGW_CASE(24) SGW_CASE(32) SGW_CASE(48) SGW_CASE(64) SGW_CASE(96)
        SGW_CASE(128) SGW_CASE(192) SGW_CASE(256) SGW_CASE(384)
#undef SGW_CASE
        default: return nullptr;
    }
}

static lean_launch_fn lean_launcher_for(int n) {
    switch (n) {
#define SGW_CASE(N) case N: return sgw_lean_launch_##N;
        SGW_CASE(8) SGW_CASE(12) SGW_CASE(16) SGW_CASE(24) SGW_CASE(32) SGW_CASE(48) SGW_CASE(64) SGW_CASE(96)
        SGW_CASE(128) SGW_CASE(192) SGW_CASE(256) SGW_CASE(384)
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

int run_plane(sgw_ctx* c, int mode, int nvec, const cd* in, cd* out, const cd* phase, bool cheb_tables) {
    if (!c->plane || nvec <= 0) return 1;
    PlaneCall call;
    call.mode = mode;
    call.a.in = in; call.a.out = out; call.a.phase = phase;
    call.a.kre_x = cheb_tables ? c->cheb_kin[0] : c->kin[0];
    call.a.kre_y = cheb_tables ? c->cheb_kin[1] : c->kin[1];
    call.a.kc_x = c->td_kin[0]; call.a.kc_y = c->td_kin[1];
    call.a.nplanes = (unsigned)((long long)c->nz * nvec);
    call.a.nz = (unsigned)c->nz;
    call.a.G = c->plane_G;
    call.tw = c->tw[0];
    call.ctas_per_sm = c->plane_ctas;
    call.stream = c->stream;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (c->prof_on && c->prof_used < 60000) {
        if (c->prof_ev.size() < 2 * (c->prof_used + 1)) {
            cudaEvent_t a, b;
            if (cudaEventCreate(&a) == cudaSuccess && cudaEventCreate(&b) == cudaSuccess) {
                c->prof_ev.push_back(a); c->prof_ev.push_back(b); c->prof_tag.push_back(0);
            }
        }
        if (c->prof_ev.size() >= 2 * (c->prof_used + 1)) {
            e0 = c->prof_ev[2 * c->prof_used]; e1 = c->prof_ev[2 * c->prof_used + 1];
            c->prof_tag[c->prof_used] = 1 * K_NKINDS + (mode == PL_TD ? K_RT_TD : K_RT_ACC);   // booked as the y pass
            cudaEventRecord(e0, c->stream);
        }
    }
    const int rc = c->plane(&call);
    if (rc == 1) return 1;
    if (rc != 0) return set_error(rc, std::string("plane launch failed: ") + cudaGetErrorString(cudaGetLastError()));
    if (e1) { cudaEventRecord(e1, c->stream); c->prof_used++; }
    c->launches++;
    return 0;
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

int run_pass(sgw_ctx* c, int axis, int kind, int nvec, const cd* in, const OpParams& p) {
    PassCall call;
    call.kind = kind;
    call.gm = geom_for_axis(c, axis, nvec, &call.ntiles);
    call.in = in;
    call.tw = c->tw[axis];
    call.p = p;
    call.stream = c->stream;
    if (call.ntiles <= 0) return 0;
    if (call.ntiles > 0x7fffffffLL) return set_error(SGW_EINVAL, "too many tiles for one launch");
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (c->prof_on && c->prof_used < 60000) {
        if (c->prof_ev.size() < 2 * (c->prof_used + 1)) {
            cudaEvent_t a, b;
            if (cudaEventCreate(&a) == cudaSuccess && cudaEventCreate(&b) == cudaSuccess) {
                c->prof_ev.push_back(a); c->prof_ev.push_back(b); c->prof_tag.push_back(0);
            }
        }
        if (c->prof_ev.size() >= 2 * (c->prof_used + 1)) {
            e0 = c->prof_ev[2 * c->prof_used]; e1 = c->prof_ev[2 * c->prof_used + 1];
            c->prof_tag[c->prof_used] = axis * K_NKINDS + kind;
            cudaEventRecord(e0, c->stream);
        }
    }
    int rc = c->pass[axis](&call);
    if (rc != 0) return set_error(rc, std::string("pass launch failed: ") + cudaGetErrorString(cudaGetLastError()));
    if (e1) { cudaEventRecord(e1, c->stream); c->prof_used++; }
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
    return sgw::eng_check_error(c);
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
        cudaFree(c->tw[a]); cudaFree(c->kin[a]); cudaFree(c->cheb_kin[a]); cudaFree(c->td_kin[a]); cudaFree(c->ws[a]);
    }
    cudaFree(c->vloc); cudaFree(c->vtab); cudaFree(c->vk3d); cudaFree(c->sph_ptr); cudaFree(c->sph_idx);
    cudaFree(c->beta); cudaFree(c->D); cudaFree(c->kbc); cudaFree(c->pois); cudaFree(c->rho); cudaFree(c->vh);
    cudaFree(c->phase); cudaFree(c->phase_last); cudaFree(c->vprev); cudaFree(c->d_segs); cudaFree(c->d_cnt); cudaFree(c->d_err);
    delete c;
    return SGW_OK;
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
    sgw_ctx* c = new sgw_ctx();
    memset((void*)&c->tw, 0, sizeof(c->tw));
    c->nx = nx; c->ny = ny; c->nz = nz; c->hx = hx; c->hy = hy; c->hz = hz;
    c->ng = (long long)nx * ny * nz;
    c->max_nvec = max_nvec;
    c->stream = (cudaStream_t)cuda_stream;
    c->B = (nx % 8 == 0) ? 8 : 4;
    c->Bx = ((long long)ny * nz) % 8 == 0 ? 8 : (((long long)ny * nz) % 4 == 0 ? 4 : 1);
    const double hh[3] = {hx, hy, hz};
    int rc = 0;
    for (int a = 0; a < 3 && !rc; ++a) {
        c->dims[a] = dims[a]; c->hs[a] = hh[a];
        c->pass[a] = launcher_for(dims[a]);
        c->kin[a] = nullptr; c->cheb_kin[a] = nullptr; c->td_kin[a] = nullptr; c->ws[a] = nullptr; c->tw[a] = nullptr;
        const int N = dims[a];
        std::vector<cd> tw(N);
        std::vector<double> kin(N);
        c->h_kin[a].resize(N);
        for (int j = 0; j < N; ++j) {
            const long double ang = -2.0L * acosl(-1.0L) * (long double)j / (long double)N;
            tw[j] = make_double2((double)cosl(ang), (double)sinl(ang));
            const int m = (2 * j >= N) ? j - N : j;
            const long double k = 2.0L * acosl(-1.0L) * (long double)m / ((long double)N * (long double)hh[a]);
            c->h_kin[a][j] = (double)(0.5L * k * k);
            kin[j] = (double)(0.5L * k * k / (long double)N);
        }
        if (!rc) rc = dev_alloc(&c->tw[a], N);
        if (!rc) rc = dev_alloc(&c->kin[a], N);
        if (!rc) rc = dev_alloc(&c->cheb_kin[a], N);
        if (!rc) rc = dev_alloc(&c->td_kin[a], N);
        if (!rc) rc = upload(c->tw[a], tw.data(), N, c->stream);
        if (!rc) rc = upload(c->kin[a], kin.data(), N, c->stream);
    }
    c->td_kin_valid = false; c->td_dt = 0;
    c->vloc = nullptr; c->vtab = nullptr; c->vk3d = nullptr;
    c->nsphere = 0; c->nproj = 0; c->sph_ptr = nullptr; c->sph_idx = nullptr; c->beta = nullptr; c->D = nullptr;
    c->kbc = nullptr; c->kbc_cap = 0;
    c->pois = nullptr; c->rho = nullptr; c->vh = nullptr; c->phase = nullptr; c->phase_last = nullptr; c->vprev = nullptr;
    c->hartree_mode = 0; c->rho_scale = 0; c->launches = 0;
    c->prof_on = false; c->prof_used = 0;
    { const char* e = getenv("SGW_L2_CHUNK"); c->l2_chunk = e ? atoi(e) : 0; }
    c->plane = nullptr; c->plane_G = 2; c->plane_ctas = 0;
    if (nx == ny && nx % 8 == 0 && !(getenv("SGW_NOPLANE") && atoi(getenv("SGW_NOPLANE")))) c->plane = plane_launcher_for(nx);
    { const char* e = getenv("SGW_PLANE_G"); if (e && atoi(e) > 0) c->plane_G = atoi(e); }
    { const char* e = getenv("SGW_PLANE_CTAS"); if (e) c->plane_ctas = atoi(e); }
    for (int a = 0; a < 3; ++a) c->lean[a] = lean_launcher_for(dims[a]);
    c->lean_G = 0; c->lean_ctas = 0;
    { const char* e = getenv("SGW_LEAN_G"); if (e) c->lean_G = atoi(e); }
    { const char* e = getenv("SGW_LEAN_CTAS"); if (e) c->lean_ctas = atoi(e); }
    for (int a = 0; a < 3; ++a) { c->eng[a] = eng_launcher_for(dims[a]); c->engB[a] = (nx % 8 == 0 && ny % 8 == 0) ? 8 : 4; }
    c->use_engine = 2; c->eng_max_ctas = 0; c->eng_resident = -1; c->eng_pc = 0;
    c->d_segs = nullptr; c->segs_cap = 0; c->d_cnt = nullptr; c->cnt_cap = 0; c->d_err = nullptr;
    cudaDeviceGetAttribute(&c->num_sms, cudaDevAttrMultiProcessorCount, 0);
    { const char* e = getenv("SGW_ENGINE"); if (e) c->use_engine = atoi(e); }
    { const char* e = getenv("SGW_ENG_CTAS"); if (e) c->eng_max_ctas = atoi(e); }
    { const char* e = getenv("SGW_ENG_RESIDENT"); if (e) c->eng_resident = atoi(e); }
    { const char* e = getenv("SGW_ENG_PC"); if (e) c->eng_pc = atoi(e); }
    c->eng_l2_prefetch = 0;
    { const char* e = getenv("SGW_ENG_L2PF"); if (e) c->eng_l2_prefetch = atoi(e); }
    { const char* e = getenv("SGW_ENG_B"); if (e && (atoi(e) == 4 || (atoi(e) == 8 && c->engB[0] == 8))) for (int a = 0; a < 3; ++a) c->engB[a] = atoi(e); }
    for (int i = 0; i < 3 * K_NKINDS; ++i) { c->prof_ms[i] = 0; c->prof_n[i] = 0; }
    if (!rc) rc = dev_alloc(&c->vtab, c->ng);
    if (!rc) rc = dev_alloc(&c->vk3d, c->ng);
    if (!rc) rc = dev_alloc(&c->pois, c->ng);
    if (!rc) rc = dev_alloc(&c->rho, c->ng);
    if (!rc) rc = dev_alloc(&c->vh, c->ng);
    if (!rc) rc = dev_alloc(&c->phase, c->ng);
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
    cudaFree(c->sph_ptr); cudaFree(c->sph_idx); cudaFree(c->beta); cudaFree(c->D);
    c->sph_ptr = nullptr; c->sph_idx = nullptr; c->beta = nullptr; c->D = nullptr; c->nsphere = 0;
    if (nsphere == 0) return SGW_OK;
    if (!d_ptr || !d_idx || !d_beta || !d_D || nproj < 1 || nproj > 8)
        return set_error(SGW_EINVAL, "sgw_set_nonlocal: bad argument");
    int64_t npts = 0;
    int rc = check_cuda(cudaMemcpy(&npts, d_ptr + nsphere, sizeof(int64_t), cudaMemcpyDeviceToHost), "read sph_ptr");
    if (rc) return rc;
    if (npts < 0) return set_error(SGW_EINVAL, "sgw_set_nonlocal: negative point count");
    if (!rc) rc = dev_alloc(&c->sph_ptr, (size_t)nsphere + 1);
    if (!rc) rc = dev_alloc(&c->sph_idx, (size_t)npts);
    if (!rc) rc = dev_alloc(&c->beta, (size_t)npts * nproj);
    if (!rc) rc = dev_alloc(&c->D, (size_t)nsphere * nproj);
    if (!rc) rc = check_cuda(cudaMemcpy(c->sph_ptr, d_ptr, (nsphere + 1) * sizeof(int64_t), cudaMemcpyDeviceToDevice), "copy");
    if (!rc && npts) rc = check_cuda(cudaMemcpy(c->sph_idx, d_idx, npts * sizeof(int32_t), cudaMemcpyDeviceToDevice), "copy");
    if (!rc && npts) rc = check_cuda(cudaMemcpy(c->beta, d_beta, npts * nproj * sizeof(double), cudaMemcpyDeviceToDevice), "copy");
    if (!rc) rc = check_cuda(cudaMemcpy(c->D, d_D, (size_t)nsphere * nproj * sizeof(double), cudaMemcpyDeviceToDevice), "copy");
    if (rc) return rc;
    c->nsphere = nsphere; c->nproj = nproj;
    return SGW_OK;
}

extern "C" int sgw_set_td(sgw_ctx* c, int hartree_mode, double rho_scale) {
    if (!c || (hartree_mode != 0 && hartree_mode != 1)) return set_error(SGW_EINVAL, "sgw_set_td: bad argument");
    c->hartree_mode = hartree_mode;
    c->rho_scale = rho_scale;
    return SGW_OK;
}
