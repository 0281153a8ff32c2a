// sgw_pass_inst.cu -- compiled once per supported axis length (-DSGW_N=<N>): instantiates every
// fused pass kernel for that length and exports one launcher, sgw_pass_launch_<N>.
#include <cstdlib>

#include "sgw_plane.cuh"
#include "sgw_engine.cuh"
#include "sgw_lean.cuh"

#ifndef SGW_N
#error "compile with -DSGW_N=<axis length>"
#endif

namespace sgw {

template <int MODE, class Op>
static int launch(const PassCall* c) {
    constexpr int N = SGW_N;
    Op op;
    op.p = c->p;
    const int threads = c->gm.B * pass_threads_per_pencil<N>();
    const size_t smem = (size_t)c->gm.B * pass_smem_per_pencil<N>();
    if (threads > 256) return -1;
    auto kern = pass_kernel<N, MODE, Op>;
    if (smem > 48 * 1024) {
        static bool attr_done = false;
        if (!attr_done) {
            if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024) != cudaSuccess)
                return -4;
            attr_done = true;
        }
    }
    kern<<<(unsigned)c->ntiles, threads, smem, c->stream>>>(c->gm, c->in, c->tw, op);
    return cudaGetLastError() == cudaSuccess ? 0 : -4;
}

// Pipelined persistent variant.  Returns 1 if it does not apply (caller falls back to launch<>).
template <int B, bool FASTN, class Op>
static int launch_pipe_b(const PassCall* c, int num_sms) {
    constexpr int N = SGW_N;
    using Cfg = PipeCfg<N, B>;
    const OpParams& p = c->p;
    PipeArgs pa;
    const void* ptrs[NSLOT] = {c->in, nullptr, nullptr, nullptr, nullptr};
    int esz[NSLOT] = {16, 16, 16, 16, 16}, grid[NSLOT] = {0, 0, 0, 0, 1};
    switch (c->kind) {
        case K_RT_STORE: break;
        case K_RT_ACC: ptrs[SLOT_ACC] = p.acc; break;
        case K_RT_HFIN: ptrs[SLOT_ACC] = p.acc; ptrs[SLOT_TAB] = p.vtab; esz[SLOT_TAB] = 8; break;
        case K_RT_CHEB:
            ptrs[SLOT_ACC] = p.acc; ptrs[SLOT_TAB] = p.vtab; esz[SLOT_TAB] = 8;
            if (p.use_prev) ptrs[SLOT_PREV] = p.prev;
            if (p.flush && !p.series_init) ptrs[SLOT_SERIES] = p.series;
            break;
        case K_RT_TD: ptrs[SLOT_TAB] = p.pro_phase ? p.pro_phase : p.epi_phase; break;
        default: return 1;
    }
    if (c->kind == K_RT_TD && p.pro_phase && p.epi_phase && p.pro_phase != p.epi_phase) return 1;
    int off = 0;
    for (int s = 0; s < NSLOT; ++s) {
        pa.src[s].ptr = (const char*)ptrs[s];
        pa.src[s].esz = esz[s];
        pa.src[s].grid = grid[s];
        pa.src[s].slot_off = off;
        if (ptrs[s]) off += B * N * esz[s];
    }
    pa.stage_bytes = off;
    pa.ntiles = (unsigned)c->ntiles;
    const size_t smem = (size_t)Cfg::FIXED_BYTES + 2 * (size_t)pa.stage_bytes;
    if (smem > 227 * 1024 || Cfg::T > 1024) return 1;
    if ((long long)N * c->gm.sN + (long long)B * c->gm.sB >= (1LL << 31)) return 1;
    auto kern = pipe_kernel<N, B, FASTN, Op>;
    static bool attr_done = false;
    if (!attr_done) {
        if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024) != cudaSuccess) return -4;
        attr_done = true;
    }
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, Cfg::T, smem) != cudaSuccess || per_sm < 1) return 1;
    long long grid_x = (long long)per_sm * num_sms;
    if (grid_x > c->ntiles) grid_x = c->ntiles;
    Op op;
    op.p = c->p;
    kern<<<(unsigned)grid_x, Cfg::T, smem, c->stream>>>(c->gm, pa, c->tw, op);
    return cudaGetLastError() == cudaSuccess ? 0 : -4;
}

template <class Op>
static int launch_pipe(const PassCall* c) {
    static int disabled = -1, num_sms = 0;
    if (disabled < 0) {
        const char* e = getenv("SGW_NOPIPE");
        disabled = (e && atoi(e)) ? 1 : 0;
        int dev = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&num_sms, cudaDevAttrMultiProcessorCount, dev);
    }
    if (disabled || c->gm.B != 8) return 1;
    return c->gm.fastn ? launch_pipe_b<8, true, Op>(c, num_sms) : launch_pipe_b<8, false, Op>(c, num_sms);
}

template <class POp, class Op>
static int launch_rt(const PassCall* c) {
    const int rc = launch_pipe<POp>(c);
    if (rc != 1) return rc;
    return launch<MODE_RT, Op>(c);
}

// rows/columns per plane tile: wide tiles keep one CTA (8-9 warps) on few planes so the x->y
// transpose stays L2-resident
#ifndef SGW_PLANE_B96
#define SGW_PLANE_B96 24
#endif
constexpr int plane_B(int n) {
    return n == 32 ? 32 : n == 48 ? 24 : n == 64 ? 32 : n == 96 ? SGW_PLANE_B96 : n == 128 ? 16 : 8;
}

template <int MODE>
static int launch_plane(const PlaneCall* c) {
    constexpr int N = SGW_N, B = plane_B(SGW_N);
    using Cfg = PlaneCfg<N, B>;
    static int num_sms = 0;
    if (!num_sms) {
        int dev = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&num_sms, cudaDevAttrMultiProcessorCount, dev);
    }
    if (Cfg::SMEM_BYTES > 227 * 1024 || N % B) return 1;
    auto kern = plane_kernel<N, B, MODE>;
    static bool attr_done = false;
    if (!attr_done) {
        if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024) != cudaSuccess) return -4;
        attr_done = true;
    }
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, Cfg::T, Cfg::SMEM_BYTES) != cudaSuccess || per_sm < 1)
        return 1;
    if (c->ctas_per_sm > 0 && c->ctas_per_sm < per_sm) per_sm = c->ctas_per_sm;
    const unsigned ngroups = (c->a.nplanes + c->a.G - 1) / c->a.G;
    long long grid_x = (long long)per_sm * num_sms;
    if (grid_x > ngroups) grid_x = ngroups;
    kern<<<(unsigned)grid_x, Cfg::T, Cfg::SMEM_BYTES, c->stream>>>(c->a, c->tw);
    return cudaGetLastError() == cudaSuccess ? 0 : -4;
}


// ---- pass engine (sgw_engine.cuh) -----------------------------------------------------------------
template <int B, bool CPLX>
static int launch_engine_b(const EngCall* c) {
    constexpr int N = SGW_N;
    using Cfg = EngCfg<N, B>;
    auto kern = engine_kernel<N, B, CPLX>;
    const size_t smem = CPLX ? Cfg::SMEM_CPLX : Cfg::SMEM_REAL;
    static int per_sm = 0, num_sms = 0;
    if (!per_sm) {
        int dev = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&num_sms, cudaDevAttrMultiProcessorCount, dev);
        cudaError_t e = smem > 48 * 1024 ? cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) : cudaSuccess;
        if (e != cudaSuccess) return -(1000 + (int)e);
        int n = 0;
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, kern, Cfg::T, smem);
        if (e != cudaSuccess) return -(2000 + (int)e);
        if (n < 1) return -2999;
        per_sm = n;
    }
    long long grid = (long long)per_sm * num_sms;
    if (c->max_ctas > 0 && c->max_ctas < grid) grid = c->max_ctas;
    if (grid > (long long)c->args.nitems) grid = c->args.nitems;
    if (grid <= 0) return 0;
    if (c->args.use_deps) {
        EngArgs args = c->args;
        void* params[] = {(void*)&args};
        cudaError_t e = cudaLaunchCooperativeKernel((const void*)kern, dim3((unsigned)grid), dim3(Cfg::T), params, smem,
                                                    c->stream);
        return e == cudaSuccess ? 0 : -(3000 + (int)e);
    }
    kern<<<(unsigned)grid, Cfg::T, smem, c->stream>>>(c->args);
    cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? 0 : -(4000 + (int)e);
}


// ---- lean passes (sgw_lean.cuh) --------------------------------------------------------------------
template <class K>
static int lean_launch_kernel(K kern, int threads, size_t smem, long long want_ctas, int ctas_per_sm, const LeanArgs& args,
                              cudaStream_t stream, int* per_sm_cache) {
    static int num_sms = 0;
    if (!num_sms) {
        int dev = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&num_sms, cudaDevAttrMultiProcessorCount, dev);
    }
    if (!*per_sm_cache) {
        cudaError_t e = smem > 48 * 1024 ? cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)
                                         : cudaSuccess;
        if (e != cudaSuccess) return -(1000 + (int)e);
        int n = 0;
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, kern, threads, smem);
        if (e != cudaSuccess) return -(2000 + (int)e);
        if (n < 1) return -2999;
        *per_sm_cache = n;
    }
    int per_sm = *per_sm_cache;
    if (ctas_per_sm > 0 && ctas_per_sm < per_sm) per_sm = ctas_per_sm;
    long long grid = (long long)per_sm * num_sms;
    if (grid > want_ctas) grid = want_ctas;
    if (grid <= 0) return 0;
    // SGW_PDL=1: programmatic dependent launch, the pass may start while its predecessor drains (it waits for the
    // predecessor's memory after loading its tables, sgw_lean.cuh).  Off by default: measured neutral on cfg1-cfg3
    // (within 0.5 %) and slower inside the cfg0 graph (0.99 -> 1.15 ms), DESIGN.md section 10
    const char* pe = getenv("SGW_PDL");
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid); cfg.blockDim = dim3((unsigned)threads); cfg.dynamicSmemBytes = smem; cfg.stream = stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = (pe && atoi(pe) == 1) ? 1 : 0;
    cudaError_t e = cudaLaunchKernelEx(&cfg, kern, args);
    if (e == cudaSuccess) e = cudaGetLastError();
    return e == cudaSuccess ? 0 : -(4000 + (int)e);
}

// cluster size for the cluster-owned plane kernel: CS * NWG groups should divide the N/B tiles of a plane
template <int N, int B> struct ClusterSize {
    static constexpr int NWG = LeanCfg<N, B, 8>::NWG, TPP = N / B;
    static constexpr int CS = (TPP % (3 * NWG) == 0 && TPP / (3 * NWG) <= 1) ? 3
                              : (TPP % (8 * NWG) == 0) ? 8 : (TPP % (4 * NWG) == 0) ? 4 : (TPP % (2 * NWG) == 0) ? 2 : 1;
};

template <int B, bool CPLX>
static int launch_plane_cluster(const LeanCall* c) {
    constexpr int N = SGW_N;
    constexpr int CS = ClusterSize<N, B>::CS;
    if (CS < 2 || N % B) return 1;
    using Cfg = LeanCfg<N, B, 8>;
    const size_t smem = CPLX ? Cfg::SMEM_CPLX : Cfg::SMEM_REAL;
    auto kern = plane_cluster_kernel<N, B, CPLX, CS>;
    static int max_clusters = 0;
    cudaLaunchConfig_t cfg = {};
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = CS; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.blockDim = dim3(Cfg::T); cfg.dynamicSmemBytes = smem; cfg.stream = c->stream; cfg.attrs = attr; cfg.numAttrs = 1;
    if (!max_clusters) {
        cudaError_t e = smem > 48 * 1024 ? cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) : cudaSuccess;
        if (e != cudaSuccess) return -(1000 + (int)e);
        if (CS > 8) { e = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1); if (e != cudaSuccess) return -(1000 + (int)e); }
        cfg.gridDim = dim3(CS * 148);
        int n = 0;
        e = cudaOccupancyMaxActiveClusters(&n, kern, &cfg);
        if (e != cudaSuccess) return -(2000 + (int)e);
        if (n < 1) return 1;
        max_clusters = n;
    }
    long long ncl = max_clusters;
    if (ncl > (long long)c->args.ntiles) ncl = c->args.ntiles;
    if (ncl <= 0) return 0;
    cfg.gridDim = dim3((unsigned)(ncl * CS));
    cudaError_t e = cudaLaunchKernelEx(&cfg, kern, c->args);
    return e == cudaSuccess ? 0 : -(4000 + (int)e);
}

template <int B, bool CPLX>
static int launch_lean_b(const LeanCall* c) {
    constexpr int N = SGW_N;
    using Cfg = LeanCfg<N, B>;
    const size_t smem = CPLX ? Cfg::SMEM_CPLX : Cfg::SMEM_REAL;
    static int occ[7] = {0, 0, 0, 0, 0, 0, 0};
    const long long tiles_ctas = ((long long)c->args.ntiles + Cfg::NWG - 1) / Cfg::NWG;
    switch (c->kind) {
        case 0: return lean_launch_kernel(axis_lean_kernel<N, B, CPLX, 0, false>, Cfg::T, smem, tiles_ctas, c->ctas_per_sm, c->args, c->stream, &occ[0]);
        case 1: return lean_launch_kernel(axis_lean_kernel<N, B, CPLX, 1, false>, Cfg::T, smem, tiles_ctas, c->ctas_per_sm, c->args, c->stream, &occ[1]);
        case 2: return lean_launch_kernel(axis_lean_kernel<N, B, CPLX, 2, false>, Cfg::T, smem, tiles_ctas, c->ctas_per_sm, c->args, c->stream, &occ[2]);
        case 5: return lean_launch_kernel(axis_lean_kernel<N, B, CPLX, 1, true>, Cfg::T, smem, tiles_ctas, c->ctas_per_sm, c->args, c->stream, &occ[5]);
        case 4: return lean_launch_kernel(axis_lean_kernel<N, B, CPLX, 2, true>, Cfg::T, smem, tiles_ctas, c->ctas_per_sm, c->args, c->stream, &occ[4]);
        case 3: {
            if (N % B) return 1;
            if (c->cluster) { const int rc = launch_plane_cluster<B, CPLX>(c); if (rc != 1) return rc; }
            const long long ngroups = ((long long)c->args.ntiles + c->args.G - 1) / c->args.G;
            if (c->wpc == 16) {
                using PCfg = LeanCfg<N, B, 16>;
                if (PCfg::T > 1024) return 1;
                return lean_launch_kernel(plane_lean_kernel<N, B, CPLX, 16>, PCfg::T, CPLX ? PCfg::SMEM_CPLX : PCfg::SMEM_REAL, ngroups,
                                          c->ctas_per_sm, c->args, c->stream, &occ[6]);
            }
            using PCfg = LeanCfg<N, B, 8>;
            return lean_launch_kernel(plane_lean_kernel<N, B, CPLX, 8>, PCfg::T, CPLX ? PCfg::SMEM_CPLX : PCfg::SMEM_REAL, ngroups,
                                      c->ctas_per_sm, c->args, c->stream, &occ[3]);
        }
    }
    return -1;
}

}  // namespace sgw

#define SGW_CAT_(a, b) a##b
#define SGW_CAT(a, b) SGW_CAT_(a, b)

extern "C" int SGW_CAT(sgw_pass_launch_, SGW_N)(const sgw::PassCall* c) {
    using namespace sgw;
    switch (c->kind) {
        case K_RT_STORE: return launch_rt<POpStore, OpStore>(c);
        case K_RT_ACC: return launch_rt<POpAcc, OpAcc>(c);
        case K_RT_HFIN: return launch_rt<POpHFin, OpHFin>(c);
        case K_RT_CHEB: return launch_rt<POpCheb, OpCheb>(c);
        case K_RT_TD: return launch_rt<POpTD, OpTD>(c);
        case K_RT_MUL3D: return launch<MODE_RT, OpMul3D>(c);
        case K_FWD: return launch<MODE_FWD, OpStore>(c);
        case K_INV: return launch<MODE_INV, OpStore>(c);
        default: return -1;
    }
}

// Fused xy-plane pass (nx == ny == SGW_N).  Returns 1 if this length has no plane kernel.
extern "C" int SGW_CAT(sgw_plane_launch_, SGW_N)(const sgw::PlaneCall* c) {
#if SGW_N >= 32
    return c->mode == sgw::PL_TD ? sgw::launch_plane<sgw::PL_TD>(c) : sgw::launch_plane<sgw::PL_SUM>(c);
#else
    (void)c;
    return 1;
#endif
}

// Pass engine: B = pencils per tile (4 or 8).
extern "C" int SGW_CAT(sgw_eng_launch_, SGW_N)(const sgw::EngCall* c, int B) {
    using namespace sgw;
    if (B == 8) return c->cplx ? launch_engine_b<8, true>(c) : launch_engine_b<8, false>(c);
    if (B == 4) return c->cplx ? launch_engine_b<4, true>(c) : launch_engine_b<4, false>(c);
    return 1;
}

// Lean passes: B = pencils per tile (4 or 8).
extern "C" int SGW_CAT(sgw_lean_launch_, SGW_N)(const sgw::LeanCall* c, int B) {
    using namespace sgw;
    if (B == 8) return c->cplx ? launch_lean_b<8, true>(c) : launch_lean_b<8, false>(c);
    if (B == 4) return c->cplx ? launch_lean_b<4, true>(c) : launch_lean_b<4, false>(c);
    return 1;
}
