// sgw_pass_inst.cu -- compiled once per supported axis length (-DSGW_N=<N>): instantiates every fused pass kernel
// for that length and exports two launchers, sgw_pass_launch_<N> (Poisson passes) and sgw_lean_launch_<N>.
#include <cstdlib>

#include "sgw_ops.cuh"
#include "sgw_lean.cuh"
#include "sgw_acc.cuh"

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
    if (smem > 48 * 1024 &&
        cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
        return -4;
    kern<<<(unsigned)c->ntiles, threads, smem, c->stream>>>(c->gm, c->in, c->tw, op);
    return cudaGetLastError() == cudaSuccess ? 0 : -4;
}

// ---- lean passes (sgw_lean.cuh) --------------------------------------------------------------------
template <class K>
static int lean_launch_kernel(K kern, int threads, size_t smem, long long want_ctas, const LeanCall* c, int* per_sm_cache) {
    const int num_sms = c->num_sms, ctas_per_sm = c->ctas_per_sm;
    const LeanArgs& args = c->args;
    cudaStream_t stream = c->stream;
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
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid); cfg.blockDim = dim3((unsigned)threads); cfg.dynamicSmemBytes = smem; cfg.stream = stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = c->pdl ? 1 : 0;
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
    int& max_clusters = c->occ[CPLX ? 8 : 7];
    cudaLaunchConfig_t cfg = {};
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = CS; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.blockDim = dim3(Cfg::T); cfg.dynamicSmemBytes = smem; cfg.stream = c->stream; cfg.attrs = attr; cfg.numAttrs = 1;
    if (!max_clusters) {
        cudaError_t e = smem > 48 * 1024 ? cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) : cudaSuccess;
        if (e != cudaSuccess) return -(1000 + (int)e);
        if (CS > 8) { e = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1); if (e != cudaSuccess) return -(1000 + (int)e); }
        cfg.gridDim = dim3(CS * c->num_sms);
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

// team-owned planes (plane_team_kernel): cooperative launch of as many CTAs as are co-resident
template <int B, bool CPLX>
static int launch_plane_team(const LeanCall* c) {
    constexpr int N = SGW_N;
    if (N % B) return 1;
    using Cfg = LeanCfg<N, B, 8>;
    const size_t smem = CPLX ? Cfg::SMEM_CPLX : Cfg::SMEM_REAL;
    auto kern = plane_team_kernel<N, B, CPLX>;
    int& per_sm = c->occ[CPLX ? 17 : 16];
    if (!per_sm) {
        cudaError_t e = smem > 48 * 1024 ? cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) : cudaSuccess;
        if (e != cudaSuccess) return -(1000 + (int)e);
        int n = 0;
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, kern, Cfg::T, smem);
        if (e != cudaSuccess) return -(2000 + (int)e);
        if (n < 1) return 1;
        per_sm = n;
    }
    int ctas = per_sm;
    if (c->ctas_per_sm > 0 && c->ctas_per_sm < ctas) ctas = c->ctas_per_sm;
    const long long grid = (long long)ctas * c->num_sms;
    if (grid * Cfg::NWG < N / B) return 1;        // not even one team
    cudaLaunchConfig_t cfg = {};
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeCooperative;
    attr[0].val.cooperative = 1;
    cfg.gridDim = dim3((unsigned)grid); cfg.blockDim = dim3(Cfg::T); cfg.dynamicSmemBytes = smem; cfg.stream = c->stream;
    cfg.attrs = attr; cfg.numAttrs = 1;
    cudaError_t e = cudaLaunchKernelEx(&cfg, kern, c->args);
    return e == cudaSuccess ? 0 : -(4000 + (int)e);
}

template <int B, bool CPLX>
static int launch_lean_b(const LeanCall* c) {
    constexpr int N = SGW_N;
    using Cfg = LeanCfg<N, B>;
    const size_t smem = CPLX ? Cfg::SMEM_CPLX : Cfg::SMEM_REAL;
    int* occ = c->occ + (CPLX ? 9 : 0);          // per context and axis length: [0..6] real kinds, [7], [8] clusters, [9..15] complex kinds, [16], [17] teams
    const long long tiles_ctas = ((long long)c->args.ntiles + Cfg::NWG - 1) / Cfg::NWG;
    switch (c->kind) {
        case 0: return lean_launch_kernel(axis_lean_kernel<N, B, CPLX, 0, false>, Cfg::T, smem, tiles_ctas, c, &occ[0]);
        case 1: return lean_launch_kernel(axis_lean_kernel<N, B, CPLX, 1, false>, Cfg::T, smem, tiles_ctas, c, &occ[1]);
        case 2: return lean_launch_kernel(axis_lean_kernel<N, B, CPLX, 2, false>, Cfg::T, smem, tiles_ctas, c, &occ[2]);
        case 5: return lean_launch_kernel(axis_lean_kernel<N, B, CPLX, 1, true>, Cfg::T, smem, tiles_ctas, c, &occ[5]);
        case 4: return lean_launch_kernel(axis_lean_kernel<N, B, CPLX, 2, true>, Cfg::T, smem, tiles_ctas, c, &occ[4]);
        case 3: {
            if (N % B) return 1;
            if (c->cluster == 2) return launch_plane_team<B, CPLX>(c);
            if (c->cluster) { const int rc = launch_plane_cluster<B, CPLX>(c); if (rc != 1) return rc; }
            const long long ngroups = ((long long)c->args.ntiles + c->args.G - 1) / c->args.G;
            if (c->wpc == 16) {
                using PCfg = LeanCfg<N, B, 16>;
                if (PCfg::T > 1024) return 1;
                return lean_launch_kernel(plane_lean_kernel<N, B, CPLX, 16>, PCfg::T, CPLX ? PCfg::SMEM_CPLX : PCfg::SMEM_REAL, ngroups,
                                          c, &occ[6]);
            }
            using PCfg = LeanCfg<N, B, 8>;
            return lean_launch_kernel(plane_lean_kernel<N, B, CPLX, 8>, PCfg::T, CPLX ? PCfg::SMEM_CPLX : PCfg::SMEM_REAL, ngroups,
                                      c, &occ[3]);
        }
    }
    return -1;
}

// ---- TMA accumulate kernel (sgw_acc.cuh): one persistent CTA per SM ---------------------------------
static int launch_acc(const AccCall* c) {
#if SGW_N >= 32 && SGW_N % 8 == 0
    constexpr int N = SGW_N;
    using Cfg = AccCfg<N>;
    const bool pz = Cfg::PAIRZ && c->args.pairz;
    auto kern = pz ? acc_tma_kernel<N, Cfg::PAIRZ> : acc_tma_kernel<N, false>;
    if (c->args.pairz && !Cfg::PAIRZ) return -(2000);
    const int fixed = Cfg::TABLES + 3 * Cfg::MAXS * 8 + 128;
    int nslots = (227 * 1024 - fixed) / Cfg::TILE;
    if (nslots > Cfg::MAXS) nslots = Cfg::MAXS;
    if (nslots < 4) return 1;
    const size_t smem = (size_t)nslots * Cfg::TILE + fixed;
    int* attr_set = c->occ + (pz ? 4 : 0);
    if (!*attr_set) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return -(1000 + (int)e);
        *attr_set = 1;
    }
    long long grid = c->num_sms;
    if (grid > (long long)c->args.ntiles) grid = c->args.ntiles;
    if (grid <= 0) return 0;
    kern<<<(unsigned)grid, Cfg::T_ACC, smem, c->stream>>>(c->args, c->cur_y, c->cur_z, c->acc_y, c->acc_z, nslots);
    cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? 0 : -(4000 + (int)e);
#else
    (void)c;
    return 1;
#endif
}

static int launch_td(const TdCall* c) {
#if SGW_N >= 32 && SGW_N % 8 == 0
    constexpr int N = SGW_N;
    using Cfg = AccCfg<N>;
    const int fixed = 3 * N * 16 + 3 * Cfg::MAXS * 8 + 128;
    int nslots = (227 * 1024 - fixed) / Cfg::TILE;
    if (nslots > Cfg::MAXS) nslots = Cfg::MAXS;
    if (nslots < 3) return 1;
    const size_t smem = (size_t)nslots * Cfg::TILE + fixed;
    const int kind = c->args.kind;
    if (kind < 0 || kind > 2) return -(2000);
    auto kern = kind == KX ? td_tma_kernel<N, KX> : (kind == KY ? td_tma_kernel<N, KY> : td_tma_kernel<N, KZ>);
    if (!c->occ[1 + kind]) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return -(1000 + (int)e);
        c->occ[1 + kind] = 1;
    }
    long long grid = c->num_sms;                              // one CTA per SM; a CTA takes whole blocks (all vectors of 8 pencils)
    const long long nblk = (Cfg::PAIRZ && kind != KX) ? (long long)N * N / 16 : (long long)N * N / 8;
    if (grid > nblk) grid = nblk;
    if (grid <= 0 || c->args.nvec <= 0) return 0;
    kern<<<(unsigned)grid, Cfg::T, smem, c->stream>>>(c->args, c->map_y, c->map_z, nslots);
    cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? 0 : -(4000 + (int)e);
#else
    (void)c;
    return 1;
#endif
}

}  // namespace sgw

#define SGW_CAT_(a, b) a##b
#define SGW_CAT(a, b) SGW_CAT_(a, b)

extern "C" int SGW_CAT(sgw_pass_launch_, SGW_N)(const sgw::PassCall* c) {
    using namespace sgw;
    switch (c->kind) {
        case K_RT_MUL3D:
            return c->variant == 1 ? launch<MODE_RT, OpMul3DC>(c) : (c->variant == 2 ? launch<MODE_RT, OpMul3DScaled>(c) : launch<MODE_RT, OpMul3D>(c));
        case K_FWD:
            return c->variant == 1 ? launch<MODE_FWD, OpFromReal>(c) : (c->variant == 3 ? launch<MODE_FWD, OpPhaseLoad>(c) : launch<MODE_FWD, OpStore>(c));
        case K_INV:
            switch (c->variant) {
                case 1: return launch<MODE_INV, OpPhaseMerge>(c);
                case 2: return launch<MODE_INV, OpToReal>(c);
                case 3: return launch<MODE_INV, OpInvAddV>(c);
                case 4: return launch<MODE_INV, OpInvCheb>(c);
                case 5: return launch<MODE_INV, OpInvPhase>(c);
                default: return launch<MODE_INV, OpStore>(c);
            }
        default: return -1;
    }
}

// Lean passes: B = pencils per tile (4 or 8).
extern "C" int SGW_CAT(sgw_lean_launch_, SGW_N)(const sgw::LeanCall* c, int B) {
    using namespace sgw;
    if (B == 8) return c->cplx ? launch_lean_b<8, true>(c) : launch_lean_b<8, false>(c);
    if (B == 4) return c->cplx ? launch_lean_b<4, true>(c) : launch_lean_b<4, false>(c);
    return 1;
}

// TMA accumulate kernel: acc += c (T + vtab) cur + e v on a cubic grid of this axis length.  Returns 1 if not built.
extern "C" int SGW_CAT(sgw_acc_launch_, SGW_N)(const sgw::AccCall* c) { return sgw::launch_acc(c); }

// TMA split-operator factor along one axis of a cubic grid of this axis length, in place.  Returns 1 if not built.
extern "C" int SGW_CAT(sgw_td_launch_, SGW_N)(const sgw::TdCall* c) { return sgw::launch_td(c); }
