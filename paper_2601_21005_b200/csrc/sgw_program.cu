// sgw_program.cu -- host side of the lean streaming passes (sgw_lean.cuh): which launches make up an H apply, a
// Chebyshev term and a split-operator step, and with which flags.
#include <cstdlib>
#include <cstring>
#include <vector>

#include "sgw_ctx.h"

using namespace sgw;

namespace {

#define SGW_TRY(expr)             \
    do {                          \
        int rc_ = (expr);         \
        if (rc_ != 0) return rc_; \
    } while (0)

__global__ void cheb_tail_kernel(cd* out, const cd* P, const cd* Q, const cd* O, double cP, double cQ, int useO, long long n) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const cd p = P[i], q = Q[i];
    cd r = make_double2(cP * p.x + cQ * q.x, cP * p.y + cQ * q.y);
    if (useO) { const cd o = O[i]; r.x += o.x; r.y += o.y; }
    out[i] = r;
}

int Fact2_R2(int n) {
    switch (n) {
        case 8: case 12: case 16: case 24: case 32: case 48: return 4;
        case 64: case 96: case 128: return 8;
        case 192: case 256: return 16;
        case 384: return 24;
    }
    return 8;
}

struct LeanOp {
    const cd* cur; cd* acc; cd* series;
    const double* vtab; const cd* phase; const cd* phase_z;
    double* rho; double dens_scale;
    double hs, c0, c1;
    int fx, ax, fy, ay, fz, az;          // flags / alpha of the x, y, z passes
    bool cplx;
    const double* kre[3];
    const cd* kc[3];
};

int lean_launch(sgw_ctx* c, int axis_n, int kind, const LeanArgs& args, bool cplx, int ctas_per_sm, int prof_tag, int wpc = 8,
                int cluster = 0) {
    LeanCall call;
    call.wpc = wpc;
    call.cluster = cluster;
    call.args = args;
    call.cplx = cplx ? 1 : 0;
    call.kind = kind;
    call.ctas_per_sm = ctas_per_sm;
    call.stream = c->stream;
    call.pdl = c->pdl;
    call.num_sms = c->num_sms;
    call.occ = c->lean_occ[axis_n];
    cudaEvent_t e1 = prof_begin(c, prof_tag);
    const int rc = c->lean[axis_n](&call, c->leanB);
    if (rc != 0)
        return set_error(rc < 0 ? SGW_ECUDA : SGW_ESIZE,
                         "lean pass launch failed: stage " + std::to_string((-rc) / 1000) + ": " +
                             cudaGetErrorString((cudaError_t)((-rc) % 1000)));
    prof_end(c, e1);
    c->launches++;
    return 0;
}

// true if the fused x+y plane kernel applies: square planes whose CTA-owned groups (cur and acc of every
// resident CTA's group) stay inside L2
bool lean_use_plane(const sgw_ctx* c, bool cplx, int* G, int* ctas, int* wpc, int* cluster) {
    if (c->nx != c->ny) return false;
    const int n = c->nx, B = c->leanB;
    if (n % B) return false;
    // bytes the resident CTAs keep live in L2 between their row tiles and their column tiles: cur and acc of
    // one plane group per CTA (one array for the complex family, which works in place).  Two 8-warp CTAs per SM
    // overlap each other's barriers and are preferred while that stays under ~90 MB (measured on cfg1: 87 MB
    // live misses 38 % of the re-reads and is still faster than one CTA per SM); then one 16-warp CTA per SM.
    const double plane_bytes = 16.0 * n * n * (cplx ? 1.0 : 2.0);
    const int g = c->lean_G > 0 ? c->lean_G : 1;
    // Cluster-owned planes (plane_cluster_kernel: 4 CTAs per 128^2 plane, 8 per 256^2 plane): measured faster for the
    // real family on those sizes (cfg2 filter 37.9 -> 38.5, cfg3 filter 31.2 -> 33.4 G units/s: 256^2 planes then
    // also transpose through L2) and slower for the complex family and for 96^2 / 384^2 planes.  SGW_LEAN_CLUSTER=0/1
    // overrides.
    int use_cluster = (!cplx && (n == 128 || n == 256)) ? 1 : 0;
    if (c->lean_cluster >= 0) use_cluster = c->lean_cluster ? 1 : 0;
    // Team-owned planes (plane_team_kernel: N/B warp groups on several SMs own a plane at a time, software-pipelined
    // arrival counters): the way 256^2 and 384^2 planes transpose through L2 (a 384^2 plane of two arrays is 4.7 MB).
    int use_team = (n >= 256) ? 1 : 0;
    if (c->lean_team >= 0) use_team = c->lean_team ? 1 : 0;
    if (c->lean_cluster == 1) use_team = 0;
    const int gw = (B * Fact2_R2(n) + 31) / 32, groups_per_cta = 8 / gw > 0 ? 8 / gw : 1;
    if (use_team && c->num_sms * groups_per_cta >= n / B) {           // at least one team even at one CTA per SM
        *cluster = 2; *G = 1; *ctas = 0; *wpc = 8;
        return true;
    }
    *cluster = use_cluster;
    if (use_cluster && (n == 256 || n == 384)) { *G = 1; *ctas = 2; *wpc = 8; return true; }
    if (use_cluster) { *G = 1; *ctas = 2; *wpc = 8; return true; }
    int w = 8, per_sm = 2;
    if (plane_bytes * g * 2 * c->num_sms > 90.0e6) { w = 16; per_sm = 1; }
    if (c->lean_ctas == 1) { w = 16; per_sm = 1; }
    if (c->lean_ctas == 2) { w = 8; per_sm = 2; }
    if (plane_bytes * g * per_sm * c->num_sms > 100.0e6) return false;
    *G = g; *ctas = per_sm; *wpc = w;
    return true;
}

// one operator application over nv vectors: x and y (one launch when the plane kernel applies), then z
int lean_apply(sgw_ctx* c, int nv, const LeanOp& op, int kind_tag, bool allow_plane = true) {
    const int B = c->leanB;
    const long long nxy = (long long)c->nx * c->ny;
    LeanArgs a;
    memset(&a, 0, sizeof(a));
    a.cur = op.cur; a.acc = op.acc; a.series = op.series; a.vtab = op.vtab; a.phase = op.phase;
    a.rho = op.rho; a.dens_scale = op.dens_scale;
    a.hs = op.hs; a.c0 = op.c0; a.c1 = op.c1;
    a.nx = c->nx; a.ny = c->ny; a.nz = c->nz;
    a.nvec = nv;
    // vectors fastest in the tile order when an N_g table is read and does not stay in L2 by itself
    const bool table = op.cplx ? (op.phase != nullptr) : (op.vtab != nullptr);
    a.vminor = (table && nv > 1 && (double)c->ng * (op.cplx ? 16.0 : 8.0) > 24.0e6) ? 1 : 0;
    if (c->lean_vminor >= 0) a.vminor = (c->lean_vminor && nv > 1) ? 1 : 0;
    a.cnt = c->team_cnt;
    int G = 1, ctas = 0, wpc = 8, cluster = 0;
    if (allow_plane && lean_use_plane(c, op.cplx, &G, &ctas, &wpc, &cluster)) {
        a.tw = c->tw[0];
        a.kre[0] = op.kre[0]; a.kre[1] = op.kre[1]; a.kc[0] = op.kc[0]; a.kc[1] = op.kc[1];
        a.flags[0] = op.fx; a.alpha[0] = op.ax; a.flags[1] = op.fy; a.alpha[1] = op.ay;
        a.ntiles = (unsigned)((long long)nv * c->nz);
        a.G = G;
        if (cluster == 2)
            SGW_TRY(check_cuda(cudaMemsetAsync(c->team_cnt, 0, (size_t)a.ntiles * sizeof(unsigned), c->stream), "team counters"));
        SGW_TRY(lean_launch(c, 0, 3, a, op.cplx, ctas, 1 * K_NKINDS + (op.cplx ? K_RT_TD : K_RT_ACC), wpc, cluster));
    } else {
        a.tw = c->tw[0];
        a.kre[0] = op.kre[0]; a.kc[0] = op.kc[0]; a.kre[1] = nullptr; a.kc[1] = nullptr;
        a.flags[0] = op.fx; a.alpha[0] = op.ax;
        a.ntiles = (unsigned)((long long)nv * c->nz * c->ny / B);
        SGW_TRY(lean_launch(c, 0, 0, a, op.cplx, 0, 0 * K_NKINDS + (op.cplx ? K_RT_TD : K_RT_STORE)));
        a.tw = c->tw[1];
        a.kre[0] = op.kre[1]; a.kc[0] = op.kc[1];
        a.flags[0] = op.fy; a.alpha[0] = op.ay;
        if (op.cplx) a.cur = op.acc;
        a.ntiles = (unsigned)((long long)nv * c->nz * (c->nx / B));
        SGW_TRY(lean_launch(c, 1, (c->nx == c->ny && c->ny == c->nz) ? 5 : 1, a, op.cplx, 0,
                            1 * K_NKINDS + (op.cplx ? K_RT_TD : K_RT_ACC)));
    }
    a.tw = c->tw[2];
    if (op.phase_z) a.phase = op.phase_z;
    a.cur = op.cplx ? (const cd*)op.acc : op.cur;
    a.kre[0] = op.kre[2]; a.kc[0] = op.kc[2]; a.kre[1] = nullptr; a.kc[1] = nullptr;
    a.flags[0] = op.fz; a.alpha[0] = op.az;
    a.ntiles = (unsigned)((long long)nv * (nxy / B));
    const bool cube = c->nx == c->ny && c->ny == c->nz;
    return lean_launch(c, 2, cube ? 4 : 2, a, op.cplx, 0, 2 * K_NKINDS + kind_tag);
}

}  // namespace

namespace {
int acc_td_step(sgw_ctx* c, int nvec, const LeanOp& op);
}

namespace sgw {

// out = (Tx + Ty + Tz + V_loc) in (the KB term is added by the caller)
int lean_apply_H(sgw_ctx* c, int nv, const cd* in, cd* out) {
    LeanOp op;
    memset(&op, 0, sizeof(op));
    op.cur = in; op.acc = out; op.vtab = c->vloc; op.hs = 1.0;
    op.fx = c->vloc ? F_VTAB : 0; op.ax = 0; op.fy = 0; op.ay = 1; op.fz = 0; op.az = 1;
    op.cplx = false;
    for (int a = 0; a < 3; ++a) op.kre[a] = c->kin[a];
    return lean_apply(c, nv, op, K_RT_HFIN);
}

// Chebyshev recurrence, accumulated in place (Eq. 3; R-1): term n takes cur = phi_{n-1},
// acc = phi_{n-2} and leaves acc = phi_n = hs (s T + vtab) cur - acc; the series is updated in the x pass of
// every even term; the tail kernel adds what is pending and writes psi.
int lean_cheb_filter(sgw_ctx* c, int nvec, cd* psi, const double* a, double s, int nterms) {
    const long long ng = c->ng;
    SGW_TRY(ensure_ws(c, 2));
    cd *Pb = psi, *Qb = c->ws[0], *Ob = c->ws[1];
    const bool kb = c->nsphere > 0;
    const int L = nterms - 1;
    // vectors per chunk: 0 = all vectors per term (streaming); c > 0 = run c vectors through all terms before the
    // next c, with separate x, y, z passes, so that cur and acc of the chunk stay in L2 (SGW_LEAN_CHUNK)
    int chunk = nvec;
    if (c->lean_chunk > 0 && !kb) chunk = c->lean_chunk < nvec ? c->lean_chunk : nvec;
    for (int v0 = 0; v0 < nvec; v0 += chunk) {
        const int nvc = (nvec - v0 < chunk) ? nvec - v0 : chunk;
        const long long voff = (long long)v0 * ng;
        for (int n = 1; n <= L; ++n) {
            const bool odd = n & 1;
            LeanOp op;
            memset(&op, 0, sizeof(op));
            op.cur = (odd ? Pb : Qb) + voff; op.acc = (odd ? Qb : Pb) + voff; op.series = Ob + voff; op.vtab = c->vtab;
            op.hs = (n == 1) ? 0.5 : 1.0;
            op.fx = F_VTAB; op.ax = (n == 1) ? 0 : -1; op.fy = 0; op.ay = 1; op.fz = 0; op.az = 1;
            if (n >= 2 && !odd) {
                op.fx |= F_FLUSH;
                if (n == 2) op.fx |= F_SINIT;
                op.c0 = a[n - 2]; op.c1 = a[n - 1];
            }
            op.cplx = false;
            for (int ax = 0; ax < 3; ++ax) op.kre[ax] = c->cheb_kin[ax];
            SGW_TRY(lean_apply(c, nvc, op, K_RT_CHEB, chunk == nvec));
            if (kb) SGW_TRY(kb_apply(c, nvc, op.cur, op.acc, 0, s * op.hs));
        }
    }
    const bool Lodd = L & 1;
    const double cL = a[L], cLm1 = Lodd ? a[L - 1] : 0.0;
    const double cP = Lodd ? cLm1 : cL, cQ = Lodd ? cL : cLm1;
    const long long n = (long long)nvec * ng;
    cheb_tail_kernel<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(Pb, Pb, Qb, Ob, cP, cQ, L >= 2 ? 1 : 0, n);
    c->launches++;
    return check_cuda(cudaGetLastError(), "cheb_tail");
}

// one split-operator step with the phase table c->phase = exp(-i V dt/2) (R-8)
// merged: c->phase holds the product of the previous step's closing and this step's opening half-step factor, and
// only the last step of a call applies a closing factor (c->phase_last) on store
int lean_td_step(sgw_ctx* c, int nvec, cd* psi, bool kb, bool accumulate_density, bool merged, bool last) {
    LeanOp op;
    memset(&op, 0, sizeof(op));
    op.cur = psi; op.acc = psi; op.phase = c->phase; op.hs = 1.0;
    op.fx = kb ? 0 : F_PRO; op.fz = kb ? 0 : F_EPI;
    if (merged && !kb) {
        if (last) op.phase_z = c->phase_last;
        else op.fz = 0;
    }
    if (accumulate_density && !kb) { op.fz |= F_DENS; op.rho = c->rho; op.dens_scale = c->rho_scale; }
    op.cplx = true;
    for (int a = 0; a < 3; ++a) op.kc[a] = c->td_kin[a];
    const bool tma = c->tdk && (c->use_acc_td >= 0 ? c->use_acc_td != 0 : c->nx >= 256);
    if (tma) return acc_td_step(c, nvec, op);
    return lean_apply(c, nvec, op, K_RT_TD);
}

}  // namespace sgw

// =====================================================================================================
// TMA accumulate kernel (sgw_acc.cuh): acc += c (T + vtab) cur + e v
// =====================================================================================================
namespace {

typedef CUresult (*tmap_encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                   const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                   CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// tensor maps of one vector array (nv vectors of a cubic N^3 grid, interleaved complex = pairs of doubles) for the
// strided tiles: y tiles (8 x-adjacent pencils along y of one plane) and z tiles (8 xy-adjacent pencils along z)
int acc_maps(sgw_ctx* c, const void* base, int nv, CUtensorMap* my, CUtensorMap* mz, CUtensorMap* mz2 = nullptr, CUtensorMap* my2 = nullptr) {
    // the recurrence alternates between three arrays: keep their maps (encoding costs a few microseconds per map)
    for (int i = 0; i < 8; ++i)
        if (c->tmap_base[i] == base && c->tmap_nv[i] == nv) {
            *my = c->tmap_y[i]; *mz = c->tmap_z[i];
            if (mz2) *mz2 = c->tmap_z2[i];
            if (my2) *my2 = c->tmap_y2[i];
            return 0;
        }
    const int slot = c->tmap_next;
    c->tmap_next = (c->tmap_next + 1) % 8;
    c->tmap_base[slot] = nullptr;
    const cuuint64_t N = (cuuint64_t)c->nx;
    tmap_encode_fn enc = (tmap_encode_fn)c->tmap_encode;
    const cuuint32_t nbox = (cuuint32_t)(N <= 256 ? N : N / 2);
    const cuuint32_t box[3] = {16, nbox, 1}, box2[3] = {32, nbox, 1}, es[3] = {1, 1, 1};
    const cuuint64_t dy[3] = {2 * N, N, N * (cuuint64_t)nv}, sy[2] = {N * 16, N * N * 16};
    const cuuint64_t dz[3] = {2 * N * N, N, (cuuint64_t)nv}, sz[2] = {N * N * 16, N * N * N * 16};
    CUresult r = enc(my, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, const_cast<void*>(base), dy, sy, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                     CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r == CUDA_SUCCESS)
        r = enc(mz, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, const_cast<void*>(base), dz, sz, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    CUtensorMap z2, y2;
    if (r == CUDA_SUCCESS)
        r = enc(&z2, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, const_cast<void*>(base), dz, sz, box2, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r == CUDA_SUCCESS)
        r = enc(&y2, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, const_cast<void*>(base), dy, sy, box2, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return set_error(SGW_ECUDA, "cuTensorMapEncodeTiled failed: " + std::to_string((int)r));
    c->tmap_base[slot] = base; c->tmap_nv[slot] = nv; c->tmap_y[slot] = *my; c->tmap_z[slot] = *mz; c->tmap_z2[slot] = z2; c->tmap_y2[slot] = y2;
    if (mz2) *mz2 = z2;
    if (my2) *my2 = y2;
    return 0;
}

// one split-operator step through the TMA kernel: three launches (x, y, z factors), each in place
int acc_td_step(sgw_ctx* c, int nvec, const LeanOp& op) {
    TdCall call;
    memset(&call, 0, sizeof(call));
    if (c->nx == 384) {           // two consumer groups: the y and z launches work on tile pairs (maps with 256-byte rows)
        CUtensorMap y1, z1;
        SGW_TRY(acc_maps(c, op.acc, nvec, &y1, &z1, &call.map_z, &call.map_y));
    } else {
        SGW_TRY(acc_maps(c, op.acc, nvec, &call.map_y, &call.map_z));
    }
    call.num_sms = c->num_sms;
    call.occ = c->acc_occ;
    call.stream = c->stream;
    const long long n = c->nx;
    const int flags[3] = {op.fx, op.fy, op.fz};
    for (int axis = 0; axis < 3; ++axis) {
        TdArgs& a = call.args;
        a.psi = op.acc;
        a.phase = (axis == 2 && op.phase_z) ? op.phase_z : op.phase;
        a.rho = op.rho; a.dens_scale = op.dens_scale;
        a.kc = op.kc[axis];
        a.tw = c->tw[axis];
        a.kind = axis;
        a.flags = flags[axis];
        a.nvec = nvec; a.nz = c->nz;
        a.ntiles = (unsigned)(n * n / 8 * nvec);
        cudaEvent_t e1 = prof_begin(c, axis * K_NKINDS + K_RT_TD);
        const int rc = c->tdk(&call);
        if (rc != 0)
            return set_error(rc < 0 ? SGW_ECUDA : SGW_ESIZE, "TMA split-operator launch failed: stage " + std::to_string((-rc) / 1000) + ": " +
                                                                 cudaGetErrorString((cudaError_t)((-rc) % 1000)));
        prof_end(c, e1);
        c->launches++;
    }
    return 0;
}

struct AccOp {
    const cd* cur; cd* acc; const cd* v;
    const double* vtab;
    const double* kre[3];
    double c, e;
    int pairz;                // z-only launch with tiles in pairs (the z maps passed are the pair maps)
};

int acc_launch_one(sgw_ctx* c, int nv, const AccOp& op, const AccCall& maps, int kinds, int plane_major, int prof_tag) {
    AccCall call = maps;
    AccArgs& a = call.args;
    memset(&a, 0, sizeof(a));
    a.cur = op.cur; a.acc = op.acc; a.v = op.v; a.vtab = op.vtab;
    for (int d = 0; d < 3; ++d) a.kre[d] = op.kre[d];
    a.tw = c->tw[0];
    a.c = op.c; a.e = op.e;
    a.nvec = nv; a.nz = c->nz;
    a.kinds = kinds; a.plane_major = plane_major;
    const long long n = c->nx, tpv = n * n / 8, nk = (kinds & 1) + ((kinds >> 1) & 1) + ((kinds >> 2) & 1);
    a.pairz = op.pairz;
    const long long ntiles = plane_major ? nk * (n / 8) * c->nz * nv : (op.pairz ? tpv / 2 * nv : nk * tpv * nv);
    if (ntiles > 0xffffffffLL - 1024) return set_error(SGW_EINVAL, "too many tiles for one launch");
    a.ntiles = (unsigned)ntiles;
    call.num_sms = c->num_sms;
    call.occ = c->acc_occ;
    call.stream = c->stream;
    cudaEvent_t e1 = prof_begin(c, prof_tag);
    const int rc = c->acc(&call);
    if (rc != 0)
        return set_error(rc < 0 ? SGW_ECUDA : SGW_ESIZE, "accumulate kernel launch failed: stage " + std::to_string((-rc) / 1000) + ": " +
                                                             cudaGetErrorString((cudaError_t)((-rc) % 1000)));
    prof_end(c, e1);
    c->launches++;
    return 0;
}

// acc += c (T + vtab) cur + e v over nv vectors.  One launch when the arrays of a vector stay in L2 together (all
// x, y and z tiles of a vector are then adjacent in the tile order: cur is read from HBM once, acc read and written
// once); otherwise the x and y tiles plane by plane, then the z tiles in a second launch.
int acc_apply(sgw_ctx* c, int nv, const AccOp& op, int z_tag) {
    AccCall maps;
    memset(&maps, 0, sizeof(maps));
    SGW_TRY(acc_maps(c, op.cur, nv, &maps.cur_y, &maps.cur_z));
    SGW_TRY(acc_maps(c, op.acc, nv, &maps.acc_y, &maps.acc_z));
    const double per_vec = 16.0 * (double)c->ng * (op.v ? 3.0 : 2.0);
    if (per_vec <= c->acc_l2_bytes) return acc_launch_one(c, nv, op, maps, 7, 0, 1 * K_NKINDS + K_RT_ACC);
    SGW_TRY(acc_launch_one(c, nv, op, maps, 3, 1, 1 * K_NKINDS + K_RT_ACC));
    // z launch: where two consumer groups work side by side (N = 384) a tile pair (16 xy-adjacent pencils, 256-byte
    // rows) is loaded and reduce-added as one tensor operation and each group takes one half: the strided rows are what
    // bounds this launch, and 256-byte rows move at 6.3 TB/s where 128-byte rows reach 4.9
    if (c->acc_pairz) {
        AccOp op2 = op;
        op2.pairz = 1;
        AccCall m2 = maps;
        CUtensorMap dummy_y, dummy_z;
        SGW_TRY(acc_maps(c, op.cur, nv, &dummy_y, &dummy_z, &m2.cur_z));
        SGW_TRY(acc_maps(c, op.acc, nv, &dummy_y, &dummy_z, &m2.acc_z));
        return acc_launch_one(c, nv, op2, m2, 4, 0, 2 * K_NKINDS + z_tag);
    }
    return acc_launch_one(c, nv, op, maps, 4, 0, 2 * K_NKINDS + z_tag);
}

__global__ void scaled_copy_kernel(cd* out, const cd* in, double a, long long n) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = cscale(in[i], a);
}

}  // namespace

namespace sgw {

// out = (Tx + Ty + Tz + V_loc) in (the KB term is added by the caller)
int acc_apply_H(sgw_ctx* c, int nv, const cd* in, cd* out) {
    SGW_TRY(check_cuda(cudaMemsetAsync(out, 0, (size_t)nv * c->ng * sizeof(cd), c->stream), "clear output"));
    AccOp op;
    memset(&op, 0, sizeof(op));
    op.cur = in; op.acc = out; op.v = nullptr; op.vtab = c->vloc;
    for (int d = 0; d < 3; ++d) op.kre[d] = c->kin[d];
    op.c = 1.0; op.e = 0.0;
    return acc_apply(c, nv, op, K_RT_HFIN);
}

// Chebyshev series sum_n a_n T_n(Ht) v (Eq. 3; R-1) by the Clenshaw recurrence
//     b_k = a_k v + 2 Ht b_{k+1} - b_{k+2}   (k = L .. 1, b_{L+1} = b_{L+2} = 0),   result = a_0 v + Ht b_1 - b_2,
// which needs the same L = nterms - 1 applications of H as the forward recurrence but only READS v every step
// instead of reading and writing a series array.  Stored are Q_k = t_k b_k with signs t = + + - - + + ... (t_k t_{k+2}
// = -1), which turns every step into a pure accumulation into the buffer that holds Q_{k+2}:
//     Q_k = Q_{k+2} + (t_k t_{k+1}) 2 Ht Q_{k+1} + (t_k a_k) v ,      result = Q_2 + (t_1 / 2) 2 Ht Q_1 + a_0 v   (t_2 = -1)
// -- the form the accumulate kernel computes.  Tables are scaled so that (T + vtab) = 2 Ht (sgw_cheb_filter).
int acc_cheb_filter(sgw_ctx* c, int nvec, cd* psi, const double* a, double s, int nterms) {
    const long long ng = c->ng, n = (long long)nvec * ng;
    SGW_TRY(ensure_ws(c, 2));
    const bool kb = c->nsphere > 0;
    const int L = nterms - 1;
    auto t = [](int k) { return ((k & 3) < 2) ? 1.0 : -1.0; };
    cd *A = c->ws[0], *Bf = c->ws[1];
    scaled_copy_kernel<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(A, psi, t(L) * a[L], n);      // Q_L
    c->launches++;
    SGW_TRY(check_cuda(cudaGetLastError(), "scaled_copy"));
    SGW_TRY(check_cuda(cudaMemsetAsync(Bf, 0, (size_t)n * sizeof(cd), c->stream), "clear"));            // Q_{L+1}
    AccOp op;
    memset(&op, 0, sizeof(op));
    op.v = psi; op.vtab = c->vtab;
    for (int d = 0; d < 3; ++d) op.kre[d] = c->cheb_kin[d];
    for (int k = L - 1; k >= 0; --k) {
        op.cur = A; op.acc = Bf;
        op.c = k > 0 ? t(k) * t(k + 1) : 0.5 * t(1);
        op.e = k > 0 ? t(k) * a[k] : a[0];
        SGW_TRY(acc_apply(c, nvec, op, K_RT_CHEB));
        if (kb) SGW_TRY(kb_apply(c, nvec, A, Bf, 0, s * op.c));
        cd* tmp = A; A = Bf; Bf = tmp;                       // A = Q_k, Bf = Q_{k+1}
    }
    return check_cuda(cudaMemcpyAsync(psi, A, (size_t)n * sizeof(cd), cudaMemcpyDeviceToDevice, c->stream), "copy result");
}

}  // namespace sgw
