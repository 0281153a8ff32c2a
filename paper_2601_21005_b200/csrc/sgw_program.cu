// sgw_program.cu -- host side of the fused passes: the lean streaming passes (sgw_lean.cuh; the default: second
// half of this file) and the pass engine (sgw_engine.cuh: programs of segments with dependency counters), each
// implementing H apply, the Chebyshev filter and the split-operator step.
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

struct Program {
    std::vector<Seg> segs;
    unsigned nitems = 0, nplanes = 0;
};

Seg blank_seg() {
    Seg s;
    memset(&s, 0, sizeof(s));
    s.dep = -1;
    s.pc = 1;
    return s;
}

bool cubic(const sgw_ctx* c) { return c->nx == c->ny && c->ny == c->nz; }

// planes per x/y group: about half a wave of tiles, a divisor of the segment's plane count
int pick_pc(const sgw_ctx* c, int nplanes, int tpp) {
    if (c->eng_pc > 0) {
        int pc = c->eng_pc < nplanes ? c->eng_pc : nplanes;
        while (nplanes % pc) --pc;
        return pc;
    }
    // a group's y tiles follow its x tiles by one slot: make a slot about a wave of tiles (measured best on
    // cfg1: 64 planes of 12 tiles), but keep the planes in flight (two slots, cur and acc) inside L2
    int target = (5 * c->num_sms) / tpp;
    const double plane_bytes = 16.0 * c->nx * c->ny;
    const int cap = (int)(40.0e6 / (4.0 * plane_bytes));
    if (target > cap) target = cap;
    if (target < 1) target = 1;
    if (target > nplanes) target = nplanes;
    while (nplanes % target) --target;
    return target;
}

// appends a segment, filling item0 / nitems / plane counters; returns its index
int add_seg(const sgw_ctx* c, Program& P, Seg s) {
    const int B = c->engB[0];
    const long long nxy = (long long)c->nx * c->ny;
    long long n = 0;
    switch (s.type) {
        case SEG_X: n = (long long)s.nvec * c->nz * (c->ny / B); break;
        case SEG_Y: n = (long long)s.nvec * c->nz * (c->nx / B); break;
        case SEG_Z: n = (long long)s.nvec * (nxy / B); break;
        case SEG_XY: {
            const int tpp = c->nx / B, planes = s.nvec * c->nz;
            s.pc = pick_pc(c, planes, tpp);
            n = 2LL * planes * tpp;
            if (s.plane_target == 0) { s.plane0 = P.nplanes; P.nplanes += planes; s.plane_target = tpp; }
            break;
        }
    }
    s.item0 = P.nitems;
    s.nitems = (unsigned)n;
    P.nitems += (unsigned)n;
    P.segs.push_back(s);
    return (int)P.segs.size() - 1;
}

int ensure_dev(sgw_ctx* c, size_t nseg, size_t ncnt) {
    if (nseg > c->segs_cap) {
        SGW_TRY(check_cuda(cudaStreamSynchronize(c->stream), "sync"));
        cudaFree(c->d_segs);
        c->d_segs = nullptr; c->segs_cap = 0;
        const size_t cap = nseg + nseg / 2 + 16;
        SGW_TRY(check_cuda(cudaMalloc((void**)&c->d_segs, cap * sizeof(Seg)), "segment buffer"));
        c->segs_cap = cap;
    }
    if (ncnt > c->cnt_cap) {
        SGW_TRY(check_cuda(cudaStreamSynchronize(c->stream), "sync"));
        cudaFree(c->d_cnt);
        c->d_cnt = nullptr; c->cnt_cap = 0;
        const size_t cap = ncnt + ncnt / 2 + 64;
        SGW_TRY(check_cuda(cudaMalloc((void**)&c->d_cnt, cap * sizeof(unsigned)), "counter buffer"));
        c->cnt_cap = cap;
    }
    if (!c->d_err) {
        SGW_TRY(check_cuda(cudaMalloc((void**)&c->d_err, sizeof(int)), "error flag"));
        SGW_TRY(check_cuda(cudaMemsetAsync(c->d_err, 0, sizeof(int), c->stream), "error flag"));
    }
    return 0;
}

struct Tables {
    const double* kre[3];
    const cd* kc[3];
    bool cplx;
};

// uploads the program once; launch_program may then be called for several vector offsets
int upload_program(sgw_ctx* c, const Program& P) {
    SGW_TRY(ensure_dev(c, P.segs.size(), P.segs.size() + P.nplanes));
    return check_cuda(cudaMemcpyAsync(c->d_segs, P.segs.data(), P.segs.size() * sizeof(Seg), cudaMemcpyHostToDevice,
                                      c->stream), "program upload");
}

// one launch executing segments [s0, s1) of the uploaded program (their item0 must be relative to s0)
int launch_segments(sgw_ctx* c, const Program& P, int s0, int s1, unsigned nitems, bool deps, const Tables& t,
                    long long voff, int axis_n) {
    EngCall call;
    memset(&call, 0, sizeof(call));
    EngArgs& a = call.args;
    a.segs = c->d_segs + s0;
    a.nseg = s1 - s0;
    a.nitems = nitems;
    a.cnt_seg = c->d_cnt;
    a.cnt_plane = c->d_cnt + P.segs.size();
    a.err = c->d_err;
    a.voff = voff;
    a.tw = c->tw[axis_n];
    for (int ax = 0; ax < 3; ++ax) {
        const bool same = c->dims[ax] == c->dims[axis_n];
        a.kre[ax] = same ? t.kre[ax] : nullptr;
        a.kc[ax] = same ? t.kc[ax] : nullptr;
    }
    a.nx = c->nx; a.ny = c->ny; a.nz = c->nz;
    a.use_deps = deps ? 1 : 0;
    a.l2_prefetch = c->eng_l2_prefetch;
    call.cplx = t.cplx ? 1 : 0;
    call.max_ctas = c->eng_max_ctas;
    call.stream = c->stream;
    if (deps)
        SGW_TRY(check_cuda(cudaMemsetAsync(c->d_cnt, 0, (P.segs.size() + P.nplanes) * sizeof(unsigned), c->stream),
                           "counter reset"));
    const int rc = c->eng[axis_n](&call, c->engB[0]);
    if (rc != 0)
        return set_error(rc < 0 ? SGW_ECUDA : SGW_ESIZE,
                         "engine launch failed: stage " + std::to_string((-rc) / 1000) + ": " +
                             cudaGetErrorString((cudaError_t)((-rc) % 1000)) + " (items " + std::to_string(nitems) + ")");
    c->launches++;
    return 0;
}

// Runs an uploaded program: one dependent launch on cubic grids, one launch per segment otherwise.
int launch_program(sgw_ctx* c, Program& P, const Tables& t, long long voff) {
    if (P.segs.empty()) return 0;
    if (cubic(c)) return launch_segments(c, P, 0, (int)P.segs.size(), P.nitems, P.segs.size() > 1 || P.nplanes, t, voff, 0);
    // per-segment launches need item0 == 0 in each segment: callers build such programs (see seg_program)
    for (size_t i = 0; i < P.segs.size(); ++i) {
        const Seg& s = P.segs[i];
        const int axis_n = s.type == SEG_XY ? 0 : s.type;
        SGW_TRY(launch_segments(c, P, (int)i, (int)i + 1, s.nitems, s.type == SEG_XY, t, voff, axis_n));
    }
    return 0;
}

// Appends the passes of one operator application over `nvec` vectors starting at vector v0 of the
// launch: x and y (fused when nx == ny), then z.  dep = segment the first pass waits for (-1: none).
// Returns the index of the z segment.  fx/fy/fz, ax/ay/az: flags and alpha per pass.
int add_apply(const sgw_ctx* c, Program& P, Seg proto, int v0, int nvec, int dep, unsigned dep_count, int fx, int ax,
              int fy, int ay, int fz, int az, unsigned plane0 = 0, unsigned plane_target = 0) {
    const long long off = (long long)v0 * c->ng;
    proto.cur += off;
    proto.acc += off;
    if (proto.series) proto.series += off;
    proto.nvec = nvec;
    const bool chain = cubic(c);       // dependencies only exist inside single launches
    int last;
    if (c->nx == c->ny) {
        Seg s = proto;
        s.type = SEG_XY; s.flags[0] = fx; s.alpha[0] = ax; s.flags[1] = fy; s.alpha[1] = ay;
        s.dep = chain ? dep : -1; s.dep_count = dep_count;
        s.plane0 = plane0; s.plane_target = plane_target;      // 0: add_seg allocates fresh counters
        last = add_seg(c, P, s);
    } else {
        Seg s = proto;
        s.type = SEG_X; s.flags[0] = fx; s.alpha[0] = ax;
        add_seg(c, P, s);
        s = proto;
        s.type = SEG_Y; s.flags[0] = fy; s.alpha[0] = ay;
        last = add_seg(c, P, s);
    }
    Seg z = proto;
    z.type = SEG_Z; z.flags[0] = fz; z.alpha[0] = az; z.series = nullptr;
    z.dep = chain ? last : -1; z.dep_count = P.segs[last].nitems;
    return add_seg(c, P, z);
}

// per-segment launches index items from 0 and use their own counters
void make_standalone(Program& P) {
    for (Seg& s : P.segs) { s.item0 = 0; s.dep = -1; if (s.type == SEG_XY) s.plane0 = 0; }
}

__global__ void cheb_tail_kernel(cd* out, const cd* P, const cd* Q, const cd* O, double cP, double cQ, int useO, long long n) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const cd p = P[i], q = Q[i];
    cd r = make_double2(cP * p.x + cQ * q.x, cP * p.y + cQ * q.y);
    if (useO) { const cd o = O[i]; r.x += o.x; r.y += o.y; }
    out[i] = r;
}

}  // namespace

namespace sgw {

int eng_check_error(sgw_ctx* c) {
    if (!c->d_err) return 0;
    int flag = 0;
    SGW_TRY(check_cuda(cudaMemcpyAsync(&flag, c->d_err, sizeof(int), cudaMemcpyDeviceToHost, c->stream), "error flag"));
    SGW_TRY(check_cuda(cudaStreamSynchronize(c->stream), "sync"));
    if (flag) {
        cudaMemsetAsync(c->d_err, 0, sizeof(int), c->stream);
        return set_error(SGW_ECUDA, "pass engine: a dependency wait gave up (internal error)");
    }
    return 0;
}

// out = (Tx + Ty + Tz + V_loc) in for nv vectors (the KB term is added by the caller)
int eng_apply_H(sgw_ctx* c, int nv, const cd* in, cd* out) {
    Program P;
    Seg s = blank_seg();
    s.cur = in; s.acc = out; s.hs = 1.0; s.vtab = c->vloc;
    const int half = (cubic(c) && nv >= 2) ? nv / 2 : nv;
    for (int v0 = 0; v0 < nv; v0 += half) {
        const int n = (nv - v0 < half) ? nv - v0 : half;
        add_apply(c, P, s, v0, n, -1, 0, c->vloc ? F_VTAB : 0, 0, 0, 1, 0, 1);
    }
    if (!cubic(c)) make_standalone(P);
    Tables t;
    for (int a = 0; a < 3; ++a) { t.kre[a] = c->kin[a]; t.kc[a] = nullptr; }
    t.cplx = false;
    SGW_TRY(upload_program(c, P));
    return launch_program(c, P, t, 0);
}


// Chebyshev recurrence (Eq. 3; R-1) on nvec <= max_nvec vectors, tables already scaled by s = 2/dE:
//   term n (n = 1..nterms-1): cur = phi_{n-1}, acc = phi_{n-2} -> acc = phi_n = hs (sT + vtab) cur - acc
//   (hs = 1/2 and no subtraction for n = 1).  The series is updated in the x pass of every even term with
//   the two vectors it has in registers; the tail kernel adds what is still pending and writes psi.
int eng_cheb_filter(sgw_ctx* c, int nvec, cd* psi, const double* a, double s, int nterms) {
    const long long ng = c->ng;
    SGW_TRY(ensure_ws(c, 2));
    cd *Pb = psi, *Qb = c->ws[0], *Ob = c->ws[1];
    const bool kb = c->nsphere > 0;
    const int L = nterms - 1;
    // vectors per launch group: L2-resident groups when at least two vectors (3 arrays each) fit
    const double bytes_vec = 16.0 * (double)ng, l2_budget = 96.0e6;
    int fit = (int)(l2_budget / (3.0 * bytes_vec));
    bool resident = false;      // measured slower than streaming all vectors per term (launches too small): opt-in
    if (c->eng_resident > 0 && cubic(c) && !kb) { resident = true; if (fit < c->eng_resident) fit = c->eng_resident; }
    int group = nvec;
    if (resident) { group = fit < nvec ? fit : nvec; if (group > 2) group &= ~1; }
    Tables t;
    for (int ax = 0; ax < 3; ++ax) { t.kre[ax] = c->cheb_kin[ax]; t.kc[ax] = nullptr; }
    t.cplx = false;

    auto build = [&](Program& P, int nvg, int n_begin, int n_end) {
        // two interleaved chunks so that a chunk's z pass (and the next term's x pass) finds its
        // predecessor long finished
        const int nch = (cubic(c) && nvg >= 2) ? 2 : 1;
        int cv0[2] = {0, nvg / 2}, cn[2] = {nch == 2 ? nvg / 2 : nvg, nvg - nvg / 2};
        int lastz[2] = {-1, -1};
        unsigned lastz_items[2] = {0, 0};
        // per-plane x counters are reused by every term of the launch with a growing target
        const unsigned tpp = (unsigned)(c->nx / c->engB[0]);
        unsigned pl0[2] = {P.nplanes, P.nplanes + (unsigned)(cn[0] * c->nz)};
        if (c->nx == c->ny) P.nplanes += (unsigned)(nvg * c->nz);
        unsigned gen = 0;
        for (int n = n_begin; n < n_end; ++n) {
            Seg sg = blank_seg();
            const bool odd = n & 1;
            sg.cur = odd ? Pb : Qb;
            sg.acc = odd ? Qb : Pb;
            sg.series = Ob;
            sg.vtab = c->vtab;
            sg.hs = (n == 1) ? 0.5 : 1.0;
            int fx = F_VTAB;
            if (n >= 2 && !odd) {
                fx |= F_FLUSH;
                if (n == 2) fx |= F_SINIT;
                sg.c0 = a[n - 2]; sg.c1 = a[n - 1];
            }
            ++gen;
            for (int ch = 0; ch < nch; ++ch) {
                lastz[ch] = add_apply(c, P, sg, cv0[ch], cn[ch], lastz[ch], lastz_items[ch], fx, n == 1 ? 0 : -1, 0, 1, 0, 1,
                                      pl0[ch], tpp * gen);
                lastz_items[ch] = P.segs[lastz[ch]].nitems;
            }
            if (nch == 2) {
                // order: XY(c0) XY(c1) Z(c0) Z(c1): move Z(c0) behind XY(c1)
                const size_t k = P.segs.size();
                // segments appended: [XY0, Z0, XY1, Z1] at k-4..k-1 -> [XY0, XY1, Z0, Z1]
                Seg xy0 = P.segs[k - 4], z0 = P.segs[k - 3], xy1 = P.segs[k - 2], z1 = P.segs[k - 1];
                const int i_xy0 = (int)k - 4, i_xy1 = (int)k - 3, i_z0 = (int)k - 2, i_z1 = (int)k - 1;
                xy1.item0 = xy0.item0 + xy0.nitems;
                z0.item0 = xy1.item0 + xy1.nitems;
                z1.item0 = z0.item0 + z0.nitems;
                z0.dep = i_xy0; z1.dep = i_xy1;
                P.segs[k - 4] = xy0; P.segs[k - 3] = xy1; P.segs[k - 2] = z0; P.segs[k - 1] = z1;
                lastz[0] = i_z0; lastz[1] = i_z1;
            }
        }
    };

    for (int g0 = 0; g0 < nvec; g0 += group) {
        const int nvg = (nvec - g0 < group) ? nvec - g0 : group;
        const long long voff = (long long)g0 * ng;
        if (kb || !cubic(c)) {
            // one term per program: the KB scatter (atomics into acc) must not overlap the passes
            for (int n = 1; n <= L; ++n) {
                Program P;
                build(P, nvg, n, n + 1);
                if (!cubic(c)) make_standalone(P);
                SGW_TRY(upload_program(c, P));
                SGW_TRY(launch_program(c, P, t, voff));
                if (kb) {
                    const bool odd = n & 1;
                    SGW_TRY(kb_apply(c, nvg, (odd ? Pb : Qb) + voff, (odd ? Qb : Pb) + voff, 0, s * (n == 1 ? 0.5 : 1.0)));
                }
            }
        } else {
            // all terms in as few launches as the counter range allows
            const int terms_per_launch = 256;
            for (int n0 = 1; n0 <= L; n0 += terms_per_launch) {
                const int n1 = (n0 + terms_per_launch <= L + 1) ? n0 + terms_per_launch : L + 1;
                Program P;
                build(P, nvg, n0, n1);
                SGW_TRY(upload_program(c, P));
                SGW_TRY(launch_program(c, P, t, voff));
            }
        }
        // tail: psi = O + pending terms.  phi_L is in the acc buffer of term L, phi_{L-1} in its cur buffer.
        const bool Lodd = L & 1;
        cd* bufL = (Lodd ? Qb : Pb) + voff;      // acc of term L
        cd* bufLm1 = (Lodd ? Pb : Qb) + voff;    // cur of term L
        double cL = a[L], cLm1 = 0.0;
        const bool useO = L >= 2;
        if (Lodd) cLm1 = a[L - 1];               // not yet flushed (flushes happen in even terms)
        const double cP = Lodd ? cLm1 : cL, cQ = Lodd ? cL : cLm1;
        (void)bufL; (void)bufLm1;
        const long long n = (long long)nvg * ng;
        cheb_tail_kernel<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(Pb + voff, Pb + voff, Qb + voff, Ob + voff, cP, cQ,
                                                                         useO ? 1 : 0, n);
        c->launches++;
        SGW_TRY(check_cuda(cudaGetLastError(), "cheb_tail"));
    }
    return 0;
}

// One split-operator step on nvec vectors with the phase table c->phase = exp(-i V dt/2) (R-8).
int eng_td_step(sgw_ctx* c, int nvec, cd* psi, bool kb) {
    Program P;
    Seg s = blank_seg();
    s.cur = psi; s.acc = psi; s.hs = 1.0; s.phase = c->phase;
    const int half = (cubic(c) && nvec >= 2) ? nvec / 2 : nvec;
    for (int v0 = 0; v0 < nvec; v0 += half) {
        const int n = (nvec - v0 < half) ? nvec - v0 : half;
        add_apply(c, P, s, v0, n, -1, 0, kb ? 0 : F_PRO, 0, 0, 0, kb ? 0 : F_EPI, 0);
    }
    if (!cubic(c)) make_standalone(P);
    Tables t;
    for (int a = 0; a < 3; ++a) { t.kre[a] = nullptr; t.kc[a] = c->td_kin[a]; }
    t.cplx = true;
    SGW_TRY(upload_program(c, P));
    return launch_program(c, P, t, 0);
}

}  // namespace sgw

// =====================================================================================================
// lean passes (sgw_lean.cuh): the default implementation
// =====================================================================================================
namespace {

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
    cudaEvent_t e1 = prof_begin(c, prof_tag);
    const int rc = c->lean[axis_n](&call, c->engB[0]);
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
    const int n = c->nx, B = c->engB[0];
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
    { const char* e = getenv("SGW_LEAN_CLUSTER"); if (e) use_cluster = atoi(e) ? 1 : 0; }
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
    const int B = c->engB[0];
    const long long nxy = (long long)c->nx * c->ny;
    LeanArgs a;
    memset(&a, 0, sizeof(a));
    a.cur = op.cur; a.acc = op.acc; a.series = op.series; a.vtab = op.vtab; a.phase = op.phase;
    a.rho = op.rho; a.dens_scale = op.dens_scale;
    a.hs = op.hs; a.c0 = op.c0; a.c1 = op.c1;
    a.nx = c->nx; a.ny = c->ny; a.nz = c->nz;
    int G = 1, ctas = 0, wpc = 8, cluster = 0;
    if (allow_plane && lean_use_plane(c, op.cplx, &G, &ctas, &wpc, &cluster)) {
        a.tw = c->tw[0];
        a.kre[0] = op.kre[0]; a.kre[1] = op.kre[1]; a.kc[0] = op.kc[0]; a.kc[1] = op.kc[1];
        a.flags[0] = op.fx; a.alpha[0] = op.ax; a.flags[1] = op.fy; a.alpha[1] = op.ay;
        a.ntiles = (unsigned)((long long)nv * c->nz);
        a.G = G;
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

// Chebyshev recurrence, accumulated in place (same scheme as eng_cheb_filter): term n takes cur = phi_{n-1},
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
    { const char* e = getenv("SGW_LEAN_CHUNK"); if (e && atoi(e) > 0 && !kb) chunk = atoi(e) < nvec ? atoi(e) : nvec; }
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
    return lean_apply(c, nvec, op, K_RT_TD);
}

}  // namespace sgw
