// sgw_engine.cuh -- the pass engine of libsgw: one persistent kernel that executes a *program* of
// round-trip passes (forward FFT along one axis, k-space multiply, inverse FFT, fused pointwise
// work) with dependency counters between passes, for sm_100a.
//
// Why this shape ("FFT pairs switch between position and momentum representations"):
//  * T = Tx + Ty + Tz is additively separable and exp(-i T dt) multiplicatively separable, so H apply,
//    a Chebyshev term and a split-operator step are each three 1D round trips, every one of the form
//        acc <- hs * RT_axis(cur) + [hs * vtab * cur] + alpha * acc            (real k table)
//        psi <- [phase] RT_axis([phase] psi)                                   (complex k table)
//    All pointwise work (potential multiply, recurrence, series accumulation, phases) is done in
//    registers on load or on store, so a pass touches cur once and acc once.
//  * A tile is B pencils of length N (B*16 bytes contiguous per row for the strided axes) and belongs
//    to one *warp group* of B*R2 threads (one warp for N = 96, B = 4).  Groups are autonomous: they
//    take items, wait for dependencies, exchange through their own slice of shared memory and publish
//    completion without any CTA-wide barrier, so the 16-24 warps of an SM are in different phases
//    and hide each other's load latency (the earlier one-CTA-per-SM kernels and the first engine with
//    CTA-wide barriers were latency bound: profiles/r01_v2_cfg1.md).
//  * Segments of a program are ordered; a segment may wait for an earlier one (whole segment, or
//    plane by plane for y after x).  All CTAs are co-resident (cooperative launch), items are dealt
//    round robin in program order, so every wait is for an item owned by a running CTA that does
//    not itself wait on later items: no deadlock.  A bounded spin sets an error flag instead of
//    hanging.  With dependencies inside one launch, the x->y transpose and (for grids whose vectors
//    fit) whole Chebyshev terms run out of the 126 MB L2 without kernel boundaries.
#pragma once
#include "sgw_fft.cuh"

namespace sgw {

// two-stage factorisation N = R1 * R2: stage A (global load/store side) keeps R1 values per thread
// with R2 threads per pencil; stage B (pure compute) is R1 independent radix-R2 round trips per pencil.
template <int N> struct Fact2;
#define SGW_FACT2(N_, R1_, R2_) \
    template <> struct Fact2<N_> { static constexpr int R1 = R1_, R2 = R2_; };
SGW_FACT2(8, 2, 4)
SGW_FACT2(12, 3, 4)
SGW_FACT2(16, 4, 4)
SGW_FACT2(24, 6, 4)
SGW_FACT2(32, 8, 4)
SGW_FACT2(48, 12, 4)
SGW_FACT2(64, 8, 8)
SGW_FACT2(96, 12, 8)
SGW_FACT2(128, 16, 8)
SGW_FACT2(192, 12, 16)
SGW_FACT2(256, 16, 16)
SGW_FACT2(384, 16, 24)
#undef SGW_FACT2

enum { SEG_X = 0, SEG_Y = 1, SEG_Z = 2, SEG_XY = 3 };
enum {
    F_VTAB = 1,      // add hs * vtab[g] * cur to the result
    F_FLUSH = 2,     // series <- [series] + c0 * acc_old + c1 * cur        (on load)
    F_SINIT = 4,     // with F_FLUSH: series is written, not accumulated
    F_PRO = 8,       // complex family: multiply by phase[g] on load
    F_EPI = 16,      // complex family: multiply by phase[g] on store
    F_DENS = 32      // complex family: rho[g] += dens_scale * |result|^2 (atomic)
};

// One pass (SEG_X, SEG_Y, SEG_Z) or an x pass and a y pass over the same planes (SEG_XY) over nvec
// vectors.  Pointers are for vector 0 of the launch; the launch adds its vector offset.
struct Seg {
    const cd* cur;
    cd* acc;
    cd* series;
    const double* vtab;
    const cd* phase;
    double* rho;
    double hs, c0, c1, dens_scale;
    int type;
    int flags[2];        // [0]: the pass (or the x half of SEG_XY); [1]: the y half
    int alpha[2];        // 0: acc is not read; +1 / -1
    int nvec;
    int pc;              // SEG_XY: planes per group (all x tiles of a group, then its y tiles)
    int dep;             // index of the segment that must be complete before this one starts, or -1
    unsigned dep_count;  // its number of items
    unsigned item0, nitems;
    unsigned plane0;     // SEG_XY: first per-plane counter
    unsigned plane_target;
};

struct EngArgs {
    const Seg* segs;
    int nseg;
    unsigned nitems;          // total over all segments
    unsigned* cnt_seg;        // [nseg]   items completed per segment (zeroed before the launch)
    unsigned* cnt_plane;      // per-plane x-tile counters
    int* err;                 // set to 1 if a wait gave up
    long long voff;           // element offset added to cur / acc / series
    const cd* tw;             // exp(-2 pi i j / N)
    const double* kre[3];     // real k tables per axis (include 1/N and any scale)
    const cd* kc[3];          // complex k tables per axis
    int nx, ny, nz;
    int use_deps;
    int l2_prefetch;          // prefetch the next item's operands into L2
};


template <int N, int B>
struct EngCfg {
    static constexpr int R1 = Fact2<N>::R1, R2 = Fact2<N>::R2;
    static constexpr int TG = B * R2;                        // threads of a group that own stage-A data
    static constexpr int GW = (TG + 31) / 32;                // warps per group
    static constexpr int GT = GW * 32;
    static constexpr int NWG = (8 / GW) > 0 ? (8 / GW) : 1;  // groups per CTA
    static constexpr int T = NWG * GT;
    static constexpr int MINB = (65536 / 128) / T > 0 ? (65536 / 128) / T : 1;   // aim at <= 128 registers
    static constexpr int TASKS = R1 * B;                     // stage-B round trips per tile
    static constexpr int ROUNDS = (TASKS + GT - 1) / GT;
    static constexpr int SK = R2 | 1;
    static constexpr int SB0 = R1 * SK;
    // pencil stride in the exchange buffer: odd for B = 8, = 2 (mod 8) for B = 4 (bank spread of the
    // strided-axis stores, where a quarter warp holds B pencils x 8/B consecutive n2)
    static constexpr int SB = (B >= 8) ? (SB0 | 1) : (SB0 + ((10 - (SB0 % 8)) % 8));
    static constexpr int XCH = B * SB;                       // complex elements per group
    static constexpr int GROUP_BYTES = ((XCH * 16 + (int)sizeof(Seg) + 16 + 15) / 16) * 16;
    static constexpr int TAB_REAL = 2 * N * 16 + 3 * N * 8;
    static constexpr int TAB_CPLX = 2 * N * 16 + 3 * N * 16;
    static constexpr int SMEM_REAL = TAB_REAL + NWG * GROUP_BYTES;
    static constexpr int SMEM_CPLX = TAB_CPLX + NWG * GROUP_BYTES;
};

__device__ __forceinline__ unsigned ld_acquire_u32(const unsigned* p) {
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];\n" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void red_release_u32(unsigned* p, unsigned v) {
    asm volatile("red.release.gpu.global.add.u32 [%0], %1;\n" ::"l"(p), "r"(v) : "memory");
}

// wait until *p >= target (relaxed polls, one acquire once satisfied); gives up (sets *err) after ~2^21 polls
__device__ __forceinline__ bool spin_until(const unsigned* p, unsigned target, int* err) {
    unsigned spins = 0, v;
    for (;;) {
        asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];\n" : "=r"(v) : "l"(p) : "memory");
        if (v >= target) break;
        __nanosleep(400);
        if (++spins > (1u << 21)) { atomicExch(err, 1); return false; }
        if ((spins & 255u) == 0 && *reinterpret_cast<volatile int*>(err)) return false;
    }
    return ld_acquire_u32(p) >= target;
}

template <int GW>
__device__ __forceinline__ void group_sync(int grp) {
    if (GW == 1) __syncwarp();
    else asm volatile("bar.sync %0, %1;\n" ::"r"(grp + 1), "r"(GW * 32) : "memory");
}

template <int N, int B, bool CPLX>
__global__ void __launch_bounds__(EngCfg<N, B>::T, EngCfg<N, B>::MINB) engine_kernel(const EngArgs a) {
    using C = EngCfg<N, B>;
    constexpr int R1 = C::R1, R2 = C::R2, TG = C::TG, GW = C::GW, GT = C::GT, NWG = C::NWG;
    constexpr int SK = C::SK, SB = C::SB, TASKS = C::TASKS, ROUNDS = C::ROUNDS;
    extern __shared__ __align__(16) char smraw[];
    cd* twA = reinterpret_cast<cd*>(smraw);                  // twA[j*R2 + n2] = W^(n2 j)
    cd* twB = twA + N;                                       // twB[m*R1 + k1] = W^(m k1)
    char* ktab = reinterpret_cast<char*>(twB + N);           // [axis][k], 8 or 16 bytes each
    const int tid = threadIdx.x, grp = tid / GT, gt = tid % GT;
    char* gbase = smraw + (CPLX ? C::TAB_CPLX : C::TAB_REAL) + grp * C::GROUP_BYTES;
    cd* xch = reinterpret_cast<cd*>(gbase);
    Seg* sg = reinterpret_cast<Seg*>(xch + C::XCH);
    int* s_ok = reinterpret_cast<int*>(sg + 1);

    for (int i = tid; i < N; i += C::T) {
        twA[i] = a.tw[(i % R2) * (i / R2)];
        twB[i] = a.tw[(i / R1) * (i % R1)];
    }
#pragma unroll
    for (int ax = 0; ax < 3; ++ax) {
        for (int k = tid; k < N; k += C::T) {
            if (CPLX) { if (a.kc[ax]) reinterpret_cast<cd*>(ktab)[ax * N + k] = a.kc[ax][k]; }
            else { if (a.kre[ax]) reinterpret_cast<double*>(ktab)[ax * N + k] = a.kre[ax][k]; }
        }
    }
    __syncthreads();                                         // the only CTA-wide barrier

    // stage-A coordinates for the contiguous axis (lanes along n) and the strided axes (lanes along b)
    const int n2_f = gt % R2, bA_f = gt / R2;
    const int bA_s = gt % B, n2_s = gt / B;
    const bool actA = gt < TG;
    const int nxy = a.nx * a.ny;
    const long long ng = (long long)nxy * a.nz;

    // item r of the cached segment -> pass axis, x/y half, plane, tile origin and strides
    auto decode = [&](unsigned r, int& axis, int& half, unsigned& plane, long long& base, int& g0, int& sN, int& sB) {
        const int type = sg->type;
        axis = type; half = 0; plane = 0;
        unsigned outer, inner;
        if (type == SEG_XY) {
            // groups of pc planes; order X(0) | X(1) Y(0) | X(2) Y(1) | ... | Y(G-1): a group's y tiles
            // come one slot after its x tiles, so they rarely have to wait
            const unsigned tpp = N / B, per = (unsigned)sg->pc * tpp;
            const unsigned G = ((unsigned)sg->nvec * (unsigned)a.nz) / (unsigned)sg->pc;
            unsigned grpi, q2;
            if (r < per) { grpi = 0; q2 = r; }
            else {
                const unsigned r1 = r - per, slot = 1 + r1 / (2 * per), q = r1 % (2 * per);
                if (slot < G && q < per) { grpi = slot; q2 = q; }
                else { half = 1; grpi = slot - 1; q2 = (slot < G) ? q - per : q; }
            }
            plane = grpi * sg->pc + q2 / tpp;
            outer = plane; inner = q2 % tpp;
            axis = half;
        } else if (type == SEG_Z) {
            const unsigned ti = (unsigned)(nxy / B);
            outer = r / ti; inner = r - outer * ti;
        } else {
            const unsigned ti = (unsigned)((type == SEG_X ? a.ny : a.nx) / B);
            outer = r / ti; inner = r - outer * ti;
            plane = outer;
        }
        if (axis == 0)      { base = (long long)outer * nxy + (long long)inner * B * a.nx; g0 = (int)(outer % (unsigned)a.nz) * nxy + (int)inner * B * a.nx; sN = 1; sB = a.nx; }
        else if (axis == 1) { base = (long long)outer * nxy + (long long)inner * B;        g0 = (int)(outer % (unsigned)a.nz) * nxy + (int)inner * B;        sN = a.nx; sB = 1; }
        else                { base = (long long)outer * ng + (long long)inner * B;         g0 = (int)inner * B;                                              sN = nxy; sB = 1; }
    };

    int si = -1, dep_ok = -1, pub_si = -1;
    unsigned seg_end = 0, pub_plane = 0xffffffffu;
    const unsigned stride = gridDim.x * NWG;
    for (unsigned it = blockIdx.x * NWG + grp; it < a.nitems; it += stride) {
        group_sync<GW>(grp);                                 // previous item: xch and sg no longer read, stores issued
        if (it >= seg_end) {
            do { ++si; } while (it >= a.segs[si].item0 + a.segs[si].nitems);
            const int* src = reinterpret_cast<const int*>(a.segs + si);
            int* dst = reinterpret_cast<int*>(sg);
            for (int i = gt; i < (int)(sizeof(Seg) / 4); i += GT) dst[i] = src[i];
            group_sync<GW>(grp);
            seg_end = sg->item0 + sg->nitems;
        }
        // ---- decode the item ------------------------------------------------------------------
        int axis, half, g0, sN, sB;
        unsigned plane;
        long long base;
        decode(it - sg->item0, axis, half, plane, base, g0, sN, sB);
        // L2 prefetch of the next item's operands (no dependency needed: L2 is the coherence point)
        if (a.l2_prefetch && it + stride < seg_end) {
            int axis2, half2, g02, sN2, sB2;
            unsigned plane2;
            long long base2;
            decode(it + stride - sg->item0, axis2, half2, plane2, base2, g02, sN2, sB2);
            const bool f2 = axis2 == 0;
            const int n22 = f2 ? n2_f : n2_s, bA2 = f2 ? bA_f : bA_s;
            if (actA && (f2 ? (n22 % 8 == 0) : (bA2 == 0))) {
                const long long o2 = a.voff + base2 + n22 * sN2 + bA2 * sB2;
                const cd* pc_ = sg->cur + o2;
                const cd* pa_ = sg->acc + o2;
                const bool want_acc = sg->alpha[half2] != 0 && sg->acc != sg->cur;
#pragma unroll
                for (int n1 = 0; n1 < R1; ++n1) {
                    asm volatile("prefetch.global.L2 [%0];\n" ::"l"(pc_ + n1 * R2 * sN2));
                    if (want_acc) asm volatile("prefetch.global.L2 [%0];\n" ::"l"(pa_ + n1 * R2 * sN2));
                }
            }
        }
        const bool fastn = axis == 0;
        const int n2 = fastn ? n2_f : n2_s, bA = fastn ? bA_f : bA_s;
        const int e0 = n2 * sN + bA * sB, estep = R2 * sN;
        const int flags = sg->flags[half], alpha = sg->alpha[half];
        const double hs = sg->hs;

        // ---- dependencies --------------------------------------------------------------------
        if (a.use_deps) {
            const unsigned* p = nullptr;
            unsigned target = 0;
            if (half) { p = a.cnt_plane + sg->plane0 + plane; target = sg->plane_target; }
            else if (sg->dep >= 0 && sg->dep != dep_ok) { p = a.cnt_seg + sg->dep; target = sg->dep_count; }
            if (p) {
                if (gt == 0) {
                    // never wait while holding an unpublished completion (another group may need it)
                    if (pub_si >= 0) {
                        red_release_u32(a.cnt_seg + pub_si, 1u);
                        if (pub_plane != 0xffffffffu) red_release_u32(a.cnt_plane + pub_plane, 1u);
                    }
                    *s_ok = spin_until(p, target, a.err) ? 1 : 0;
                }
                pub_si = -1;
                group_sync<GW>(grp);
                if (!*s_ok) return;
                if (!half) dep_ok = sg->dep;
            }
        }

        // ---- load, pointwise work on load ----------------------------------------------------
        const cd* cur = sg->cur + a.voff + base + e0;
        cd* acc = sg->acc + a.voff + base + e0;
        cd x[R1], ad[R1];
        if (actA) {
#pragma unroll
            for (int n1 = 0; n1 < R1; ++n1) x[n1] = __ldcg(cur + n1 * estep);
            if (CPLX) {
                if (flags & (F_PRO | F_EPI)) {
                    const cd* ph = sg->phase + g0 + e0;
#pragma unroll
                    for (int n1 = 0; n1 < R1; ++n1) ad[n1] = __ldg(ph + n1 * estep);
                    if (flags & F_PRO) {
#pragma unroll
                        for (int n1 = 0; n1 < R1; ++n1) x[n1] = cmul(x[n1], ad[n1]);
                    }
                }
            } else {
                if (alpha != 0) {
#pragma unroll
                    for (int n1 = 0; n1 < R1; ++n1) ad[n1] = __ldcg(acc + n1 * estep);
                } else {
#pragma unroll
                    for (int n1 = 0; n1 < R1; ++n1) ad[n1] = make_double2(0.0, 0.0);
                }
                if (flags & F_FLUSH) {
                    cd* ser = sg->series + a.voff + base + e0;
                    const double c0 = sg->c0, c1 = sg->c1;
#pragma unroll
                    for (int n1 = 0; n1 < R1; ++n1) {
                        cd s = make_double2(c0 * ad[n1].x + c1 * x[n1].x, c0 * ad[n1].y + c1 * x[n1].y);
                        if (!(flags & F_SINIT)) s = cadd(s, __ldcs(ser + n1 * estep));
                        __stcs(ser + n1 * estep, s);
                    }
                }
                const double al = (double)alpha;
                if (flags & F_VTAB) {
                    const double* vt = sg->vtab + g0 + e0;
#pragma unroll
                    for (int n1 = 0; n1 < R1; ++n1) {
                        const double v = hs * __ldg(vt + n1 * estep);
                        ad[n1] = make_double2(v * x[n1].x + al * ad[n1].x, v * x[n1].y + al * ad[n1].y);
                    }
                } else {
#pragma unroll
                    for (int n1 = 0; n1 < R1; ++n1) ad[n1] = cscale(ad[n1], al);
                }
            }
        }

        // ---- round trip: A | exchange | B, multiply, B^-1 | exchange | A^-1 --------------------
        cd* xA = xch + bA * SB + n2;
        if (actA) {
            Dft<R1, -1>::run(x);
            xA[0] = x[0];
#pragma unroll
            for (int j = 1; j < R1; ++j) xA[j * SK] = cmul(x[j], twA[j * R2 + n2]);
        }
        group_sync<GW>(grp);
        // publish the previous item here: its stores were issued a whole load + stage A ago, so the
        // release does not wait for them
        if (a.use_deps && pub_si >= 0 && gt == 0) {
            red_release_u32(a.cnt_seg + pub_si, 1u);
            if (pub_plane != 0xffffffffu) red_release_u32(a.cnt_plane + pub_plane, 1u);
        }
        pub_si = -1;
#pragma unroll
        for (int rd = 0; rd < ROUNDS; ++rd) {
            const int task = gt + rd * GT;
            if (task < TASKS) {
                const int bB = task % B, k1 = task / B;      // pencils fastest: bank-conflict free (odd pencil stride)
                cd* xB = xch + bB * SB + k1 * SK;
                cd y[R2];
#pragma unroll
                for (int m = 0; m < R2; ++m) y[m] = xB[m];
                Dft<R2, -1>::run(y);
                if (CPLX) {
                    const cd* kt = reinterpret_cast<const cd*>(ktab) + axis * N + k1;
#pragma unroll
                    for (int k2 = 0; k2 < R2; ++k2) y[k2] = cmul(y[k2], kt[R1 * k2]);
                } else {
                    const double* kt = reinterpret_cast<const double*>(ktab) + axis * N + k1;
#pragma unroll
                    for (int k2 = 0; k2 < R2; ++k2) y[k2] = cscale(y[k2], kt[R1 * k2]);
                }
                Dft<R2, +1>::run(y);
                xB[0] = y[0];
#pragma unroll
                for (int m = 1; m < R2; ++m) xB[m] = cmulc(y[m], twB[m * R1 + k1]);
            }
        }
        group_sync<GW>(grp);
        if (actA) {
#pragma unroll
            for (int j = 0; j < R1; ++j) x[j] = xA[j * SK];
            Dft<R1, +1>::run(x);

            // ---- pointwise work on store ---------------------------------------------------------
            if (CPLX) {
                if (flags & F_EPI) {
#pragma unroll
                    for (int n1 = 0; n1 < R1; ++n1) x[n1] = cmul(x[n1], ad[n1]);
                }
                if (flags & F_DENS) {
                    double* rho = sg->rho + g0 + e0;
                    const double ds = sg->dens_scale;
#pragma unroll
                    for (int n1 = 0; n1 < R1; ++n1)
                        atomicAdd(rho + n1 * estep, ds * (x[n1].x * x[n1].x + x[n1].y * x[n1].y));
                }
#pragma unroll
                for (int n1 = 0; n1 < R1; ++n1) __stcg(acc + n1 * estep, x[n1]);
            } else {
#pragma unroll
                for (int n1 = 0; n1 < R1; ++n1)
                    __stcg(acc + n1 * estep, make_double2(hs * x[n1].x + ad[n1].x, hs * x[n1].y + ad[n1].y));
            }
        }
        pub_si = si;
        pub_plane = (sg->type == SEG_XY && !half) ? sg->plane0 + plane : 0xffffffffu;
    }
    group_sync<GW>(grp);
    if (a.use_deps && pub_si >= 0 && gt == 0) {
        red_release_u32(a.cnt_seg + pub_si, 1u);
        if (pub_plane != 0xffffffffu) red_release_u32(a.cnt_plane + pub_plane, 1u);
    }
}

struct EngCall {
    EngArgs args;
    int cplx;
    int max_ctas;             // 0 = fill the device
    cudaStream_t stream;
};
// returns 0, a negative sgw error code, or 1 if this (N, B) is not instantiated
typedef int (*eng_launch_fn)(const EngCall*, int B);

}  // namespace sgw
