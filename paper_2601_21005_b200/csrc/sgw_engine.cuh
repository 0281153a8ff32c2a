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
//  * A tile is B pencils of length N (B*16 bytes contiguous per row for the strided axes); a CTA is
//    only B*R2 threads (96 for N = 96) and needs ~20 KB of shared memory, so 5-7 CTAs share an SM
//    and hide each other's load latency and barrier waits (the earlier one-CTA-per-SM kernels were
//    latency bound: profiles/r01_v2_cfg1.md).
//  * Segments of a program are ordered; a segment may wait for an earlier one (whole segment, or
//    plane by plane for y after x).  All CTAs are co-resident (cooperative launch), items are dealt
//    round robin in program order, so every wait is for an item owned by a running CTA that does
//    not itself wait on later items: no deadlock.  A bounded spin sets an error flag instead of
//    hanging.  With dependencies inside one launch, the x->y transpose and (for grids whose vectors
//    fit) whole Chebyshev terms run out of the 126 MB L2 without kernel boundaries.
#pragma once
#include "sgw_fft.cuh"

namespace sgw {

// two-stage factorisation with the SMALL radix first: stage A (global load/store side) keeps R1
// values per thread, stage B (pure compute) R2 values; R2 threads per pencil.
template <int N> struct Fact2;
#define SGW_FACT2(N_, R1_, R2_) \
    template <> struct Fact2<N_> { static constexpr int R1 = R1_, R2 = R2_; };
SGW_FACT2(8, 2, 4)
SGW_FACT2(12, 3, 4)
SGW_FACT2(16, 4, 4)
SGW_FACT2(24, 4, 6)
SGW_FACT2(32, 4, 8)
SGW_FACT2(48, 6, 8)
SGW_FACT2(64, 8, 8)
SGW_FACT2(96, 8, 12)
SGW_FACT2(128, 8, 16)
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
};

template <int N, int B>
struct EngCfg {
    static constexpr int R1 = Fact2<N>::R1, R2 = Fact2<N>::R2;
    static constexpr int T = B * R2;
    static constexpr int SK = R2 | 1;
    static constexpr int SB = (R1 * SK) | 1;
    static constexpr int XCH = B * SB;                       // complex elements
    static constexpr int SMEM_REAL = (XCH + 2 * N) * 16 + 3 * N * 8;
    static constexpr int SMEM_CPLX = (XCH + 2 * N) * 16 + 3 * N * 16;
};

__device__ __forceinline__ unsigned ld_acquire_u32(const unsigned* p) {
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];\n" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void red_release_u32(unsigned* p, unsigned v) {
    asm volatile("red.release.gpu.global.add.u32 [%0], %1;\n" ::"l"(p), "r"(v) : "memory");
}

// wait until *p >= target; gives up (sets *err) after ~2^22 polls
__device__ __forceinline__ bool spin_until(const unsigned* p, unsigned target, int* err) {
    unsigned spins = 0;
    while (ld_acquire_u32(p) < target) {
        __nanosleep(200);
        if (++spins > (1u << 22)) { atomicExch(err, 1); return false; }
        if ((spins & 255u) == 0 && *reinterpret_cast<volatile int*>(err)) return false;
    }
    return true;
}

template <int N, int B, bool CPLX>
__global__ void __launch_bounds__(EngCfg<N, B>::T) engine_kernel(const EngArgs a) {
    using C = EngCfg<N, B>;
    constexpr int R1 = C::R1, R2 = C::R2, T = C::T, SK = C::SK, SB = C::SB;
    extern __shared__ __align__(16) char smraw[];
    cd* xch = reinterpret_cast<cd*>(smraw);
    cd* twA = xch + C::XCH;                                  // twA[j*R2 + n2] = W^(n2 j)
    cd* twB = twA + N;                                       // twB[m*R1 + k1] = W^(m k1)
    char* ktab = reinterpret_cast<char*>(twB + N);           // [axis][k], 8 or 16 bytes each
    __shared__ Seg s_seg;
    __shared__ int s_abort;
    const int tid = threadIdx.x;

    for (int i = tid; i < N; i += T) {
        twA[i] = a.tw[(i % R2) * (i / R2)];
        twB[i] = a.tw[(i / R1) * (i % R1)];
    }
    for (int i = tid; i < 3 * N; i += T) {
        const int ax = i / N, k = i - ax * N;
        if (CPLX) { if (a.kc[ax]) reinterpret_cast<cd*>(ktab)[i] = a.kc[ax][k]; }
        else { if (a.kre[ax]) reinterpret_cast<double*>(ktab)[i] = a.kre[ax][k]; }
    }
    if (tid == 0) s_abort = 0;

    // thread coordinates for the contiguous axis (lanes along n) and the strided axes (lanes along b)
    const int n2_f = tid % R2, bA_f = tid / R2, k1_f = tid % R1, bB_f = tid / R1;
    const int bA_s = tid % B, n2_s = tid / B;
    const long long nxy = (long long)a.nx * a.ny, ng = nxy * a.nz;

    int si = -1;
    unsigned seg_end = 0;
    for (unsigned it = blockIdx.x; it < a.nitems; it += gridDim.x) {
        __syncthreads();                                    // previous item done with xch and s_seg
        if (it >= seg_end) {
            do { ++si; } while (it >= a.segs[si].item0 + a.segs[si].nitems);
            const int* src = reinterpret_cast<const int*>(a.segs + si);
            int* dst = reinterpret_cast<int*>(&s_seg);
            for (int i = tid; i < (int)(sizeof(Seg) / 4); i += T) dst[i] = src[i];
            __syncthreads();
            seg_end = s_seg.item0 + s_seg.nitems;
        }
        // ---- decode the item ------------------------------------------------------------------
        const unsigned r = it - s_seg.item0;
        int axis = s_seg.type, half = 0;
        unsigned outer, inner, plane = 0;
        if (s_seg.type == SEG_XY) {
            const unsigned tpp = N / B, per = (unsigned)s_seg.pc * tpp;
            const unsigned grp = r / (2 * per), q = r - grp * 2 * per;
            half = q >= per;
            const unsigned q2 = half ? q - per : q;
            plane = grp * s_seg.pc + q2 / tpp;
            outer = plane; inner = q2 % tpp;
            axis = half;
        } else if (s_seg.type == SEG_Z) {
            const unsigned ti = (unsigned)(nxy / B);
            outer = r / ti; inner = r - outer * ti;
        } else {
            const unsigned ti = (unsigned)((s_seg.type == SEG_X ? a.ny : a.nx) / B);
            outer = r / ti; inner = r - outer * ti;
            plane = outer;
        }
        long long base, g0, sN, sB;
        if (axis == 0)      { base = (long long)outer * nxy + (long long)inner * B * a.nx; g0 = base % ng; sN = 1; sB = a.nx; }
        else if (axis == 1) { base = (long long)outer * nxy + (long long)inner * B;        g0 = base % ng; sN = a.nx; sB = 1; }
        else                { base = (long long)outer * ng + (long long)inner * B;         g0 = (long long)inner * B; sN = nxy; sB = 1; }
        const bool fastn = axis == 0;
        const int n2 = fastn ? n2_f : n2_s, bA = fastn ? bA_f : bA_s;
        const int k1 = fastn ? k1_f : n2_s, bB = fastn ? bB_f : bA_s;
        const bool actB = fastn ? (tid < B * R1) : (n2_s < R1);
        const long long e0 = (long long)n2 * sN + (long long)bA * sB, estep = (long long)R2 * sN;
        const int flags = s_seg.flags[half], alpha = s_seg.alpha[half];
        const double hs = s_seg.hs;

        // ---- dependencies --------------------------------------------------------------------
        if (a.use_deps) {
            if (tid == 0) {
                bool ok = true;
                if (*reinterpret_cast<volatile int*>(a.err)) ok = false;
                if (ok && s_seg.dep >= 0 && !half) ok = spin_until(a.cnt_seg + s_seg.dep, s_seg.dep_count, a.err);
                if (ok && half) ok = spin_until(a.cnt_plane + s_seg.plane0 + plane, s_seg.plane_target, a.err);
                if (!ok) s_abort = 1;
            }
            __syncthreads();
            if (s_abort) return;
        }

        // ---- load, pointwise work on load ----------------------------------------------------
        const cd* cur = s_seg.cur + a.voff + base + e0;
        cd* acc = s_seg.acc + a.voff + base + e0;
        cd x[R1], ad[R1];
#pragma unroll
        for (int n1 = 0; n1 < R1; ++n1) x[n1] = __ldcg(cur + n1 * estep);
        if (CPLX) {
            if (flags & (F_PRO | F_EPI)) {
                const cd* ph = s_seg.phase + g0 + e0;
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
                cd* ser = s_seg.series + a.voff + base + e0;
                const double c0 = s_seg.c0, c1 = s_seg.c1;
#pragma unroll
                for (int n1 = 0; n1 < R1; ++n1) {
                    cd s = make_double2(c0 * ad[n1].x + c1 * x[n1].x, c0 * ad[n1].y + c1 * x[n1].y);
                    if (!(flags & F_SINIT)) s = cadd(s, __ldcs(ser + n1 * estep));
                    __stcs(ser + n1 * estep, s);
                }
            }
            const double al = (double)alpha;
            if (flags & F_VTAB) {
                const double* vt = s_seg.vtab + g0 + e0;
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

        // ---- round trip: A | exchange | B, multiply, B^-1 | exchange | A^-1 --------------------
        cd* xA = xch + bA * SB + n2;
        cd* xB = xch + bB * SB + k1 * SK;
        Dft<R1, -1>::run(x);
        xA[0] = x[0];
#pragma unroll
        for (int j = 1; j < R1; ++j) xA[j * SK] = cmul(x[j], twA[j * R2 + n2]);
        __syncthreads();
        if (actB) {
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
        __syncthreads();
#pragma unroll
        for (int j = 0; j < R1; ++j) x[j] = xA[j * SK];
        Dft<R1, +1>::run(x);

        // ---- pointwise work on store ------------------------------------------------------------
        if (CPLX) {
            if (flags & F_EPI) {
#pragma unroll
                for (int n1 = 0; n1 < R1; ++n1) x[n1] = cmul(x[n1], ad[n1]);
            }
            if (flags & F_DENS) {
                double* rho = s_seg.rho + g0 + e0;
                const double ds = s_seg.dens_scale;
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

        // ---- publish -----------------------------------------------------------------------------
        if (a.use_deps) {
            __threadfence();
            __syncthreads();
            if (tid == 0) {
                red_release_u32(a.cnt_seg + si, 1u);
                if (s_seg.type == SEG_XY && !half) red_release_u32(a.cnt_plane + s_seg.plane0 + plane, 1u);
            }
        }
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
