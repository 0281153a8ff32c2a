// sgw_lean.cuh -- lean streaming round-trip passes for sm_100a (the default implementation).
//
// One pass = for every tile of B pencils: acc <- hs * RT_axis(cur) [+ hs * V * cur] + alpha * acc (real k
// table: H apply, Chebyshev term) or psi <- [phase] RT_axis([phase] psi) (complex k table:
// split-operator factor).  What the profiles of the earlier kernels showed (profiles/
// r01_lean_cfg1.md) shaped this one:
//  * a tile belongs to an autonomous warp group (B * R2 threads, two warps for N = 96) with its own slice
//    of shared memory and its own named barrier; 16 warps per SM in different phases hide each other's
//    latency, nothing is staged through shared memory, and the only per-item work outside the
//    transforms is one multiply-add for the tile origin;
//  * the input is loaded straight into the registers of the first butterfly stage; everything the
//    epilogue needs (old accumulator, potential, series) is loaded late, after the inverse transform, so
//    it never lives across the transforms (no spills at 128 registers);
//  * measured alone on 64 x 96^3 such a pass runs at 6.2 TB/s (acc += RT(cur), 48 B per point), i.e. at
//    the measured HBM copy peak.
// plane_lean_kernel runs the x and the y pass of whole xy planes in one launch: a CTA owns a group of
// planes, does their row tiles, __syncthreads, then their column tiles, so the x->y transpose goes
// through L2 and HBM sees cur once and acc once for the two passes.
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

// per-pass flags
enum {
    F_VTAB = 1,      // add hs * vtab[g] * cur to the result
    F_FLUSH = 2,     // series <- [series] + c0 * acc_old + c1 * cur        (on load)
    F_SINIT = 4,     // with F_FLUSH: series is written, not accumulated
    F_PRO = 8,       // complex family: multiply by phase[g] on load
    F_EPI = 16,      // complex family: multiply by phase[g] on store
    F_DENS = 32      // complex family: rho[g] += dens_scale * |result|^2 (atomic)
};

struct LeanArgs {
    const cd* cur;            // input vectors
    cd* acc;                  // accumulator / output vectors (may alias cur for the complex family)
    cd* series;               // Chebyshev series accumulator (F_FLUSH)
    const double* vtab;       // N_g real table (F_VTAB)
    const cd* phase;          // N_g complex table (F_PRO / F_EPI)
    double* rho;              // N_g doubles: density accumulator (F_DENS)
    double dens_scale;
    const cd* tw;             // exp(-2 pi i j / N)
    const double* kre[2];     // real k tables (include 1/N and any scale): [0] first pass, [1] second pass (y of a plane launch)
    const cd* kc[2];          // complex k tables
    double hs, c0, c1;
    int flags[2], alpha[2];   // per pass
    int nx, ny, nz;
    unsigned ntiles;          // axis kernel: tiles; plane kernel: planes (nz * nvec)
    int G;                    // plane kernel: planes per CTA-owned group
    int nvec;                 // vectors of the launch
    int vminor;               // 1: consecutive tiles / planes run over the vectors at one grid location, so the N_g tables
                              //    (potential, phases) are read from HBM once per launch instead of once per vector
    unsigned* cnt;            // team plane kernel: one arrival counter per plane (zeroed before the launch)
};

template <int N, int B, int WPC_ = 8>
struct LeanCfg {
    static constexpr int R1 = Fact2<N>::R1, R2 = Fact2<N>::R2;
    static constexpr int TG = B * R2;                        // threads of a group that own stage-A data
    static constexpr int GW = (TG + 31) / 32;                // warps per group
    static constexpr int GT = GW * 32;
    static constexpr int WPC = WPC_;                         // warps per CTA (axis kernels: 8, two CTAs per SM)
    static constexpr int NWG = (WPC / GW) > 0 ? (WPC / GW) : 1;
    static constexpr int T = NWG * GT;
    static constexpr int MINB = (65536 / 128) / T > 0 ? (65536 / 128) / T : 1;   // <= 128 registers when two CTAs fit
    static constexpr int TASKS = R1 * B;
    static constexpr int ROUNDS = (TASKS + GT - 1) / GT;
    static constexpr int SK = R2 | 1;
    static constexpr int SB = (R1 * SK) | 1;
    static constexpr int XCH = B * SB;
    static constexpr int SMEM_REAL = 2 * N * 16 + 2 * N * 8 + NWG * XCH * 16;
    static constexpr int SMEM_CPLX = 2 * N * 16 + 2 * N * 16 + NWG * XCH * 16;
};

// L2 residency hints.  The plane kernel re-reads in its y pass what its x pass touched a few microseconds
// earlier, while 2 x 148 planes of two arrays (~87 MB on cfg1) are in flight: x-pass traffic is marked
// evict_last, everything that will not be touched again before it leaves L2 anyway evict_first.
enum { H_STREAM = 0, H_KEEP = 1 };
template <int H>
__device__ __forceinline__ unsigned long long l2_policy() {
    unsigned long long pol;
    if (H == H_KEEP) asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;\n" : "=l"(pol));
    else asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;\n" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ cd ld_hint(const cd* p, unsigned long long pol) {
    cd v;
    asm volatile("ld.global.L1::no_allocate.L2::cache_hint.v2.f64 {%0,%1}, [%2], %3;\n"
                 : "=d"(v.x), "=d"(v.y) : "l"(p), "l"(pol) : "memory");
    return v;
}
__device__ __forceinline__ void st_hint(cd* p, cd v, unsigned long long pol) {
    asm volatile("st.global.L2::cache_hint.v2.f64 [%0], {%1,%2}, %3;\n" ::"l"(p), "d"(v.x), "d"(v.y), "l"(pol) : "memory");
}

template <int GW>
__device__ __forceinline__ void lean_sync(int grp) {
    if (GW == 1) __syncwarp();
    else asm volatile("bar.sync %0, %1;\n" ::"r"(grp + 1), "r"(GW * 32) : "memory");
}

// One tile.  cur/acc/series point at this thread's first element of the tile, vt/ph at the same grid point
// of the N_g tables; element n1 of the thread is n1 * estep further.  ktab: this pass's k table (already + 0).
template <int N, int B, int WPC, bool CPLX, bool FIRST, int HIN, int HOUT>
__device__ __forceinline__ void lean_tile(const LeanArgs& a, int pass, const cd* cur, cd* acc,
                                          cd* ser, const double* __restrict__ vt, const cd* __restrict__ ph,
                                          int estep, cd* xch, const cd* twA, const cd* twB, const void* ktab, int grp,
                                          int gt, int n2, int bA) {
    using C = LeanCfg<N, B, WPC>;
    constexpr int R1 = C::R1, R2 = C::R2, TG = C::TG, GW = C::GW, GT = C::GT, SK = C::SK, SB = C::SB;
    constexpr int TASKS = C::TASKS, ROUNDS = C::ROUNDS;
    constexpr bool WCACHE = R2 <= 8;     // stage B keeps its twiddles in registers and applies both directions
    const bool actA = gt < TG;
    const int flags = a.flags[pass], alpha = a.alpha[pass];
    const unsigned long long pin = l2_policy<HIN>(), pout = l2_policy<HOUT>(), pstream = l2_policy<H_STREAM>();
    cd x[R1];
    cd* xA = xch + bA * SB + n2;
    if (actA) {
#pragma unroll
        for (int n1 = 0; n1 < R1; ++n1) x[n1] = ld_hint(cur + n1 * estep, pin);
        if (CPLX && (flags & F_PRO)) {
#pragma unroll
            for (int n1 = 0; n1 < R1; ++n1) x[n1] = cmul(x[n1], __ldg(ph + n1 * estep));
        }
        Dft<R1, -1>::run(x);
        if (WCACHE) {
#pragma unroll
            for (int j = 0; j < R1; ++j) xA[j * SK] = x[j];  // the twiddle W^(n2 k1) is applied by stage B
        } else {
            xA[0] = x[0];
#pragma unroll
            for (int j = 1; j < R1; ++j) xA[j * SK] = cmul(x[j], twA[j * R2 + n2]);
        }
    }
    lean_sync<GW>(grp);
#pragma unroll
    for (int rd = 0; rd < ROUNDS; ++rd) {
        const int task = gt + rd * GT;
        if (task < TASKS) {
            const int bB = task % B, k1 = task / B;          // pencils fastest: a quarter warp reads B = 8 distinct banks (odd pencil stride)
            cd* xB = xch + bB * SB + k1 * SK;
            // one twiddle table read serves both directions: forward y[m] *= W^(m k1), inverse y[m] *= conj(W^(m k1))
            // (small R2 only: for R2 >= 12 the cached twiddles would not fit the register budget)
            cd y[R2], w[WCACHE ? R2 : 1];
            y[0] = xB[0];
            if (WCACHE) {
#pragma unroll
                for (int m = 1; m < R2; ++m) { w[m] = twB[m * R1 + k1]; y[m] = cmul(xB[m], w[m]); }
            } else {
#pragma unroll
                for (int m = 1; m < R2; ++m) y[m] = xB[m];
            }
            Dft<R2, -1>::run(y);
            if (CPLX) {
                const cd* kt = reinterpret_cast<const cd*>(ktab) + k1;
#pragma unroll
                for (int k2 = 0; k2 < R2; ++k2) y[k2] = cmul(y[k2], kt[R1 * k2]);
            } else {
                const double* kt = reinterpret_cast<const double*>(ktab) + k1;
#pragma unroll
                for (int k2 = 0; k2 < R2; ++k2) y[k2] = cscale(y[k2], kt[R1 * k2]);
            }
            Dft<R2, +1>::run(y);
            xB[0] = y[0];
#pragma unroll
            for (int m = 1; m < R2; ++m) xB[m] = cmulc(y[m], WCACHE ? w[m] : twB[m * R1 + k1]);
        }
    }
    lean_sync<GW>(grp);
    if (actA) {
#pragma unroll
        for (int j = 0; j < R1; ++j) x[j] = xA[j * SK];
        Dft<R1, +1>::run(x);
        if (CPLX) {
            if (flags & F_EPI) {
#pragma unroll
                for (int n1 = 0; n1 < R1; ++n1) x[n1] = cmul(x[n1], __ldg(ph + n1 * estep));
            }
            if (flags & F_DENS) {
                // rho += rho_scale |psi|^2 of the finished step, so the next step's Hartree rebuild does
                // not have to read the vectors again; one FP64 reduction per point and vector
                double* rp = a.rho + (ph - a.phase);
                const double ds = a.dens_scale;
#pragma unroll
                for (int n1 = 0; n1 < R1; ++n1) atomicAdd(rp + n1 * estep, ds * (x[n1].x * x[n1].x + x[n1].y * x[n1].y));
            }
#pragma unroll
            for (int n1 = 0; n1 < R1; ++n1) st_hint(acc + n1 * estep, x[n1], pout);
        } else {
            const double hs = a.hs;
            if (FIRST && (flags & (F_VTAB | F_FLUSH))) {
                // first pass of an operator application: needs the input again (L2 hit) with the potential,
                // and (every second Chebyshev term) adds the two vectors at hand to the series
                const double al = (double)alpha, c0 = a.c0, c1 = a.c1;
                constexpr int CH = (R1 % 4 == 0) ? 4 : ((R1 % 3 == 0) ? 3 : ((R1 % 2 == 0) ? 2 : 1));
#pragma unroll
                for (int c = 0; c < R1; c += CH) {
                    cd vin[CH], ao[CH], so[CH];
                    double v[CH];
#pragma unroll
                    for (int q = 0; q < CH; ++q) {
                        const int o = (c + q) * estep;
                        vin[q] = ld_hint(cur + o, pin);
                        ao[q] = alpha != 0 ? ld_hint(acc + o, pstream) : make_double2(0.0, 0.0);
                        v[q] = (flags & F_VTAB) ? __ldg(vt + o) : 0.0;
                        so[q] = ((flags & F_FLUSH) && !(flags & F_SINIT)) ? __ldcs(ser + o) : make_double2(0.0, 0.0);
                    }
#pragma unroll
                    for (int q = 0; q < CH; ++q) {
                        const int n1 = c + q, o = n1 * estep;
                        if (flags & F_FLUSH)
                            __stcs(ser + o, make_double2(so[q].x + c0 * ao[q].x + c1 * vin[q].x,
                                                         so[q].y + c0 * ao[q].y + c1 * vin[q].y));
                        const double hv = hs * v[q];
                        st_hint(acc + o, make_double2(hs * x[n1].x + hv * vin[q].x + al * ao[q].x,
                                                            hs * x[n1].y + hv * vin[q].y + al * ao[q].y), pout);
                    }
                }
            } else if (alpha != 0) {
                cd ad[R1];
#pragma unroll
                for (int n1 = 0; n1 < R1; ++n1) ad[n1] = ld_hint(acc + n1 * estep, pstream);
                const double al = (double)alpha;
#pragma unroll
                for (int n1 = 0; n1 < R1; ++n1)
                    st_hint(acc + n1 * estep, make_double2(hs * x[n1].x + al * ad[n1].x, hs * x[n1].y + al * ad[n1].y), pout);
            } else {
#pragma unroll
                for (int n1 = 0; n1 < R1; ++n1) st_hint(acc + n1 * estep, cscale(x[n1], hs), pout);
            }
        }
    }
    lean_sync<GW>(grp);                                       // the exchange buffer is free for the next tile
}

template <int N, int B, int WPC, bool CPLX>
__device__ __forceinline__ void lean_tables(const LeanArgs& a, cd* twA, cd* twB, char* ktab) {
    using C = LeanCfg<N, B, WPC>;
    for (int i = threadIdx.x; i < N; i += C::T) {
        twA[i] = a.tw[(i % C::R2) * (i / C::R2)];
        twB[i] = a.tw[(i / C::R1) * (i % C::R1)];
    }
#pragma unroll
    for (int p = 0; p < 2; ++p) {
        for (int k = threadIdx.x; k < N; k += C::T) {
            if (CPLX) { if (a.kc[p]) reinterpret_cast<cd*>(ktab)[p * N + k] = a.kc[p][k]; }
            else { if (a.kre[p]) reinterpret_cast<double*>(ktab)[p * N + k] = a.kre[p][k]; }
        }
    }
    __syncthreads();
}

// Programmatic dependent launch (opt-in, SGW_PDL=1: lean_launch_kernel sets the stream-serialization attribute): a pass lets the next
// launch start at once and loads its own constant tables (twiddles, k-space multipliers: written before any pass of
// the call) before it waits for the preceding grid's memory.  Both are no-ops for a plain launch.
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// One pass along AXIS (0 x, 1 y, 2 z) over all tiles; groups take tiles round robin.
//   x: tile t = B consecutive rows (rows are contiguous across planes and vectors)
//   y: tile t = (plane, column block);  z: tile t = (vector, xy block)
//   CUBE: nx == ny == N as well (compile-time strides)
template <int N, int B, bool CPLX, int AXIS, bool CUBE>
__global__ void __launch_bounds__(LeanCfg<N, B>::T, LeanCfg<N, B>::MINB) axis_lean_kernel(const LeanArgs a) {
    using C = LeanCfg<N, B>;
    constexpr int R2 = C::R2, GT = C::GT, NWG = C::NWG;
    extern __shared__ __align__(16) char smraw[];
    cd* twA = reinterpret_cast<cd*>(smraw);
    cd* twB = twA + N;
    char* ktab = reinterpret_cast<char*>(twB + N);
    const int tid = threadIdx.x, grp = tid / GT, gt = tid % GT;
    cd* xch = reinterpret_cast<cd*>(ktab + 2 * N * (CPLX ? 16 : 8)) + grp * C::XCH;
    pdl_launch_dependents();
    lean_tables<N, B, 8, CPLX>(a, twA, twB, ktab);
    pdl_wait();

    const int nxy = CUBE ? N * N : a.nx * a.ny;
    const long long ng = (long long)nxy * a.nz;
    int n2, bA, e0, estep;
    if (AXIS == 0) { n2 = gt % R2; bA = gt / R2; e0 = bA * a.nx + n2; estep = R2; }
    else { bA = gt % B; n2 = gt / B; const int sN = (AXIS == 1) ? (CUBE ? N : a.nx) : nxy; e0 = n2 * sN + bA; estep = R2 * sN; }
    const unsigned stride = gridDim.x * NWG;
    const unsigned cb_per_plane = (unsigned)(a.nx / B);
    const unsigned nvec = (unsigned)a.nvec;
    // tile -> offset of its first element in the vector arrays (vectors fastest when vminor) and in the N_g tables
    auto locate = [&](unsigned t, int& g0) -> long long {
        unsigned v, q;
        if (a.vminor) { q = t / nvec; v = t - q * nvec; }
        else { const unsigned tpv = a.ntiles / nvec; v = t / tpv; q = t - v * tpv; }
        if (AXIS == 0) {
            g0 = (int)q * (B * a.nx);
        } else if (AXIS == 1) {
            const unsigned z = q / cb_per_plane, cb = q - z * cb_per_plane;
            g0 = (int)z * nxy + (int)cb * B;
        } else {
            g0 = (int)q * B;
        }
        return (long long)v * ng + g0;
    };
    for (unsigned t = blockIdx.x * NWG + grp; t < a.ntiles; t += stride) {
        int g0;
        const long long o = locate(t, g0) + e0;
        lean_tile<N, B, 8, CPLX, AXIS == 0, H_STREAM, H_STREAM>(a, 0, a.cur + o, a.acc + o, a.series + o, a.vtab + g0 + e0, a.phase + g0 + e0, estep,
                                         xch, twA, twB, ktab, grp, gt, n2, bA);
    }
}

// k-th plane of a launch -> plane index p = v * nz + z (vminor: consecutive k run over the vectors at one z)
__device__ __forceinline__ unsigned plane_of(const LeanArgs& a, unsigned k) {
    if (!a.vminor) return k;
    const unsigned nvec = (unsigned)a.nvec, z = k / nvec, v = k - z * nvec;
    return v * (unsigned)a.nz + z;
}

// x pass then y pass of whole xy planes (nx == ny == N) in one launch.  A CTA owns planes [pg*G, pg*G + G): its
// groups do the row tiles of those planes, the CTA synchronises (which also makes the stores visible to the
// whole CTA), then the column tiles; the transpose goes through L2.  (A barrier-free variant that pipelines
// planes inside a CTA with shared-memory counters was tried: it needs both a producer and a consumer
// throttle to bound the planes in flight, keeps more of them live than L2 holds, and was slower.)
template <int N, int B, bool CPLX, int WPC>
__global__ void __launch_bounds__(LeanCfg<N, B, WPC>::T, LeanCfg<N, B, WPC>::MINB) plane_lean_kernel(const LeanArgs a) {
    using C = LeanCfg<N, B, WPC>;
    constexpr int R2 = C::R2, GT = C::GT, NWG = C::NWG;
    constexpr unsigned TPP = N / B;
    constexpr int NXY = N * N;
    extern __shared__ __align__(16) char smraw[];
    cd* twA = reinterpret_cast<cd*>(smraw);
    cd* twB = twA + N;
    char* ktab = reinterpret_cast<char*>(twB + N);
    const int tid = threadIdx.x, grp = tid / GT, gt = tid % GT;
    cd* xch = reinterpret_cast<cd*>(ktab + 2 * N * (CPLX ? 16 : 8)) + grp * C::XCH;
    pdl_launch_dependents();
    lean_tables<N, B, WPC, CPLX>(a, twA, twB, ktab);
    pdl_wait();
    const char* ktab_y = ktab + N * (CPLX ? 16 : 8);

    const int n2x = gt % R2, bAx = gt / R2, e0x = bAx * N + n2x;                 // x: lanes along n
    const int bAy = gt % B, n2y = gt / B, e0y = n2y * N + bAy;                   // y: lanes along b
    const unsigned G = (unsigned)a.G;
    const unsigned ngroups = (a.ntiles + G - 1) / G;
    for (unsigned pg = blockIdx.x; pg < ngroups; pg += gridDim.x) {
        const unsigned p0 = pg * G, np = (a.ntiles - p0 < G) ? a.ntiles - p0 : G;
        for (unsigned q = grp; q < np * TPP; q += NWG) {
            const unsigned p = plane_of(a, p0 + q / TPP), rb = q % TPP;
            const long long o = (long long)p * NXY + (long long)rb * (B * N) + e0x;
            const int g = (int)(p % (unsigned)a.nz) * NXY + (int)rb * (B * N) + e0x;
            lean_tile<N, B, WPC, CPLX, true, H_KEEP, H_KEEP>(a, 0, a.cur + o, a.acc + o, a.series + o, a.vtab + g, a.phase + g, R2, xch, twA, twB,
                                        ktab, grp, gt, n2x, bAx);
        }
        __syncthreads();                                     // every row tile of the group is stored (to L2)
        for (unsigned q = grp; q < np * TPP; q += NWG) {
            const unsigned p = plane_of(a, p0 + q / TPP), cb = q % TPP;
            const long long o = (long long)p * NXY + (long long)cb * B + e0y;
            const int g = (int)(p % (unsigned)a.nz) * NXY + (int)cb * B + e0y;
            // the y pass reads what the x pass left in acc; for the complex family cur == acc
            lean_tile<N, B, WPC, CPLX, false, H_STREAM, H_STREAM>(a, 1, a.cur + o, a.acc + o, a.series + o, a.vtab + g, a.phase + g, R2 * N, xch, twA,
                                         twB, ktab_y, grp, gt, n2y, bAy);
        }
    }
}

// Cluster variant of the plane kernel: a thread-block cluster of CS CTAs (CS SMs' worth of warp groups) owns one
// plane at a time, so the planes in flight - what has to stay in L2 between the row tiles and the column tiles -
// are 1/CS of the resident CTAs, and CS * NWG groups share a plane's N/B tiles (12 groups for the 12 tiles of a
// 96^2 plane with CS = 3).  The x->y handoff is a cluster barrier with release/acquire semantics.
__device__ __forceinline__ void cluster_barrier() {
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;\n" ::: "memory");
}
template <int N, int B, bool CPLX, int CS>
__global__ void __launch_bounds__(LeanCfg<N, B, 8>::T, LeanCfg<N, B, 8>::MINB) plane_cluster_kernel(const LeanArgs a) {
    using C = LeanCfg<N, B, 8>;
    constexpr int R2 = C::R2, GT = C::GT, NWG = C::NWG;
    constexpr unsigned TPP = N / B;
    constexpr int NXY = N * N;
    extern __shared__ __align__(16) char smraw[];
    cd* twA = reinterpret_cast<cd*>(smraw);
    cd* twB = twA + N;
    char* ktab = reinterpret_cast<char*>(twB + N);
    const int tid = threadIdx.x, grp = tid / GT, gt = tid % GT;
    cd* xch = reinterpret_cast<cd*>(ktab + 2 * N * (CPLX ? 16 : 8)) + grp * C::XCH;
    lean_tables<N, B, 8, CPLX>(a, twA, twB, ktab);
    const char* ktab_y = ktab + N * (CPLX ? 16 : 8);
    unsigned crank, cid, ncl;
    asm volatile("mov.u32 %0, %%cluster_ctarank;\n" : "=r"(crank));
    asm volatile("mov.u32 %0, %%clusterid.x;\n" : "=r"(cid));
    asm volatile("mov.u32 %0, %%nclusterid.x;\n" : "=r"(ncl));
    const int n2x = gt % R2, bAx = gt / R2, e0x = bAx * N + n2x;                 // x: lanes along n
    const int bAy = gt % B, n2y = gt / B, e0y = n2y * N + bAy;                   // y: lanes along b
    const unsigned me = crank * NWG + grp, gsz = CS * NWG;
    for (unsigned k = cid; k < a.ntiles; k += ncl) {
        const unsigned p = plane_of(a, k);
        const int gp = (int)(p % (unsigned)a.nz) * NXY;
        for (unsigned q = me; q < TPP; q += gsz) {
            const long long o = (long long)p * NXY + (long long)q * (B * N) + e0x;
            const int g = gp + (int)q * (B * N) + e0x;
            lean_tile<N, B, 8, CPLX, true, H_KEEP, H_KEEP>(a, 0, a.cur + o, a.acc + o, a.series + o, a.vtab + g, a.phase + g, R2, xch,
                                                           twA, twB, ktab, grp, gt, n2x, bAx);
        }
        cluster_barrier();                                   // every row tile of the plane is stored and visible
        for (unsigned q = me; q < TPP; q += gsz) {
            const long long o = (long long)p * NXY + (long long)q * B + e0y;
            const int g = gp + (int)q * B + e0y;
            lean_tile<N, B, 8, CPLX, false, H_STREAM, H_STREAM>(a, 1, a.cur + o, a.acc + o, a.series + o, a.vtab + g, a.phase + g,
                                                                R2 * N, xch, twA, twB, ktab_y, grp, gt, n2y, bAy);
        }
    }
}

// Team variant of the plane kernel, for planes too large for CTA- or cluster-owned transposes through L2 (256^2,
// 384^2): a TEAM of TPP = N/B warp groups (on as many SMs as that takes: 24 SMs for 384^2) owns one plane at a
// time, one row tile and one column tile per group, so only (groups / TPP) planes are in flight and the x->y
// transpose of a 2.4 MB plane stays in L2.  The teams are software constructs: the x->y handoff is one arrival
// counter per plane in global memory (release: group barrier, fence, atomic; acquire: one lane polls, group barrier),
// software-pipelined so that a group does its row tile of plane k+1 before it waits for plane k.  All CTAs must be
// co-resident: the launcher uses a cooperative launch sized by the occupancy query.
__device__ __forceinline__ unsigned ld_acquire_u32(const unsigned* p) {
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];\n" : "=r"(v) : "l"(p) : "memory");
    return v;
}
template <int N, int B, bool CPLX>
__global__ void __launch_bounds__(LeanCfg<N, B, 8>::T, LeanCfg<N, B, 8>::MINB) plane_team_kernel(const LeanArgs a) {
    using C = LeanCfg<N, B, 8>;
    constexpr int R2 = C::R2, GT = C::GT, NWG = C::NWG, GW = C::GW;
    constexpr unsigned TPP = N / B;
    constexpr int NXY = N * N;
    extern __shared__ __align__(16) char smraw[];
    cd* twA = reinterpret_cast<cd*>(smraw);
    cd* twB = twA + N;
    char* ktab = reinterpret_cast<char*>(twB + N);
    const int tid = threadIdx.x, grp = tid / GT, gt = tid % GT;
    cd* xch = reinterpret_cast<cd*>(ktab + 2 * N * (CPLX ? 16 : 8)) + grp * C::XCH;
    lean_tables<N, B, 8, CPLX>(a, twA, twB, ktab);
    const char* ktab_y = ktab + N * (CPLX ? 16 : 8);
    const int n2x = gt % R2, bAx = gt / R2, e0x = bAx * N + n2x;                 // x: lanes along n
    const int bAy = gt % B, n2y = gt / B, e0y = n2y * N + bAy;                   // y: lanes along b
    const unsigned gid = blockIdx.x * NWG + grp, nteams = (gridDim.x * NWG) / TPP;
    const unsigned team = gid / TPP, slot = gid - team * TPP;
    if (team >= nteams) return;                                                // left-over groups
    long long prev = -1;
    for (unsigned k = team;; k += nteams) {
        const bool have = k < a.ntiles;
        if (have) {
            const unsigned p = plane_of(a, k);
            const long long o = (long long)p * NXY + (long long)slot * (B * N) + e0x;
            const int g = (int)(p % (unsigned)a.nz) * NXY + (int)slot * (B * N) + e0x;
            lean_tile<N, B, 8, CPLX, true, H_KEEP, H_KEEP>(a, 0, a.cur + o, a.acc + o, a.series + o, a.vtab + g, a.phase + g, R2, xch,
                                                           twA, twB, ktab, grp, gt, n2x, bAx);
            // lean_tile ends with a group barrier: every store of the tile precedes this release
            if (gt == 0) { __threadfence(); atomicAdd(a.cnt + k, 1u); }
        }
        if (prev >= 0) {
            if (gt == 0) { while (ld_acquire_u32(a.cnt + prev) < TPP) __nanosleep(64); }
            lean_sync<GW>(grp);
            const unsigned p = plane_of(a, (unsigned)prev);
            const long long o = (long long)p * NXY + (long long)slot * B + e0y;
            const int g = (int)(p % (unsigned)a.nz) * NXY + (int)slot * B + e0y;
            lean_tile<N, B, 8, CPLX, false, H_STREAM, H_STREAM>(a, 1, a.cur + o, a.acc + o, a.series + o, a.vtab + g, a.phase + g,
                                                                R2 * N, xch, twA, twB, ktab_y, grp, gt, n2y, bAy);
        }
        if (!have) break;
        prev = k;
    }
}

struct LeanCall {
    LeanArgs args;
    int cplx;
    int kind;                 // 0..2: axis pass along x, y, z; 3: plane pass (x then y); 4 / 5: z / y pass on a cubic grid
    int ctas_per_sm;          // 0 = as many as fit
    int wpc;                  // plane kernel: warps per CTA, 8 (two CTAs per SM) or 16 (one)
    int cluster;              // plane kernel: 1 = cluster-owned planes (plane_cluster_kernel), 2 = team-owned, 0 = CTA-owned
    int pdl;                  // 1 = programmatic dependent launch (SGW_PDL=1)
    int num_sms;              // of the context's device
    int* occ;                 // context-owned cache of occupancy results for this axis length, 18 ints, zero-initialised
    cudaStream_t stream;
};
// returns 0, -(stage*1000 + cudaError) on failure, or 1 if this (N, B) is not instantiated
typedef int (*lean_launch_fn)(const LeanCall*, int B);

}  // namespace sgw
