// sgw_acc.cuh -- TMA accumulate kernel for sm_100a: acc += c * (T_x + T_y + T_z + vtab) cur + e * v, one launch.
//
// Why it exists (profiles/r02_*.md): in the register-operand passes of sgw_lean.cuh every global operand goes through
// the LSU (and, for the late operands of the first pass, exposes its latency); the x+y plane pass was bound by that
// path.  Here no consumer thread touches global memory for the vectors at all:
//   * a LOADER thread brings tiles of B = 8 pencils into a ring of shared-memory slots with bulk asynchronous copies
//     (cp.async.bulk for the contiguous x tiles, cp.async.bulk.tensor.3d through a tensor map for the strided y / z
//     tiles), completion on an mbarrier per slot;
//   * consumer warp groups run the two-stage round trip IN PLACE in the slot: the dense TMA layout is
//     bank-conflict free for 16-byte elements with the pencils-fastest thread mapping, and every thread reads and
//     writes the same slots in stage A, so the tile is its own exchange buffer;
//   * a STORER thread sends the finished tile to the accumulator with bulk REDUCE-ADD operations
//     (cp.reduce.async.bulk[.tensor].add.f64): the read-modify-write of acc happens in L2, the SM never loads it.
// Because every direction's contribution is a pure sum into acc, the x, y and z tiles of a term have NO mutual
// dependency: one launch, no x->y handoff, no barrier between directions; the order of the tiles only decides what
// stays in L2 (all tiles of a vector together when its arrays fit, else planes then z columns).
// The Chebyshev recurrence is run in Clenshaw form with sign-folded buffers so that every step is such a sum
// (sgw_program.cu: acc_cheb_filter; Eq. 3).
#pragma once
#include <cuda.h>

#include "sgw_lean.cuh"

namespace sgw {

struct AccArgs {
    const cd* cur;            // input vectors
    cd* acc;                  // accumulated into
    const cd* v;              // second input added with coefficient e in the x tiles (Clenshaw start vector) or NULL
    const double* vtab;       // N_g real table or NULL
    const double* kre[3];     // real k tables per axis (include 1/N and any scale)
    const cd* tw;             // exp(-2 pi i j / N)
    double c, e;
    int nvec, nz;             // cubic grids only: nx = ny = nz = N
    int kinds;                // bit 0: x tiles, bit 1: y tiles, bit 2: z tiles
    int plane_major;          // 1: x and y tiles interleaved plane by plane (z tiles, if any, after all planes)
    int pairz;                // z-only launch whose tiles are PAIRS (16 xy-adjacent pencils): ntiles counts pairs, the z maps
                              // passed have 256-byte rows, and each of the two consumer groups takes one half of a pair
    unsigned ntiles;
};

template <int N>
struct AccCfg {
    static constexpr int B = 8;
    static constexpr int R1 = Fact2<N>::R1, R2 = Fact2<N>::R2;
    static constexpr int TG = B * R2;                        // threads of a consumer group
    static constexpr int GW = (TG + 31) / 32, GT = GW * 32;
    static constexpr int TASKS = R1 * B, ROUNDS = (TASKS + GT - 1) / GT;
    static constexpr int XP = N + 1;                         // x tile: row pitch in elements (odd pitch: bank-conflict free)
    static constexpr int TILE = ((XP * B * 16 + 127) / 128) * 128;   // slot bytes (>= N * B * 16 of the dense y / z tile)
    static constexpr int TABLES = 2 * N * 16 + 3 * N * 8;
    static constexpr int NBOX = N <= 256 ? N : N / 2;        // tensor-map box rows (at most 256 per dimension)
    static constexpr int NOPS = N / NBOX;
    // consumer groups: as many as leave each thread ~128-146 registers
    static constexpr int NG = (GW == 1) ? 8 : (GW == 2 ? 7 : (GW <= 4 ? 3 : 2));
    // warp-specialised register budget (setmaxnreg): where the consumers fill whole warpgroups, the CTA is 16 warps at
    // 128 registers, the first warpgroup (loader warp, storer warp, two idle warps) hands back all but 40 registers per
    // thread and the consumer warpgroups take 152
    static constexpr bool WS = (NG * GT) % 128 == 0 && NG * GT <= 384;
    static constexpr int PRODT = WS ? 128 : 64;              // threads before the consumers
    static constexpr int T = PRODT + NG * GT;                // loader warp, storer warp, consumers
    // the accumulate kernel keeps the plain layout at N = 384 (measured: its x tiles lose with the larger budget)
    // split-operator x launch: how many of a thread's R1 phases stay in registers across the tiles of a block (the rest
    // are read again for every tile); all of them where the register budget allows
    static constexpr int NPRO = N > 256 ? R1 / 2 : R1;
    static constexpr bool WS_ACC = WS && N <= 256;
    static constexpr int PRODT_ACC = WS_ACC ? 128 : 64;
    static constexpr int T_ACC = PRODT_ACC + NG * GT;
    static constexpr int MAXS = 24;
    static constexpr bool PAIRZ = NG == 2;                   // tile pairs need exactly two consumer groups
    // x tiles: the pointwise part w = (c vtab) cur + e v either goes through a second slot of the tile (v is brought in
    // by the loader) or, where a slot is too precious (few, large slots), is read from global memory after the inverse
    // stage (cur is an L2 hit then)
    static constexpr bool LATEW = N > 256;
};

__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* b, unsigned n) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(smem_u32(b)), "r"(n));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* b, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* b) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"(smem_u32(b)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* b, unsigned parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "ACC_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra ACC_DONE;\n"
        "bra ACC_WAIT;\n"
        "ACC_DONE:\n"
        "}\n" ::"r"(smem_u32(b)), "r"(parity) : "memory");
}
__device__ __forceinline__ bool mbar_test(uint64_t* b, unsigned parity) {
    unsigned ok;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n" : "=r"(ok) : "r"(smem_u32(b)), "r"(parity) : "memory");
    return ok != 0;
}
__device__ __forceinline__ void bulk_load(void* dst, const void* src, unsigned bytes, uint64_t* b) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n" ::"r"(smem_u32(dst)), "l"(src),
                 "r"(bytes), "r"(smem_u32(b)) : "memory");
}
__device__ __forceinline__ void bulk_red_add(void* gdst, const void* ssrc, unsigned bytes) {
    asm volatile("cp.reduce.async.bulk.global.shared::cta.bulk_group.add.f64 [%0], [%1], %2;\n" ::"l"(gdst), "r"(smem_u32(ssrc)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void tma_load_3d(void* dst, const CUtensorMap* m, int c0, int c1, int c2, uint64_t* b) {
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];\n" ::"r"(
                     smem_u32(dst)), "l"(m), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(b)) : "memory");
}
__device__ __forceinline__ void tma_red_add_3d(const CUtensorMap* m, const void* src, int c0, int c1, int c2) {
    asm volatile("cp.reduce.async.bulk.tensor.3d.global.shared::cta.add.tile.bulk_group [%0, {%2, %3, %4}], [%1];\n" ::"l"(m),
                 "r"(smem_u32(src)), "r"(c0), "r"(c1), "r"(c2) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;\n" ::: "memory"); }
template <int K>
__device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read %0;\n" ::"n"(K) : "memory"); }
__device__ __forceinline__ void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory"); }

// Tile sequence of one CTA (tiles blockIdx.x, blockIdx.x + gridDim.x, ...) without per-tile integer divisions.
//   vector-major: the tiles of a vector are [x tiles | y tiles | z tiles] (kinds present in the launch), vector after vector
//   plane-major (x and y kinds only): the tiles of a plane are [x tiles | y tiles], plane after plane
// kind 0 x: rows [j*8, j*8+8) of plane p;  1 y: columns [j*8, ..) of plane p;  2 z: xy points [j*8, ..) of vector v.
template <int N, bool PZ = false>
struct AccIter {
    static constexpr unsigned TPP = N / 8, TPV = (unsigned)N * N / 8;
    unsigned t, q, u, period, step, seg; // u = vector (vector-major) or plane (plane-major), q = offset inside it
    bool hasx;
    int kind;
    unsigned v, p, j;
    __device__ __forceinline__ void init(const AccArgs& a, unsigned t0, unsigned stride) {
        const unsigned nk = (unsigned)((a.kinds & 1) + ((a.kinds >> 1) & 1) + ((a.kinds >> 2) & 1));
        seg = a.plane_major ? TPP : (PZ ? TPV / 2 : TPV);
        hasx = a.kinds & 1;
        period = nk * seg;
        t = t0; step = stride;
        u = t0 / period; q = t0 - u * period;
    }
    // x tiles are the first segment of a period when the launch has any
    __device__ __forceinline__ bool is_x() const { return hasx && q < seg; }
    __device__ __forceinline__ void decode(const AccArgs& a) {
        if (PZ) { kind = 2; v = u; j = q; p = 0; return; }   // pair j of vector u: xy points [16 j, 16 j + 16)
        if (a.plane_major) {
            const unsigned k = q / TPP;
            kind = (a.kinds & 1) ? (int)k : 1;
            j = q - k * TPP; p = u; v = 0;
        } else {
            const unsigned k = q / TPV, i = q - k * TPV;
            int kd = 0, seen = 0;
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                if ((a.kinds >> d) & 1) { if (seen == (int)k) kd = d; ++seen; }
            }
            kind = kd; v = u;
            if (kd == 2) { j = i; p = 0; }
            else { const unsigned z = i / TPP; p = u * (unsigned)a.nz + z; j = i - z * TPP; }
        }
    }
    __device__ __forceinline__ void next() {
        t += step; q += step;
        while (q >= period) { q -= period; ++u; }
    }
};

// the round trip of one tile, in place in its slot.  XK: x tile (rows of pitch XP, lanes along the row) or y / z tile
// (dense [point][pencil], lanes along the pencils).
//   wtile (x tiles): second slot of the tile.  On entry it holds the v tile (hasv) or nothing; the thread replaces its
//   elements by w = (c * vtab) * cur + e * v, what the x tiles add besides the transform, and reads them back after the
//   inverse stage, so that w costs no registers across the transform.
template <int N, bool XK, int PITCH = AccCfg<N>::B>
__device__ __forceinline__ void acc_tile_compute(const AccArgs& a, cd* tile, cd* wtile, bool hasv, const double* __restrict__ vt, const cd* twA,
                                                 const cd* twB, const double* ktab, int gt, int bar_id, const cd* __restrict__ gcur = nullptr,
                                                 const cd* __restrict__ gv = nullptr) {
    using C = AccCfg<N>;
    constexpr int R1 = C::R1, R2 = C::R2, TG = C::TG, GW = C::GW, GT = C::GT, TASKS = C::TASKS, ROUNDS = C::ROUNDS, B = C::B;
    constexpr bool WCACHE = R2 <= 8;
    constexpr int SB = XK ? C::XP : 1, SI = XK ? 1 : PITCH;  // element strides of (pencil, point) inside the slot (PITCH = 2 B: half of a tile pair)
    const bool actA = gt < TG;
    const int n2 = XK ? gt % R2 : gt / B, bA = XK ? gt / R2 : gt % B;
    cd* eA = tile + bA * SB + n2 * SI;
    cd x[R1];
    constexpr bool LATEW = C::LATEW;
    cd* eW = (XK && !LATEW) ? wtile + bA * SB + n2 * SI : nullptr;
    if (actA) {
#pragma unroll
        for (int n1 = 0; n1 < R1; ++n1) x[n1] = eA[n1 * R2 * SI];
        if (XK && !LATEW) {
            const double c = a.c, e = a.e;
#pragma unroll
            for (int n1 = 0; n1 < R1; ++n1) {
                const double cv = vt ? c * __ldg(vt + n1 * R2) : 0.0;
                cd w = make_double2(cv * x[n1].x, cv * x[n1].y);
                if (hasv) { const cd u = eW[n1 * R2 * SI]; w.x += e * u.x; w.y += e * u.y; }
                eW[n1 * R2 * SI] = w;
            }
        }
        Dft<R1, -1>::run(x);
        if (WCACHE) {
#pragma unroll
            for (int j = 0; j < R1; ++j) eA[j * R2 * SI] = x[j];
        } else {
            eA[0] = x[0];
#pragma unroll
            for (int j = 1; j < R1; ++j) eA[j * R2 * SI] = cmul(x[j], twA[j * R2 + n2]);
        }
    }
    lean_sync<GW>(bar_id);
#pragma unroll
    for (int rd = 0; rd < ROUNDS; ++rd) {
        const int task = gt + rd * GT;
        if (task < TASKS) {
            const int bB = task % B, k1 = task / B;
            cd* eB = tile + bB * SB + k1 * R2 * SI;
            cd y[R2], wc[WCACHE ? R2 : 1];
            y[0] = eB[0];
            if (WCACHE) {
#pragma unroll
                for (int m = 1; m < R2; ++m) { wc[m] = twB[m * R1 + k1]; y[m] = cmul(eB[m * SI], wc[m]); }
            } else {
#pragma unroll
                for (int m = 1; m < R2; ++m) y[m] = eB[m * SI];
            }
            Dft<R2, -1>::run(y);
            const double* kt = ktab + k1;
#pragma unroll
            for (int k2 = 0; k2 < R2; ++k2) y[k2] = cscale(y[k2], kt[R1 * k2]);
            Dft<R2, +1>::run(y);
            eB[0] = y[0];
#pragma unroll
            for (int m = 1; m < R2; ++m) eB[m * SI] = cmulc(y[m], WCACHE ? wc[m] : twB[m * R1 + k1]);
        }
    }
    lean_sync<GW>(bar_id);
    if (actA) {
#pragma unroll
        for (int j = 0; j < R1; ++j) x[j] = eA[j * R2 * SI];
        Dft<R1, +1>::run(x);
        const double c = a.c;
        if (XK && LATEW) {
            const double e = a.e;
            constexpr int CH = (R1 % 4 == 0) ? 4 : ((R1 % 3 == 0) ? 3 : 1);
#pragma unroll
            for (int c0 = 0; c0 < R1; c0 += CH) {
                cd cu[CH], vv[CH];
                double tv[CH];
#pragma unroll
                for (int q = 0; q < CH; ++q) {
                    const int o = (c0 + q) * R2;
                    tv[q] = vt ? __ldg(vt + o) : 0.0;
                    cu[q] = vt ? __ldg(gcur + o) : make_double2(0.0, 0.0);
                    vv[q] = hasv ? __ldg(gv + o) : make_double2(0.0, 0.0);
                }
#pragma unroll
                for (int q = 0; q < CH; ++q) {
                    const int n1 = c0 + q;
                    const double cv = c * tv[q];
                    eA[n1 * R2 * SI] = make_double2(c * x[n1].x + cv * cu[q].x + e * vv[q].x, c * x[n1].y + cv * cu[q].y + e * vv[q].y);
                }
            }
        } else {
#pragma unroll
            for (int n1 = 0; n1 < R1; ++n1) {
                cd r = cscale(x[n1], c);
                if (XK) { const cd w = eW[n1 * R2 * SI]; r.x += w.x; r.y += w.y; }
                eA[n1 * R2 * SI] = r;
            }
        }
        fence_proxy_async_smem();                            // the bulk reduce-add reads the slot through the async proxy
    }
    lean_sync<GW>(bar_id);
}

// PZ: the z-only launch in tile pairs, a separate instantiation so that the code of the other launches is untouched by it
template <int N, bool PZ = false>
__global__ void __launch_bounds__(AccCfg<N>::T_ACC, 1)
acc_tma_kernel(const AccArgs a, const __grid_constant__ CUtensorMap cur_y, const __grid_constant__ CUtensorMap cur_z,
               const __grid_constant__ CUtensorMap acc_y, const __grid_constant__ CUtensorMap acc_z, int nslots) {
    using C = AccCfg<N>;
    constexpr int GT = C::GT, NG = C::NG, B = C::B, TILE = C::TILE;
    constexpr unsigned ROWB = N * 16, YZB = N * B * 16;
    extern __shared__ __align__(128) char smraw[];
    char* slots = smraw;                                      // nslots * TILE, 128-byte aligned
    cd* twA = reinterpret_cast<cd*>(smraw + (size_t)nslots * TILE);
    cd* twB = twA + N;
    double* ktab = reinterpret_cast<double*>(twB + N);        // [3][N]
    uint64_t* full = reinterpret_cast<uint64_t*>(ktab + 3 * N);
    uint64_t* done = full + C::MAXS;
    uint64_t* empty = done + C::MAXS;
    unsigned* ticket = reinterpret_cast<unsigned*>(empty + C::MAXS);   // [0]: next tile of the CTA's sequence; [1 + g]: the one group g took
    const int tid = threadIdx.x;
    for (int i = tid; i < N; i += C::T_ACC) {
        twA[i] = a.tw[(i % C::R2) * (i / C::R2)];
        twB[i] = a.tw[(i / C::R1) * (i % C::R1)];
#pragma unroll
        for (int d = 0; d < 3; ++d) ktab[d * N + i] = a.kre[d][i];
    }
    if (tid == 0) {
        for (int s = 0; s < nslots; ++s) { mbar_init(full + s, 1); mbar_init(done + s, 1); mbar_init(empty + s, 1); }
        ticket[0] = 0;
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    __syncthreads();
    const unsigned S = (unsigned)nslots;
    const bool usev = a.v != nullptr;
    const long long ng = (long long)N * N * a.nz;

    if (tid < C::PRODT_ACC) {
        if (C::WS_ACC) asm volatile("setmaxnreg.dec.sync.aligned.u32 40;\n");
        if (tid == 0) {
            // ---------------- loader: one slot per tile (two for an x tile with a v operand), in tile order
            unsigned seq = 0;
            AccIter<N, PZ> tl;
            for (tl.init(a, blockIdx.x, gridDim.x); tl.t < a.ntiles; tl.next()) {
                tl.decode(a);
                if (PZ) {
                    // a pair fills two adjacent slots (rows of 16 pencils = 256 bytes); only the first slot's barriers are used
                    const unsigned s = seq % S, round = seq / S;
                    if (round > 0) mbar_wait(empty + s, (round - 1) & 1);
                    char* dst = slots + (size_t)s * TILE;
                    mbar_expect_tx(full + s, 2 * YZB);
#pragma unroll
                    for (int o = 0; o < C::NOPS; ++o)
                        tma_load_3d(dst + (size_t)o * C::NBOX * 2 * B * 16, &cur_z, (int)tl.j * 32, o * C::NBOX, (int)tl.v, full + s);
                    seq += 2;
                    continue;
                }
                const int nops = (tl.kind == 0 && !C::LATEW) ? 2 : 1;   // an x tile takes a second slot: the v tile, then scratch
                for (int op = 0; op < nops; ++op, ++seq) {
                    const unsigned s = seq % S, round = seq / S;
                    if (round > 0) mbar_wait(empty + s, (round - 1) & 1);
                    char* dst = slots + (size_t)s * TILE;
                    if (op == 1 && !usev) { mbar_arrive(full + s); continue; }
                    if (tl.kind == 0) {
                        mbar_expect_tx(full + s, B * ROWB);
                        const cd* src = (op == 0 ? a.cur : a.v) + (long long)tl.p * (N * N) + (long long)tl.j * (B * N);
#pragma unroll
                        for (int b = 0; b < B; ++b) bulk_load(dst + (size_t)b * C::XP * 16, src + b * N, ROWB, full + s);
                    } else {
                        mbar_expect_tx(full + s, YZB);
                        const CUtensorMap* m = tl.kind == 1 ? &cur_y : &cur_z;
                        const int c2 = tl.kind == 1 ? (int)tl.p : (int)tl.v;
#pragma unroll
                        for (int o = 0; o < C::NOPS; ++o)
                            tma_load_3d(dst + (size_t)o * C::NBOX * B * 16, m, (int)tl.j * 16, o * C::NBOX, c2, full + s);
                    }
                }
            }
        } else if (tid == 32) {
            // ---------------- storer: reduce-add of finished tiles, slots released when the engine has read them
            unsigned seq = 0, pend[2], npend = 0;
            AccIter<N, PZ> tl;
            for (tl.init(a, blockIdx.x, gridDim.x); tl.t < a.ntiles; tl.next()) {
                tl.decode(a);
                const unsigned s = seq % S, round = seq / S;
                constexpr bool pair = PZ;
                seq += (pair || (tl.kind == 0 && !C::LATEW)) ? 2 : 1;
                if (!mbar_test(done + s, round & 1)) {
                    // about to block: first hand back every slot whose reduce-add has been issued (with few slots the
                    // loader may need exactly those to bring in the tile this thread waits for)
                    if (npend) {
                        bulk_wait_read<0>();
                        for (unsigned k = 0; k < npend; ++k) mbar_arrive(empty + pend[k]);
                        npend = 0;
                    }
                    mbar_wait(done + s, round & 1);
                }
                if (pair) mbar_wait(done + s + 1, round & 1);            // the second group's half (it arrives on the second slot's barrier;
                                                                         // that tile is loaded, so this wait cannot depend on the loader)
                const char* src = slots + (size_t)s * TILE;
                if (tl.kind == 0) {
                    cd* dst = a.acc + (long long)tl.p * (N * N) + (long long)tl.j * (B * N);
#pragma unroll
                    for (int b = 0; b < B; ++b) bulk_red_add(dst + b * N, src + (size_t)b * C::XP * 16, ROWB);
                } else {
                    const CUtensorMap* m = tl.kind == 1 ? &acc_y : &acc_z;
                    const int c2 = tl.kind == 1 ? (int)tl.p : (int)tl.v;
                    if (pair) {
#pragma unroll
                        for (int o = 0; o < C::NOPS; ++o) tma_red_add_3d(m, src + (size_t)o * C::NBOX * 2 * B * 16, (int)tl.j * 32, o * C::NBOX, c2);
                    } else {
#pragma unroll
                        for (int o = 0; o < C::NOPS; ++o) tma_red_add_3d(m, src + (size_t)o * C::NBOX * B * 16, (int)tl.j * 16, o * C::NBOX, c2);
                    }
                }
                bulk_commit();
                if (npend == 2) {
                    bulk_wait_read<2>();                      // all but the two newest groups have been read: tile k-2 is free
                    mbar_arrive(empty + pend[0]);
                    pend[0] = pend[1]; npend = 1;
                }
                pend[npend++] = s;
            }
            asm volatile("cp.async.bulk.wait_group 0;\n" ::: "memory");      // every reduce-add has been performed
        }
        return;
    }

    // ---------------- consumers.  DYN (N <= 256): a free group takes the next tile of the CTA's sequence (an x tile costs
    // more than a y / z tile); tiles are taken in order, so every earlier tile is finished or in progress and the ring
    // cannot deadlock (cfg1: 0.954 -> 0.884 ms per term).  N = 384: group g keeps the tiles g, g + NG, ... -- in the
    // plane-major launch that hands one group the x tiles (latency-bound on their late operands) and the other the y
    // tiles for long stretches, which measured better than mixing them (31.3 against 36.2 ms).
    if (C::WS_ACC) asm volatile("setmaxnreg.inc.sync.aligned.u32 152;\n");
    const int ct = tid - C::PRODT_ACC, grp = ct / GT, gt = ct % GT;
    unsigned seq = 0, i = 0;
    AccIter<N, PZ> tl;
    tl.init(a, blockIdx.x, gridDim.x);
    // one tile: the slot(s) follow from its position seq in the CTA's slot sequence
    auto process = [&](unsigned seq) {
        const unsigned s = seq % S, round = seq / S;
        const unsigned s2 = (seq + 1) % S, round2 = (seq + 1) / S;
        tl.decode(a);
        cd* tile = reinterpret_cast<cd*>(slots + (size_t)s * TILE);
        if (tl.kind == 0) {
            const int n2 = gt % C::R2, bA = gt / C::R2;
            const long long g0 = (long long)(tl.p % (unsigned)a.nz) * (N * N) + (long long)tl.j * (B * N);
            const double* vt = a.vtab ? a.vtab + g0 + bA * N + n2 : nullptr;
            mbar_wait(full + s, round & 1);
            if (C::LATEW) {
                const long long o = (long long)tl.p * (N * N) + (long long)tl.j * (B * N) + bA * N + n2;
                acc_tile_compute<N, true>(a, tile, nullptr, usev, vt, twA, twB, ktab, gt, grp, a.cur + o, usev ? a.v + o : nullptr);
            } else {
                mbar_wait(full + s2, round2 & 1);
                acc_tile_compute<N, true>(a, tile, reinterpret_cast<cd*>(slots + (size_t)s2 * TILE), usev, vt, twA, twB, ktab, gt, grp);
                // the second slot is free again (its `done` barrier is advanced too: the phase of every barrier of a slot
                // is the number of times the slot has been used)
                if (gt == 0) { mbar_arrive(done + s2); mbar_arrive(empty + s2); }
            }
        } else {
            mbar_wait(full + s, round & 1);
            acc_tile_compute<N, false>(a, tile, nullptr, false, nullptr, twA, twB, ktab + tl.kind * N, gt, grp);
        }
        if (gt == 0) mbar_arrive(done + s);
    };
    if constexpr (!C::LATEW) {
        for (;;) {
            if (gt == 0) ticket[1 + grp] = atomicAdd(ticket, 1u);
            lean_sync<C::GW>(grp);
            const unsigned mine = ticket[1 + grp];
            for (; i < mine && tl.t < a.ntiles; ++i, tl.next()) seq += tl.is_x() ? 2 : 1;
            if (tl.t >= a.ntiles) break;
            process(seq);
        }
    } else {
        if (PZ) {
            // every pair is worked on by both groups: group g takes pencils [8 g, 8 g + 8) of the 16, in place, rows 256 bytes apart
            for (; tl.t < a.ntiles; tl.next(), seq += 2) {
                const unsigned s = seq % S, round = seq / S;
                cd* tile = reinterpret_cast<cd*>(slots + (size_t)s * TILE) + grp * B;
                mbar_wait(full + s, round & 1);
                acc_tile_compute<N, false, 2 * B>(a, tile, nullptr, false, nullptr, twA, twB, ktab + 2 * N, gt, grp);
                if (gt == 0) mbar_arrive(done + s + grp);
            }
            return;
        }
        for (; tl.t < a.ntiles; tl.next(), ++i, ++seq) {
            if ((int)(i % NG) != grp) continue;
            process(seq);
        }
    }
}

// =====================================================================================================================
// Split-operator factors through the same slot ring: psi <- [phase] F^-1 exp(-i T_axis dt) F [phase] psi for
// one axis per launch, in place: TMA load of a tile, round trip with the complex k table in the slot, plain bulk store
// back to where it came from.  The potential phases (an N_g table shared by all vectors) are read from global memory by
// the thread that owns the element; the tiles run over the vectors first, so the table comes from HBM once per launch.
// =====================================================================================================================
enum { KX = 0, KY = 1, KZ = 2 };          // tile kinds = axes

struct TdArgs {
    cd* psi;
    const cd* phase;          // N_g table applied on load (F_PRO) or on store (F_EPI)
    double* rho;              // F_DENS: rho[g] += dens_scale * |result|^2
    double dens_scale;
    const cd* kc;             // complex k table of the axis: exp(-i 1/2 k^2 dt) / N
    const cd* tw;
    int kind;                 // KX, KY or KZ
    int flags;                // F_PRO / F_EPI / F_DENS
    int nvec, nz;
    unsigned ntiles;          // nvec * N * N / 8
};

// pro: the thread's phases applied on load (x launch only); racc: its sums of |psi|^2 over the vectors of the block (z
// launch only); both live in registers across the tiles of a block
template <int N, int KIND>
__device__ __forceinline__ void td_tile_compute(const TdArgs& a, cd* tile, const cd* __restrict__ ph, long long gstep,
                                                const cd* twA, const cd* twB, const cd* ktab, int gt, int bar_id,
                                                const cd (&pro)[KIND == KX ? AccCfg<N>::NPRO : 1], double (&racc)[KIND == KZ ? AccCfg<N>::R1 : 1]) {
    using C = AccCfg<N>;
    constexpr bool XK = KIND == KX;
    constexpr int R1 = C::R1, R2 = C::R2, TG = C::TG, GW = C::GW, GT = C::GT, TASKS = C::TASKS, ROUNDS = C::ROUNDS, B = C::B;
    constexpr bool WCACHE = R2 <= 8;
    constexpr int SB = XK ? C::XP : 1, SI = XK ? 1 : ((C::PAIRZ && !XK) ? 2 * B : B);   // y / z tiles in pairs: rows of 16 pencils
    const bool actA = gt < TG;
    const int n2 = XK ? gt % R2 : gt / B, bA = XK ? gt / R2 : gt % B;
    cd* eA = tile + bA * SB + n2 * SI;
    cd x[R1];
    if (actA) {
#pragma unroll
        for (int n1 = 0; n1 < R1; ++n1) x[n1] = eA[n1 * R2 * SI];
        if (KIND == KX && (a.flags & F_PRO)) {
            constexpr int NP = KIND == KX ? C::NPRO : 0;
#pragma unroll
            for (int n1 = NP; n1 < R1; ++n1) x[n1] = cmul(x[n1], __ldg(ph + (long long)n1 * gstep));
#pragma unroll
            for (int n1 = 0; n1 < NP; ++n1) x[n1] = cmul(x[n1], pro[n1]);
        }
        Dft<R1, -1>::run(x);
        if (WCACHE) {
#pragma unroll
            for (int j = 0; j < R1; ++j) eA[j * R2 * SI] = x[j];
        } else {
            eA[0] = x[0];
#pragma unroll
            for (int j = 1; j < R1; ++j) eA[j * R2 * SI] = cmul(x[j], twA[j * R2 + n2]);
        }
    }
    lean_sync<GW>(bar_id);
#pragma unroll
    for (int rd = 0; rd < ROUNDS; ++rd) {
        const int task = gt + rd * GT;
        if (task < TASKS) {
            const int bB = task % B, k1 = task / B;
            cd* eB = tile + bB * SB + k1 * R2 * SI;
            cd y[R2], wc[WCACHE ? R2 : 1];
            y[0] = eB[0];
            if (WCACHE) {
#pragma unroll
                for (int m = 1; m < R2; ++m) { wc[m] = twB[m * R1 + k1]; y[m] = cmul(eB[m * SI], wc[m]); }
            } else {
#pragma unroll
                for (int m = 1; m < R2; ++m) y[m] = eB[m * SI];
            }
            Dft<R2, -1>::run(y);
            const cd* kt = ktab + k1;
#pragma unroll
            for (int k2 = 0; k2 < R2; ++k2) y[k2] = cmul(y[k2], kt[R1 * k2]);
            Dft<R2, +1>::run(y);
            eB[0] = y[0];
#pragma unroll
            for (int m = 1; m < R2; ++m) eB[m * SI] = cmulc(y[m], WCACHE ? wc[m] : twB[m * R1 + k1]);
        }
    }
    lean_sync<GW>(bar_id);
    if (actA) {
#pragma unroll
        for (int j = 0; j < R1; ++j) x[j] = eA[j * R2 * SI];
        Dft<R1, +1>::run(x);
        if (KIND == KZ && (a.flags & F_EPI)) {               // closing factor of the last step of a call
#pragma unroll
            for (int n1 = 0; n1 < R1; ++n1) x[n1] = cmul(x[n1], __ldg(ph + (long long)n1 * gstep));
        }
        if (KIND == KZ && (a.flags & F_DENS)) {
#pragma unroll
            for (int n1 = 0; n1 < R1; ++n1) racc[KIND == KZ ? n1 : 0] += x[n1].x * x[n1].x + x[n1].y * x[n1].y;
        }
#pragma unroll
        for (int n1 = 0; n1 < R1; ++n1) eA[n1 * R2 * SI] = x[n1];
        fence_proxy_async_smem();
    }
    lean_sync<GW>(bar_id);
}

__device__ __forceinline__ void bulk_store(void* gdst, const void* ssrc, unsigned bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;\n" ::"l"(gdst), "r"(smem_u32(ssrc)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void tma_store_3d(const CUtensorMap* m, const void* src, int c0, int c1, int c2) {
    asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.tile.bulk_group [%0, {%2, %3, %4}], [%1];\n" ::"l"(m), "r"(smem_u32(src)),
                 "r"(c0), "r"(c1), "r"(c2) : "memory");
}

// one instantiation per axis (KIND): the kind-specific address arithmetic and tile layout are compile-time, which
// keeps the consumers within the register budget
template <int N, int KIND>
__global__ void __launch_bounds__(AccCfg<N>::T, 1)
td_tma_kernel(const TdArgs a, const __grid_constant__ CUtensorMap map_y, const __grid_constant__ CUtensorMap map_z, int nslots) {
    using C = AccCfg<N>;
    constexpr int GT = C::GT, NG = C::NG, B = C::B, TILE = C::TILE;
    constexpr unsigned ROWB = N * 16, TILEB = N * B * 16, TPV = (unsigned)N * N / 8;
    extern __shared__ __align__(128) char smraw[];
    char* slots = smraw;
    cd* twA = reinterpret_cast<cd*>(smraw + (size_t)nslots * TILE);
    cd* twB = twA + N;
    cd* ktab = twB + N;
    uint64_t* full = reinterpret_cast<uint64_t*>(ktab + N);
    uint64_t* done = full + C::MAXS;
    uint64_t* empty = done + C::MAXS;
    const int tid = threadIdx.x;
    for (int i = tid; i < N; i += C::T) {
        twA[i] = a.tw[(i % C::R2) * (i / C::R2)];
        twB[i] = a.tw[(i / C::R1) * (i % C::R1)];
        ktab[i] = a.kc[i];
    }
    if (tid == 0) {
        for (int s = 0; s < nslots; ++s) { mbar_init(full + s, 1); mbar_init(done + s, 1); mbar_init(empty + s, 1); }
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    __syncthreads();
    const unsigned S = (unsigned)nslots, nvec = (unsigned)a.nvec, G = gridDim.x;
    // Tile sequence of a CTA: block q = blockIdx.x, blockIdx.x + G, ... of a vector's blocks (x: 8 rows; y: plane z, 8
    // columns; z: 8 xy points), and for each block all nvec vectors in turn.  One CTA therefore sees every vector of a
    // block back to back: the owning thread reads its phases once per block (not once per tile) and sums |psi|^2 over the
    // vectors in registers, one atomic per element and block; and at any moment the CTAs work on G adjacent blocks of the
    // same few vectors (contiguous in memory).  The phase table comes from HBM once per launch.
    // PAIR (y and z launches with two consumer groups, N = 384): a block is 16 pencils, loaded and stored as one tensor
    // operation with 256-byte rows into two adjacent slots; both groups work on every tile, each on its 8 pencils (the
    // strided 128-byte rows are what bounds these launches; only the first slot's full / empty barriers are used, group g
    // arrives on done[s + g]).
    constexpr bool PAIR = C::PAIRZ && KIND != KX;
    constexpr unsigned NBLK = PAIR ? TPV / 2 : TPV, STEP = PAIR ? 2 : 1, PB = PAIR ? 2 * B : B;
    constexpr unsigned TPPB = N / PB;                          // y blocks per plane
    if (tid < C::PRODT) {
        if (C::WS) asm volatile("setmaxnreg.dec.sync.aligned.u32 40;\n");
        if (tid == 0) {
            unsigned seq = 0, q = blockIdx.x, v = 0;
            for (; q < NBLK; seq += STEP) {
                const unsigned s = seq % S, round = seq / S;
                if (round > 0) mbar_wait(empty + s, (round - 1) & 1);
                char* dst = slots + (size_t)s * TILE;
                mbar_expect_tx(full + s, STEP * TILEB);
                if (KIND == KX) {
                    const cd* row0 = a.psi + ((long long)v * a.nz * N + (long long)q * B) * N;
#pragma unroll
                    for (int b = 0; b < B; ++b) bulk_load(dst + (size_t)b * C::XP * 16, row0 + b * N, ROWB, full + s);
                } else {
                    const CUtensorMap* m = KIND == KY ? &map_y : &map_z;
                    const int c0 = KIND == KY ? (int)(q % TPPB) * (2 * PB) : (int)q * (2 * PB);
                    const int c2 = KIND == KY ? (int)(v * (unsigned)a.nz + q / TPPB) : (int)v;
#pragma unroll
                    for (int o = 0; o < C::NOPS; ++o) tma_load_3d(dst + (size_t)o * C::NBOX * PB * 16, m, c0, o * C::NBOX, c2, full + s);
                }
                if (++v == nvec) { v = 0; q += G; }
            }
        } else if (tid == 32) {
            unsigned seq = 0, pend[2], npend = 0, q = blockIdx.x, v = 0;
            for (; q < NBLK; seq += STEP) {
                const unsigned s = seq % S, round = seq / S;
                if (!mbar_test(done + s, round & 1)) {
                    if (npend) {
                        bulk_wait_read<0>();
                        for (unsigned k = 0; k < npend; ++k) mbar_arrive(empty + pend[k]);
                        npend = 0;
                    }
                    mbar_wait(done + s, round & 1);
                }
                if (PAIR) mbar_wait(done + s + 1, round & 1);          // the second group's half (loaded already: cannot depend on the loader)
                const char* src = slots + (size_t)s * TILE;
                if (KIND == KX) {
                    cd* row0 = a.psi + ((long long)v * a.nz * N + (long long)q * B) * N;
#pragma unroll
                    for (int b = 0; b < B; ++b) bulk_store(row0 + b * N, src + (size_t)b * C::XP * 16, ROWB);
                } else {
                    const CUtensorMap* m = KIND == KY ? &map_y : &map_z;
                    const int c0 = KIND == KY ? (int)(q % TPPB) * (2 * PB) : (int)q * (2 * PB);
                    const int c2 = KIND == KY ? (int)(v * (unsigned)a.nz + q / TPPB) : (int)v;
#pragma unroll
                    for (int o = 0; o < C::NOPS; ++o) tma_store_3d(m, src + (size_t)o * C::NBOX * PB * 16, c0, o * C::NBOX, c2);
                }
                bulk_commit();
                if (npend == 2) {
                    bulk_wait_read<2>();
                    mbar_arrive(empty + pend[0]);
                    pend[0] = pend[1]; npend = 1;
                }
                pend[npend++] = s;
                if (++v == nvec) { v = 0; q += G; }
            }
            asm volatile("cp.async.bulk.wait_group 0;\n" ::: "memory");
        }
        return;
    }
    if (C::WS) asm volatile("setmaxnreg.inc.sync.aligned.u32 152;\n");
    const int ct = tid - C::PRODT, grp = ct / GT, gt = ct % GT;
    const bool act = gt < C::TG;                              // owns elements in the first / last stage
    const int half = PAIR ? grp * B : 0;                      // this group's pencils inside a pair
    // grid index of this thread's first element inside block 0 and the step between its elements (phase table, density)
    long long goff, gstep;
    if (KIND == KX) { goff = (long long)(gt / C::R2) * N + gt % C::R2; gstep = C::R2; }
    else if (KIND == KY) { goff = half + gt % B + (long long)(gt / B) * N; gstep = (long long)C::R2 * N; }
    else { goff = half + gt % B + (long long)(gt / B) * (N * N); gstep = (long long)C::R2 * N * N; }
    auto block_base = [&](unsigned q) -> long long {
        if (KIND == KX) return (long long)q * (B * N);
        if (KIND == KY) { const unsigned z = q / TPPB, cb = q - z * TPPB; return (long long)z * (N * N) + (long long)cb * PB; }
        return (long long)q * PB;
    };
    constexpr int NPRO = KIND == KX ? C::NPRO : 1, NRHO = KIND == KZ ? C::R1 : 1;
    cd pro[NPRO];
    double racc[NRHO];
#pragma unroll
    for (int n1 = 0; n1 < NPRO; ++n1) pro[n1] = make_double2(1.0, 0.0);
#pragma unroll
    for (int n1 = 0; n1 < NRHO; ++n1) racc[n1] = 0.0;
    auto flush = [&](unsigned q) {                            // one atomic per element for all the vectors of the block
        if (KIND != KZ || !(a.flags & F_DENS) || !act) return;
        double* rp = a.rho + block_base(q) + goff;
        const double ds = a.dens_scale;
#pragma unroll
        for (int n1 = 0; n1 < NRHO; ++n1) { atomicAdd(rp + n1 * gstep, ds * racc[n1]); racc[n1] = 0.0; }
    };
    // without pairs group g takes the CTA's tiles g, g + NG, ...; with pairs both groups take every tile
    unsigned q = blockIdx.x, v = PAIR ? 0u : (unsigned)grp, qcur = 0xffffffffu;
    constexpr unsigned VSTEP = PAIR ? 1 : NG;
    while (v >= nvec) { v -= nvec; q += G; }
    for (unsigned seq = PAIR ? 0u : (unsigned)grp; q < NBLK; seq += PAIR ? 2 : NG) {
        const unsigned s = seq % S, round = seq / S;
        cd* tile = reinterpret_cast<cd*>(slots + (size_t)s * TILE) + half;
        if (q != qcur) {
            if (qcur != 0xffffffffu) flush(qcur);
            qcur = q;
            if (KIND == KX && (a.flags & F_PRO) && act) {
                const cd* ph = a.phase + block_base(q) + goff;
#pragma unroll
                for (int n1 = 0; n1 < NPRO; ++n1) pro[n1] = __ldg(ph + n1 * gstep);
            }
        }
        mbar_wait(full + s, round & 1);
        td_tile_compute<N, KIND>(a, tile, a.phase + block_base(q) + goff, gstep, twA, twB, ktab, gt, grp, pro, racc);
        if (gt == 0) mbar_arrive(done + s + (PAIR ? grp : 0));
        v += VSTEP;
        while (v >= nvec) { v -= nvec; q += G; }
    }
    if (qcur != 0xffffffffu) flush(qcur);
}

struct TdCall {
    TdArgs args;
    CUtensorMap map_y, map_z;
    int num_sms;
    int* occ;                 // context-owned: [1] = 1 once the kernel attribute is set
    cudaStream_t stream;
};
typedef int (*td_launch_fn)(const TdCall*);

struct AccCall {
    AccArgs args;
    CUtensorMap cur_y, cur_z, acc_y, acc_z;
    int num_sms;
    int* occ;                 // context-owned: [0] = 1 once the kernel attribute is set
    cudaStream_t stream;
};
// returns 0, -(stage*1000 + cudaError) on failure, 1 if this length has no accumulate kernel
typedef int (*acc_launch_fn)(const AccCall*);

}  // namespace sgw
