// sgw_pipe.cuh -- persistent, software-pipelined round-trip pass for sm_100a.
//
// Each CTA loops over tiles (B pencils of length N).  All operands of tile i+1 (the input vector
// and every array the fused epilogue needs: accumulator, phi_{n-1}, series, potential or phase
// table) are copied global->shared with cp.async while tile i is transformed, so HBM latency is
// hidden by the copy path rather than by occupancy (the first, non-pipelined kernel ran at
// 11 warps/SM and ~45 % of HBM bandwidth: profiles/r01_v1_ncu_summary.md).  The transform itself
// is the two-stage register FFT of sgw_fft.cuh; results go from registers straight to HBM.
// Everything that depends only on the thread (element offsets, twiddle addresses) is hoisted out
// of the tile loop; tile arithmetic is 32-bit.
#pragma once
#include "sgw_ops.cuh"

namespace sgw {

enum { SLOT_IN = 0, SLOT_ACC = 1, SLOT_PREV = 2, SLOT_SERIES = 3, SLOT_TAB = 4, NSLOT = 5 };

struct StageSrc {
    const char* ptr;     // NULL = slot unused
    int esz;             // element bytes: 16 (complex) or 8 (real)
    int grid;            // 1: indexed by grid point g (shared by all vectors); 0: by vector element
    int slot_off;        // byte offset of this slot inside a stage
};

struct PipeArgs {
    StageSrc src[NSLOT];
    int stage_bytes;     // bytes of one stage (all used slots)
    unsigned ntiles;
};

__device__ __forceinline__ void cp_async16(unsigned smem, const void* gmem) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(smem), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async8(unsigned smem, const void* gmem) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n" ::"r"(smem), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;\n" ::: "memory"); }

// Staged operands of the current tile as seen by the functors: slot base pointers already offset to
// this thread's first element; element n1 of the thread is at index n1*STEP.
struct StageView {
    const char* slot[NSLOT];
    __device__ __forceinline__ cd c16(int s, int i) const { return reinterpret_cast<const cd*>(slot[s])[i]; }
    __device__ __forceinline__ double r8(int s, int i) const { return reinterpret_cast<const double*>(slot[s])[i]; }
};

// ---- functors (pipelined form) ------------------------------------------------------------------
//   cd   pro(cd v, const StageView&, int i)                    i = element index inside the slot
//   cd   mult(cd X, const double* mre, const cd* mc, int k)    tables already offset by k1
//   void epi(cd r, const StageView&, int i, cd* out, cd* series, long long o)
struct POpBase {
    OpParams p;
    static constexpr bool CPLX_MULT = false;
    __device__ __forceinline__ cd pro(cd v, const StageView&, int) const { return v; }
};
struct POpStore : POpBase {
    __device__ __forceinline__ void epi(cd r, const StageView&, int, cd* out, cd*, long long o) const { out[o] = r; }
};
struct POpAcc : POpBase {
    __device__ __forceinline__ void epi(cd r, const StageView& sv, int i, cd* out, cd*, long long o) const {
        out[o] = cadd(r, sv.c16(SLOT_ACC, i));
    }
};
struct POpHFin : POpBase {
    __device__ __forceinline__ void epi(cd r, const StageView& sv, int i, cd* out, cd*, long long o) const {
        const cd a = sv.c16(SLOT_ACC, i), vin = sv.c16(SLOT_IN, i);
        const double v = p.vtab ? sv.r8(SLOT_TAB, i) : 0.0;
        out[o] = make_double2(r.x + a.x + v * vin.x, r.y + a.y + v * vin.y);
    }
};
struct POpCheb : POpBase {
    __device__ __forceinline__ void epi(cd r, const StageView& sv, int i, cd* out, cd* series, long long o) const {
        const cd a = sv.c16(SLOT_ACC, i), vin = sv.c16(SLOT_IN, i);
        const double v = sv.r8(SLOT_TAB, i);
        cd nx = make_double2(p.hs * (r.x + a.x + v * vin.x), p.hs * (r.y + a.y + v * vin.y));
        cd pv = make_double2(0.0, 0.0);
        if (p.use_prev) { pv = sv.c16(SLOT_PREV, i); nx = csub(nx, pv); }
        out[o] = nx;
        if (p.flush) {
            cd s = make_double2(p.c0 * pv.x + p.c1 * vin.x + p.c2 * nx.x, p.c0 * pv.y + p.c1 * vin.y + p.c2 * nx.y);
            if (!p.series_init) s = cadd(s, sv.c16(SLOT_SERIES, i));
            series[o] = s;
        }
    }
};
struct POpTD {
    OpParams p;
    static constexpr bool CPLX_MULT = true;
    __device__ __forceinline__ cd pro(cd v, const StageView& sv, int i) const {
        return p.pro_phase ? cmul(v, sv.c16(SLOT_TAB, i)) : v;
    }
    __device__ __forceinline__ void epi(cd r, const StageView& sv, int i, cd* out, cd*, long long o) const {
        out[o] = p.epi_phase ? cmul(r, sv.c16(SLOT_TAB, i)) : r;
    }
};

template <int N, int B>
struct PipeCfg {
    static constexpr int R1 = Fact<N>::R1, R2 = Fact<N>::R2;
    static constexpr int TP = R1 > R2 ? R1 : R2;       // threads per pencil
    static constexpr int T = B * TP;                   // threads per CTA
    static constexpr int CP = (B * N) / T;             // cp.async per thread per slot ( = min(R1,R2) )
    static constexpr int SK = R2 | 1;
    static constexpr int SB = (R1 * SK) | 1;
    static constexpr int XCH_BYTES = ((B * SB * 16) + 15) & ~15;
    static constexpr int TW_BYTES = 2 * N * 16 + N * 16;   // twA, twB, k-space table (complex-sized)
    static constexpr int FIXED_BYTES = XCH_BYTES + TW_BYTES;
};

// One round trip (forward, k-space multiply, inverse) of the staged tile: the three register phases
// with their two shared-memory exchanges.  Contains two __syncthreads.
template <int N, int B, bool FASTN, class Op>
__device__ __forceinline__ void tile_roundtrip(const Op& op, const StageView& sv, cd* xA, cd* xB, const cd* twAp,
                                               const cd* twBp, const cd* ktp, const double* ktr, bool actA, bool actB,
                                               cd* out, cd* series, long long ostep) {
    constexpr int R1 = Fact<N>::R1, R2 = Fact<N>::R2;
    constexpr int SK = R2 | 1;
    constexpr int ESTEP = FASTN ? R2 : R2 * B;
    cd x[R1];
    if (actA) {
#pragma unroll
        for (int n1 = 0; n1 < R1; ++n1) x[n1] = op.pro(sv.c16(SLOT_IN, n1 * ESTEP), sv, n1 * ESTEP);
        Dft<R1, -1>::run(x);
        xA[0] = x[0];
#pragma unroll
        for (int j = 1; j < R1; ++j) xA[j * SK] = cmul(x[j], twAp[j * R2]);
    }
    __syncthreads();
    if (actB) {
        cd y[R2];
#pragma unroll
        for (int m = 0; m < R2; ++m) y[m] = xB[m];
        Dft<R2, -1>::run(y);
#pragma unroll
        for (int k2 = 0; k2 < R2; ++k2) {
            if (Op::CPLX_MULT) y[k2] = cmul(y[k2], ktp[R1 * k2]);
            else y[k2] = cscale(y[k2], ktr[R1 * k2]);
        }
        Dft<R2, +1>::run(y);
        xB[0] = y[0];
#pragma unroll
        for (int m = 1; m < R2; ++m) xB[m] = cmulc(y[m], twBp[m * R1]);
    }
    __syncthreads();
    if (actA) {
#pragma unroll
        for (int j = 0; j < R1; ++j) x[j] = xA[j * SK];
        Dft<R1, +1>::run(x);
#pragma unroll
        for (int n1 = 0; n1 < R1; ++n1) op.epi(x[n1], sv, n1 * ESTEP, out, series, n1 * ostep);
    }
}

template <int N, int B, bool FASTN, class Op>
__global__ void __launch_bounds__(PipeCfg<N, B>::T) pipe_kernel(PassGeom gm, PipeArgs pa, const cd* __restrict__ twN, Op op) {
    using Cfg = PipeCfg<N, B>;
    constexpr int R1 = Cfg::R1, R2 = Cfg::R2, T = Cfg::T, CP = Cfg::CP, SK = Cfg::SK, SB = Cfg::SB;
    constexpr int ESTEP = FASTN ? R2 : R2 * B;         // slot-index step between a thread's elements
    extern __shared__ __align__(16) char smraw[];
    cd* xch = reinterpret_cast<cd*>(smraw);
    cd* twA = reinterpret_cast<cd*>(smraw + Cfg::XCH_BYTES);   // twA[j*R2 + n2] = W^(n2 j)
    cd* twB = twA + N;                                          // twB[m*R1 + k1] = W^(m k1)
    cd* ktab = twB + N;                                         // k-space multiplier, [k]
    char* stages = smraw + Cfg::FIXED_BYTES;
    const int tid = threadIdx.x;

    for (int i = tid; i < N; i += T) {
        twA[i] = twN[(i % R2) * (i / R2)];
        twB[i] = twN[(i / R1) * (i % R1)];
        if (Op::CPLX_MULT) ktab[i] = op.p.mul_c[i];
        else reinterpret_cast<double*>(ktab)[i] = op.p.mul_re[i];
    }

    int bA, n2, bB, k1;
    if (FASTN) { n2 = tid % R2; bA = tid / R2; k1 = tid % R1; bB = tid / R1; }
    else       { bA = tid % B;  n2 = tid / B;  bB = bA;       k1 = n2; }
    const bool actA = tid < B * R2, actB = tid < B * R1;

    // thread-invariant offsets (elements) of the CP elements this thread copies per slot
    int cpo[CP];
#pragma unroll
    for (int j = 0; j < CP; ++j) {
        const int idx = tid + j * T;
        cpo[j] = FASTN ? (idx / N) * (int)gm.sB + (idx % N) : (idx / B) * (int)gm.sN + (idx % B);
    }
    const int eA = FASTN ? bA * N + n2 : n2 * B + bA;                 // slot index of this thread's element n1 = 0
    const long long oA = (long long)n2 * gm.sN + (long long)bA * gm.sB;
    const long long ostep = (long long)R2 * gm.sN;
    const unsigned smem_stage0 = (unsigned)__cvta_generic_to_shared(stages);
    const cd* twAp = twA + n2;
    const cd* twBp = twB + k1;
    const cd* ktp = ktab + k1;
    const double* ktr = reinterpret_cast<const double*>(ktab) + k1;
    cd* xA = xch + bA * SB + n2;
    cd* xB = xch + bB * SB + k1 * SK;

    auto tile_base = [&](unsigned t, long long& base, long long& g0) {
        const unsigned outer = t / (unsigned)gm.TI, inner = t - outer * (unsigned)gm.TI;
        base = (long long)outer * gm.SO + (long long)inner * gm.SI;
        g0 = (long long)(outer % (unsigned)gm.GO) * gm.SO + (long long)inner * gm.SI;
    };
    auto prefetch = [&](unsigned t, int stage) {
        long long base, g0;
        tile_base(t, base, g0);
        const unsigned st = smem_stage0 + (unsigned)stage * (unsigned)pa.stage_bytes;
#pragma unroll
        for (int s = 0; s < NSLOT; ++s) {
            const StageSrc src = pa.src[s];
            if (!src.ptr) continue;
            if (src.esz == 16) {
                const char* gp = src.ptr + (src.grid ? g0 : base) * 16;
                const unsigned dst = st + src.slot_off + tid * 16;
#pragma unroll
                for (int j = 0; j < CP; ++j) cp_async16(dst + j * T * 16, gp + (long long)cpo[j] * 16);
            } else {
                const char* gp = src.ptr + (src.grid ? g0 : base) * 8;
                const unsigned dst = st + src.slot_off + tid * 8;
#pragma unroll
                for (int j = 0; j < CP; ++j) cp_async8(dst + j * T * 8, gp + (long long)cpo[j] * 8);
            }
        }
        cp_async_commit();
    };

    unsigned t = blockIdx.x;
    if (t >= pa.ntiles) return;
    prefetch(t, 0);
    int stage = 0;
    for (; t < pa.ntiles; t += gridDim.x, stage ^= 1) {
        cp_async_wait_all();
        __syncthreads();                       // stage data (and tables) visible; previous tile fully consumed
        const unsigned tn = t + gridDim.x;
        if (tn < pa.ntiles) prefetch(tn, stage ^ 1);

        long long base, g0;
        tile_base(t, base, g0);
        StageView sv;
        const char* st = stages + (size_t)stage * pa.stage_bytes;
#pragma unroll
        for (int s = 0; s < NSLOT; ++s) sv.slot[s] = st + pa.src[s].slot_off + eA * pa.src[s].esz;

        tile_roundtrip<N, B, FASTN, Op>(op, sv, xA, xB, twAp, twBp, ktp, ktr, actA, actB, op.p.out + base + oA,
                                        op.p.series + base + oA, ostep);
    }
}

}  // namespace sgw
