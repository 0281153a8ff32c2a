// sgw_plane.cuh -- fused x+y pass: one persistent CTA owns whole xy planes (nx == ny == N).
//
// The kinetic operator is additively separable (T = Tx + Ty + Tz) and exp(-i T dt) multiplicatively
// separable, so neither H apply nor the split-operator step needs a 3D transform: an xy-plane pass
// plus a z-pencil pass suffice.  Here the plane pass runs as two tile phases inside ONE kernel:
//   phase X: row tiles (B contiguous rows)   W = RTx(phi)           | psi = RTx(phase * psi)
//   phase Y: column tiles (B columns)        W = W + RTy(phi)       | psi = RTy(psi)
// The CTA that wrote a plane's rows in phase X reads them back by columns in phase Y, a few
// microseconds later, so the transpose happens in L2 and HBM sees each array once (32 B per
// grid point for the plane pass instead of 80 B for separate x and y passes).  Planes are taken in
// groups of G >= 2 (all X tiles of the group, then all Y tiles) so the cp.async prefetch of the first
// Y tile never races the stores of the last X tile of the same plane.
#pragma once
#include "sgw_pipe.cuh"

namespace sgw {

enum { PL_SUM = 0, PL_TD = 1 };

struct PlaneArgs {
    const cd* in;          // phi (PL_SUM) or psi (PL_TD, == out)
    cd* out;               // W (PL_SUM) or psi (PL_TD)
    const cd* phase;       // PL_TD: complex N_g table applied on load in phase X, or NULL
    const double* kre_x;   // PL_SUM: real k-space tables (incl. 1/N)
    const double* kre_y;
    const cd* kc_x;        // PL_TD: complex k-space tables (incl. 1/N)
    const cd* kc_y;
    unsigned nplanes;      // nz * nvec
    unsigned nz;
    int G;                 // planes per group
};

struct PlaneCall {
    int mode;
    PlaneArgs a;
    const cd* tw;
    int ctas_per_sm;       // 0 = as many as fit
    cudaStream_t stream;
};
typedef int (*plane_launch_fn)(const PlaneCall*);

template <int N, int B>
struct PlaneCfg {
    using P = PipeCfg<N, B>;
    static constexpr int T = P::T;
    static constexpr int SLOT_BYTES = B * N * 16;
    static constexpr int STAGE_BYTES = 2 * SLOT_BYTES;               // in + (acc | phase)
    static constexpr int TAB_BYTES = 4 * N * 16;                     // twA, twB, ktab x, ktab y
    static constexpr int FIXED_BYTES = P::XCH_BYTES + TAB_BYTES;
    static constexpr int SMEM_BYTES = FIXED_BYTES + 2 * STAGE_BYTES;
    static constexpr int TPP = N / B;                                // tiles per plane per phase
};

struct PlaneOpSumX {
    OpParams p;
    static constexpr bool CPLX_MULT = false;
    __device__ __forceinline__ cd pro(cd v, const StageView&, int) const { return v; }
    __device__ __forceinline__ void epi(cd r, const StageView&, int, cd* out, cd*, long long o) const { out[o] = r; }
};
struct PlaneOpSumY {
    OpParams p;
    static constexpr bool CPLX_MULT = false;
    __device__ __forceinline__ cd pro(cd v, const StageView&, int) const { return v; }
    __device__ __forceinline__ void epi(cd r, const StageView& sv, int i, cd* out, cd*, long long o) const {
        out[o] = cadd(r, sv.c16(SLOT_ACC, i));
    }
};
struct PlaneOpTDX {
    OpParams p;
    static constexpr bool CPLX_MULT = true;
    __device__ __forceinline__ cd pro(cd v, const StageView& sv, int i) const {
        return p.pro_phase ? cmul(v, sv.c16(SLOT_ACC, i)) : v;
    }
    __device__ __forceinline__ void epi(cd r, const StageView&, int, cd* out, cd*, long long o) const { out[o] = r; }
};
struct PlaneOpTDY {
    OpParams p;
    static constexpr bool CPLX_MULT = true;
    __device__ __forceinline__ cd pro(cd v, const StageView&, int) const { return v; }
    __device__ __forceinline__ void epi(cd r, const StageView&, int, cd* out, cd*, long long o) const { out[o] = r; }
};

template <int N, int B, int MODE>
__global__ void __launch_bounds__(PlaneCfg<N, B>::T) plane_kernel(PlaneArgs a, const cd* __restrict__ twN) {
    using Cfg = PlaneCfg<N, B>;
    using PC = PipeCfg<N, B>;
    constexpr int R1 = PC::R1, R2 = PC::R2, T = PC::T, CP = PC::CP, SK = PC::SK, SB = PC::SB, TP = PC::TP;
    constexpr int TPP = Cfg::TPP;
    constexpr long long NXY = (long long)N * N;
    extern __shared__ __align__(16) char smraw[];
    cd* xch = reinterpret_cast<cd*>(smraw);
    cd* twA = reinterpret_cast<cd*>(smraw + PC::XCH_BYTES);
    cd* twB = twA + N;
    cd* ktx = twB + N;
    cd* kty = ktx + N;
    char* stages = smraw + Cfg::FIXED_BYTES;
    const unsigned smem_stage0 = (unsigned)__cvta_generic_to_shared(stages);
    const int tid = threadIdx.x;

    for (int i = tid; i < N; i += T) {
        twA[i] = twN[(i % R2) * (i / R2)];
        twB[i] = twN[(i / R1) * (i % R1)];
        if (MODE == PL_TD) { ktx[i] = a.kc_x[i]; kty[i] = a.kc_y[i]; }
        else { reinterpret_cast<double*>(ktx)[i] = a.kre_x[i]; reinterpret_cast<double*>(kty)[i] = a.kre_y[i]; }
    }

    // thread coordinates in the two phases
    const int n2x = tid % R2, bAx = tid / R2, k1x = tid % R1, bBx = tid / R1;   // X: lanes along n
    const int bAy = tid % B, n2y = tid / B;                                       // Y: lanes along b
    const bool actA = tid < B * R2, actB = tid < B * R1;

    // ---- CTA-local iterator over (group, item): item < np*TPP are X tiles, the rest Y tiles ----------
    const unsigned G = (unsigned)a.G;
    const unsigned ngroups = (a.nplanes + G - 1) / G;
    struct It { unsigned grp, item; };
    auto np_of = [&](unsigned grp) { const unsigned r = a.nplanes - grp * G; return r < G ? r : G; };
    auto advance = [&](It& it) {
        if (++it.item == 2 * np_of(it.grp) * TPP) { it.item = 0; it.grp += gridDim.x; }
    };
    auto decode = [&](const It& it, bool& phaseY, unsigned& plane, unsigned& tile) {
        const unsigned half = np_of(it.grp) * TPP;
        phaseY = it.item >= half;
        const unsigned r = phaseY ? it.item - half : it.item;
        plane = it.grp * G + r / TPP;
        tile = r % TPP;
    };
    auto prefetch = [&](const It& it, int stage) {
        bool py; unsigned plane, tile;
        decode(it, py, plane, tile);
        const unsigned st = smem_stage0 + (unsigned)stage * Cfg::STAGE_BYTES;
        const long long pbase = (long long)plane * NXY;
        if (!py) {                                  // B contiguous rows
            const long long base = pbase + (long long)tile * (B * N);
            const char* gp = reinterpret_cast<const char*>(a.in + base) + tid * 16;
            const unsigned dst = st + tid * 16;
#pragma unroll
            for (int j = 0; j < CP; ++j) cp_async16(dst + j * T * 16, gp + j * T * 16);
            if (MODE == PL_TD && a.phase) {
                const long long g0 = (long long)(plane % a.nz) * NXY + (long long)tile * (B * N);
                const char* gq = reinterpret_cast<const char*>(a.phase + g0) + tid * 16;
#pragma unroll
                for (int j = 0; j < CP; ++j) cp_async16(dst + Cfg::SLOT_BYTES + j * T * 16, gq + j * T * 16);
            }
        } else {                                    // B columns: element (y, b) at base + y*N + b
            const long long base = pbase + (long long)tile * B;
            const long long o0 = (long long)(tid / B) * N + (tid % B);
            const unsigned dst = st + tid * 16;
            const char* gp = reinterpret_cast<const char*>((MODE == PL_TD ? a.out : a.in) + base + o0);
#pragma unroll
            for (int j = 0; j < CP; ++j) cp_async16(dst + j * T * 16, gp + (long long)j * (TP * N * 16));
            if (MODE == PL_SUM) {
                const char* gq = reinterpret_cast<const char*>(a.out + base + o0);
#pragma unroll
                for (int j = 0; j < CP; ++j)
                    cp_async16(dst + Cfg::SLOT_BYTES + j * T * 16, gq + (long long)j * (TP * N * 16));
            }
        }
        cp_async_commit();
    };

    It cur{blockIdx.x, 0};
    if (cur.grp >= ngroups) return;
    prefetch(cur, 0);
    int stage = 0;
    OpParams pp;
    pp.pro_phase = a.phase;
    while (cur.grp < ngroups) {
        cp_async_wait_all();
        __syncthreads();
        It nxt = cur;
        advance(nxt);
        bool late = false;
        if (nxt.grp < ngroups) {
            // a lone plane (ragged last group): its first Y tile must wait for the X tile in flight
            late = (np_of(nxt.grp) == 1 && nxt.item == TPP);
            if (!late) prefetch(nxt, stage ^ 1);
        }
        bool py; unsigned plane, tile;
        decode(cur, py, plane, tile);
        const long long pbase = (long long)plane * NXY;
        const char* st = stages + (size_t)stage * Cfg::STAGE_BYTES;
        StageView sv;
        if (!py) {
            const int eA = bAx * N + n2x;
            sv.slot[SLOT_IN] = st + eA * 16;
            sv.slot[SLOT_ACC] = st + Cfg::SLOT_BYTES + eA * 16;
            cd* out = a.out + pbase + (long long)tile * (B * N) + (long long)bAx * N + n2x;
            if (MODE == PL_TD) {
                PlaneOpTDX op; op.p = pp;
                tile_roundtrip<N, B, true, PlaneOpTDX>(op, sv, xch + bAx * SB + n2x, xch + bBx * SB + k1x * SK, twA + n2x,
                                                       twB + k1x, ktx + k1x, nullptr, actA, actB, out, nullptr, R2);
            } else {
                PlaneOpSumX op; op.p = pp;
                tile_roundtrip<N, B, true, PlaneOpSumX>(op, sv, xch + bAx * SB + n2x, xch + bBx * SB + k1x * SK, twA + n2x,
                                                        twB + k1x, nullptr, reinterpret_cast<const double*>(ktx) + k1x,
                                                        actA, actB, out, nullptr, R2);
            }
        } else {
            const int eA = n2y * B + bAy;
            sv.slot[SLOT_IN] = st + eA * 16;
            sv.slot[SLOT_ACC] = st + Cfg::SLOT_BYTES + eA * 16;
            cd* out = a.out + pbase + (long long)tile * B + (long long)n2y * N + bAy;
            if (MODE == PL_TD) {
                PlaneOpTDY op; op.p = pp;
                tile_roundtrip<N, B, false, PlaneOpTDY>(op, sv, xch + bAy * SB + n2y, xch + bAy * SB + n2y * SK, twA + n2y,
                                                        twB + n2y, kty + n2y, nullptr, actA, actB, out, nullptr,
                                                        (long long)R2 * N);
            } else {
                PlaneOpSumY op; op.p = pp;
                tile_roundtrip<N, B, false, PlaneOpSumY>(op, sv, xch + bAy * SB + n2y, xch + bAy * SB + n2y * SK, twA + n2y,
                                                         twB + n2y, nullptr, reinterpret_cast<const double*>(kty) + n2y,
                                                         actA, actB, out, nullptr, (long long)R2 * N);
            }
        }
        if (late) {
            __syncthreads();                        // this tile's stores are ordered before the Y prefetch
            prefetch(nxt, stage ^ 1);
        }
        cur = nxt;
        stage ^= 1;
    }
}

}  // namespace sgw
