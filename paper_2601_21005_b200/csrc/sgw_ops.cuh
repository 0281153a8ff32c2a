// sgw_ops.cuh -- prologue / k-space / epilogue functors fused into the FFT passes, and the plain
// struct through which the library core asks a per-length translation unit to launch a pass.
#pragma once
#include "sgw_fft.cuh"

namespace sgw {

enum PassKind {
    K_RT_STORE = 0,    // out = RT(in)                      RT multiplies by a real 1D table
    K_RT_ACC = 1,      // out = RT(in) + acc
    K_RT_HFIN = 2,     // out = RT(in) + acc + V*in                        (last pass of H apply)
    K_RT_CHEB = 3,     // Chebyshev recurrence + series accumulation       (last pass of a term)
    K_RT_TD = 4,       // out = [phase] RT([phase] in), complex 1D table   (split-operator factor)
    K_RT_MUL3D = 5,    // out = RT(in) with a real 3D k-space table        (Poisson kernel)
    K_FWD = 6,         // out = forward transform along the axis, natural k order
    K_INV = 7,         // out = inverse transform (unnormalised)
    K_NKINDS = 8
};

struct OpParams {
    cd* out;                 // result
    const cd* acc;           // added to the result (may alias out)
    const cd* prev;          // Chebyshev phi_{n-1} (may alias out)
    cd* series;              // Chebyshev series accumulator
    const double* vtab;      // real N_g table multiplying the input in the epilogue
    const double* mul_re;    // real [N] k-space table (includes 1/N)
    const cd* mul_c;         // complex [N] k-space table (includes 1/N)
    const double* mul3d;     // real N_g k-space table
    const cd* pro_phase;     // complex N_g table applied on load (or NULL)
    const cd* epi_phase;     // complex N_g table applied on store (or NULL)
    double hs, c0, c1, c2;   // Chebyshev: scale of H term; series coefficients for prev, cur, next
    int use_prev, flush, series_init;
};

struct PassCall {
    int kind;
    PassGeom gm;
    long long ntiles;
    const cd* in;
    const cd* tw;            // exp(-2 pi i j / N), j < N
    OpParams p;
    cudaStream_t stream;
};

typedef int (*pass_launch_fn)(const PassCall*);

// ---- functors -------------------------------------------------------------------------------
struct OpBase {
    OpParams p;
    __device__ __forceinline__ cd pro(cd v, long long, long long) const { return v; }
    __device__ __forceinline__ cd mult(cd X, int k, long long) const { return cscale(X, __ldg(p.mul_re + k)); }
};
struct OpStore : OpBase {
    __device__ __forceinline__ void epi(cd r, cd, long long off, long long) const { p.out[off] = r; }
};
struct OpAcc : OpBase {
    __device__ __forceinline__ void epi(cd r, cd, long long off, long long) const {
        p.out[off] = cadd(r, p.acc[off]);
    }
};
struct OpHFin : OpBase {
    __device__ __forceinline__ void epi(cd r, cd vin, long long off, long long g) const {
        cd a = p.acc[off];
        const double v = p.vtab ? __ldg(p.vtab + g) : 0.0;
        p.out[off] = make_double2(r.x + a.x + v * vin.x, r.y + a.y + v * vin.y);
    }
};
struct OpCheb : OpBase {
    __device__ __forceinline__ void epi(cd r, cd vin, long long off, long long g) const {
        cd a = p.acc[off];
        const double v = __ldg(p.vtab + g);
        cd nx = make_double2(p.hs * (r.x + a.x + v * vin.x), p.hs * (r.y + a.y + v * vin.y));
        cd pv = make_double2(0.0, 0.0);
        if (p.use_prev) { pv = p.prev[off]; nx = csub(nx, pv); }
        p.out[off] = nx;
        if (p.flush) {
            cd s = make_double2(p.c0 * pv.x + p.c1 * vin.x + p.c2 * nx.x, p.c0 * pv.y + p.c1 * vin.y + p.c2 * nx.y);
            if (!p.series_init) s = cadd(s, p.series[off]);
            p.series[off] = s;
        }
    }
};
struct OpTD {
    OpParams p;
    __device__ __forceinline__ cd pro(cd v, long long, long long g) const {
        return p.pro_phase ? cmul(v, __ldg(p.pro_phase + g)) : v;
    }
    __device__ __forceinline__ cd mult(cd X, int k, long long) const { return cmul(X, __ldg(p.mul_c + k)); }
    __device__ __forceinline__ void epi(cd r, cd, long long off, long long g) const {
        p.out[off] = p.epi_phase ? cmul(r, __ldg(p.epi_phase + g)) : r;
    }
};
struct OpMul3D {
    OpParams p;
    __device__ __forceinline__ cd pro(cd v, long long, long long) const { return v; }
    __device__ __forceinline__ cd mult(cd X, int, long long gk) const { return cscale(X, __ldg(p.mul3d + gk)); }
    __device__ __forceinline__ void epi(cd r, cd, long long off, long long) const { p.out[off] = r; }
};

}  // namespace sgw
