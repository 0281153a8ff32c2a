// sgw_fft.cuh -- FP64 complex FFT building blocks for sm_100a.
//
// A length-N transform is done in two register-resident stages N = R1 * R2 (Cooley-Tukey "four
// step"): stage A = radix-R1 butterflies over n1 for fixed n2, twiddle by W_N^(n2 k1), exchange
// through shared memory, stage B = radix-R2 butterflies over n2 for fixed k1.  A *round trip*
// (forward, pointwise multiply in k-space, inverse) runs A B | mult | B^-1 A^-1 with only two
// shared-memory exchanges and the data back in the registers of the thread that loaded it, so
// prologue/epilogue work (potential multiply, Chebyshev recurrence, phases) fuses for free.
// The operator structure this serves is P:84 of the paper ("FFT pairs switch between position and
// momentum representations").
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "sgw_twiddles.h"

namespace sgw {

typedef double2 cd;

__device__ __forceinline__ cd cadd(cd a, cd b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ cd csub(cd a, cd b) { return make_double2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ cd cmul(cd a, cd b) {
    return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
__device__ __forceinline__ cd cmulc(cd a, cd b) {   // a * conj(b)
    return make_double2(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y);
}
__device__ __forceinline__ cd cscale(cd a, double s) { return make_double2(a.x * s, a.y * s); }
// a * (SIGN * i)
template <int SIGN>
__device__ __forceinline__ cd mul_i(cd a) {
    return SIGN > 0 ? make_double2(-a.y, a.x) : make_double2(a.y, -a.x);
}

// a * exp(SIGN * 2 pi i j / R), j a compile-time constant after unrolling; R divides 96.
template <int R, int SIGN>
__device__ __forceinline__ cd mul_w(cd a, int j) {
    static_assert(96 % R == 0, "small-DFT radix must divide 96");
    const int q = (j % R) * (96 / R);
    if (q == 0) return a;
    if (q == 48) return make_double2(-a.x, -a.y);
    if (q == 24) return mul_i<SIGN>(a);
    if (q == 72) return mul_i<-SIGN>(a);
    const double c = tw96_cos(q), s = (SIGN > 0 ? 1.0 : -1.0) * tw96_sin(q);
    if (q == 12 || q == 36 || q == 60 || q == 84) {        // |c| == |s| == sqrt(1/2)
        const double h = 0.7071067811865476;
        const double sc = c > 0 ? 1.0 : -1.0, ss = s > 0 ? 1.0 : -1.0;
        return make_double2((sc * a.x - ss * a.y) * h, (ss * a.x + sc * a.y) * h);
    }
    return make_double2(a.x * c - a.y * s, a.x * s + a.y * c);
}

// In-register DFT of length R, natural order in and out: X[k] = sum_n x[n] exp(SIGN 2 pi i n k / R)
template <int R, int SIGN>
struct Dft {
    static __device__ __forceinline__ void run(cd* x) {
        constexpr int P = (R % 4 == 0) ? 4 : ((R % 2 == 0) ? 2 : 3);
        constexpr int Q = R / P;
        cd sub[P][Q];
#pragma unroll
        for (int p = 0; p < P; ++p)
#pragma unroll
            for (int q = 0; q < Q; ++q) sub[p][q] = x[P * q + p];
#pragma unroll
        for (int p = 0; p < P; ++p) Dft<Q, SIGN>::run(sub[p]);
#pragma unroll
        for (int k = 0; k < Q; ++k) {
            cd t[P];
#pragma unroll
            for (int p = 0; p < P; ++p) t[p] = mul_w<R, SIGN>(sub[p][k], p * k);
            Dft<P, SIGN>::run(t);
#pragma unroll
            for (int j = 0; j < P; ++j) x[k + Q * j] = t[j];
        }
    }
};
template <int SIGN>
struct Dft<1, SIGN> {
    static __device__ __forceinline__ void run(cd*) {}
};
template <int SIGN>
struct Dft<2, SIGN> {
    static __device__ __forceinline__ void run(cd* x) {
        cd a = x[0], b = x[1];
        x[0] = cadd(a, b);
        x[1] = csub(a, b);
    }
};
template <int SIGN>
struct Dft<3, SIGN> {
    static __device__ __forceinline__ void run(cd* x) {
        const double h = 0.8660254037844386;   // sqrt(3)/2
        cd t = cadd(x[1], x[2]);
        cd m = make_double2(x[0].x - 0.5 * t.x, x[0].y - 0.5 * t.y);
        cd d = cscale(csub(x[1], x[2]), h);
        cd id = mul_i<SIGN>(d);
        x[0] = cadd(x[0], t);
        x[1] = cadd(m, id);
        x[2] = csub(m, id);
    }
};
template <int SIGN>
struct Dft<4, SIGN> {
    static __device__ __forceinline__ void run(cd* x) {
        cd a = cadd(x[0], x[2]), b = csub(x[0], x[2]);
        cd c = cadd(x[1], x[3]), d = mul_i<SIGN>(csub(x[1], x[3]));
        x[0] = cadd(a, c);
        x[2] = csub(a, c);
        x[1] = cadd(b, d);
        x[3] = csub(b, d);
    }
};

// ---------------------------------------------------------------------------------------------
// two-stage factorisation per supported length
// ---------------------------------------------------------------------------------------------
template <int N> struct Fact;
#define SGW_FACT(N_, R1_, R2_) \
    template <> struct Fact<N_> { static constexpr int R1 = R1_, R2 = R2_; };
SGW_FACT(8, 4, 2)
SGW_FACT(12, 4, 3)
SGW_FACT(16, 4, 4)
SGW_FACT(24, 6, 4)
SGW_FACT(32, 8, 4)
SGW_FACT(48, 8, 6)
SGW_FACT(64, 8, 8)
SGW_FACT(96, 12, 8)
SGW_FACT(128, 16, 8)
SGW_FACT(192, 16, 12)
SGW_FACT(256, 16, 16)
SGW_FACT(384, 24, 16)
#undef SGW_FACT

// Geometry of one pass: which pencils a CTA owns and how they sit in memory.
//   tile t -> base = (t / TI) * SO + (t % TI) * SI;   element (n, b) at base + n*sN + b*sB
//   fastn != 0: the transform axis is the contiguous one (x); lanes run along n for coalescing.
//   grid index of the tile's first element: g0 = ((t / TI) % GO) * SO + (t % TI) * SI
struct PassGeom {
    long long SO, SI, sN, sB, ng;
    int TI, GO, B, fastn;
};

enum { MODE_RT = 0, MODE_FWD = 1, MODE_INV = 2 };

// One CTA = B pencils of length N.  Op supplies (sgw_ops.cuh):
//   cd   load(const cd* in, long long off, long long g)     input element (off: in the vector arrays, g: on the grid)
//   cd   mult(cd X, int k, long long gk)                    k-space multiply (RT only)
//   void epi(cd r, long long off, long long g)              store
template <int N, int MODE, class Op>
__global__ void __launch_bounds__(256) pass_kernel(PassGeom gm, const cd* __restrict__ in,
                                                    const cd* __restrict__ twN, Op op) {
    constexpr int R1 = Fact<N>::R1, R2 = Fact<N>::R2;
    constexpr int SK = R2 | 1;
    constexpr int SB = (R1 * SK) | 1;
    extern __shared__ double2 sm[];
    const int tid = threadIdx.x, B = gm.B;
    const long long t = blockIdx.x;
    const long long base = (t / gm.TI) * gm.SO + (t % gm.TI) * gm.SI;
    const long long g0 = base % gm.ng;

    // stage-A coordinates (b, n2) and stage-B coordinates (b, k1) of this thread
    int bA, n2, bB, k1;
    if (gm.fastn) { n2 = tid % R2; bA = tid / R2; k1 = tid % R1; bB = tid / R1; }
    else          { bA = tid % B;  n2 = tid / B;  bB = tid % B;  k1 = tid / B; }
    const bool actA = tid < B * R2, actB = tid < B * R1;

    cd x[R1];
    if (MODE != MODE_INV) {
        if (actA) {
#pragma unroll
            for (int n1 = 0; n1 < R1; ++n1) {
                const long long o = (long long)(n1 * R2 + n2) * gm.sN + (long long)bA * gm.sB;
                x[n1] = op.load(in, base + o, g0 + o);
            }
            Dft<R1, -1>::run(x);
#pragma unroll
            for (int j = 0; j < R1; ++j) {
                cd w = twN[n2 * j];                       // exp(-2 pi i n2 j / N)
                sm[bA * SB + j * SK + n2] = (j == 0) ? x[0] : cmul(x[j], w);
            }
        }
        __syncthreads();
    }
    if (actB) {
        cd y[R2];
        if (MODE != MODE_INV) {
#pragma unroll
            for (int m = 0; m < R2; ++m) y[m] = sm[bB * SB + k1 * SK + m];
            Dft<R2, -1>::run(y);
        }
        if (MODE == MODE_FWD) {
#pragma unroll
            for (int k2 = 0; k2 < R2; ++k2) {
                const long long o = (long long)(k1 + R1 * k2) * gm.sN + (long long)bB * gm.sB;
                op.epi(y[k2], base + o, g0 + o);
            }
        } else {
            if (MODE == MODE_RT) {
#pragma unroll
                for (int k2 = 0; k2 < R2; ++k2) {
                    const int k = k1 + R1 * k2;
                    y[k2] = op.mult(y[k2], k, g0 + (long long)k * gm.sN + (long long)bB * gm.sB);
                }
            } else {
#pragma unroll
                for (int k2 = 0; k2 < R2; ++k2) {
                    const long long o = (long long)(k1 + R1 * k2) * gm.sN + (long long)bB * gm.sB;
                    y[k2] = op.load(in, base + o, g0 + o);
                }
            }
            Dft<R2, +1>::run(y);
#pragma unroll
            for (int m = 0; m < R2; ++m) {
                cd w = twN[m * k1];
                sm[bB * SB + k1 * SK + m] = (m == 0) ? y[0] : cmulc(y[m], w);   // * exp(+2 pi i m k1/N)
            }
        }
    }
    if (MODE != MODE_FWD) {
        __syncthreads();
        if (actA) {
#pragma unroll
            for (int j = 0; j < R1; ++j) x[j] = sm[bA * SB + j * SK + n2];
            Dft<R1, +1>::run(x);
#pragma unroll
            for (int n1 = 0; n1 < R1; ++n1) {
                const long long o = (long long)(n1 * R2 + n2) * gm.sN + (long long)bA * gm.sB;
                op.epi(x[n1], base + o, g0 + o);
            }
        }
    }
}

template <int N>
constexpr int pass_threads_per_pencil() {
    return Fact<N>::R1 > Fact<N>::R2 ? Fact<N>::R1 : Fact<N>::R2;
}
template <int N>
constexpr int pass_smem_per_pencil() {       // bytes
    return ((Fact<N>::R1 * (Fact<N>::R2 | 1)) | 1) * 16;
}

}  // namespace sgw
