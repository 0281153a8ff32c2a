// fftcore_bench.cu -- standalone measurement program (not part of libsgw): bare two-stage register FFT round-trip core (no global traffic): element*round-trips per second for several factorisations / group shapes.
// It exercises the same building blocks as the library (sgw_fft.cuh) so that design choices can be measured in
// isolation; results of round 1 are in profiles/r01_microbench.md.
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -std=c++17 -I.. fftcore_bench.cu -o fftcore_bench && ./fftcore_bench
#include <cstdio>
#include <cstdlib>
#include <vector>
#include "sgw_fft.cuh"
using namespace sgw;

template <int GW>
__device__ __forceinline__ void gsync(int grp) {
    if (GW == 1) __syncwarp();
    else asm volatile("bar.sync %0, %1;\n" ::"r"(grp + 1), "r"(GW * 32) : "memory");
}

// two-stage core, R1 values per thread in stage A (R2 threads per pencil), B pencils per group
template <int R1, int R2, int B, int NWG, int MINB>
__global__ void __launch_bounds__(NWG * (((B * R2 + 31) / 32) * 32), MINB)
core2(const cd* __restrict__ tw, const double* __restrict__ ktab_g, cd* out, int iters) {
    constexpr int N = R1 * R2, TG = B * R2, GW = (TG + 31) / 32, GT = GW * 32;
    constexpr int SK = R2 | 1, SB = (R1 * SK) | 1, TASKS = R1 * B, ROUNDS = (TASKS + GT - 1) / GT;
    extern __shared__ __align__(16) char smraw[];
    cd* twA = reinterpret_cast<cd*>(smraw);
    cd* twB = twA + N;
    double* ktab = reinterpret_cast<double*>(twB + N);
    const int tid = threadIdx.x, grp = tid / GT, gt = tid % GT;
    cd* xch = reinterpret_cast<cd*>(ktab + N) + grp * (B * SB);
    for (int i = tid; i < N; i += blockDim.x) {
        twA[i] = tw[(i % R2) * (i / R2)];
        twB[i] = tw[(i / R1) * (i % R1)];
        ktab[i] = ktab_g[i];
    }
    __syncthreads();
    const int n2 = gt % R2, bA = gt / R2;
    const bool actA = gt < TG;
    cd x[R1];
#pragma unroll
    for (int j = 0; j < R1; ++j) x[j] = make_double2(1.0 + j + gt, 0.5 * gt - j);
    cd* xA = xch + bA * SB + n2;
    for (int it = 0; it < iters; ++it) {
        if (actA) {
            Dft<R1, -1>::run(x);
            xA[0] = x[0];
#pragma unroll
            for (int j = 1; j < R1; ++j) xA[j * SK] = cmul(x[j], twA[j * R2 + n2]);
        }
        gsync<GW>(grp);
#pragma unroll
        for (int rd = 0; rd < ROUNDS; ++rd) {
            const int task = gt + rd * GT;
            if (task < TASKS) {
                const int k1 = task % R1, bB = task / R1;
                cd* xB = xch + bB * SB + k1 * SK;
                cd y[R2];
#pragma unroll
                for (int m = 0; m < R2; ++m) y[m] = xB[m];
                Dft<R2, -1>::run(y);
                const double* kt = ktab + k1;
#pragma unroll
                for (int k2 = 0; k2 < R2; ++k2) y[k2] = cscale(y[k2], kt[R1 * k2]);
                Dft<R2, +1>::run(y);
                xB[0] = y[0];
#pragma unroll
                for (int m = 1; m < R2; ++m) xB[m] = cmulc(y[m], twB[m * R1 + k1]);
            }
        }
        gsync<GW>(grp);
        if (actA) {
#pragma unroll
            for (int j = 0; j < R1; ++j) x[j] = xA[j * SK];
            Dft<R1, +1>::run(x);
        }
        gsync<GW>(grp);
    }
    if (actA) {
        cd s = make_double2(0, 0);
#pragma unroll
        for (int j = 0; j < R1; ++j) s = cadd(s, x[j]);
        out[(size_t)blockIdx.x * blockDim.x + tid] = s;
    }
}

template <int R1, int R2, int B, int NWG, int MINB>
void run(const char* name, int iters) {
    constexpr int N = R1 * R2, TG = B * R2, GW = (TG + 31) / 32, GT = GW * 32, T = NWG * GT;
    constexpr int SK = R2 | 1, SB = (R1 * SK) | 1;
    const size_t smem = 2 * N * 16 + N * 8 + (size_t)NWG * B * SB * 16;
    auto kern = core2<R1, R2, B, NWG, MINB>;
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    int per_sm = 0;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, T, smem);
    cudaFuncAttributes fa; cudaFuncGetAttributes(&fa, kern);
    std::vector<cd> tw(N); std::vector<double> kt(N);
    for (int j = 0; j < N; ++j) { double a = -2 * M_PI * j / N; tw[j] = make_double2(cos(a), sin(a)); kt[j] = 1.0 / N; }
    cd* dtw; double* dkt; cd* dout;
    cudaMalloc(&dtw, N * 16); cudaMalloc(&dkt, N * 8);
    cudaMemcpy(dtw, tw.data(), N * 16, cudaMemcpyHostToDevice); cudaMemcpy(dkt, kt.data(), N * 8, cudaMemcpyHostToDevice);
    const int grid = 148 * per_sm;
    cudaMalloc(&dout, (size_t)grid * T * 16);
    kern<<<grid, T, smem>>>(dtw, dkt, dout, 10);
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    cudaEventRecord(e0);
    kern<<<grid, T, smem>>>(dtw, dkt, dout, iters);
    cudaEventRecord(e1); cudaEventSynchronize(e1);
    float ms; cudaEventElapsedTime(&ms, e0, e1);
    const double elems = (double)grid * NWG * B * N * iters;
    printf("%-28s N=%3d R1=%2d R2=%2d B=%d GW=%d NWG=%d regs=%3d spill=%zu ctas/SM=%d warps/SM=%2d  %8.3f ms  %7.1f G el*RT/s  (%s)\n",
           name, N, R1, R2, B, GW, NWG, fa.numRegs, (size_t)fa.localSizeBytes, per_sm, per_sm * T / 32, ms, elems / ms / 1e6,
           cudaGetErrorString(cudaGetLastError()));
    cudaFree(dtw); cudaFree(dkt); cudaFree(dout);
}

int main(int argc, char** argv) {
    const int iters = argc > 1 ? atoi(argv[1]) : 2000;
    run<12, 8, 8, 4, 2>("v3 96=12x8 B8 2w", iters);
    run<12, 8, 8, 4, 1>("96=12x8 B8 2w nocap", iters);
    run<12, 8, 4, 8, 2>("96=12x8 B4 1w", iters);
    run<12, 8, 4, 8, 1>("96=12x8 B4 1w nocap", iters);
    run<8, 12, 8, 2, 3>("96=8x12 B8 3w cap3", iters);
    run<8, 12, 8, 2, 2>("96=8x12 B8 3w cap2", iters);
    run<8, 12, 8, 3, 2>("96=8x12 B8 3w nwg3", iters);
    run<6, 16, 4, 4, 3>("96=6x16 B4 2w", iters);
    run<16, 8, 8, 4, 2>("128=16x8 B8 2w", iters);
    run<8, 16, 8, 2, 2>("128=8x16 B8 4w", iters);
    run<16, 16, 4, 4, 2>("256=16x16 B4 2w", iters);
    run<8, 8, 8, 4, 2>("64=8x8 B8 2w", iters);
    run<8, 4, 8, 8, 2>("32=8x4 B8 1w", iters);
    return 0;
}
