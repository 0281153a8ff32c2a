// pass_bench.cu -- standalone measurement program (not part of libsgw): one lean streaming pass acc += RT(cur) on nvec x 96^3: early / late accumulator load, x / z axis, B = 4 / 8.
// It exercises the same building blocks as the library (sgw_fft.cuh) so that design choices can be measured in
// isolation; results of round 1 are in profiles/r01_microbench.md.
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -std=c++17 -I.. pass_bench.cu -o pass_bench && ./pass_bench
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

// MODE 0: acc loaded with x (early);  1: acc loaded after the inverse transform (late);  2: no acc (out = RT(cur))
// AXIS 2: z pencils (stride nxy);  0: x pencils (contiguous rows)
template <int R1, int R2, int B, int NWG, int MINB, int MODE, int AXIS>
__global__ void __launch_bounds__(NWG * (((B * R2 + 31) / 32) * 32), MINB)
passk(const cd* __restrict__ tw, const double* __restrict__ ktab_g, const cd* __restrict__ cur, cd* __restrict__ acc,
      int nvec, unsigned ntiles) {
    constexpr int N = R1 * R2, TG = B * R2, GW = (TG + 31) / 32, GT = GW * 32;
    constexpr int SK = R2 | 1, SB = (R1 * SK) | 1, TASKS = R1 * B, ROUNDS = (TASKS + GT - 1) / GT;
    constexpr int NXY = N * N;
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
    int n2, bA, e0, estep;
    if (AXIS == 0) { n2 = gt % R2; bA = gt / R2; e0 = bA * N + n2; estep = R2; }
    else           { bA = gt % B; n2 = gt / B; e0 = n2 * NXY + bA; estep = R2 * NXY; }
    const bool actA = gt < TG;
    cd* xA = xch + bA * SB + n2;
    constexpr unsigned TPV = NXY / B;
    const unsigned stride = gridDim.x * NWG;
    for (unsigned t = blockIdx.x * NWG + grp; t < ntiles; t += stride) {
        long long base;
        if (AXIS == 0) base = (long long)t * (B * N);
        else { const unsigned v = t / TPV, i = t - v * TPV; base = (long long)v * ((long long)NXY * N) + (long long)i * B; }
        const cd* cp = cur + base + e0;
        cd* ap = acc + base + e0;
        cd x[R1], ad[R1];
        if (actA) {
#pragma unroll
            for (int j = 0; j < R1; ++j) x[j] = __ldcg(cp + j * estep);
            if (MODE == 0) {
#pragma unroll
                for (int j = 0; j < R1; ++j) ad[j] = __ldcg(ap + j * estep);
            }
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
            if (MODE == 1) {
#pragma unroll
                for (int j = 0; j < R1; ++j) ad[j] = __ldcg(ap + j * estep);
            }
#pragma unroll
            for (int j = 0; j < R1; ++j)
                __stcg(ap + j * estep, MODE == 2 ? x[j] : cadd(x[j], ad[j]));
        }
        gsync<GW>(grp);
    }
}

template <int R1, int R2, int B, int NWG, int MINB, int MODE, int AXIS>
void run(const char* name, int nvec, cd* cur, cd* acc) {
    constexpr int N = R1 * R2, TG = B * R2, GW = (TG + 31) / 32, GT = GW * 32, T = NWG * GT;
    constexpr int SK = R2 | 1, SB = (R1 * SK) | 1;
    const size_t smem = 2 * N * 16 + N * 8 + (size_t)NWG * B * SB * 16;
    auto kern = passk<R1, R2, B, NWG, MINB, MODE, AXIS>;
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    int per_sm = 0;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, T, smem);
    cudaFuncAttributes fa; cudaFuncGetAttributes(&fa, kern);
    std::vector<cd> tw(N); std::vector<double> kt(N);
    for (int j = 0; j < N; ++j) { double a = -2 * M_PI * j / N; tw[j] = make_double2(cos(a), sin(a)); kt[j] = 1.0 / N; }
    cd* dtw; double* dkt;
    cudaMalloc(&dtw, N * 16); cudaMalloc(&dkt, N * 8);
    cudaMemcpy(dtw, tw.data(), N * 16, cudaMemcpyHostToDevice); cudaMemcpy(dkt, kt.data(), N * 8, cudaMemcpyHostToDevice);
    const unsigned ntiles = (unsigned)((size_t)nvec * N * N * N / (B * N));
    const int grid = 148 * per_sm;
    kern<<<grid, T, smem>>>(dtw, dkt, cur, acc, nvec, ntiles);
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    float best = 1e30f;
    for (int rep = 0; rep < 3; ++rep) {
        cudaEventRecord(e0);
        kern<<<grid, T, smem>>>(dtw, dkt, cur, acc, nvec, ntiles);
        cudaEventRecord(e1); cudaEventSynchronize(e1);
        float ms; cudaEventElapsedTime(&ms, e0, e1);
        if (ms < best) best = ms;
    }
    const double elems = (double)nvec * N * N * N;
    const double bytes = elems * (MODE == 2 ? 32.0 : 48.0);
    printf("%-26s N=%3d R1=%2d R2=%2d B=%d GW=%d NWG=%d mode=%d axis=%d regs=%3d spill=%zu warps/SM=%2d  %7.3f ms  %6.1f G el*RT/s  %6.0f GB/s (%s)\n",
           name, N, R1, R2, B, GW, NWG, MODE, AXIS, fa.numRegs, (size_t)fa.localSizeBytes, per_sm * T / 32, best, elems / best / 1e6,
           bytes / best / 1e6, cudaGetErrorString(cudaGetLastError()));
    cudaFree(dtw); cudaFree(dkt);
}

int main(int argc, char** argv) {
    const int nvec = argc > 1 ? atoi(argv[1]) : 64;
    const size_t n = (size_t)nvec * 96 * 96 * 96;
    cd *cur, *acc;
    cudaMalloc(&cur, n * 16); cudaMalloc(&acc, n * 16);
    cudaMemset(cur, 0, n * 16); cudaMemset(acc, 0, n * 16);
    run<12, 8, 8, 4, 2, 0, 2>("z early-acc B8", nvec, cur, acc);
    run<12, 8, 8, 4, 2, 1, 2>("z late-acc B8", nvec, cur, acc);
    run<12, 8, 8, 4, 2, 2, 2>("z no-acc B8", nvec, cur, acc);
    run<12, 8, 4, 8, 2, 1, 2>("z late-acc B4", nvec, cur, acc);
    run<12, 8, 8, 4, 1, 0, 2>("z early-acc B8 nocap", nvec, cur, acc);
    run<8, 12, 8, 2, 3, 1, 2>("z late 8x12 3w cap3", nvec, cur, acc);
    run<8, 12, 8, 2, 3, 0, 2>("z early 8x12 3w cap3", nvec, cur, acc);
    run<8, 12, 8, 3, 2, 0, 2>("z early 8x12 nwg3", nvec, cur, acc);
    run<12, 8, 8, 4, 2, 0, 0>("x early-acc B8", nvec, cur, acc);
    run<12, 8, 8, 4, 2, 1, 0>("x late-acc B8", nvec, cur, acc);
    run<12, 8, 8, 4, 2, 2, 0>("x no-acc B8", nvec, cur, acc);
    return 0;
}
