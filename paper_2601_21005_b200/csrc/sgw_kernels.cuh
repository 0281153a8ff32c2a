// sgw_kernels.cuh -- the non-FFT kernels of the hot path: counter RNG, density, phases, the sparse
// Kleinman-Bylander gather-dot-scatter, segmented norms.
#pragma once
#include "sgw_fft.cuh"

namespace sgw {

// ---- a1: white-noise vectors (R-4, R-5) -------------------------------------------------
__host__ __device__ __forceinline__ uint64_t sm64(uint64_t x) {
    x += 0x9E3779B97F4A7C15ULL;
    x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ULL;
    x = (x ^ (x >> 27)) * 0x94D049BB133111EBULL;
    return x ^ (x >> 31);
}

// grid (ceil(ng/ (256*4)), nvec): each thread writes 4 consecutive elements (64 B)
static __global__ void rng_kernel(cd* __restrict__ psi, uint64_t seed_mixed, int first_vec, long long ng) {
    const int v = blockIdx.y;
    const uint64_t key = sm64(seed_mixed ^ (uint64_t)(first_vec + v));
    const long long g0 = ((long long)blockIdx.x * blockDim.x + threadIdx.x) * 4;
    cd* dst = psi + (long long)v * ng;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const long long g = g0 + j;
        if (g < ng) {
            const uint64_t h = sm64(key ^ (uint64_t)g);
            dst[g] = make_double2((h >> 63) ? -1.0 : 1.0, 0.0);
        }
    }
}

// ---- a9: density --------------------------------------------------------------------
static __global__ void density_kernel(const cd* __restrict__ psi, int nvec, long long ng, double scale,
                                      double* __restrict__ rho, double* __restrict__ rho2) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= ng) return;
    double s = 0.0;
    for (int v = 0; v < nvec; ++v) {
        const cd a = psi[(long long)v * ng + i];
        s += a.x * a.x + a.y * a.y;
    }
    s *= scale;
    rho[i] = s;
    if (rho2) rho2[i] = s;
}

// rho[g] += scale * sum_v |psi_v[g]|^2 at the listed (distinct) grid points only: corrects a density accumulated by the
// last pass of a step for the points the closing nonlocal factor changes afterwards (scale < 0 before it, > 0 after)
static __global__ void density_points_kernel(const cd* __restrict__ psi, int nvec, long long ng, const int32_t* __restrict__ pts,
                                             long long npts, double scale, double* __restrict__ rho) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= npts) return;
    const long long g = pts[i];
    double s = 0.0;
    for (int v = 0; v < nvec; ++v) {
        const cd a = psi[(long long)v * ng + g];
        s += a.x * a.x + a.y * a.y;
    }
    rho[g] += scale * s;
}

// phase[g] = exp(-i (vloc[g] + vh[g]) * half_dt)
static __global__ void phase_kernel(const double* __restrict__ vloc, const double* __restrict__ vh, double half_dt,
                                    cd* __restrict__ phase, long long n) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    double v = vloc ? vloc[i] : 0.0;
    if (vh) v += vh[i];
    double s, c;
    sincos(v * half_dt, &s, &c);
    phase[i] = make_double2(c, -s);
}

// Merged half-step phases for consecutive split-operator steps (R-8): the closing factor exp(-i V_{n-1} dt/2) of
// step n-1 and the opening factor exp(-i V_n dt/2) of step n are applied together on load in step n:
//   table[g] = exp(-i (V_n + V_{n-1}) half_dt)   (first step of a call: exp(-i V_n half_dt));   vprev <- V_n
//   last[g]  = exp(-i V_n half_dt)               (only for the last step of a call, applied on store)
// Frozen-potential form (V = V_loc); with the Hartree rebuild the same tables are written by the last pass of the
// Poisson solve (OpPhaseMerge, sgw_ops.cuh).
static __global__ void phase_merge_kernel(const double* __restrict__ vloc, double* __restrict__ vprev,
                                          double half_dt, int first, cd* __restrict__ table, cd* __restrict__ last, long long n) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double v = vloc ? vloc[i] : 0.0;
    double s, c;
    sincos((first ? v : v + vprev[i]) * half_dt, &s, &c);
    table[i] = make_double2(c, -s);
    vprev[i] = v;
    if (last) {
        sincos(v * half_dt, &s, &c);
        last[i] = make_double2(c, -s);
    }
}

static __global__ void scale_kernel(cd* __restrict__ psi, double a, long long n) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) psi[i] = cscale(psi[i], a);
}

// vtab[g] = s * (vloc[g] - Eb)
static __global__ void vtab_kernel(const double* __restrict__ vloc, double s, double Eb, double* __restrict__ vtab,
                                   long long n) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) vtab[i] = s * ((vloc ? vloc[i] : 0.0) - Eb);
}

// out[j] = exp(-i kin[j] dt) / n   (split-operator kinetic factor per axis; 1/n = inverse-transform scale)
static __global__ void td_table_kernel(const double* __restrict__ kin, double dt, cd* __restrict__ out, int n) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    double s, c;
    sincos(kin[i] * dt, &s, &c);
    out[i] = make_double2(c / n, -s / n);
}

static __global__ void scale_table_kernel(const double* __restrict__ in, double s, double* __restrict__ out, int n) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = s * in[i];
}

// ---- norms as segmented sums + one atomic per segment -------------------------------
static __global__ void norms_kernel(const cd* __restrict__ psi, long long ng, double* __restrict__ out) {
    const int v = blockIdx.y;
    const cd* p = psi + (long long)v * ng;
    double s = 0.0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < ng; i += (long long)gridDim.x * blockDim.x) {
        const cd a = p[i];
        s += a.x * a.x + a.y * a.y;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
    __shared__ double part[8];
    if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) t += part[w];
        atomicAdd(out + v, t);
    }
}

// ---- spectral bounds by shifted power iteration (R-20) ------------------------------------
// y -= shift * x;  red[0] += Re<x|y>,  red[1] += |y|^2   (segmented sums + one atomic per block)
static __global__ void power_reduce_kernel(const cd* __restrict__ x, cd* __restrict__ y, double shift, long long n,
                                           double* __restrict__ red) {
    double a = 0.0, b = 0.0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const cd xv = x[i];
        cd yv = y[i];
        yv.x -= shift * xv.x; yv.y -= shift * xv.y;
        y[i] = yv;
        a += xv.x * yv.x + xv.y * yv.y;
        b += yv.x * yv.x + yv.y * yv.y;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        a += __shfl_down_sync(0xffffffffu, a, o);
        b += __shfl_down_sync(0xffffffffu, b, o);
    }
    __shared__ double pa[8], pb[8];
    if ((threadIdx.x & 31) == 0) { pa[threadIdx.x >> 5] = a; pb[threadIdx.x >> 5] = b; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double ta = 0.0, tb = 0.0;
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) { ta += pa[w]; tb += pb[w]; }
        atomicAdd(red, ta);
        atomicAdd(red + 1, tb);
    }
}
// x = y / sqrt(red[1]);  lambda_out[0] = red[0] (Rayleigh quotient of the normalised x);  then red is cleared by the host
static __global__ void power_scale_kernel(cd* __restrict__ x, const cd* __restrict__ y, const double* __restrict__ red,
                                          long long n, double* __restrict__ lambda_out) {
    const double inv = 1.0 / sqrt(red[1]);
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i == 0) lambda_out[0] = red[0];
    if (i < n) x[i] = cscale(y[i], inv);
}

// ---- NEXT-2: perturbed copy and sparse stochastic projection (R-21..R-23) -------------------------
// psi[v][g] *= exp(-i lambda vpert[g])
static __global__ void kick_kernel(cd* __restrict__ psi, const double* __restrict__ vpert, double lambda, long long ng) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= ng) return;
    double s, c;
    sincos(lambda * vpert[i], &s, &c);
    cd* p = psi + (long long)blockIdx.y * ng;
    p[i] = cmul(p[i], make_double2(c, -s));
}

// out[m * stride] = dV * sum over the nfrag fragments of xi_m (32 consecutive grid points each, start 32 * (h(seed, 2m, f)
// mod N_g/32), signs from the top bit of h(seed, 2m+1, 32 f + j)) of sign * field.  One warp per fragment (a coalesced
// 256-byte read), a shuffle sum per segment of L = 32 and one atomic add per segment ("each xi function is
// processed in segments of length L = 32"; one atomic add per segment).  grid (nxi), out zeroed by the caller.
static __global__ void __launch_bounds__(256) xi_project_kernel(const double* __restrict__ field, long long ng, uint64_t seed_mixed, int nfrag,
                                                                 double dV, double* __restrict__ out, int stride) {
    const int m = blockIdx.x, lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
    const uint64_t kpos = sm64(seed_mixed ^ (uint64_t)(2 * m)), ksgn = sm64(seed_mixed ^ (uint64_t)(2 * m + 1));
    const uint64_t nblocks = (uint64_t)(ng / 32);
    for (int f = warp; f < nfrag; f += nwarps) {
        const uint64_t b = sm64(kpos ^ (uint64_t)f) % nblocks;
        const double sg = (sm64(ksgn ^ ((uint64_t)f * 32 + lane)) >> 63) ? -1.0 : 1.0;
        double a = sg * field[b * 32 + lane];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) a += __shfl_down_sync(0xffffffffu, a, o);
        if (lane == 0) atomicAdd(out + (long long)m * stride, a * dV);
    }
}

// ---- NEXT-4: zeta-pair projections, time-ordering, Sigma(t) (R-24..R-26) ----------------------
// out[m * stride] = dV * sum over xi_m's fragments of sign * phi(point) * psi(point): the complex, phi-weighted form of
// xi_project_kernel (same xi, same segments of L = 32, one atomic pair per segment).  grid (nxi), out zeroed by the caller.
static __global__ void __launch_bounds__(256) xi_project_weighted_kernel(const cd* __restrict__ psi, const double* __restrict__ phi, long long ng,
                                                                          uint64_t seed_mixed, int nfrag, double dV, cd* __restrict__ out,
                                                                          int stride) {
    const int m = blockIdx.x, lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
    const uint64_t kpos = sm64(seed_mixed ^ (uint64_t)(2 * m)), ksgn = sm64(seed_mixed ^ (uint64_t)(2 * m + 1));
    const uint64_t nblocks = (uint64_t)(ng / 32);
    for (int f = warp; f < nfrag; f += nwarps) {
        const uint64_t b = sm64(kpos ^ (uint64_t)f) % nblocks;
        const double sg = (sm64(ksgn ^ ((uint64_t)f * 32 + lane)) >> 63) ? -1.0 : 1.0;
        const long long i = (long long)(b * 32 + lane);
        const cd z = psi[i];
        const double w = sg * phi[i];
        double ar = w * z.x, ai = w * z.y;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) { ar += __shfl_down_sync(0xffffffffu, ar, o); ai += __shfl_down_sync(0xffffffffu, ai, o); }
        if (lane == 0) {
            double* dst = reinterpret_cast<double*>(out + (long long)m * stride);
            atomicAdd(dst, ar * dV);
            atomicAdd(dst + 1, ai * dV);
        }
    }
}

// Time-ordering of one coefficient series per block (R-24): C(w_k) = sum_n c(t_n) e^{+2 pi i k n / M} on the zero-padded
// series (M = 2 nt), conjugate for k < 0, c^T(t_n) = (1/M) sum_k C^T(w_k) e^{-2 pi i k n / M}.  Direct sums with exactly
// reduced angles (nt is N_tau ~ 1000 in the paper, not an FFT-friendly length; the step is a vanishing share of the
// work: P:104).  dynamic shared memory: nt doubles + M complex.
static __global__ void time_order_kernel(const double* __restrict__ cr, long long stride_n, long long stride_m, int nt, int nxi,
                                         cd* __restrict__ ct) {
    extern __shared__ double tsm[];
    const int m = blockIdx.x, M = 2 * nt;
    double* c = tsm;
    cd* Cw = reinterpret_cast<cd*>(tsm + nt + (nt & 1));
    for (int n = threadIdx.x; n < nt; n += blockDim.x) c[n] = cr[n * stride_n + m * stride_m];
    __syncthreads();
    for (int kk = threadIdx.x; kk < M; kk += blockDim.x) {
        const int k = kk - M / 2;
        double re = 0.0, im = 0.0;
        for (int n = 0; n < nt; ++n) {
            long long r = ((long long)k * n) % M;
            if (r < 0) r += M;
            double s, co;
            sincospi(2.0 * (double)r / (double)M, &s, &co);
            re += c[n] * co; im += c[n] * s;
        }
        Cw[kk] = make_double2(re, k < 0 ? -im : im);
    }
    __syncthreads();
    for (int n = threadIdx.x; n < nt; n += blockDim.x) {
        double re = 0.0, im = 0.0;
        for (int kk = 0; kk < M; ++kk) {
            const int k = kk - M / 2;
            long long r = ((long long)k * n) % M;
            if (r < 0) r += M;
            double s, co;
            sincospi(-2.0 * (double)r / (double)M, &s, &co);
            const cd z = Cw[kk];
            re += z.x * co - z.y * s; im += z.x * s + z.y * co;
        }
        ct[(long long)n * nxi + m] = make_double2(re / M, im / M);
    }
}

// sigma[n][k] = norm * sum_m ct[n][m] * p[n][m][k]   (Eq. 5 in the xi basis, R-26); grid (nt), one block per time
static __global__ void sigma_kernel(const cd* __restrict__ ct, const cd* __restrict__ p, int nxi, double norm, cd* __restrict__ sigma) {
    const int n = blockIdx.x;
    double a[4] = {0.0, 0.0, 0.0, 0.0};
    for (int m = threadIdx.x; m < nxi; m += blockDim.x) {
        const cd c = ct[(long long)n * nxi + m];
#pragma unroll
        for (int k = 0; k < 2; ++k) {
            const cd z = p[((long long)n * nxi + m) * 2 + k];
            a[2 * k] += c.x * z.x - c.y * z.y;
            a[2 * k + 1] += c.x * z.y + c.y * z.x;
        }
    }
    __shared__ double red[8][4];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) a[q] += __shfl_down_sync(0xffffffffu, a[q], o);
        if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5][q] = a[q];
    }
    __syncthreads();
    if (threadIdx.x < 4) {
        double t = 0.0;
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) t += red[w][threadIdx.x];
        reinterpret_cast<double*>(sigma + (long long)n * 2)[threadIdx.x] = t * norm;
    }
}

// ---- a6: Kleinman-Bylander gather-dot (R-12) --------------------------------------------
// grid (nsphere, ceil(nvec / KB_VB)), 128 threads: c[v][s][p] = dV * sum_j beta[j][p] * psi_v[idx[j]].  A block takes
// KB_VB vectors of one sphere: the point list, the projector values and (propagator) the phases are read once for all
// of them.
constexpr int KB_VB = 4;

template <int NP>
static __global__ void __launch_bounds__(128) kb_project_kernel(const cd* __restrict__ psi, long long ng, int nvec,
                                                                 const int64_t* __restrict__ ptr,
                                                                 const int32_t* __restrict__ idx,
                                                                 const double* __restrict__ beta, double dV,
                                                                 cd* __restrict__ cout, int nsphere,
                                                                 const cd* __restrict__ phase = nullptr, int phase_conj = 0) {
    const int s = blockIdx.x, v0 = blockIdx.y * KB_VB;
    const int nv = nvec - v0 < KB_VB ? nvec - v0 : KB_VB;
    const cd* p = psi + (long long)v0 * ng;
    double ar[KB_VB][NP], ai[KB_VB][NP];
#pragma unroll
    for (int u = 0; u < KB_VB; ++u)
#pragma unroll
        for (int q = 0; q < NP; ++q) ar[u][q] = ai[u][q] = 0.0;
    for (int64_t j = ptr[s] + threadIdx.x; j < ptr[s + 1]; j += blockDim.x) {
        const long long g = idx[j];
        double b[NP];
#pragma unroll
        for (int q = 0; q < NP; ++q) b[q] = beta[j * NP + q];
        cd ph = make_double2(1.0, 0.0);
        if (phase) ph = phase[g];  // the projections are those of phase * psi (or conj(phase) * psi): see sgw_td_propagate
#pragma unroll
        for (int u = 0; u < KB_VB; ++u) {
            if (u < nv) {
                cd a = p[(long long)u * ng + g];
                if (phase) a = phase_conj ? cmulc(a, ph) : cmul(a, ph);
#pragma unroll
                for (int q = 0; q < NP; ++q) {
                    ar[u][q] += b[q] * a.x;
                    ai[u][q] += b[q] * a.y;
                }
            }
        }
    }
    __shared__ double red[4][KB_VB][2 * NP];
#pragma unroll
    for (int u = 0; u < KB_VB; ++u)
#pragma unroll
        for (int q = 0; q < NP; ++q) {
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                ar[u][q] += __shfl_down_sync(0xffffffffu, ar[u][q], o);
                ai[u][q] += __shfl_down_sync(0xffffffffu, ai[u][q], o);
            }
            if ((threadIdx.x & 31) == 0) { red[threadIdx.x >> 5][u][2 * q] = ar[u][q]; red[threadIdx.x >> 5][u][2 * q + 1] = ai[u][q]; }
        }
    __syncthreads();
    if (threadIdx.x < KB_VB * NP) {
        const int u = threadIdx.x / NP, q = threadIdx.x % NP;
        if (u < nv) {
            double re = 0.0, im = 0.0;
            for (int w = 0; w < 4; ++w) { re += red[w][u][2 * q]; im += red[w][u][2 * q + 1]; }
            cout[((long long)(v0 + u) * nsphere + s) * NP + q] = make_double2(re * dV, im * dV);
        }
    }
}

// scatter: dst_v[idx[j]] += sum_p beta[j][p] * f_p * c[v][s][p], atomics where spheres overlap
//   mode 0: f_p = scale * D[s][p]                         (H apply / Chebyshev term)
//   mode 1: f_p = exp(-i D[s][p] tau) - 1                 (propagator factor NL(tau), R-11)
template <int NP>
static __global__ void __launch_bounds__(128) kb_scatter_kernel(cd* __restrict__ dst, long long ng, int nvec,
                                                                 const int64_t* __restrict__ ptr,
                                                                 const int32_t* __restrict__ idx,
                                                                 const double* __restrict__ beta,
                                                                 const double* __restrict__ D,
                                                                 const cd* __restrict__ cin, int nsphere, int mode,
                                                                 double scale_or_tau, const cd* __restrict__ phase = nullptr,
                                                                 int phase_conj = 0) {
    const int s = blockIdx.x, v0 = blockIdx.y * KB_VB;
    const int nv = nvec - v0 < KB_VB ? nvec - v0 : KB_VB;
    __shared__ cd f[KB_VB][NP];
    if (threadIdx.x < KB_VB * NP) {
        const int u = threadIdx.x / NP, q = threadIdx.x % NP;
        if (u < nv) {
            const cd c = cin[((long long)(v0 + u) * nsphere + s) * NP + q];
            const double d = D[s * NP + q];
            if (mode == 0) f[u][q] = cscale(c, scale_or_tau * d);
            else {
                double sn, cs;
                sincos(d * scale_or_tau, &sn, &cs);
                f[u][q] = cmul(make_double2(cs - 1.0, -sn), c);
            }
        }
    }
    __syncthreads();
    for (int64_t j = ptr[s] + threadIdx.x; j < ptr[s + 1]; j += blockDim.x) {
        const long long g = idx[j];
        double b[NP];
#pragma unroll
        for (int q = 0; q < NP; ++q) b[q] = beta[j * NP + q];
        cd ph = make_double2(1.0, 0.0);
        if (phase) ph = phase[g];  // the contribution is added to phase^-1 * (...) or phase * (...): |phase| = 1
#pragma unroll
        for (int u = 0; u < KB_VB; ++u) {
            if (u < nv) {
                double re = 0.0, im = 0.0;
#pragma unroll
                for (int q = 0; q < NP; ++q) {
                    re += b[q] * f[u][q].x;
                    im += b[q] * f[u][q].y;
                }
                if (phase) {
                    const cd t = phase_conj ? cmulc(make_double2(re, im), ph) : cmul(make_double2(re, im), ph);
                    re = t.x; im = t.y;
                }
                double* out = reinterpret_cast<double*>(dst + (long long)(v0 + u) * ng);
                atomicAdd(out + 2 * g, re);
                atomicAdd(out + 2 * g + 1, im);
            }
        }
    }
}

}  // namespace sgw
