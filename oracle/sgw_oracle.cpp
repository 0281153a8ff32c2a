// sgw_oracle.cpp -- plain, slow CPU oracle for the sGW hot path.  TEST INFRASTRUCTURE ONLY.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
// load this.  It shares no code with the CUDA path (paper_2601_21005_b200/csrc) and imports
// nothing from it.  Every function follows a passage of /root/reference/PAPER.md ("P:NN") or a
// reading listed in DESIGN.md ("R-n", taken from SURVEY.md section 8(c)).
//
// What it computes ("Fourier grid representation ... FFT pairs switch between position and
// momentum representations where the potential energy and kinetic energy operators are
// diagonal"):
//   H psi = F^-1[ 1/2 |k|^2 F[psi] ] + V_loc psi + sum_{s,p} |beta_sp> D_sp dV <beta_sp|psi>
//   Chebyshev series (Eq. 3)  out = sum_{n<nterms} a_n T_n(Ht) v,  Ht = (H - Eb)/dE
//   split-operator step with time-dependent Hartree
//   Hartree potential by FFT Poisson solve with a spherically cut Coulomb kernel (R-10)
//   +-1 white-noise vectors from a splitmix64 keyed hash (R-4, R-5)
//
// Layout: vectors [nvec][nz][ny][nx], x fastest, complex interleaved (re,im) doubles.
// Arithmetic: template parameter T = double (the timed baseline) or long double (the parity
// reference); inputs and outputs are always double.  Compile with -ffp-contract=off (R-17).
// OpenMP over vectors only.
//
// Pins (tests/test_oracle_*.py): splitmix64 published stream; FFT vs O(N^2) DFT and numpy.fft;
// plane-wave eigenvalues; dense-H built independently with numpy; eigh brute force; Hartree erf
// closed form; TD closed forms and order-2 convergence; TD-Hartree energy drift proportional to dt; overlapping KB
// spheres converge to the dense propagator; power-iteration bounds vs dense eigenvalues.  "parity unpinned": config-level
// outputs; the TD-Hartree trajectory and the KB factor NL(tau) inside the propagator are pinned to first order in the
// step only (sign, scale, per-step rebuild), their O(tau^2) terms are defined by the algorithm below (R-8, R-9, R-11).
#include <cmath>
#include <complex>
#include <cstdint>
#include <cstring>
#include <vector>

namespace {

template <class T> using C = std::complex<T>;

template <class T> inline T pi_v() { return std::acos((T)-1); }

// ---------------------------------------------------------------------------------------------
// RNG (R-5): key = sm64(sm64(seed) ^ vec); h = sm64(key ^ g); value = top bit ? -1 : +1
// ---------------------------------------------------------------------------------------------
inline uint64_t sm64(uint64_t x) {
    x += 0x9E3779B97F4A7C15ULL;
    x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ULL;
    x = (x ^ (x >> 27)) * 0x94D049BB133111EBULL;
    return x ^ (x >> 31);
}
inline uint64_t keyed_hash(uint64_t seed, uint64_t vec, uint64_t g) {
    uint64_t key = sm64(sm64(seed) ^ vec);
    return sm64(key ^ g);
}

// ---------------------------------------------------------------------------------------------
// 1D DFT, textbook recursive decimation in time over the smallest prime factor.
//   X[k] = sum_n x[n] w^(n k),  w = exp(sign * 2 pi i / N)
// tw[j] = exp(sign*2*pi*i*j/N) for j < N, each evaluated directly with cos/sin.
// ---------------------------------------------------------------------------------------------
template <class T>
void make_twiddles(int N, int sign, std::vector<C<T>>& tw) {
    tw.resize(N);
    for (int j = 0; j < N; ++j) {
        T a = (T)sign * (T)2 * pi_v<T>() * (T)j / (T)N;
        tw[j] = C<T>(std::cos(a), std::sin(a));
    }
}

inline int smallest_factor(int n) {
    for (int p = 2; p * p <= n; ++p)
        if (n % p == 0) return p;
    return n;
}

// in: n elements at stride `is`; out: n contiguous.  tw has N entries, ts = N/n.
template <class T>
void dft_rec(int n, const C<T>* in, int is, C<T>* out, const C<T>* tw, int N, int ts) {
    if (n == 1) { out[0] = in[0]; return; }
    const int p = smallest_factor(n), m = n / p;
    for (int r = 0; r < p; ++r) dft_rec(m, in + (size_t)r * is, is * p, out + (size_t)r * m, tw, N, ts * p);
    C<T> ysmall[8];
    std::vector<C<T>> ybig;
    C<T>* y = ysmall;
    if (p > 8) { ybig.resize(p); y = ybig.data(); }
    for (int k = 0; k < m; ++k) {
        for (int r = 0; r < p; ++r) y[r] = out[r * m + k] * tw[((long)r * k * ts) % N];
        for (int q = 0; q < p; ++q) {
            C<T> s(0, 0);
            for (int r = 0; r < p; ++r) s += y[r] * tw[((long)r * q * m * ts) % N];
            out[q * m + k] = s;   // safe: y holds the inputs of this k; slots q*m+k are only read for this k
        }
    }
}

template <class T>
void fft1d(int N, int sign, const C<T>* in, int is, C<T>* out, const std::vector<C<T>>& tw) {
    dft_rec<T>(N, in, is, out, tw.data(), N, 1);
    (void)sign;
}

// 3D transform, unnormalised, in place on a[nz][ny][nx]; sign -1 = forward e^{-ik.r} (R: a2).
template <class T>
void fft3(int nx, int ny, int nz, int sign, C<T>* a) {
    std::vector<C<T>> tw, buf, line;
    const int dims[3] = {nx, ny, nz};
    const size_t strides[3] = {1, (size_t)nx, (size_t)nx * ny};
    for (int ax = 0; ax < 3; ++ax) {
        const int N = dims[ax];
        make_twiddles<T>(N, sign, tw);
        buf.resize(N);
        line.resize(N);
        const int a1 = (ax + 1) % 3, a2 = (ax + 2) % 3;
        for (int i2 = 0; i2 < dims[a2]; ++i2)
            for (int i1 = 0; i1 < dims[a1]; ++i1) {
                C<T>* base = a + i1 * strides[a1] + i2 * strides[a2];
                for (int j = 0; j < N; ++j) line[j] = base[j * strides[ax]];
                fft1d<T>(N, sign, line.data(), 1, buf.data(), tw);
                for (int j = 0; j < N; ++j) base[j * strides[ax]] = buf[j];
            }
    }
}

// k_i = 2 pi m / (N h), m in [-N/2, N/2)  (R: a3).  Index j >= N/2 (N even) or > (N-1)/2 maps to j-N.
template <class T>
void kvals(int N, double h, std::vector<T>& k) {
    k.resize(N);
    for (int j = 0; j < N; ++j) {
        int m = (2 * j >= N) ? j - N : j;     // for even N the Nyquist index N/2 -> -N/2
        k[j] = (T)2 * pi_v<T>() * (T)m / ((T)N * (T)h);
    }
}

struct Grid { int nx, ny, nz; double hx, hy, hz; };

// Kinetic-energy cutoff ("apply an energy cutoff of 28 Hartrees to the kinetic energy operator"; a cutoff
// bounds the spectral width and with it N_chb; R-14): when g_ecut > 0 the kinetic operator is diagonal in k
// with values min(1/2 |k|^2, E_cut) instead of 1/2 |k|^2, in H and in the propagator.  0 = no cutoff (the configs).
double g_ecut = 0.0;
template <class T>
inline T kinetic(T k2) {
    const T t = (T)0.5 * k2;
    return (g_ecut > 0.0 && t > (T)g_ecut) ? (T)g_ecut : t;
}
struct KBList {
    int nsphere, nproj;
    const int64_t* ptr; const int32_t* idx; const double* beta; const double* D;
};

// ---------------------------------------------------------------------------------------------
// H apply on one vector (SURVEY 8(c) "applyH")
// ---------------------------------------------------------------------------------------------
template <class T>
void apply_H_one(const Grid& g, const double* vloc, const KBList& kb, const C<T>* psi, C<T>* out) {
    const size_t ng = (size_t)g.nx * g.ny * g.nz;
    std::vector<T> kx, ky, kz;
    kvals<T>(g.nx, g.hx, kx); kvals<T>(g.ny, g.hy, ky); kvals<T>(g.nz, g.hz, kz);
    std::vector<C<T>> t(psi, psi + ng);
    fft3<T>(g.nx, g.ny, g.nz, -1, t.data());
    for (int iz = 0; iz < g.nz; ++iz)
        for (int iy = 0; iy < g.ny; ++iy)
            for (int ix = 0; ix < g.nx; ++ix) {
                T k2 = kx[ix] * kx[ix] + ky[iy] * ky[iy] + kz[iz] * kz[iz];
                t[ix + (size_t)g.nx * (iy + (size_t)g.ny * iz)] *= kinetic<T>(k2);
            }
    fft3<T>(g.nx, g.ny, g.nz, +1, t.data());
    const T inv = (T)1 / (T)ng;
    for (size_t i = 0; i < ng; ++i) out[i] = t[i] * inv;
    if (vloc)
        for (size_t i = 0; i < ng; ++i) out[i] += (T)vloc[i] * psi[i];
    const T dV = (T)g.hx * (T)g.hy * (T)g.hz;
    for (int s = 0; s < kb.nsphere; ++s)
        for (int p = 0; p < kb.nproj; ++p) {
            C<T> c(0, 0);
            for (int64_t j = kb.ptr[s]; j < kb.ptr[s + 1]; ++j)
                c += (T)kb.beta[j * kb.nproj + p] * psi[kb.idx[j]];
            c *= dV;
            const T D = (T)kb.D[s * kb.nproj + p];
            for (int64_t j = kb.ptr[s]; j < kb.ptr[s + 1]; ++j)
                out[kb.idx[j]] += (T)kb.beta[j * kb.nproj + p] * D * c;
        }
}

template <class T>
void load_vec(const double* src, size_t ng, std::vector<C<T>>& v) {
    v.resize(ng);
    for (size_t i = 0; i < ng; ++i) v[i] = C<T>((T)src[2 * i], (T)src[2 * i + 1]);
}
template <class T>
void store_vec(const std::vector<C<T>>& v, double* dst) {
    for (size_t i = 0; i < v.size(); ++i) { dst[2 * i] = (double)v[i].real(); dst[2 * i + 1] = (double)v[i].imag(); }
}

template <class T>
void apply_H_batch(const Grid& g, const double* vloc, const KBList& kb, int nvec, const double* in, double* out) {
    const size_t ng = (size_t)g.nx * g.ny * g.nz;
#pragma omp parallel for schedule(dynamic)
    for (int v = 0; v < nvec; ++v) {
        std::vector<C<T>> a, b(ng);
        load_vec<T>(in + 2 * ng * v, ng, a);
        apply_H_one<T>(g, vloc, kb, a.data(), b.data());
        store_vec<T>(b, out + 2 * ng * v);
    }
}

// ---------------------------------------------------------------------------------------------
// Chebyshev filter (Eq. 3; R-1: nterms coefficients, degrees 0..nterms-1)
// ---------------------------------------------------------------------------------------------
template <class T>
void cheb_batch(const Grid& g, const double* vloc, const KBList& kb, int nvec, double* psi,
                const double* coeffs, double Emin, double Emax, int nterms) {
    const size_t ng = (size_t)g.nx * g.ny * g.nz;
    const T Eb = ((T)Emax + (T)Emin) / (T)2, dE = ((T)Emax - (T)Emin) / (T)2;
#pragma omp parallel for schedule(dynamic)
    for (int v = 0; v < nvec; ++v) {
        std::vector<C<T>> p0, p1(ng), p2(ng), out(ng), h(ng);
        load_vec<T>(psi + 2 * ng * v, ng, p0);
        for (size_t i = 0; i < ng; ++i) out[i] = (T)coeffs[0] * p0[i];
        if (nterms > 1) {
            apply_H_one<T>(g, vloc, kb, p0.data(), h.data());
            for (size_t i = 0; i < ng; ++i) p1[i] = (h[i] - Eb * p0[i]) / dE;
            for (size_t i = 0; i < ng; ++i) out[i] += (T)coeffs[1] * p1[i];
        }
        for (int n = 2; n < nterms; ++n) {
            apply_H_one<T>(g, vloc, kb, p1.data(), h.data());
            for (size_t i = 0; i < ng; ++i) p2[i] = (T)2 * ((h[i] - Eb * p1[i]) / dE) - p0[i];
            for (size_t i = 0; i < ng; ++i) out[i] += (T)coeffs[n] * p2[i];
            p0.swap(p1);
            p1.swap(p2);
        }
        store_vec<T>(out, psi + 2 * ng * v);
    }
}

// ---------------------------------------------------------------------------------------------
// Hartree (R-9, R-10): rho = rho_scale sum_l |psi_l|^2;  V_H = Re F^-1[ v(k) F[rho] ],
// v(k) = 4 pi (1 - cos(|k| Rc)) / |k|^2, v(0) = 2 pi Rc^2, Rc = min(Lx,Ly,Lz)/2
// ---------------------------------------------------------------------------------------------
template <class T>
void density(const Grid& g, int nvec, const double* psi, double rho_scale, std::vector<T>& rho) {
    const size_t ng = (size_t)g.nx * g.ny * g.nz;
    rho.assign(ng, (T)0);
    for (int v = 0; v < nvec; ++v)
        for (size_t i = 0; i < ng; ++i) {
            T re = (T)psi[2 * (ng * v + i)], im = (T)psi[2 * (ng * v + i) + 1];
            rho[i] += re * re + im * im;
        }
    for (size_t i = 0; i < ng; ++i) rho[i] *= (T)rho_scale;
}

template <class T>
void poisson(const Grid& g, const std::vector<T>& rho, std::vector<T>& vh) {
    const size_t ng = (size_t)g.nx * g.ny * g.nz;
    std::vector<T> kx, ky, kz;
    kvals<T>(g.nx, g.hx, kx); kvals<T>(g.ny, g.hy, ky); kvals<T>(g.nz, g.hz, kz);
    T Lmin = std::fmin((T)g.nx * (T)g.hx, std::fmin((T)g.ny * (T)g.hy, (T)g.nz * (T)g.hz));
    const T Rc = Lmin / (T)2;
    std::vector<C<T>> t(ng);
    for (size_t i = 0; i < ng; ++i) t[i] = C<T>(rho[i], 0);
    fft3<T>(g.nx, g.ny, g.nz, -1, t.data());
    for (int iz = 0; iz < g.nz; ++iz)
        for (int iy = 0; iy < g.ny; ++iy)
            for (int ix = 0; ix < g.nx; ++ix) {
                T k2 = kx[ix] * kx[ix] + ky[iy] * ky[iy] + kz[iz] * kz[iz];
                T vk = (k2 == (T)0) ? (T)2 * pi_v<T>() * Rc * Rc
                                    : (T)4 * pi_v<T>() * ((T)1 - std::cos(std::sqrt(k2) * Rc)) / k2;
                t[ix + (size_t)g.nx * (iy + (size_t)g.ny * iz)] *= vk;
            }
    fft3<T>(g.nx, g.ny, g.nz, +1, t.data());
    vh.resize(ng);
    for (size_t i = 0; i < ng; ++i) vh[i] = t[i].real() / (T)ng;
}

// ---------------------------------------------------------------------------------------------
// split-operator propagation (R-8, R-9, R-11):
//   V = V_loc + (mode ? V_H[rho(psi_n)] : 0), frozen over the step
//   psi <- e^{-iV dt/2} NL(dt/2) F^-1 e^{-i k^2 dt/2} F NL(dt/2) e^{-iV dt/2} psi
//   NL(tau): psi[idx] += sum_p beta (e^{-i D tau} - 1) c_sp, all c_sp = dV <beta_sp|psi> from the SAME input
// ---------------------------------------------------------------------------------------------
template <class T>
void nl_phase(const Grid& g, const KBList& kb, T tau, std::vector<C<T>>& psi) {
    if (kb.nsphere == 0) return;
    const T dV = (T)g.hx * (T)g.hy * (T)g.hz;
    std::vector<C<T>> c((size_t)kb.nsphere * kb.nproj);
    for (int s = 0; s < kb.nsphere; ++s)
        for (int p = 0; p < kb.nproj; ++p) {
            C<T> a(0, 0);
            for (int64_t j = kb.ptr[s]; j < kb.ptr[s + 1]; ++j) a += (T)kb.beta[j * kb.nproj + p] * psi[kb.idx[j]];
            c[(size_t)s * kb.nproj + p] = a * dV;
        }
    for (int s = 0; s < kb.nsphere; ++s)
        for (int p = 0; p < kb.nproj; ++p) {
            const T D = (T)kb.D[s * kb.nproj + p];
            const C<T> f = C<T>(std::cos(D * tau) - (T)1, -std::sin(D * tau)) * c[(size_t)s * kb.nproj + p];
            for (int64_t j = kb.ptr[s]; j < kb.ptr[s + 1]; ++j) psi[kb.idx[j]] += (T)kb.beta[j * kb.nproj + p] * f;
        }
}

template <class T>
void td_batch(const Grid& g, const double* vloc, const KBList& kb, int nvec, double* psi, double dt,
              int nsteps, int hartree_mode, double rho_scale) {
    const size_t ng = (size_t)g.nx * g.ny * g.nz;
    std::vector<T> kx, ky, kz;
    kvals<T>(g.nx, g.hx, kx); kvals<T>(g.ny, g.hy, ky); kvals<T>(g.nz, g.hz, kz);
    std::vector<T> rho, vh, V(ng);
    for (int step = 0; step < nsteps; ++step) {
        for (size_t i = 0; i < ng; ++i) V[i] = vloc ? (T)vloc[i] : (T)0;
        if (hartree_mode) {
            density<T>(g, nvec, psi, rho_scale, rho);
            poisson<T>(g, rho, vh);
            for (size_t i = 0; i < ng; ++i) V[i] += vh[i];
        }
#pragma omp parallel for schedule(dynamic)
        for (int v = 0; v < nvec; ++v) {
            std::vector<C<T>> a;
            load_vec<T>(psi + 2 * ng * v, ng, a);
            const T half = (T)dt / (T)2;
            for (size_t i = 0; i < ng; ++i) a[i] *= C<T>(std::cos(V[i] * half), -std::sin(V[i] * half));
            nl_phase<T>(g, kb, half, a);
            fft3<T>(g.nx, g.ny, g.nz, -1, a.data());
            for (int iz = 0; iz < g.nz; ++iz)
                for (int iy = 0; iy < g.ny; ++iy)
                    for (int ix = 0; ix < g.nx; ++ix) {
                        T ph = kinetic<T>(kx[ix] * kx[ix] + ky[iy] * ky[iy] + kz[iz] * kz[iz]) * (T)dt;
                        a[ix + (size_t)g.nx * (iy + (size_t)g.ny * iz)] *= C<T>(std::cos(ph), -std::sin(ph));
                    }
            fft3<T>(g.nx, g.ny, g.nz, +1, a.data());
            for (size_t i = 0; i < ng; ++i) a[i] /= (T)ng;
            nl_phase<T>(g, kb, half, a);
            for (size_t i = 0; i < ng; ++i) a[i] *= C<T>(std::cos(V[i] * half), -std::sin(V[i] * half));
            store_vec<T>(a, psi + 2 * ng * v);
        }
    }
}

// ---------------------------------------------------------------------------------------------
// NEXT-2: perturbed / unperturbed pair propagation and the sparse stochastic projection of the retarded response
// ("create a perturbed copy of each eta (eta^lambda) and propagate both perturbed and unperturbed copies in time
// under the action of the time-dependent Hamiltonian ... accumulate the causal response function u^R(r,t) as the
// difference of the perturbed and unperturbed time-dependent potentials"; "projecting u^R(r,t) onto a set of N_xi
// randomly chosen functions xi on short, fragmented segments of the spatial grid"; "(N_xi x N_g f_g) and
// (N_g f_g x 2) ... each xi function is processed in segments of length L = 32").  Readings R-21..R-23:
//   * the caller supplies both copies (the perturbed one is exp(-i lambda v_pert(r)) eta, sgwo_apply_kick);
//   * each copy is propagated with the split-operator step of td_batch under ITS OWN Hartree potential
//     V_loc + V_H[rho_copy(t_n)];
//   * xi_m (m < nxi) lives on nfrag fragments of L = 32 consecutive grid points; fragment f starts at grid index
//     32 * (h(seed, 2m, f) mod (N_g / 32)) and carries the signs (top bit of h(seed, 2m+1, 32 f + j) ? -1 : +1);
//   * at the start of step n: out[n][m][copy] = dV * sum_{f,j} sign * V_H[rho_copy(t_n)](point), copy 0 = unperturbed,
//     1 = perturbed; the coefficients of u^R are (out[..][1] - out[..][0]) / lambda.
// ---------------------------------------------------------------------------------------------
constexpr int XI_L = 32;

template <class T>
void xi_project(const Grid& g, const std::vector<T>& field, uint64_t seed, int nxi, int nfrag, double* out, int stride) {
    const size_t ng = (size_t)g.nx * g.ny * g.nz;
    const uint64_t nblocks = ng / XI_L;
    const T dV = (T)g.hx * (T)g.hy * (T)g.hz;
    for (int m = 0; m < nxi; ++m) {
        T acc = 0;
        for (int f = 0; f < nfrag; ++f) {
            const uint64_t b = keyed_hash(seed, 2 * (uint64_t)m, (uint64_t)f) % nblocks;
            for (int j = 0; j < XI_L; ++j) {
                const T sg = (keyed_hash(seed, 2 * (uint64_t)m + 1, (uint64_t)f * XI_L + j) >> 63) ? (T)-1 : (T)1;
                acc += sg * field[b * XI_L + j];
            }
        }
        out[(size_t)m * stride] = (double)(acc * dV);
    }
}

template <class T>
void td_pair(const Grid& g, const double* vloc, const KBList& kb, int nvec, double* psi, double* psi_lam, double dt, int nsteps,
             double rho_scale, uint64_t xi_seed, int nxi, int nfrag, double* out) {
    std::vector<T> rho, vh;
    for (int n = 0; n < nsteps; ++n) {
        for (int copy = 0; copy < 2; ++copy) {
            density<T>(g, nvec, copy ? psi_lam : psi, rho_scale, rho);
            poisson<T>(g, rho, vh);
            xi_project<T>(g, vh, xi_seed, nxi, nfrag, out + ((size_t)n * nxi) * 2 + copy, 2);
        }
        td_batch<T>(g, vloc, kb, nvec, psi, dt, 1, 1, rho_scale);
        td_batch<T>(g, vloc, kb, nvec, psi_lam, dt, 1, 1, rho_scale);
    }
}

// ---------------------------------------------------------------------------------------------
// NEXT-4: time-ordering of the retarded response, and the zeta pair with its sparse projections
// ("we time-order the accumulated u^R(r,t) to produce the effective polarization potential u(r,t)"; "calling
// the cuFFT library before and after an OpenACC kernel used for performing the complex conjugation step"; Eq. 4:
// "propagating the filtered zeta backwards in time while simultaneously propagating its orthogonal complement forwards in
// time"; "(N_g x 2)"; Eq. 5: <phi|Sigma(t)|phi> = (1/N_zeta) sum_zeta int phi(r) zeta(r,t) u(r,t) dr).
// Readings R-24..R-26:
//   * time-ordering acts on each coefficient series c^R(t_n), n < nt (real, causal: zero for t < 0), zero-padded to
//     M = 2 nt samples: C(w_k) = sum_n c^R(t_n) e^{+i w_k t_n}, w_k = 2 pi k / (M dt), k = -M/2 .. M/2-1;
//     C^T(w) = Re C(w) + i sgn(w) Im C(w) (= C(w) for w >= 0 and its conjugate for w < 0: the conjugation step);
//     c^T(t_n) = (1/M) sum_k C^T(w_k) e^{-i w_k t_n}, n < nt;
//   * the pair (psi_0 = filtered zeta, psi_1 = its complement) is propagated with the split-operator step under the
//     frozen potential V_loc, psi_0 with -dt and psi_1 with +dt; at the start of step n the projections
//     p[n][m][k] = dV sum_{f,j} sign * phi(point) * psi_k(point, t_n) onto the same xi_m as in td_pair are recorded;
//   * Sigma(t_n) then is (N_g / (N_xi nfrag 32 dV)) sum_m c^T_m(t_n) p[n][m][k] (resolution of the identity in the xi
//     basis), a contraction the tests do with numpy.
// ---------------------------------------------------------------------------------------------
template <class T>
void time_order(int nxi, int nt, const double* cr, int cr_stride_n, int cr_stride_m, double* ct) {
    const int M = 2 * nt;
    std::vector<C<T>> Cw(M);
    for (int m = 0; m < nxi; ++m) {
        for (int kk = 0; kk < M; ++kk) {
            const int k = kk - M / 2;
            C<T> acc(0, 0);
            for (int n = 0; n < nt; ++n) {
                const T ang = (T)2 * pi_v<T>() * (T)(((long long)k * n) % M) / (T)M;
                acc += (T)cr[(size_t)n * cr_stride_n + (size_t)m * cr_stride_m] * C<T>(std::cos(ang), std::sin(ang));
            }
            Cw[kk] = k < 0 ? std::conj(acc) : acc;          // Re C + i sgn(w) Im C
        }
        for (int n = 0; n < nt; ++n) {
            C<T> acc(0, 0);
            for (int kk = 0; kk < M; ++kk) {
                const int k = kk - M / 2;
                const T ang = -(T)2 * pi_v<T>() * (T)(((long long)k * n) % M) / (T)M;
                acc += Cw[kk] * C<T>(std::cos(ang), std::sin(ang));
            }
            ct[2 * ((size_t)n * nxi + m)] = (double)(acc.real() / (T)M);
            ct[2 * ((size_t)n * nxi + m) + 1] = (double)(acc.imag() / (T)M);
        }
    }
}

template <class T>
void td_zeta(const Grid& g, const double* vloc, const KBList& kb, double* pair, const double* phi, double dt, int nsteps,
             uint64_t xi_seed, int nxi, int nfrag, double* out) {
    const size_t ng = (size_t)g.nx * g.ny * g.nz;
    const uint64_t nblocks = ng / XI_L;
    const T dV = (T)g.hx * (T)g.hy * (T)g.hz;
    for (int n = 0; n < nsteps; ++n) {
        for (int k = 0; k < 2; ++k) {
            const double* psi = pair + 2 * ng * k;
            for (int m = 0; m < nxi; ++m) {
                C<T> acc(0, 0);
                for (int f = 0; f < nfrag; ++f) {
                    const uint64_t b = keyed_hash(xi_seed, 2 * (uint64_t)m, (uint64_t)f) % nblocks;
                    for (int j = 0; j < XI_L; ++j) {
                        const T sg = (keyed_hash(xi_seed, 2 * (uint64_t)m + 1, (uint64_t)f * XI_L + j) >> 63) ? (T)-1 : (T)1;
                        const size_t i = b * XI_L + j;
                        acc += sg * (T)phi[i] * C<T>((T)psi[2 * i], (T)psi[2 * i + 1]);
                    }
                }
                out[2 * (((size_t)n * nxi + m) * 2 + k)] = (double)(acc.real() * dV);
                out[2 * (((size_t)n * nxi + m) * 2 + k) + 1] = (double)(acc.imag() * dV);
            }
        }
        td_batch<T>(g, vloc, kb, 1, pair, -dt, 1, 0, 0.0);
        td_batch<T>(g, vloc, kb, 1, pair + 2 * ng, dt, 1, 0, 0.0);
    }
}

}  // namespace

// =============================================================================================
// C entry points (ctypes).  use_ld != 0 selects the long double instantiation.
// =============================================================================================
// ---------------------------------------------------------------------------------------------
// Spectral bounds by shifted power iteration ("the upper and lower spectral bounds of the
// Kohn-Sham Hamiltonian ... a shifted power iteration"; R-20 in DESIGN.md fixes the details the
// paper leaves open).  power(shift, x0): x = x0/|x0|; repeat niter times: y = H x - shift x;
// lambda = Re<x|y> (Rayleigh quotient of H - shift, |x| = 1); x = y/|y|.  Returns lambda + shift.
// Run 1 (shift 0, start vector `seed`,0) converges to the eigenvalue of largest magnitude la; run 2
// (shift la, start vector `seed`,1) to the other end of the spectrum.  Plain sums over grid points.
// ---------------------------------------------------------------------------------------------
template <class T>
T power_iteration(const Grid& g, const double* vloc, const KBList& kb, T shift, int niter, uint64_t seed, uint64_t vec) {
    const size_t ng = (size_t)g.nx * g.ny * g.nz;
    std::vector<C<T>> x(ng), y(ng);
    for (size_t i = 0; i < ng; ++i) x[i] = C<T>((keyed_hash(seed, vec, i) >> 63) ? (T)-1 : (T)1, (T)0);
    T nrm = 0;
    for (size_t i = 0; i < ng; ++i) nrm += std::norm(x[i]);
    nrm = std::sqrt(nrm);
    for (size_t i = 0; i < ng; ++i) x[i] /= nrm;
    T lambda = 0;
    for (int it = 0; it < niter; ++it) {
        apply_H_one<T>(g, vloc, kb, x.data(), y.data());
        T a = 0, b = 0;
        for (size_t i = 0; i < ng; ++i) {
            y[i] -= shift * x[i];
            a += x[i].real() * y[i].real() + x[i].imag() * y[i].imag();
            b += std::norm(y[i]);
        }
        lambda = a;
        const T inv = (T)1 / std::sqrt(b);
        for (size_t i = 0; i < ng; ++i) x[i] = y[i] * inv;
    }
    return lambda + shift;
}

template <class T>
void spectral_bounds(const Grid& g, const double* vloc, const KBList& kb, int niter, uint64_t seed, double* emin, double* emax) {
    const T la = power_iteration<T>(g, vloc, kb, (T)0, niter, seed, 0);
    const T lb = power_iteration<T>(g, vloc, kb, la, niter, seed, 1);
    *emin = (double)(la < lb ? la : lb);
    *emax = (double)(la < lb ? lb : la);
}

extern "C" {
void sgwo_set_kinetic_cutoff(double ecut) { g_ecut = ecut > 0.0 ? ecut : 0.0; }

uint64_t sgwo_splitmix64_next(uint64_t* state) {   // the standard generator: state += gamma; mix
    uint64_t s = *state;
    uint64_t out = sm64(s);
    *state = s + 0x9E3779B97F4A7C15ULL;
    return out;
}
uint64_t sgwo_hash(uint64_t seed, uint64_t vec, uint64_t g) { return keyed_hash(seed, vec, g); }

void sgwo_random_vectors(uint64_t seed, int first_vec, int nvec, int64_t ng, double* psi) {
    for (int v = 0; v < nvec; ++v)
        for (int64_t i = 0; i < ng; ++i) {
            uint64_t h = keyed_hash(seed, (uint64_t)(first_vec + v), (uint64_t)i);
            psi[2 * ((int64_t)v * ng + i)] = (h >> 63) ? -1.0 : 1.0;
            psi[2 * ((int64_t)v * ng + i) + 1] = 0.0;
        }
}

void sgwo_fft1d(int n, int sign, const double* in, double* out, int use_ld) {
    if (use_ld) {
        std::vector<C<long double>> a, b(n), tw;
        load_vec<long double>(in, n, a);
        make_twiddles<long double>(n, sign, tw);
        fft1d<long double>(n, sign, a.data(), 1, b.data(), tw);
        store_vec<long double>(b, out);
    } else {
        std::vector<C<double>> a, b(n), tw;
        load_vec<double>(in, n, a);
        make_twiddles<double>(n, sign, tw);
        fft1d<double>(n, sign, a.data(), 1, b.data(), tw);
        store_vec<double>(b, out);
    }
}

void sgwo_fft3(int nx, int ny, int nz, int sign, double* a, int use_ld) {
    size_t ng = (size_t)nx * ny * nz;
    if (use_ld) {
        std::vector<C<long double>> t; load_vec<long double>(a, ng, t);
        fft3<long double>(nx, ny, nz, sign, t.data()); store_vec<long double>(t, a);
    } else {
        std::vector<C<double>> t; load_vec<double>(a, ng, t);
        fft3<double>(nx, ny, nz, sign, t.data()); store_vec<double>(t, a);
    }
}

#define GRID_ARGS int nx, int ny, int nz, double hx, double hy, double hz
#define KB_ARGS int nsphere, const int64_t* sph_ptr, const int32_t* sph_idx, int nproj, const double* beta, const double* D
#define MK Grid g{nx, ny, nz, hx, hy, hz}; KBList kb{nsphere, nproj, sph_ptr, sph_idx, beta, D};

void sgwo_apply_H(GRID_ARGS, const double* vloc, KB_ARGS, int nvec, const double* in, double* out, int use_ld) {
    MK
    if (use_ld) apply_H_batch<long double>(g, vloc, kb, nvec, in, out);
    else apply_H_batch<double>(g, vloc, kb, nvec, in, out);
}

void sgwo_cheb_filter(GRID_ARGS, const double* vloc, KB_ARGS, int nvec, double* psi, const double* coeffs,
                      double Emin, double Emax, int nterms, int use_ld) {
    MK
    if (use_ld) cheb_batch<long double>(g, vloc, kb, nvec, psi, coeffs, Emin, Emax, nterms);
    else cheb_batch<double>(g, vloc, kb, nvec, psi, coeffs, Emin, Emax, nterms);
}

void sgwo_hartree(GRID_ARGS, int nvec, const double* psi, double rho_scale, double* vh, double* rho_out, int use_ld) {
    Grid g{nx, ny, nz, hx, hy, hz};
    size_t ng = (size_t)nx * ny * nz;
    if (use_ld) {
        std::vector<long double> rho, v;
        density<long double>(g, nvec, psi, rho_scale, rho); poisson<long double>(g, rho, v);
        for (size_t i = 0; i < ng; ++i) { vh[i] = (double)v[i]; if (rho_out) rho_out[i] = (double)rho[i]; }
    } else {
        std::vector<double> rho, v;
        density<double>(g, nvec, psi, rho_scale, rho); poisson<double>(g, rho, v);
        for (size_t i = 0; i < ng; ++i) { vh[i] = v[i]; if (rho_out) rho_out[i] = rho[i]; }
    }
}

// Poisson solve alone on a given real density (for the erf closed-form pin).
void sgwo_poisson(GRID_ARGS, const double* rho, double* vh, int use_ld) {
    Grid g{nx, ny, nz, hx, hy, hz};
    size_t ng = (size_t)nx * ny * nz;
    if (use_ld) {
        std::vector<long double> r(rho, rho + ng), v; poisson<long double>(g, r, v);
        for (size_t i = 0; i < ng; ++i) vh[i] = (double)v[i];
    } else {
        std::vector<double> r(rho, rho + ng), v; poisson<double>(g, r, v);
        for (size_t i = 0; i < ng; ++i) vh[i] = v[i];
    }
}

void sgwo_td_propagate(GRID_ARGS, const double* vloc, KB_ARGS, int nvec, double* psi, double dt, int nsteps,
                       int hartree_mode, double rho_scale, int use_ld) {
    MK
    if (use_ld) td_batch<long double>(g, vloc, kb, nvec, psi, dt, nsteps, hartree_mode, rho_scale);
    else td_batch<double>(g, vloc, kb, nvec, psi, dt, nsteps, hartree_mode, rho_scale);
}

// psi <- exp(-i lambda v_pert(r)) psi for nvec vectors (the perturbed copy of P:57; R-21)
void sgwo_apply_kick(int64_t ng, int nvec, double* psi, const double* vpert, double lambda) {
    for (int v = 0; v < nvec; ++v)
        for (int64_t i = 0; i < ng; ++i) {
            const long double ph = (long double)lambda * (long double)vpert[i];
            const std::complex<long double> z((long double)psi[2 * (ng * v + i)], (long double)psi[2 * (ng * v + i) + 1]);
            const std::complex<long double> r = z * std::complex<long double>(std::cos(ph), -std::sin(ph));
            psi[2 * (ng * v + i)] = (double)r.real();
            psi[2 * (ng * v + i) + 1] = (double)r.imag();
        }
}

void sgwo_td_pair(GRID_ARGS, const double* vloc, KB_ARGS, int nvec, double* psi, double* psi_lam, double dt, int nsteps,
                  double rho_scale, uint64_t xi_seed, int nxi, int nfrag, double* out, int use_ld) {
    MK
    if (use_ld) td_pair<long double>(g, vloc, kb, nvec, psi, psi_lam, dt, nsteps, rho_scale, xi_seed, nxi, nfrag, out);
    else td_pair<double>(g, vloc, kb, nvec, psi, psi_lam, dt, nsteps, rho_scale, xi_seed, nxi, nfrag, out);
}

// cr: [nt][nxi] real (element (n, m) at cr[n * stride_n + m * stride_m]); ct: [nt][nxi] complex
void sgwo_time_order(int nxi, int nt, const double* cr, int stride_n, int stride_m, double* ct, int use_ld) {
    if (use_ld) time_order<long double>(nxi, nt, cr, stride_n, stride_m, ct);
    else time_order<double>(nxi, nt, cr, stride_n, stride_m, ct);
}

void sgwo_td_zeta(GRID_ARGS, const double* vloc, KB_ARGS, double* pair, const double* phi, double dt, int nsteps, uint64_t xi_seed,
                  int nxi, int nfrag, double* out, int use_ld) {
    MK
    if (use_ld) td_zeta<long double>(g, vloc, kb, pair, phi, dt, nsteps, xi_seed, nxi, nfrag, out);
    else td_zeta<double>(g, vloc, kb, pair, phi, dt, nsteps, xi_seed, nxi, nfrag, out);
}

void sgwo_spectral_bounds(GRID_ARGS, const double* vloc, KB_ARGS, int niter, uint64_t seed, double* emin, double* emax,
                          int use_ld) {
    MK
    if (use_ld) spectral_bounds<long double>(g, vloc, kb, niter, seed, emin, emax);
    else spectral_bounds<double>(g, vloc, kb, niter, seed, emin, emax);
}

void sgwo_norms(int64_t ng, int nvec, const double* psi, double* out) {   // sum_g |psi|^2 (no dV)
    for (int v = 0; v < nvec; ++v) {
        long double s = 0;
        for (int64_t i = 0; i < ng; ++i) {
            long double re = psi[2 * (v * ng + i)], im = psi[2 * (v * ng + i) + 1];
            s += re * re + im * im;
        }
        out[v] = (double)s;
    }
}

int sgwo_max_threads(void);
}

#ifdef _OPENMP
#include <omp.h>
extern "C" int sgwo_max_threads(void) { return omp_get_max_threads(); }
extern "C" void sgwo_set_threads(int n) { omp_set_num_threads(n); }
#else
extern "C" int sgwo_max_threads(void) { return 1; }
extern "C" void sgwo_set_threads(int) {}
#endif
