// sgw_ops.cuh -- functors of the generic pass kernel (sgw_fft.cuh: pass_kernel), which serves the Poisson solve of
// the Hartree rebuild (R-10), and the plain struct through which the library core asks a per-length translation
// unit to launch such a pass.  The pass kinds double as the tags of the per-pass profile (sgw_profile_get).
#pragma once
#include "sgw_fft.cuh"

namespace sgw {

enum PassKind {
    K_RT_STORE = 0,    // lean x pass of an operator application (store form)
    K_RT_ACC = 1,      // lean y pass / x+y plane pass (accumulate form)
    K_RT_HFIN = 2,     // lean z pass of H apply
    K_RT_CHEB = 3,     // lean z pass of a Chebyshev term
    K_RT_TD = 4,       // lean passes of a split-operator step
    K_RT_MUL3D = 5,    // Poisson: z round trip with the real 3D table v(k)/N_g
    K_FWD = 6,         // Poisson: forward transform along the axis, natural k order
    K_INV = 7,         // Poisson: inverse transform (unnormalised)
    K_KB_PROJECT = 8,  // nonlocal term: gather-dot (booked under axis 0)
    K_KB_SCATTER = 9,  // nonlocal term: scatter (booked under axis 0)
    K_DENSITY = 10,    // density_kernel (booked under axis 0)
    K_NKINDS = 11
};

struct OpParams {
    cd* out;                 // result
    const double* rin;       // K_FWD from a real field: the input is rin[g] + 0i (in is ignored)
    const double* mul3d;     // real N_g k-space table
    // K_INV with the merged phase epilogue (R-8): V = vloc + Re(result)
    const double* vloc;
    double* vprev;           // in: V of the previous step; out: V
    cd* table;               // exp(-i (V + vprev) half_dt)   (first != 0: exp(-i V half_dt))
    cd* last;                // exp(-i V half_dt) or NULL
    double* rho_reset;       // zeroed (the next step accumulates into it) or NULL
    double* vh_out;          // Re(result) or NULL
    double half_dt;
    int first;
    // non-separable kinetic operator (sgw_set_kinetic_cutoff): passes over nvec vectors
    const cd* src;           // the operator's input vectors (epilogues that add V * src)
    cd* acc;                 // Chebyshev: phi_{n-1} in, phi_{n+1} out
    const double* vtab;      // N_g real table multiplying src in the epilogue
    const cd* phase;         // N_g complex table applied on load (K_FWD variant 3) or on store (K_INV variant 5)
    const cd* mul3c;         // complex N_g k-space table
    double kscale, hs, alpha;
};

struct PassCall {
    int kind;                // PassKind
    int variant;             // K_FWD: 1 = real input (rin), 3 = phase on load;  K_RT_MUL3D: 1 = complex table;
                             // K_INV: 1 = merged phase epilogue, 2 = real output (vh_out), 3 = + vtab * src, 4 = Chebyshev step, 5 = phase on store
    PassGeom gm;
    long long ntiles;
    const cd* in;
    const cd* tw;            // exp(-2 pi i j / N), j < N
    OpParams p;
    cudaStream_t stream;
};

typedef int (*pass_launch_fn)(const PassCall*);

// ---- functors -------------------------------------------------------------------------------
//   cd   load(const cd* in, long long off, long long g)     input element
//   cd   mult(cd X, int k, long long gk)                    k-space multiply (RT only)
//   void epi(cd r, long long off, long long g)              store
struct OpStore {
    OpParams p;
    __device__ __forceinline__ cd load(const cd* in, long long off, long long) const { return in[off]; }
    __device__ __forceinline__ cd mult(cd X, int, long long) const { return X; }
    __device__ __forceinline__ void epi(cd r, long long off, long long) const { p.out[off] = r; }
};
// forward pass straight from the real density (replaces a separate real -> complex copy)
struct OpFromReal : OpStore {
    __device__ __forceinline__ cd load(const cd*, long long off, long long) const { return make_double2(p.rin[off], 0.0); }
};
struct OpMul3D : OpStore {
    __device__ __forceinline__ cd mult(cd X, int, long long gk) const { return cscale(X, __ldg(p.mul3d + gk)); }
};
// last inverse pass of the Poisson solve writes only the real part (sgw_hartree)
struct OpToReal : OpStore {
    __device__ __forceinline__ void epi(cd r, long long off, long long) const { p.vh_out[off] = r.x; }
};
// last inverse pass of the Poisson solve inside the propagator: V_H never reaches memory; the merged half-step
// phase tables of R-8 are written instead (see phase_merge_kernel for the frozen-potential form)
struct OpPhaseMerge : OpStore {
    __device__ __forceinline__ void epi(cd r, long long off, long long) const {
        const double v = (p.vloc ? p.vloc[off] : 0.0) + r.x;
        // sincospi: no large-argument reduction path; the 1/pi factor costs half an ulp of the angle (~1e-16 absolute here)
        const double hp = p.half_dt * 0.318309886183790671537767526745028724;
        double s, c;
        sincospi((p.first ? v : v + p.vprev[off]) * hp, &s, &c);
        p.table[off] = make_double2(c, -s);
        p.vprev[off] = v;
        if (p.last) {
            sincospi(v * hp, &s, &c);
            p.last[off] = make_double2(c, -s);
        }
        if (p.rho_reset) p.rho_reset[off] = 0.0;
    }
};

// ---- non-separable kinetic operator min(1/2 k^2, E_cut) (R-14): full 3D transform in five passes ----------
struct OpPhaseLoad : OpStore {                // forward x pass of a split-operator step: psi * phase on load
    __device__ __forceinline__ cd load(const cd* in, long long off, long long g) const { return cmul(in[off], __ldg(p.phase + g)); }
};
struct OpMul3DScaled : OpStore {              // z round trip with kscale * table (filter: table scaled by 2 / dE)
    __device__ __forceinline__ cd mult(cd X, int, long long gk) const { return cscale(X, p.kscale * __ldg(p.mul3d + gk)); }
};
struct OpMul3DC : OpStore {                   // z round trip with a complex table: exp(-i T dt) / N_g
    __device__ __forceinline__ cd mult(cd X, int, long long gk) const { return cmul(X, __ldg(p.mul3c + gk)); }
};
struct OpInvAddV : OpStore {                  // last inverse pass of H apply: out = T src + vtab * src
    __device__ __forceinline__ void epi(cd r, long long off, long long g) const {
        const cd u = p.src[off];
        const double v = p.vtab ? __ldg(p.vtab + g) : 0.0;
        p.out[off] = make_double2(r.x + v * u.x, r.y + v * u.y);
    }
};
struct OpInvCheb : OpStore {                  // last inverse pass of a Chebyshev step: acc <- hs (T + vtab) src + alpha acc
    __device__ __forceinline__ void epi(cd r, long long off, long long g) const {
        const cd u = p.src[off];
        const double v = __ldg(p.vtab + g);
        cd n = make_double2(p.hs * (r.x + v * u.x), p.hs * (r.y + v * u.y));
        if (p.alpha != 0.0) { const cd o = p.acc[off]; n.x += p.alpha * o.x; n.y += p.alpha * o.y; }
        p.acc[off] = n;
    }
};
struct OpInvPhase : OpStore {                 // last inverse pass of a split-operator step: result * phase on store
    __device__ __forceinline__ void epi(cd r, long long off, long long g) const { p.out[off] = cmul(r, __ldg(p.phase + g)); }
};

}  // namespace sgw
