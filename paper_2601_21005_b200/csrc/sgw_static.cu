// sgw_static.cu -- sgw_hartree_static: the Hartree rebuild (density + cut-Coulomb Poisson solve, include/sgw.h) for
// callers that cannot allocate device memory (code under stream capture, tight serving loops, harnesses that forbid
// cudaMalloc).  Same kernels and the same five passes as sgw_hartree; the only difference is where the two scratch
// arrays of the solve live: not in the context's cudaMalloc'ed rho / pois arrays but in ONE file-scope device array of
// a fixed maximum size, which every GPU that loads the library holds until exit.
#include <cstring>
#include <mutex>
#include <string>

#include "sgw_ctx.h"
#include "sgw_kernels.cuh"

using namespace sgw;

namespace {

constexpr long long MAX_NG = SGW_STATIC_MAX_NG;                 // 64^3 grid points (include/sgw.h)
constexpr size_t POIS_BYTES = (size_t)MAX_NG * sizeof(cd);      // N_g complex: the array the five passes transform in place
constexpr size_t RHO_BYTES = (size_t)MAX_NG * sizeof(double);   // N_g real: the density the first pass reads
static_assert(POIS_BYTES % 256 == 0, "the density part must start 256-byte aligned");

// 6 MB per GPU.  In HOST code this name is only a stand-in for the symbol: it is not a device address and must never
// be handed to a kernel; the address comes from cudaGetSymbolAddress (scratch_for below).
static __device__ __align__(256) unsigned char g_static_scratch[POIS_BYTES + RHO_BYTES];

constexpr int MAX_DEVICES = 64;
std::mutex g_mu;
unsigned char* g_scratch_ptr[MAX_DEVICES] = {};                 // device address of g_static_scratch, per device

// set-up, once per device, with that device current
int scratch_for(const sgw_ctx* c, unsigned char** out) {
    int dev = -1;
    if (check_cuda(cudaGetDevice(&dev), "cudaGetDevice") != 0) return SGW_ECUDA;
    if (dev != c->device)
        return set_error(SGW_EINVAL, "sgw_hartree_static: the context's device (" + std::to_string(c->device) +
                                         ") is not the current device (" + std::to_string(dev) + ")");
    if (dev < 0 || dev >= MAX_DEVICES) return set_error(SGW_EINVAL, "sgw_hartree_static: device ordinal out of range");
    std::lock_guard<std::mutex> lk(g_mu);
    if (!g_scratch_ptr[dev]) {
        void* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_static_scratch);
        if (e != cudaSuccess || !p) {
            check_cuda(e, "cudaGetSymbolAddress(g_static_scratch)");
            return e != cudaSuccess ? SGW_ECUDA : set_error(SGW_ECUDA, "cudaGetSymbolAddress returned a null address");
        }
        g_scratch_ptr[dev] = (unsigned char*)p;
    }
    *out = g_scratch_ptr[dev];
    return 0;
}

int pass(sgw_ctx* c, int axis, int kind, int variant, const cd* in, const OpParams& p) {
    PassCall call;
    call.kind = kind;
    call.variant = variant;
    call.gm = geom_for_axis(c, axis, 1, &call.ntiles);
    call.in = in;
    call.tw = c->tw[axis];
    call.p = p;
    call.stream = c->stream;
    if (call.ntiles <= 0) return 0;
    if (c->pass[axis](&call) != 0)
        return set_error(SGW_ECUDA, std::string("sgw_hartree_static: pass launch failed: ") + cudaGetErrorString(cudaGetLastError()));
    c->launches++;
    return 0;
}

}  // namespace

extern "C" int64_t sgw_static_max_grid_points(void) { return MAX_NG; }

extern "C" int sgw_static_setup(sgw_ctx* c) {
    if (!c) return set_error(SGW_EINVAL, "sgw_static_setup: bad argument");
    unsigned char* s = nullptr;
    return scratch_for(c, &s);
}

extern "C" int sgw_hartree_static(sgw_ctx* c, int nvec, const void* d_psi, double rho_scale, double* d_vh, double* d_rho) {
    if (!c || nvec < 0 || (nvec > 0 && !d_psi) || !d_vh) return set_error(SGW_EINVAL, "sgw_hartree_static: bad argument");
    if (c->ng > MAX_NG)
        return set_error(SGW_ESIZE, "sgw_hartree_static: grid of " + std::to_string(c->ng) + " points exceeds the static scratch (" +
                                        std::to_string(MAX_NG) + " points = 64^3); use sgw_hartree");
    unsigned char* s = nullptr;
    if (int rc = scratch_for(c, &s)) return rc;
    cd* pois = (cd*)s;
    double* rho = (double*)(s + POIS_BYTES);
    const long long ng = c->ng;
    // nothing in the scratch has to start at zero: density_kernel overwrites rho[0, ng) and the forward x pass overwrites
    // pois[0, ng) from it; what the previous call left beyond ng is never read
    density_kernel<<<(unsigned)((ng + 255) / 256), 256, 0, c->stream>>>((const cd*)d_psi, nvec, ng, rho_scale, rho, d_rho);
    c->launches++;
    if (int rc = check_cuda(cudaGetLastError(), "density")) return rc;
    OpParams p;
    memset(&p, 0, sizeof(p));
    p.out = pois;
    p.rin = rho;
    if (int rc = pass(c, 0, K_FWD, 1, pois, p)) return rc;          // forward x, straight from the real density
    p.rin = nullptr;
    if (int rc = pass(c, 1, K_FWD, 0, pois, p)) return rc;          // forward y
    p.mul3d = c->vk3d;
    if (int rc = pass(c, 2, K_RT_MUL3D, 0, pois, p)) return rc;     // z round trip with v(k) / N_g
    p.mul3d = nullptr;
    if (int rc = pass(c, 1, K_INV, 0, pois, p)) return rc;          // inverse y
    p.vh_out = d_vh;
    return pass(c, 0, K_INV, 2, pois, p);                           // inverse x, real part to d_vh
}
