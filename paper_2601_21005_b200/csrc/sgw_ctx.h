// sgw_ctx.h -- the library context (host-side state) shared by the translation units of libsgw.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "../../include/sgw.h"
#include "sgw_plane.cuh"
#include "sgw_engine.cuh"
#include "sgw_lean.cuh"

struct sgw_ctx {
    int nx, ny, nz;
    double hx, hy, hz;
    long long ng;
    int max_nvec;
    cudaStream_t stream;
    int B;                                   // pencils per CTA on the strided axes (y, z)
    int Bx;                                  // pencils per CTA on the contiguous axis (x)
    sgw::pass_launch_fn pass[3];             // per-axis launcher (x, y, z)
    sgw::plane_launch_fn plane;              // fused xy-plane launcher (nx == ny) or NULL
    int plane_G, plane_ctas;                 // planes per group, CTAs per SM (0 = auto)
    int dims[3];
    double hs[3];
    sgw::cd* tw[3];                          // exp(-2 pi i j/N) per axis
    std::vector<double> h_kin[3];            // 1/2 k^2 per axis (host)
    double* kin[3];                          // 1/2 k^2 / N per axis (device)
    double* cheb_kin[3];                     // s * 1/2 k^2 / N (rebuilt per filter call)
    sgw::cd* td_kin[3];                      // exp(-i 1/2 k^2 dt)/N (rebuilt when dt changes)
    double td_dt;
    bool td_kin_valid;
    double* vloc;                            // N_g or NULL
    double* vtab;                            // scaled potential for the filter, N_g
    double* vk3d;                            // Poisson kernel v(k)/N_g, N_g
    // Kleinman-Bylander lists
    int nsphere, nproj;
    int64_t* sph_ptr;
    int32_t* sph_idx;
    double* beta;
    double* D;
    sgw::cd* kbc;                            // [nvec][nsphere][nproj] projections
    long long kbc_cap;
    // workspace
    sgw::cd* ws[3];
    sgw::cd* pois;                           // N_g complex scratch for the Poisson solve
    double* rho;
    double* vh;
    sgw::cd* phase;                          // exp(-i V dt/2), N_g (merged table of two half steps in the lean TD path)
    sgw::cd* phase_last;                     // closing exp(-i V dt/2) of the last step of a call (lean TD path, lazy)
    double* vprev;                           // total potential of the previous step (lean TD path, lazy)
    int hartree_mode;
    double rho_scale;
    int64_t launches;
    // pass engine (sgw_engine.cuh)
    sgw::eng_launch_fn eng[3];               // per-axis launcher
    int engB[3];                             // pencils per tile per axis
    sgw::lean_launch_fn lean[3];             // per-axis launcher of the lean passes
    int lean_G, lean_ctas;                   // plane kernel: planes per CTA-owned group, CTAs per SM (0 = auto)
    int use_engine;                          // 0: v2 kernels (plane/pipe), 1: engine, 2: lean passes (default)
    int eng_max_ctas;                        // 0 = fill the device
    int eng_resident;                        // -1 auto, 0 stream all vectors per term, 1 force L2-resident groups
    int eng_l2_prefetch;                     // 1: prefetch the next item's operands into L2
    int eng_pc;                              // planes per x/y group (0 = auto)
    int num_sms;
    sgw::Seg* d_segs;
    size_t segs_cap;
    unsigned* d_cnt;
    size_t cnt_cap;
    int* d_err;
    int l2_chunk;                            // vectors per L2-resident chunk (0 = whole batch)
    // launch-bound grids: one whole sgw_cheb_filter call captured as a CUDA graph and cached (sgw_solvers.cu)
    cudaStream_t gstream;                    // internal capture stream (lazy)
    cudaGraphExec_t fgraph;                  // instantiated graph of the last small filter call, or NULL
    void* fg_psi;                            // its key: vector block, counts, window, coefficients
    int fg_nvec, fg_nterms;
    double fg_emin, fg_emax;
    std::vector<double> fg_coeffs;
    int64_t fg_launches;                     // kernel nodes in the graph
    // optional per-pass device timing (sgw_profile_*): event pairs around pass launches
    bool prof_on;
    std::vector<cudaEvent_t> prof_ev;        // 2 per recorded launch
    std::vector<int> prof_tag;               // axis * K_NKINDS + kind
    size_t prof_used;                        // pairs recorded since the last collect
    double prof_ms[3 * sgw::K_NKINDS];
    long long prof_n[3 * sgw::K_NKINDS];
};

namespace sgw {
int set_error(int code, const std::string& msg);
int check_cuda(cudaError_t e, const char* what);
PassGeom geom_for_axis(const sgw_ctx* c, int axis, int nvec, long long* ntiles);
int run_pass(sgw_ctx* c, int axis, int kind, int nvec, const cd* in, const OpParams& p);
// fused x+y pass; returns 1 when unavailable for this grid (caller runs the two passes instead)
int run_plane(sgw_ctx* c, int mode, int nvec, const cd* in, cd* out, const cd* phase, bool cheb_tables);
// engine-based implementations (sgw_program.cu)
int eng_apply_H(sgw_ctx* c, int nv, const cd* in, cd* out);
int eng_cheb_filter(sgw_ctx* c, int nvec, cd* psi, const double* h_coeffs, double s, int nterms);
int eng_td_step(sgw_ctx* c, int nvec, cd* psi, bool kb);
int eng_check_error(sgw_ctx* c);
// lean-pass implementations (sgw_program.cu)
int lean_apply_H(sgw_ctx* c, int nv, const cd* in, cd* out);
int lean_cheb_filter(sgw_ctx* c, int nvec, cd* psi, const double* h_coeffs, double s, int nterms);
int lean_td_step(sgw_ctx* c, int nvec, cd* psi, bool kb, bool accumulate_density, bool merged, bool last);
cudaEvent_t prof_begin(sgw_ctx* c, int tag);
void prof_end(sgw_ctx* c, cudaEvent_t e1);
int kb_apply(sgw_ctx* c, int nvec, const cd* src, cd* dst, int mode, double scale_or_tau, const cd* phase = nullptr,
             int fold = 0);
int ensure_ws(sgw_ctx* c, int n);
// forget the cached filter graph (the operator or its buffers changed)
void drop_filter_graph(sgw_ctx* c);
}  // namespace sgw
