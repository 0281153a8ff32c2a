// sgw_ctx.h -- the library context (host-side state) shared by the translation units of libsgw.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "../../include/sgw.h"
#include "sgw_ops.cuh"
#include "sgw_lean.cuh"
#include "sgw_acc.cuh"

struct sgw_ctx {
    int nx, ny, nz;
    double hx, hy, hz;
    long long ng;
    int max_nvec;
    cudaStream_t stream;
    int device, num_sms;                     // the device current at sgw_init_grid
    int B;                                   // Poisson passes: pencils per CTA on the strided axes (y, z)
    int Bx;                                  // Poisson passes: pencils per CTA on the contiguous axis (x)
    int leanB;                               // lean passes: pencils per tile (8, or 4 when nx or ny is not a multiple of 8)
    sgw::pass_launch_fn pass[3];             // per-axis launcher of the Poisson passes (x, y, z)
    sgw::lean_launch_fn lean[3];             // per-axis launcher of the lean passes
    sgw::acc_launch_fn acc;                  // TMA accumulate kernel (cubic grids) or NULL
    sgw::td_launch_fn tdk;                   // TMA split-operator kernel (cubic grids) or NULL
    int use_acc_td;                          // complex family through it (SGW_ACC_TD; default: from 256 points per axis)
    int acc_occ[5];                          // kernel attribute set: accumulate, split-operator x / y / z, accumulate in tile pairs
    int acc_pairz;                           // z launch of the accumulate kernel in tile pairs (N = 384; SGW_ACC_PAIRZ=0 disables)
    int use_acc;                             // real family through the TMA accumulate kernel (SGW_ACC; default: where it is built and measured faster)
    double acc_l2_bytes;                     // one-launch terms when cur + acc + v of a vector are at most this (SGW_ACC_L2_MB)
    const void* tmap_base[8];                // small cache of tensor maps: (array, vectors) -> y and z maps
    int tmap_nv[8], tmap_next;
    CUtensorMap tmap_y[8], tmap_z[8], tmap_z2[8], tmap_y2[8];   // z2 / y2: tiles in pairs (16 adjacent pencils, 256-byte rows)
    void* tmap_encode;                       // cuTensorMapEncodeTiled (driver entry point)
    int lean_occ[3][18];                     // occupancy results of the lean kernels, per axis length (filled on first use)
    int lean_G, lean_ctas;                   // plane kernel: planes per CTA-owned group, CTAs per SM (0 = auto)
    int lean_cluster;                        // -1 auto, 0 / 1 forced (SGW_LEAN_CLUSTER)
    int lean_team;                           // -1 auto, 0 / 1 forced (SGW_LEAN_TEAM): team-owned planes
    int lean_vminor;                         // -1 auto, 0 / 1 forced (SGW_LEAN_VMINOR): vectors fastest in the tile order
    unsigned* team_cnt;                      // max_nvec * nz plane arrival counters of the team plane kernel
    int lean_chunk;                          // filter: vectors per L2-resident chunk (SGW_LEAN_CHUNK; 0 = whole batch)
    int l2_chunk;                            // TD: vectors per L2-resident chunk (SGW_L2_CHUNK; 0 = whole batch)
    int pdl;                                 // programmatic dependent launch (SGW_PDL=1)
    int graph_on;                            // cached filter graph allowed (SGW_GRAPH != 0)
    double graph_bytes;                      // largest vector block that takes the graph path (SGW_GRAPH_BYTES)
    int dims[3];
    double hs[3];
    sgw::cd* tw[3];                          // exp(-2 pi i j/N) per axis
    double* kin[3];                          // 1/2 k^2 / N per axis (device)
    double* kin_raw[3];                      // 1/2 k^2 per axis (device)
    double* cheb_kin[3];                     // s * 1/2 k^2 / N (rebuilt per filter call)
    sgw::cd* td_kin[3];                      // exp(-i 1/2 k^2 dt)/N (rebuilt on the device when dt changes)
    double td_dt;
    bool td_kin_valid;
    double* vloc;                            // N_g or NULL
    double* vtab;                            // scaled potential for the filter, N_g
    double* vk3d;                            // Poisson kernel v(k)/N_g, N_g
    // Kleinman-Bylander lists
    int nsphere, nproj;
    int64_t* sph_ptr;
    int32_t* sph_idx;
    int32_t* sph_uniq;                       // the distinct grid points of all spheres, ascending (density correction of the propagator)
    int64_t nuniq;
    double* beta;
    double* D;
    sgw::cd* kbc;                            // [max_nvec][nsphere][nproj] projections (allocated by sgw_set_nonlocal)
    // workspace
    sgw::cd* ws[2];                          // max_nvec vectors each, allocated by the first call that needs them
    sgw::cd* pois;                           // N_g complex scratch for the Poisson solve
    double* rho;
    double* vh;
    sgw::cd* phase;                          // exp(-i V dt/2), N_g (merged table of two half steps without KB)
    sgw::cd* phase_last;                     // closing exp(-i V dt/2) of the last step of a call
    double* vprev;                           // total potential of the previous step
    // kinetic-energy cutoff (sgw_set_kinetic_cutoff): non-separable kinetic operator min(1/2 k^2, E_cut)
    double ecut;                             // 0 = off
    double* kin3d;                           // min(1/2 |k|^2, E_cut) / N_g on the grid's k layout
    sgw::cd* td_kin3d;                       // exp(-i min(1/2 |k|^2, E_cut) dt) / N_g (rebuilt when dt changes)
    double td3d_dt;
    bool td3d_valid;
    sgw::cd* wcut;                           // max_nvec vectors of scratch for the five-pass route
    double* red;                             // 4 doubles: reductions of sgw_spectral_bounds
    int hartree_mode;
    double rho_scale;
    int64_t launches;
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
// one Poisson pass on a single N_g array (variant: see PassCall)
int run_pass(sgw_ctx* c, int axis, int kind, int variant, const cd* in, const OpParams& p, int nvec = 1);
// non-separable kinetic operator (sgw_cut.cu)
int cut_apply_H(sgw_ctx* c, int nv, const cd* in, cd* out);
int cut_cheb_filter(sgw_ctx* c, int nvec, cd* psi, const double* h_coeffs, double s, int nterms);
int cut_td_propagate(sgw_ctx* c, int nvec, cd* psi, double dt, int nsteps);
// lean-pass implementations (sgw_program.cu)
int lean_apply_H(sgw_ctx* c, int nv, const cd* in, cd* out);
int lean_cheb_filter(sgw_ctx* c, int nvec, cd* psi, const double* h_coeffs, double s, int nterms);
int lean_td_step(sgw_ctx* c, int nvec, cd* psi, bool kb, bool accumulate_density, bool merged, bool last);
// TMA accumulate implementations (sgw_program.cu)
int acc_apply_H(sgw_ctx* c, int nv, const cd* in, cd* out);
int acc_cheb_filter(sgw_ctx* c, int nvec, cd* psi, const double* h_coeffs, double s, int nterms);
cudaEvent_t prof_begin(sgw_ctx* c, int tag);
void prof_end(sgw_ctx* c, cudaEvent_t e1);
int kb_apply(sgw_ctx* c, int nvec, const cd* src, cd* dst, int mode, double scale_or_tau, const cd* phase = nullptr,
             int fold = 0);
int ensure_ws(sgw_ctx* c, int n);
// forget the cached filter graph (the operator or its buffers changed)
void drop_filter_graph(sgw_ctx* c);
}  // namespace sgw
