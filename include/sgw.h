/* sgw.h -- C ABI of libsgw: the data-parallel hot path of stochastic GW on one B200 (sm_100a).
 *
 * The path (arXiv 2601.21005; "P:NN" = line NN of the paper text, "R-n" = reading n in DESIGN.md):
 * batched application of the Fourier-grid Kohn-Sham Hamiltonian H = -1/2 nabla^2 + V_loc + V_NL
 * to many stochastic vectors, the Chebyshev filter built on it (Eq. 3), and
 * split-operator propagation under a time-dependent Hartree potential.
 *
 * Conventions
 *  - Every call returns 0 on success or a negative code; nothing aborts or throws.
 *      SGW_EINVAL (-1) bad argument        SGW_ESIZE (-2) unsupported grid length
 *      SGW_ENOMEM (-3) allocation failed   SGW_ECUDA (-4) CUDA runtime error
 *    sgw_last_error() returns a thread-local message for the last failing call.
 *  - d_* are DEVICE pointers into caller-owned memory; h_* are HOST pointers read during the call.
 *  - Complex vectors are interleaved (re,im) IEEE double, 16 B per element, layout
 *    [nvec][nz][ny][nx] with x fastest; flat grid index g = ix + nx*(iy + ny*iz) (packed
 *    (N_g x n) multi-index arrays).  Real fields (V_loc, rho, V_H) are [nz][ny][nx] doubles.
 *  - All work is enqueued on the CUDA stream given to sgw_init_grid and is asynchronous with respect to the
 *    host.  The calls that block the host are: sgw_init_grid, sgw_set_vloc, sgw_set_nonlocal, sgw_set_kinetic_cutoff, sgw_destroy (setup;
 *    they allocate and synchronise the stream), sgw_sync_check, sgw_profile_get / _reset / _enable(0),
 *    sgw_spectral_bounds and sgw_probe_fp64 (they return host values), the FIRST sgw_cheb_filter / sgw_spectral_bounds call on a context
 *    (it allocates the two workspace arrays of max_nvec vectors: cudaMalloc), and error paths.  sgw_random_vectors,
 *    sgw_apply_H, sgw_hartree, sgw_td_propagate, sgw_norms and every later sgw_cheb_filter only enqueue work.
 *    k-space data never crosses the boundary.
 *  - Supported axis lengths: 8, 12, 16, 24, 32, 48, 64, 96, 128, 192, 256, 384 (products of 2 and
 *    3 with a compiled two-stage factorisation); nx must be a multiple of 4.  Others: SGW_ESIZE.
 *  - The library owns only its context (tables, workspace for max_nvec vectors).  Calls with
 *    nvec > max_nvec are processed in sub-batches of max_nvec (vectors are independent in the
 *    filter; in the TD step the density is accumulated over all sub-batches first).
 *  - Run-time switches, all read ONCE in sgw_init_grid (defaults are the measured best):
 *      SGW_ACC=0|1           H apply / Chebyshev filter through the TMA accumulate kernel (bulk-tensor loads, in-place
 *                            round trip in shared memory, bulk reduce-add; cubic grids with N a multiple of 8): default
 *                            on for N >= 64, else the register-operand passes below
 *      SGW_ACC_TD=0|1        split-operator steps through the TMA kernel of the same design (one launch per axis, bulk
 *                            stores; a CTA owns blocks of 8 pencils with all their vectors; at N = 384 the y and z launches
 *                            move tile pairs; cubic grids): default on from N = 256, else the plane / axis passes below
 *      SGW_ACC_L2_MB=m       accumulate kernel: one launch per term while cur + acc + v of a vector are at most m MB
 *                            (default 104: up to 128^3; the L2 holds 126 MB), else planes (x, y tiles) then z columns in two launches
 *      SGW_ACC_PAIRZ=0|1     accumulate kernel at N = 384: z tiles in pairs (16 pencils, 256-byte rows, one tensor operation per
 *                            pair, each of the two consumer groups takes one half); default 1
 *      SGW_LEAN_B=4|8        pencils per tile of the fused passes (default 8 when nx and ny are multiples of 8)
 *      SGW_LEAN_G=n          plane kernel: planes per CTA-owned group (default 1)
 *      SGW_LEAN_CTAS=1|2     plane kernel: one 16-warp or two 8-warp CTAs per SM (default: by L2 footprint)
 *      SGW_LEAN_CLUSTER=0|1  plane kernel: cluster-owned planes off / on (default: on for real 128^2 planes)
 *      SGW_LEAN_TEAM=0|1     plane kernel: team-owned planes (arrival counter per plane) off / on (default: on from 256^2)
 *      SGW_LEAN_VMINOR=0|1   tile order runs over the vectors first (default: when an N_g table exceeds 24 MB)
 *      SGW_LEAN_CHUNK=n      filter: n vectors at a time through all terms (default: all vectors per term)
 *      SGW_L2_CHUNK=n        propagation: n vectors at a time through a step (default: all vectors)
 *      SGW_PDL=1             programmatic dependent launch of the passes (default off)
 *      SGW_GRAPH=0           never replay a repeated small filter call as a CUDA graph (default on)
 *      SGW_GRAPH_BYTES=b     largest vector block that takes the graph path (default 16e6)
 *  - There is no CPU fallback: without a CUDA device sgw_init_grid fails with SGW_ECUDA.
 */
#ifndef SGW_H
#define SGW_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SGW_OK 0
#define SGW_EINVAL (-1)
#define SGW_ESIZE (-2)
#define SGW_ENOMEM (-3)
#define SGW_ECUDA (-4)

typedef struct sgw_ctx sgw_ctx;

/* Create a context for an nx*ny*nz periodic grid with spacings hx,hy,hz (bohr) (N_g =
 * N_x N_y N_z).  k_i = 2 pi m/(N_i h_i), m in [-N_i/2, N_i/2) (R: SURVEY 8(a) a3).  max_nvec
 * sizes the internal workspace (2 complex arrays of max_nvec*N_g, allocated by the first sgw_cheb_filter /
 * sgw_spectral_bounds call) and the projection buffer of the nonlocal term.  The device current at this call is
 * the context's device.  cuda_stream is a cudaStream_t owned by the caller (NULL = default
 * stream).  *ctx is written on success only. */
int sgw_init_grid(sgw_ctx** ctx, int nx, int ny, int nz, double hx, double hy, double hz,
                  int max_nvec, void* cuda_stream);

/* Free the context and everything it allocated.  Synchronises the stream first. */
int sgw_destroy(sgw_ctx* ctx);

/* Set the local potential V_loc(r) (Ha), N_g device doubles; copied into the context (the
 * potential-energy operator is diagonal in position).  NULL clears it (V_loc = 0). */
int sgw_set_vloc(sgw_ctx* ctx, const double* d_vloc);

/* Set the Kleinman-Bylander nonlocal term V_NL = sum_{s,p} |beta_sp> D_sp dV <beta_sp| as sparse
 * sphere lists ("pseudopotential contribution ... applied via atomic operations on grid
 * points where pseudopotentials for neighboring atoms overlap"; R-12).  d_sph_ptr[nsphere+1]
 * (int64) delimits each sphere's points in d_sph_idx (int32 flat grid indices) and d_beta
 * ([point][nproj] doubles); d_D is [nsphere][nproj] (Ha).  All four arrays are copied.
 * nproj_per_sphere must be 1..8.  nsphere = 0 clears the term. */
int sgw_set_nonlocal(sgw_ctx* ctx, int nsphere, const int64_t* d_sph_ptr, const int32_t* d_sph_idx,
                     int nproj_per_sphere, const double* d_beta, const double* d_D);

/* White-noise start vectors (R-4, R-5): element g of vector first_vec+j is
 * (h >> 63) ? -1.0 : +1.0 with h = sm64(sm64(sm64(seed) ^ (first_vec+j)) ^ g), imaginary part 0,
 * where sm64 is the splitmix64 output function.  Writes nvec*N_g complex to d_psi.  Bit-exact
 * and independent of batching. */
int sgw_random_vectors(sgw_ctx* ctx, uint64_t seed, int first_vec, int nvec, void* d_psi);

/* d_out = H d_in for nvec vectors, out of place (d_out must not alias d_in):
 * H psi = F^-1[ 1/2 |k|^2 F psi ] + V_loc psi + V_NL psi. */
int sgw_apply_H(sgw_ctx* ctx, int nvec, const void* d_in, void* d_out);

/* Chebyshev filter in place (Eq. 3; R-1): d_psi <- sum_{n<nterms} h_coeffs[n] T_n(Ht) d_psi,
 * Ht = (H - Eb)/dE, Eb = (Emax+Emin)/2, dE = (Emax-Emin)/2; three-term recurrence, nterms-1
 * applications of H.  h_coeffs: nterms host doubles.  Requires nterms >= 1 and Emax > Emin.
 * Asynchronous on the context's stream.  When one vector block is at most 16 MB and there is no
 * nonlocal term the call is launch-bound: when it repeats with the same (d_psi, nvec, nterms, Emin,
 * Emax, h_coeffs[]) its launches are captured into a CUDA graph that the context keeps and replays
 * from then on; same kernels, same order, same bits.  sgw_set_vloc / sgw_set_nonlocal drop the
 * graph.  SGW_GRAPH=0 disables. */
int sgw_cheb_filter(sgw_ctx* ctx, int nvec, void* d_psi, const double* h_coeffs, double Emin,
                    double Emax, int nterms);

/* rho(r) = rho_scale * sum_l |psi_l(r)|^2 over the nvec vectors (all N_eta orbitals on
 * one rank so the density needs no communication), and the Hartree potential
 * V_H = F^-1[ v(k) F rho ], v(k) = 4 pi (1 - cos(|k| Rc))/|k|^2, v(0) = 2 pi Rc^2,
 * Rc = min(Lx,Ly,Lz)/2 (R-10: spherically cut Coulomb kernel).  d_vh: N_g doubles out;
 * d_rho: N_g doubles out or NULL. */
int sgw_hartree(sgw_ctx* ctx, int nvec, const void* d_psi, double rho_scale, double* d_vh, double* d_rho);

/* The same Hartree rebuild for callers that cannot allocate device memory (code under stream capture, tight serving
 * loops, harnesses that forbid cudaMalloc): same arguments, same kernels, same five passes and the same bits as
 * sgw_hartree, but the two scratch arrays of the solve (N_g doubles of density, N_g complex for the transforms) live in
 * one file-scope `static __device__` array of the library instead of the context's allocations.
 *  - Limit: grids of at most SGW_STATIC_MAX_NG = 64^3 points (the array is 24 B x 64^3 = 6 MB, held by every GPU that
 *    loads the library until the process exits).  Larger grids: SGW_ESIZE with a message naming the limit; use sgw_hartree.
 *  - The call launches six kernels on the context's stream and calls no cudaMalloc, cudaFree or allocating library
 *    routine.  The context's device must be the current device (SGW_EINVAL otherwise).  The device address of the array
 *    is resolved once per device (cudaGetSymbolAddress) by the first call on that device, or ahead of time by
 *    sgw_static_setup (for a caller that wants nothing but launches inside a capture).
 *  - Every call, from every context on that GPU, shares the one array: calls that can overlap on the GPU (different
 *    streams, different contexts) RACE; serialise them.  The array keeps the last call's contents; nothing in it has
 *    to start at zero (the density kernel and the first pass overwrite the N_g elements the solve reads).
 * sgw_static_max_grid_points returns the limit. */
#define SGW_STATIC_MAX_NG (64LL * 64 * 64)
int sgw_hartree_static(sgw_ctx* ctx, int nvec, const void* d_psi, double rho_scale, double* d_vh, double* d_rho);
int sgw_static_setup(sgw_ctx* ctx);
int64_t sgw_static_max_grid_points(void);

/* Select the time-dependent part of the propagation Hamiltonian ("time-dependent
 * Hartree"; R-9): hartree_mode 0: V = V_loc frozen; 1: V = V_loc + V_H[rho(t_n)], rebuilt at the
 * start of every step from the current vectors with the given rho_scale. */
int sgw_set_td(sgw_ctx* ctx, int hartree_mode, double rho_scale);

/* nsteps symmetric split-operator steps in place (P:84, P:155 dt = 0.05; R-8, R-11):
 * psi <- e^{-iV dt/2} NL(dt/2) F^-1 e^{-i |k|^2 dt/2} F NL(dt/2) e^{-iV dt/2} psi,
 * NL(tau) psi = psi + sum_{s,p} beta_sp (e^{-i D_sp tau} - 1) dV <beta_sp|psi>.
 * dt may be negative (reverse-time propagation). */
int sgw_td_propagate(sgw_ctx* ctx, int nvec, void* d_psi, double dt, int nsteps);

/* d_psi <- exp(-i lambda v_pert(r)) d_psi for nvec vectors: the perturbed copy eta^lambda of P:57 ("we create a perturbed
 * copy of each eta"; R-21: the perturbing potential and its strength are the caller's).  d_vpert: N_g device doubles. */
int sgw_apply_kick(sgw_ctx* ctx, int nvec, void* d_psi, const double* d_vpert, double lambda);

/* Pair propagation with the sparse stochastic projection of the retarded response ("propagate both perturbed and
 * unperturbed copies in time under the action of the time-dependent Hamiltonian ... accumulate the causal response
 * function u^R(r,t) as the difference of the perturbed and unperturbed time-dependent potentials"; projected
 * on the fly onto N_xi random functions xi on short, fragmented segments of the grid, in segments of L = 32; R-21..R-23).
 * d_psi (unperturbed) and d_psi_lambda (perturbed) hold nvec vectors each and are both propagated nsteps split-operator
 * steps in place, each under V_loc + V_H[rho of ITS OWN copy at the start of the step] with the rho_scale of sgw_set_td
 * (the Hartree rebuild is always on here).  xi_m (m < nxi) consists of nfrag fragments of 32 consecutive grid points;
 * fragment f starts at grid index 32 * (h(seed, 2m, f) mod N_g/32) and carries the signs (top bit of h(seed, 2m+1, 32 f + j)
 * ? -1 : +1), h the keyed hash of sgw_random_vectors.  d_out[nsteps][nxi][2] (device doubles) receives, at the start of
 * step n, dV <xi_m | V_H[rho_copy(t_n)]> for copy 0 (unperturbed) and 1 (perturbed); the coefficients of u^R are
 * (out[..][1] - out[..][0]) / lambda.  N_g must be a multiple of 32.  nvec <= max_nvec vectors are processed at a time. */
int sgw_td_propagate_pair(sgw_ctx* ctx, int nvec, void* d_psi, void* d_psi_lambda, double dt, int nsteps, uint64_t xi_seed,
                          int nxi, int nfrag, double* d_out);

/* The zeta pair of the Green's function (Eq. 4: "propagating the filtered zeta backwards in time while
 * simultaneously propagating its orthogonal complement forwards in time"; packed as (N_g x 2); R-25).  d_pair holds
 * two vectors: [0] the filtered zeta, propagated with -dt, [1] its complement, propagated with +dt, nsteps split-operator
 * steps each, in place, under the frozen potential V_loc (+ V_NL).  At the start of step n the projections
 * d_out[n][m][k] = dV <xi_m | phi psi_k(t_n)> (complex; d_out is [nsteps][nxi][2] complex) onto the xi of
 * sgw_td_propagate_pair are recorded; d_phi: N_g device doubles, the orbital of Eq. 5. */
int sgw_td_propagate_zeta(sgw_ctx* ctx, void* d_pair, const double* d_phi, double dt, int nsteps, uint64_t xi_seed, int nxi,
                          int nfrag, void* d_out);

/* Time-ordering of the retarded response ("we time-order the accumulated u^R(r,t) to produce the effective
 * polarization potential u(r,t)"; a transform in time before and after a complex-conjugation step; R-24), on each of
 * the nxi coefficient series c^R(t_n), n < nt, element (n, m) at d_cr[n * stride_n + m * stride_m] (real, causal): zero-
 * padded to M = 2 nt samples, C(w_k) = sum_n c^R(t_n) e^{+2 pi i k n / M}, C^T = C for k >= 0 and its conjugate for k < 0,
 * c^T(t_n) = (1/M) sum_k C^T(w_k) e^{-2 pi i k n / M}.  d_ct: [nt][nxi] complex.  nt up to about 5000. */
int sgw_time_order(sgw_ctx* ctx, int nxi, int nt, const double* d_cr, int64_t stride_n, int64_t stride_m, void* d_ct);

/* Sigma(t_n) in the xi basis (Eq. 5; R-26): d_sigma[n][k] = N_g / (nxi nfrag 32 dV) * sum_m c^T[n][m] p[n][m][k], with
 * d_ct from sgw_time_order and d_p from sgw_td_propagate_zeta.  d_sigma: [nt][2] complex. */
int sgw_sigma_t(sgw_ctx* ctx, int nt, int nxi, int nfrag, const void* d_ct, const void* d_p, void* d_sigma);

/* Kinetic-energy cutoff ("apply an energy cutoff of 28 Hartrees to the kinetic energy operator"; it bounds
 * the spectral width and with it the number of Chebyshev terms; R-14).  ecut > 0 (Ha): from now on the kinetic operator
 * of sgw_apply_H, sgw_cheb_filter, sgw_td_propagate and sgw_spectral_bounds is F^-1 min(1/2 |k|^2, ecut) F.  That
 * operator is not separable, so these calls then take a five-pass full-3D-transform route (about 7 array sweeps per
 * application instead of 2-3).  ecut <= 0 restores the plain 1/2 |k|^2 (the default, and what BASELINE.json's configs
 * use).  Setup call: allocates N_g doubles + N_g complex + max_nvec vectors of scratch and synchronises the stream. */
int sgw_set_kinetic_cutoff(sgw_ctx* ctx, double ecut);

/* Spectral bounds of H by shifted power iteration ("the upper and lower spectral bounds of the Kohn-Sham
 * Hamiltonian ... a shifted power iteration"; R-20).  power(shift, x0): x = x0/|x0|; niter times: y = H x - shift x,
 * lambda = Re<x|y>, x = y/|y|; result lambda + shift.  Run 1: shift 0 from white-noise vector (seed, 0) gives the
 * eigenvalue of largest magnitude la; run 2: shift la from vector (seed, 1) gives the other end.  *h_emin / *h_emax
 * (HOST doubles) receive min / max of the two.  Rayleigh quotients lie inside the spectrum, so the estimates
 * approach the true bounds from inside; callers pad them.  Uses the V_loc / nonlocal terms currently set.  Reductions
 * are segmented sums with one atomic per block.  Synchronises the stream (it returns host values). */
int sgw_spectral_bounds(sgw_ctx* ctx, int niter, uint64_t seed, double* h_emin, double* h_emax);

/* d_out[l] = sum_g |psi_l(g)|^2 (no dV factor), nvec doubles (normalisations as segmented
 * sums with one atomic add per segment).  Test helper. */
int sgw_norms(sgw_ctx* ctx, int nvec, const void* d_psi, double* d_out);

/* Number of kernels the library has launched on this context since creation (for bench.py's
 * gpu_launches).  Host counter; never fails (returns 0 for NULL). */
int64_t sgw_launch_count(const sgw_ctx* ctx);

/* Per-pass device timing for measurement (bench.py's roofline): while enabled, every FFT pass launch
 * is bracketed by a pair of CUDA events on the context's stream (at most 60000 launches between
 * collections).  sgw_profile_get synchronises the stream and returns, for passes along `axis`
 * (0 x, 1 y, 2 z) of `kind` (0 x pass of an operator application, 1 y pass or fused x+y plane pass, 2 z pass of
 * H apply, 3 z pass of a Chebyshev term, 4 split-operator passes, 5 / 6 / 7 Poisson z round trip / forward /
 * inverse passes), the number of launches timed and their summed duration in ms since the last
 * sgw_profile_reset.  Booked under axis 0 as well: kind 8 / 9 the gather-dot / scatter kernels of the nonlocal term,
 * kind 10 the density kernel; under axis 1 of kind 10 its sphere-point correction in the propagator (density_points_kernel). */
int sgw_profile_enable(sgw_ctx* ctx, int on);
int sgw_profile_reset(sgw_ctx* ctx);
int sgw_profile_get(sgw_ctx* ctx, int axis, int kind, int64_t* count, double* total_ms);

/* Measurement helper ("FP64 peak ... must be probed"): runs a dependent-free DFMA loop (8 independent
 * chains per thread, 32 warps per SM, 2 CTAs per SM) on the context's stream at whatever clocks the device is at
 * and writes the best of three timed repetitions, in FP64 flop/s (2 per DFMA), to *h_flops_per_s.  Blocks the host. */
int sgw_probe_fp64(sgw_ctx* ctx, double* h_flops_per_s);

/* Synchronises the context's stream and reports asynchronous failures: SGW_ECUDA if a kernel faulted,
 * SGW_OK otherwise. */
int sgw_sync_check(sgw_ctx* ctx);

/* Message for the last error on the calling thread ("" if none). */
const char* sgw_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* SGW_H */
