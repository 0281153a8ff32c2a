/* c_abi_consumer.c -- a plain C consumer of include/sgw.h, compiled by tests/test_abi_exports.py with gcc and linked
 * against libsgw.so: proves the header compiles as C and that every declared entry point links with the declared
 * signature.  Without a CUDA device it checks the documented error behaviour (SGW_ECUDA from sgw_init_grid,
 * SGW_EINVAL for a NULL context, nothing aborts); with one it runs every entry point once on an 8^3 grid. */
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <cuda_runtime_api.h>

#include "sgw.h"

#define CHECK(cond)                                                           \
    do {                                                                      \
        if (!(cond)) {                                                        \
            printf("FAILED line %d: %s (%s)\n", __LINE__, #cond, sgw_last_error()); \
            return 1;                                                         \
        }                                                                     \
    } while (0)

int main(void) {
    sgw_ctx* ctx = NULL;
    double emin = 0, emax = 0, ms = 0;
    int64_t cnt = 0;
    const double coeffs[3] = {0.5, 0.25, 0.125};
    /* argument errors never need a device */
    CHECK(sgw_init_grid(NULL, 8, 8, 8, 0.5, 0.5, 0.5, 1, NULL) == SGW_EINVAL);
    CHECK(sgw_init_grid(&ctx, 10, 8, 8, 0.5, 0.5, 0.5, 1, NULL) == SGW_ESIZE);
    CHECK(strlen(sgw_last_error()) > 0);
    CHECK(sgw_set_vloc(NULL, NULL) == SGW_EINVAL);
    CHECK(sgw_set_nonlocal(NULL, 0, NULL, NULL, 4, NULL, NULL) == SGW_EINVAL);
    CHECK(sgw_random_vectors(NULL, 1, 0, 1, NULL) == SGW_EINVAL);
    CHECK(sgw_apply_H(NULL, 1, NULL, NULL) == SGW_EINVAL);
    CHECK(sgw_cheb_filter(NULL, 1, NULL, coeffs, 0.0, 1.0, 3) == SGW_EINVAL);
    CHECK(sgw_hartree(NULL, 1, NULL, 1.0, NULL, NULL) == SGW_EINVAL);
    CHECK(sgw_set_td(NULL, 0, 0.0) == SGW_EINVAL);
    CHECK(sgw_td_propagate(NULL, 1, NULL, 0.05, 1) == SGW_EINVAL);
    CHECK(sgw_spectral_bounds(NULL, 1, 1, &emin, &emax) == SGW_EINVAL);
    CHECK(sgw_norms(NULL, 1, NULL, NULL) == SGW_EINVAL);
    CHECK(sgw_profile_enable(NULL, 1) == SGW_EINVAL);
    CHECK(sgw_profile_reset(NULL) == SGW_EINVAL);
    CHECK(sgw_profile_get(NULL, 0, 0, &cnt, &ms) == SGW_EINVAL);
    CHECK(sgw_td_propagate_zeta(NULL, NULL, NULL, 0.05, 1, 1, 1, 1, NULL) == SGW_EINVAL);
    CHECK(sgw_time_order(NULL, 1, 1, NULL, 1, 1, NULL) == SGW_EINVAL);
    CHECK(sgw_sigma_t(NULL, 1, 1, 1, NULL, NULL, NULL) == SGW_EINVAL);
    CHECK(sgw_set_kinetic_cutoff(NULL, 28.0) == SGW_EINVAL);
    CHECK(sgw_apply_kick(NULL, 1, NULL, NULL, 0.1) == SGW_EINVAL);
    CHECK(sgw_td_propagate_pair(NULL, 1, NULL, NULL, 0.05, 1, 1, 1, 1, NULL) == SGW_EINVAL);
    CHECK(sgw_probe_fp64(NULL, &ms) == SGW_EINVAL);
    CHECK(sgw_hartree_static(NULL, 1, NULL, 1.0, NULL, NULL) == SGW_EINVAL);
    CHECK(sgw_static_setup(NULL) == SGW_EINVAL);
    CHECK(sgw_static_max_grid_points() == SGW_STATIC_MAX_NG);
    CHECK(sgw_sync_check(NULL) == SGW_EINVAL);
    CHECK(sgw_launch_count(NULL) == 0);
    CHECK(sgw_destroy(NULL) == SGW_OK);

    int rc = sgw_init_grid(&ctx, 8, 8, 8, 0.5, 0.5, 0.5, 2, NULL);
    if (rc == SGW_ECUDA) {                      /* no device: the product path fails loudly, there is no fallback */
        CHECK(ctx == NULL);
        printf("nogpu ok\n");
        return 0;
    }
    CHECK(rc == SGW_OK && ctx != NULL);
    const size_t ng = 512;
    void *psi = NULL, *out = NULL;
    double *vloc = NULL, *vh = NULL, *nrm = NULL;
    CHECK(cudaMalloc(&psi, 2 * ng * 16) == cudaSuccess && cudaMalloc(&out, 2 * ng * 16) == cudaSuccess);
    CHECK(cudaMalloc((void**)&vloc, ng * 8) == cudaSuccess && cudaMalloc((void**)&vh, ng * 8) == cudaSuccess);
    CHECK(cudaMalloc((void**)&nrm, 4 * 8) == cudaSuccess);
    CHECK(cudaMemset(vloc, 0, ng * 8) == cudaSuccess);
    CHECK(sgw_set_vloc(ctx, vloc) == SGW_OK);
    CHECK(sgw_set_nonlocal(ctx, 0, NULL, NULL, 4, NULL, NULL) == SGW_OK);
    CHECK(sgw_random_vectors(ctx, 20260121u, 0, 2, psi) == SGW_OK);
    CHECK(sgw_apply_H(ctx, 2, psi, out) == SGW_OK);
    CHECK(sgw_apply_H(ctx, 2, psi, psi) == SGW_EINVAL);           /* out of place only */
    CHECK(sgw_cheb_filter(ctx, 2, psi, coeffs, -1.0, 80.0, 3) == SGW_OK);
    CHECK(sgw_hartree(ctx, 2, psi, 1.0, vh, NULL) == SGW_OK);
    CHECK(sgw_set_td(ctx, 1, 0.01) == SGW_OK);
    CHECK(sgw_td_propagate(ctx, 2, psi, 0.05, 2) == SGW_OK);
    CHECK(sgw_norms(ctx, 2, psi, nrm) == SGW_OK);
    CHECK(sgw_spectral_bounds(ctx, 3, 7, &emin, &emax) == SGW_OK && emin <= emax);
    CHECK(sgw_profile_enable(ctx, 1) == SGW_OK && sgw_profile_reset(ctx) == SGW_OK);
    CHECK(sgw_apply_H(ctx, 1, psi, out) == SGW_OK);
    CHECK(sgw_profile_get(ctx, 2, 2, &cnt, &ms) == SGW_OK && cnt == 1);
    CHECK(sgw_profile_enable(ctx, 0) == SGW_OK);
    CHECK(sgw_apply_kick(ctx, 2, out, vloc, 0.01) == SGW_OK);
    CHECK(sgw_td_propagate_pair(ctx, 2, psi, out, 0.05, 2, 7, 1, 3, nrm) == SGW_OK);    /* nrm: 2 steps x 1 xi x 2 = 4 doubles */
    {   /* NEXT-4: 3 steps, 2 xi of 2 fragments */
        void *zp = NULL, *ct = NULL, *sg = NULL;
        double* cr = NULL;
        CHECK(cudaMalloc(&zp, 3 * 2 * 2 * 16) == cudaSuccess && cudaMalloc(&ct, 3 * 2 * 16) == cudaSuccess);
        CHECK(cudaMalloc(&sg, 3 * 2 * 16) == cudaSuccess && cudaMalloc((void**)&cr, 3 * 2 * 8) == cudaSuccess);
        CHECK(cudaMemset(cr, 0, 3 * 2 * 8) == cudaSuccess);
        CHECK(sgw_td_propagate_zeta(ctx, psi, vloc, 0.05, 3, 7, 2, 2, zp) == SGW_OK);
        CHECK(sgw_time_order(ctx, 2, 3, cr, 2, 1, ct) == SGW_OK);
        CHECK(sgw_sigma_t(ctx, 3, 2, 2, ct, zp, sg) == SGW_OK);
        CHECK(sgw_sync_check(ctx) == SGW_OK);
        cudaFree(zp); cudaFree(ct); cudaFree(sg); cudaFree(cr);
    }
    CHECK(sgw_set_kinetic_cutoff(ctx, 5.0) == SGW_OK);
    CHECK(sgw_apply_H(ctx, 2, psi, out) == SGW_OK);
    CHECK(sgw_cheb_filter(ctx, 2, psi, coeffs, -1.0, 20.0, 3) == SGW_OK);
    CHECK(sgw_td_propagate(ctx, 2, psi, 0.05, 2) == SGW_OK);
    CHECK(sgw_set_kinetic_cutoff(ctx, 0.0) == SGW_OK);
    CHECK(sgw_probe_fp64(ctx, &ms) == SGW_OK && ms > 1e11);
    CHECK(sgw_sync_check(ctx) == SGW_OK);
    double h[2] = {0, 0};
    CHECK(cudaMemcpy(h, nrm, 16, cudaMemcpyDeviceToHost) == cudaSuccess);
    CHECK(h[0] > 0 && h[1] > 0 && isfinite(h[0]) && isfinite(h[1]));
    CHECK(sgw_launch_count(ctx) > 0);
    CHECK(sgw_destroy(ctx) == SGW_OK);
    cudaFree(psi); cudaFree(out); cudaFree(vloc); cudaFree(vh); cudaFree(nrm);
    printf("gpu ok\n");
    return 0;
}
