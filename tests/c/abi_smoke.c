/* Plain C client of the C ABI (include/wpgrid.h): create -> wkernel_build -> grid -> dirty_image -> destroy, with
 * device memory from the CUDA runtime's C API and nothing else — no Python, no torch.  Pins the boundary itself:
 * the header compiles as C, the library links, workspaces are caller-owned, errors come back as codes.
 * Checks: counters of a two-visibility input (one off the grid); flux conservation P11 (sum of the grid = weight *
 * vis * sum of the slice, and K5 makes the on-cell slice of a w = 0 stack sum to 1: here w_max = 0); a too-small
 * workspace is WPG_ENOMEM.  Exit code 0 = pass.  Built and run by tests/test_c_abi.py. */
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <cuda_runtime_api.h>

#include "wpgrid.h"

#define CHECK(cond, ...) do { if (!(cond)) { fprintf(stderr, "FAIL %s:%d: ", __FILE__, __LINE__); fprintf(stderr, __VA_ARGS__); fprintf(stderr, "\n"); return 1; } } while (0)

int main(void) {
    wpg_ctx *ctx = NULL;
    int rc = wpg_create(&ctx, 0, NULL);
    CHECK(rc == WPG_OK, "wpg_create rc=%d (%s)", rc, wpg_last_error(NULL));

    wpg_kdesc d;
    memset(&d, 0, sizeof d);
    d.Nw = 2; d.oversample = 8; d.grid_N = 64; d.w_max = 0.0; d.cell = 0.08 / 64; d.support_max = 8;
    d.support = NULL; d.plane_offset = NULL;
    const long long nk = wpg_wkernel_elems(d.Nw, 8, d.oversample);
    CHECK(nk == 2LL * 64 * 64, "wpg_wkernel_elems = %lld", nk);

    void *dK = NULL, *dws = NULL, *dgrid = NULL, *dimg = NULL;
    const size_t kws = wpg_wkernel_workspace_bytes(&d);
    CHECK(kws > 0, "wkernel workspace 0");
    CHECK(cudaMalloc(&dK, (size_t)nk * 8) == cudaSuccess && cudaMalloc(&dws, kws) == cudaSuccess, "cudaMalloc");
    rc = wpg_wkernel_build(ctx, &d, WPG_F32, dK, dws, kws);
    CHECK(rc == WPG_OK, "wpg_wkernel_build rc=%d (%s)", rc, wpg_last_error(ctx));
    rc = wpg_wkernel_build(ctx, &d, WPG_F32, dK, dws, 16);
    CHECK(rc == WPG_ENOMEM, "small workspace: rc=%d, expected WPG_ENOMEM", rc);
    cudaFree(dws);

    /* two rows, one channel at wavelength units (freq = c0): (0, 0, 0) on a cell, and one far off the grid */
    const double uvw[6] = {0.0, 0.0, 0.0, 1.0e6, 0.0, 0.0};
    const float vis[4] = {2.0f, -1.0f, 5.0f, 5.0f};
    const float wt[2] = {0.5f, 1.0f};
    const double freq[1] = {299792458.0};
    void *dv, *du, *dw, *df;
    CHECK(cudaMalloc(&dv, sizeof vis) == cudaSuccess && cudaMalloc(&du, sizeof uvw) == cudaSuccess &&
          cudaMalloc(&dw, sizeof wt) == cudaSuccess && cudaMalloc(&df, sizeof freq) == cudaSuccess, "cudaMalloc");
    cudaMemcpy(dv, vis, sizeof vis, cudaMemcpyHostToDevice); cudaMemcpy(du, uvw, sizeof uvw, cudaMemcpyHostToDevice);
    cudaMemcpy(dw, wt, sizeof wt, cudaMemcpyHostToDevice); cudaMemcpy(df, freq, sizeof freq, cudaMemcpyHostToDevice);
    const size_t gbytes = (size_t)64 * 64 * 8;
    CHECK(cudaMalloc(&dgrid, gbytes) == cudaSuccess, "cudaMalloc grid");
    cudaMemset(dgrid, 0, gbytes);
    const size_t gws = wpg_grid_workspace_bytes(ctx, 2, 1, &d, WPG_F32);
    CHECK(gws > 0 && cudaMalloc(&dws, gws) == cudaSuccess, "grid workspace");
    wpg_stats st;
    rc = wpg_grid(ctx, dv, (const double *)du, (const float *)dw, (const double *)df, 2, 1, dK, &d, WPG_F32, dgrid, dws, gws, &st);
    CHECK(rc == WPG_OK, "wpg_grid rc=%d (%s)", rc, wpg_last_error(ctx));
    CHECK(st.n_gridded == 1 && st.n_skipped_oob == 1 && st.n_skipped_zero_weight == 0 && st.n_updates == 64,
          "stats %lld %lld %lld %lld", (long long)st.n_gridded, (long long)st.n_skipped_oob,
          (long long)st.n_skipped_zero_weight, (long long)st.n_updates);
    float *hg = (float *)malloc(gbytes);
    cudaMemcpy(hg, dgrid, gbytes, cudaMemcpyDeviceToHost);
    double sre = 0.0, sim = 0.0; int nz = 0;
    for (int i = 0; i < 64 * 64; ++i) { sre += hg[2 * i]; sim += hg[2 * i + 1]; nz += (hg[2 * i] != 0.0f || hg[2 * i + 1] != 0.0f); }
    /* on-cell slice of a w = 0 stack sums to 1 (K5): sum of the grid = weight * vis */
    CHECK(fabs(sre - 1.0) < 1e-5 && fabs(sim + 0.5) < 1e-5, "flux: %.8f %+.8f, expected 1 -0.5", sre, sim);
    CHECK(nz > 0 && nz <= 64, "%d non-zero cells, expected 1..64", nz);
    rc = wpg_grid(ctx, dv, (const double *)du, (const float *)dw, (const double *)df, 2, 1, dK, &d, WPG_F32, dgrid, dws, 64, NULL);
    CHECK(rc == WPG_ENOMEM, "small grid workspace: rc=%d", rc);
    cudaFree(dws);

    const size_t iws = wpg_dirty_image_workspace_bytes(64, WPG_F32);
    CHECK(iws > 0 && cudaMalloc(&dws, iws) == cudaSuccess && cudaMalloc(&dimg, (size_t)64 * 64 * 4) == cudaSuccess, "image buffers");
    rc = wpg_dirty_image(ctx, dgrid, &d, 0.5, WPG_F32, dimg, dws, iws);
    CHECK(rc == WPG_OK, "wpg_dirty_image rc=%d (%s)", rc, wpg_last_error(ctx));
    float *himg = (float *)malloc((size_t)64 * 64 * 4);
    CHECK(cudaMemcpy(himg, dimg, (size_t)64 * 64 * 4, cudaMemcpyDeviceToHost) == cudaSuccess, "copy image");
    /* a visibility 2 - i at (u, v) = 0 with weight 1/2, normalised by the weight sum: a flat image of value Re(vis) = 2
     * where the taper correction is defined (centre pixel: exact up to the kernel's truncation) */
    CHECK(fabs(himg[32 * 64 + 32] - 2.0f) < 2e-3f, "image centre %.6f, expected 2", himg[32 * 64 + 32]);

    rc = wpg_set_option(ctx, "no_such_option", 1);
    CHECK(rc == WPG_EINVAL, "unknown option rc=%d", rc);
    free(hg); free(himg);
    cudaFree(dK); cudaFree(dws); cudaFree(dgrid); cudaFree(dimg); cudaFree(dv); cudaFree(du); cudaFree(dw); cudaFree(df);
    wpg_destroy(ctx);
    printf("abi_smoke OK\n");
    return 0;
}
