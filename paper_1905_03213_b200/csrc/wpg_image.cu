// Step a3 — dirty image: centre-origin inverse 2-D FFT of the grid, real part, / sum of weights,
// / taper ("the master node performs an IFFT on the ... gridding result";
// DESIGN.md O5, R11).  The fftshift/ifftshift pair is (-1)^(i+j) sign checkerboards before and after a
// plain transform (N even): img[n] = (-1)^(n1+n2) * IFFT_unnormalised[(-1)^(k1+k2) g[k]]  (the constant
// (-1)^N is 1).  The transform is cuFFT, out of place from the caller's grid (which is not modified).
#include "wpg_common.h"

namespace {

constexpr double kTaperFloor = 1e-3;

// f = plain (origin at index 0) unnormalised inverse FFT of the UNMODIFIED grid.  Modulating the input by
// (-1)^(k1+k2) is a shift of the output by N/2 in both axes, so the input checkerboard is an index offset
// here and costs no pass over the data; the output checkerboard is the sign below.
template <typename C, typename T>
__global__ void __launch_bounds__(256)
correct_kernel(const C *__restrict__ f, T *__restrict__ img, const double *__restrict__ taper, int N, double inv_wsum) {
    int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y;
    if (i >= N) return;
    const int h = N >> 1;
    const int is = i < h ? i + h : i - h, js = j < h ? j + h : j - h;
    double t = taper[i] * taper[j];
    double v = (double)f[(size_t)js * N + is].x;
    if ((i + j) & 1) v = -v;
    img[(size_t)j * N + i] = t >= kTaperFloor ? (T)(v * inv_wsum / t) : (T)0;
}

const char *cufft_str(cufftResult r) {
    switch (r) {
        case CUFFT_SUCCESS: return "CUFFT_SUCCESS";
        case CUFFT_ALLOC_FAILED: return "CUFFT_ALLOC_FAILED";
        case CUFFT_INVALID_VALUE: return "CUFFT_INVALID_VALUE";
        case CUFFT_INTERNAL_ERROR: return "CUFFT_INTERNAL_ERROR";
        case CUFFT_EXEC_FAILED: return "CUFFT_EXEC_FAILED";
        case CUFFT_SETUP_FAILED: return "CUFFT_SETUP_FAILED";
        case CUFFT_INVALID_SIZE: return "CUFFT_INVALID_SIZE";
        default: return "CUFFT error";
    }
}

}  // namespace

// workspace: the transform's output [N][N] complex, then the taper table psi[N] (fp64)
static size_t fft_bytes(int N, wpg_prec prec) { return (((size_t)N * N * (prec == WPG_F32 ? 8 : 16)) + 255) & ~(size_t)255; }
extern "C" size_t wpg_dirty_image_workspace_bytes(int grid_N, wpg_prec prec) {
    if (grid_N < 2) return 0;
    return fft_bytes(grid_N, prec) + (size_t)grid_N * 8;
}

extern "C" int wpg_dirty_image(wpg_ctx *ctx, const void *d_grid, const wpg_kdesc *desc, double weight_sum,
                               wpg_prec prec, void *d_image, void *d_workspace, size_t workspace_bytes) {
    if (!ctx) return WPG_EINVAL;
    int rc = wpg_check_desc(ctx, desc);
    if (rc) return rc;
    if (!d_grid || !d_image) return wpg_fail(ctx, WPG_EINVAL, "grid or image pointer is NULL");
    if (prec != WPG_F32 && prec != WPG_F64) return wpg_fail(ctx, WPG_EINVAL, "bad precision");
    const int N = desc->grid_N;
    if (N % 2) return wpg_fail(ctx, WPG_EINVAL, "dirty_image needs an even grid size, got %d", N);
    if (!(weight_sum > 0.0)) return wpg_fail(ctx, WPG_EINVAL, "weight_sum must be > 0");
    size_t need = wpg_dirty_image_workspace_bytes(N, prec);
    if (!d_workspace || workspace_bytes < need)
        return wpg_fail(ctx, WPG_ENOMEM, "workspace of %zu bytes given, %zu needed", workspace_bytes, need);
    WPG_DEVICE(ctx);
    if (ctx->plan_N != N || ctx->plan_prec != (int)prec) {
        if (ctx->plan) { cufftDestroy(ctx->plan); ctx->plan = 0; ctx->plan_N = 0; }
        cufftResult r = cufftPlan2d(&ctx->plan, N, N, prec == WPG_F32 ? CUFFT_C2C : CUFFT_Z2Z);
        if (r != CUFFT_SUCCESS) { ctx->plan = 0; return wpg_fail(ctx, WPG_ECUDA, "cufftPlan2d: %s", cufft_str(r)); }
        ctx->plan_N = N; ctx->plan_prec = (int)prec;
    }
    cufftResult r = cufftSetStream(ctx->plan, ctx->stream);
    if (r != CUFFT_SUCCESS) return wpg_fail(ctx, WPG_ECUDA, "cufftSetStream: %s", cufft_str(r));
    // taper psi(2 l_j / FoV), l_j = (j - N/2) cell: evaluated on the device into the caller's workspace (N values)
    double *d_taper = (double *)((char *)d_workspace + fft_bytes(N, prec));
    if ((rc = wpg_launch_taper(ctx, d_taper, N, 1.0 / N))) return rc;
    dim3 gr((N + 255) / 256, N);
    cudaStream_t s = ctx->stream;
    if (prec == WPG_F32) {
        r = cufftExecC2C(ctx->plan, (cufftComplex *)const_cast<void *>(d_grid), (cufftComplex *)d_workspace, CUFFT_INVERSE);
        if (r != CUFFT_SUCCESS) return wpg_fail(ctx, WPG_ECUDA, "cufftExecC2C: %s", cufft_str(r));
        correct_kernel<float2, float><<<gr, 256, 0, s>>>((const float2 *)d_workspace, (float *)d_image, d_taper, N, 1.0 / weight_sum);
    } else {
        r = cufftExecZ2Z(ctx->plan, (cufftDoubleComplex *)const_cast<void *>(d_grid), (cufftDoubleComplex *)d_workspace, CUFFT_INVERSE);
        if (r != CUFFT_SUCCESS) return wpg_fail(ctx, WPG_ECUDA, "cufftExecZ2Z: %s", cufft_str(r));
        correct_kernel<double2, double><<<gr, 256, 0, s>>>((const double2 *)d_workspace, (double *)d_image, d_taper, N, 1.0 / weight_sum);
    }
    ctx->n_launches += 1;
    WPG_CUDA(ctx, cudaGetLastError());
    return WPG_OK;
}
