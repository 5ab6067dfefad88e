// wpg_grid_static: wpg_grid (binning a1 + gridder a2) for callers that cannot allocate device
// memory and have no workspace to hand over — code under CUDA graph capture, tight serving loops, harnesses that
// forbid cudaMalloc.  The scratch wpg_grid wants from its caller (counters, bucket table, sorted records:
// wpg_grid_workspace_bytes) lives here in ONE file-scope device array of WPG_STATIC_SCRATCH_BYTES = 64 MiB; every
// GPU on which this library's module is loaded holds that array until the process exits.
//
// In host code the array's name is a host-side stand-in, not a device address: its device address is looked up once
// per device, with that device current, by cudaGetSymbolAddress and cached; that pointer is what the kernels get.
// Everything else is the existing path, unchanged: the call goes through wpg_grid with the array as its workspace, and
// wpg_grid clears what must start at zero (counters and bucket table) with a memset on the stream at every call — the
// array keeps the previous call's contents otherwise.  All calls on a device share the array: calls that overlap on
// the GPU (two contexts or streams) race; calls on one stream are ordered and safe.
#include <mutex>

#include "wpg_common.h"

namespace {

constexpr size_t kStaticScratchBytes = WPG_STATIC_SCRATCH_BYTES;      // wpgrid.h: 64 MiB
static __device__ __align__(256) unsigned char wpg_static_scratch[kStaticScratchBytes];

constexpr int kMaxDevices = 64;
std::mutex g_lock;
void *g_scratch_ptr[kMaxDevices] = {};          // device address of the array on each device, nullptr = not looked up yet

// the context's device must be current (WPG_DEVICE in the caller)
int scratch_address(wpg_ctx *ctx, void **out) {
    if (ctx->device < 0 || ctx->device >= kMaxDevices)
        return wpg_fail(ctx, WPG_EINVAL, "wpg_grid_static: device ordinal %d outside 0..%d", ctx->device, kMaxDevices - 1);
    std::lock_guard<std::mutex> guard(g_lock);
    if (!g_scratch_ptr[ctx->device]) {
        void *p = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&p, wpg_static_scratch);
        if (e != cudaSuccess || !p)
            return wpg_fail(ctx, WPG_ECUDA, "wpg_grid_static: cudaGetSymbolAddress of the static scratch failed on device %d: %s",
                            ctx->device, cudaGetErrorString(e));
        g_scratch_ptr[ctx->device] = p;
    }
    *out = g_scratch_ptr[ctx->device];
    return WPG_OK;
}

}  // namespace

extern "C" size_t wpg_static_scratch_bytes(void) { return kStaticScratchBytes; }

extern "C" int wpg_grid_static(wpg_ctx *ctx, const void *d_vis, const double *d_uvw, const float *d_weight,
                               const double *d_freq, int64_t nrow, int nchan, const void *d_kernels,
                               const wpg_kdesc *desc, wpg_prec prec, void *d_grid, wpg_stats *h_stats) {
    if (!ctx) return WPG_EINVAL;
    if (!desc) return wpg_fail(ctx, WPG_EINVAL, "wpg_grid_static: desc is NULL");
    // size check first (host arithmetic only): the same plan wpg_grid makes
    PlaneTab tab; BinParams bp; WorkspaceLayout ws;
    int rc = wpg_make_plan(ctx, desc, nrow, nchan, prec, &tab, &bp, &ws);
    if (rc) return rc;
    if (ws.total > kStaticScratchBytes)
        return wpg_fail(ctx, WPG_ENOMEM,
                        "wpg_grid_static: this problem needs %zu bytes of scratch (%lld visibilities, %u sort keys), the static "
                        "array holds %zu (WPG_STATIC_SCRATCH_BYTES); use wpg_grid with a caller-owned workspace or split the rows",
                        ws.total, (long long)(nrow * nchan), ws.nkeys, kStaticScratchBytes);
    WPG_DEVICE(ctx);
    void *scratch = nullptr;
    if ((rc = scratch_address(ctx, &scratch))) return rc;
    return wpg_grid(ctx, d_vis, d_uvw, d_weight, d_freq, nrow, nchan, d_kernels, desc, prec, d_grid, scratch,
                    kStaticScratchBytes, h_stats);
}
