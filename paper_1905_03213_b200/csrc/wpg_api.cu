// C-ABI entry points of libwpgrid.so: context, argument checks, workspace planning, sequencing.
// The arithmetic lives in wpg_bin.cu (a1), wpg_grid.cu (a2), wpg_wkernel.cu (a0), wpg_image.cu (a3).
#include <algorithm>
#include <cstdarg>
#include <cstdio>
#include <cstring>

#include "wpg_common.h"

static thread_local std::string g_create_err;

int wpg_fail(wpg_ctx *ctx, int code, const char *fmt, ...) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    if (ctx) ctx->err = buf; else g_create_err = buf;
    return code;
}

extern "C" int wpg_version(void) { return 100; }

extern "C" int wpg_create(wpg_ctx **out, int device, void *cuda_stream) {
    if (!out) return wpg_fail(nullptr, WPG_EINVAL, "wpg_create: out is NULL");
    *out = nullptr;
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev == 0)
        return wpg_fail(nullptr, WPG_ECUDA, "wpg_create: no CUDA device (%s); there is no CPU fallback",
                        e == cudaSuccess ? "count = 0" : cudaGetErrorString(e));
    if (device < 0 || device >= ndev) return wpg_fail(nullptr, WPG_EINVAL, "wpg_create: bad device %d", device);
    wpg_ctx *ctx = new wpg_ctx();
    ctx->device = device;
    ctx->stream = (cudaStream_t)cuda_stream;
    DeviceGuard guard(device);             // the caller's current device is restored on return
    if (guard.err != cudaSuccess ||
        cudaDeviceGetAttribute(&ctx->sm_count, cudaDevAttrMultiProcessorCount, device) != cudaSuccess) {
        delete ctx;
        return wpg_fail(nullptr, WPG_ECUDA, "wpg_create: cannot select device %d", device);
    }
    *out = ctx;
    return WPG_OK;
}

extern "C" void wpg_destroy(wpg_ctx *ctx) {
    if (!ctx) return;
    DeviceGuard guard(ctx->device);
    for (auto &e : ctx->ev) cudaEventDestroy(e);
    for (int i = 0; i < 3; ++i) {
        if (ctx->side[i]) cudaStreamDestroy(ctx->side[i]);
        if (ctx->ev_join[i]) cudaEventDestroy(ctx->ev_join[i]);
    }
    if (ctx->ev_fork) cudaEventDestroy(ctx->ev_fork);
    if (ctx->copy_stream) cudaStreamDestroy(ctx->copy_stream);
    if (ctx->ev_start) cudaEventDestroy(ctx->ev_start);
    for (int i = 0; i < 4; ++i) if (ctx->ev_chunk[i]) cudaEventDestroy(ctx->ev_chunk[i]);
    if (ctx->plan) cufftDestroy(ctx->plan);
    if (ctx->d_host_scratch) cudaFree(ctx->d_host_scratch);
    delete ctx;
}

extern "C" const char *wpg_last_error(const wpg_ctx *ctx) {
    return ctx ? ctx->err.c_str() : g_create_err.c_str();
}

extern "C" int wpg_set_option(wpg_ctx *ctx, const char *name, int64_t value) {
    if (!ctx || !name) return WPG_EINVAL;
    if (!strcmp(name, "segment")) { if (value < 0 || value > (1 << 20)) return wpg_fail(ctx, WPG_EINVAL, "segment must be 0..2^20"); ctx->opt_segment = (int)value; }
    else if (!strcmp(name, "ctas_per_sm")) { if (value < 0 || value > 32) return wpg_fail(ctx, WPG_EINVAL, "ctas_per_sm must be 0..32"); ctx->opt_ctas_per_sm = (int)value; }
    else if (!strcmp(name, "key_bits")) { if (value != 0 && (value < 8 || value > 28)) return wpg_fail(ctx, WPG_EINVAL, "key_bits must be 0 or 8..28"); ctx->opt_key_bits = (int)value; }
    else if (!strcmp(name, "timing")) { ctx->opt_timing = value != 0; }
    else if (!strcmp(name, "no_pairs")) { ctx->opt_no_pairs = value != 0; }
    else if (!strcmp(name, "compress")) { ctx->opt_compress = value != 0; }
    else if (!strcmp(name, "chunk_sort")) { ctx->opt_chunk_sort = value != 0; }
    else if (!strcmp(name, "bin_tile")) { if (value < 0 || value > 65536) return wpg_fail(ctx, WPG_EINVAL, "bin_tile must be 0..65536"); ctx->opt_bin_tile = (int)value; }
    else if (!strcmp(name, "row_block")) { if (value < 0) return wpg_fail(ctx, WPG_EINVAL, "row_block must be >= 0"); ctx->opt_row_block = value; }
    else return wpg_fail(ctx, WPG_EINVAL, "unknown option '%s'", name);
    return WPG_OK;
}

int wpg_check_desc(wpg_ctx *ctx, const wpg_kdesc *d) {
    if (!d) return wpg_fail(ctx, WPG_EINVAL, "kernel descriptor is NULL");
    if (d->Nw < 1 || d->Nw > WPG_MAX_NW) return wpg_fail(ctx, WPG_EINVAL, "Nw = %d outside 1..%d", d->Nw, WPG_MAX_NW);
    if (d->oversample < 1 || d->oversample > 64) return wpg_fail(ctx, WPG_EINVAL, "oversample = %d outside 1..64", d->oversample);
    if (d->grid_N < 2 || d->grid_N > WPG_MAX_N) return wpg_fail(ctx, WPG_EINVAL, "grid_N = %d outside 2..%d", d->grid_N, WPG_MAX_N);
    if (!(d->cell > 0.0)) return wpg_fail(ctx, WPG_EINVAL, "cell must be > 0");
    if (!(d->w_max >= 0.0)) return wpg_fail(ctx, WPG_EINVAL, "w_max must be >= 0");
    if ((d->support == nullptr) != (d->plane_offset == nullptr))
        return wpg_fail(ctx, WPG_EINVAL, "support and plane_offset must both be given or both be NULL");
    int64_t off = 0;
    for (int p = 0; p < d->Nw; ++p) {
        int S = d->support ? d->support[p] : d->support_max;
        if (S < 1 || S > WPG_MAX_S) return wpg_fail(ctx, WPG_EINVAL, "support[%d] = %d outside 1..%d", p, S, WPG_MAX_S);
        if (S > d->grid_N) return wpg_fail(ctx, WPG_EINVAL, "support %d larger than the grid %d", S, d->grid_N);
        if ((S * d->oversample) % 2) return wpg_fail(ctx, WPG_EINVAL, "support*oversample = %d*%d must be even", S, d->oversample);
        if (S > d->support_max) return wpg_fail(ctx, WPG_EINVAL, "support[%d] = %d exceeds support_max %d", p, S, d->support_max);
        if (d->plane_offset && d->plane_offset[p] != off)
            return wpg_fail(ctx, WPG_EINVAL, "plane_offset[%d] = %lld, expected %lld (planes are concatenated)", p,
                            (long long)d->plane_offset[p], (long long)off);
        off += (int64_t)d->oversample * d->oversample * S * S;
    }
    if (d->plane_offset && d->plane_offset[d->Nw] != off) return wpg_fail(ctx, WPG_EINVAL, "plane_offset[Nw] inconsistent");
    if (off >= (int64_t)1 << 31) return wpg_fail(ctx, WPG_EINVAL, "kernel stack has %lld elements, limit 2^31", (long long)off);
    return WPG_OK;
}

static size_t align_up(size_t x) { return (x + 255) & ~(size_t)255; }

int wpg_make_plan(wpg_ctx *ctx, const wpg_kdesc *d, int64_t nrow, int nchan, wpg_prec prec,
                  PlaneTab *tab, BinParams *bp, WorkspaceLayout *ws) {
    int rc = wpg_check_desc(ctx, d);
    if (rc) return rc;
    if (nrow < 0 || nchan < 1) return wpg_fail(ctx, WPG_EINVAL, "nrow = %lld, nchan = %d", (long long)nrow, nchan);
    if (prec != WPG_F32 && prec != WPG_F64) return wpg_fail(ctx, WPG_EINVAL, "bad precision %d", (int)prec);
    int64_t nvis = nrow * nchan;
    if (nvis >= ((int64_t)1 << 32) - 2) return wpg_fail(ctx, WPG_EINVAL, "nrow*nchan = %lld exceeds 2^32 - 2 per call; chunk the input", (long long)nvis);
    memset(tab, 0, sizeof *tab);
    int64_t off = 0;
    std::vector<int> distinct;
    for (int p = 0; p < d->Nw; ++p) {
        int S = d->support ? d->support[p] : d->support_max;
        tab->off[p] = (int32_t)off;
        tab->S[p] = (uint8_t)S;
        off += (int64_t)d->oversample * d->oversample * S * S;
        if (std::find(distinct.begin(), distinct.end(), S) == distinct.end()) distinct.push_back(S);
    }
    tab->off[d->Nw] = (int32_t)off;
    std::sort(distinct.begin(), distinct.end());
    if ((int)distinct.size() > WPG_MAX_CLS)
        return wpg_fail(ctx, WPG_EINVAL, "%d distinct supports, limit %d", (int)distinct.size(), WPG_MAX_CLS);
    for (int p = 0; p < d->Nw; ++p)
        tab->cls[p] = (uint8_t)(std::find(distinct.begin(), distinct.end(), (int)tab->S[p]) - distinct.begin());
    for (size_t c = 0; c < distinct.size(); ++c) tab->clsS[c] = (uint8_t)distinct[c];

    memset(bp, 0, sizeof *bp);
    bp->nrow = nrow; bp->nchan = nchan;
    // time-coherent thread mapping only if it is well formed and leaves enough parallelism
    bp->vis_block = 0;
    if (ctx->opt_row_block > 0 && ctx->opt_row_block * nchan < ((int64_t)1 << 31) && nvis >= 64 * ctx->opt_row_block * nchan)
        bp->vis_block = (uint32_t)(ctx->opt_row_block * nchan);
    bp->row_block = bp->vis_block ? (uint32_t)ctx->opt_row_block : 0u;
    bp->vis_nbx = (bp->vis_block + 255u) / 256u;
    bp->vis_ngroups = bp->vis_block ? (uint32_t)(((nvis + bp->vis_block - 1) / bp->vis_block + 3) / 4) : 0u;     // kVpt = 4 (wpg_bin.cu)
    // block tile of the binning passes: a power of two, default 16, raised until the number of tiles fits grid.y
    bp->vis_tile_shift = 4;
    if (ctx->opt_bin_tile > 0) { bp->vis_tile_shift = 0; while ((2u << bp->vis_tile_shift) <= (uint32_t)ctx->opt_bin_tile) bp->vis_tile_shift++; }
    while (bp->vis_tile_shift < 30 && ((bp->vis_ngroups + (1u << bp->vis_tile_shift) - 1) >> bp->vis_tile_shift) > 65535u) bp->vis_tile_shift++;
    bp->vis_tile = 1u << bp->vis_tile_shift;
    bp->chan_shift = -1;
    for (int sft = 0; sft < 16; ++sft) if ((1 << sft) == nchan) bp->chan_shift = sft;
    bp->N = d->grid_N; bp->Q = d->oversample; bp->Nw = d->Nw;
    bp->w_max = d->w_max;
    bp->dw = 2.0 * d->w_max / (double)d->Nw;
    double fov = (double)d->grid_N * d->cell;
    bp->du = 1.0 / fov;
    bp->halfN = (double)(d->grid_N / 2);
    bp->rdu = 1.0 / bp->du;
    bp->rdw = bp->dw > 0.0 ? 1.0 / bp->dw : 0.0;
    bp->invQ = 1.0 / (double)d->oversample;
    bp->qshift = -1;
    for (int sft = 0; sft < 7; ++sft) if ((1 << sft) == d->oversample) bp->qshift = sft;
    bp->ncls = (int)distinct.size();
    bp->compress = ctx->opt_compress;
    bp->S0 = distinct[0];
    // sort key = (class, j0u, j0v >> kshift): the visibilities are swept column by column of window starts,
    // down the v axis, so a window that moves on leaves whole grid-row segments behind (contiguous write-outs)
    // and keeps its column ownership (the parity of j0u is fixed within a sweep); full resolution unless the
    // key space would exceed 2^key_bits
    // (ragged stacks multiply the key space by the number of support classes: their budget is set further down)
    // Default cap of a uniform stack: 2^24 keys (a 64 MB offset table; at 2^26 the binning of N = 8192 takes twice as
    // long).  Where full resolution does not fit (N > 4096) the cap follows the data instead — about 16 records per
    // key, 2^20 .. 2^24 — and the chunk sort (wpg_bin.cu, pass 4) restores the fine order inside the buckets: measured
    // on config 3 at N = 8192, 2^22 keys + chunk sort beat 2^24 keys without it by 10 % of the step.
    int def_bits = 24;
    if (bp->ncls == 1 && ctx->opt_chunk_sort && (int64_t)d->grid_N * d->grid_N > ((int64_t)1 << 24)) {
        def_bits = 20;
        while (def_bits < 24 && ((int64_t)16 << def_bits) < nvis) ++def_bits;
    }
    const int64_t cap = (int64_t)1 << (ctx->opt_key_bits ? ctx->opt_key_bits : (bp->ncls > 1 ? 26 : def_bits));
    int kshift = 0;
    while ((int64_t)bp->ncls * d->grid_N * (((int64_t)d->grid_N + (1 << kshift) - 1) >> kshift) > cap && kshift < 13) ++kshift;
    bp->kshift = kshift;
    bp->nkg = (d->grid_N + (1 << kshift) - 1) >> kshift;
    bp->keys_per_class = (uint32_t)((int64_t)d->grid_N * bp->nkg);
    int64_t nkeys = (int64_t)bp->ncls * bp->keys_per_class;
    // ragged stacks: the key space is a budget (see below, or 2^key_bits) split among the classes on
    // the device, after a census, so that the classes that hold the visibilities get the resolution
    bp->dyn_keys = bp->ncls > 1;
    if (bp->dyn_keys) {
        // default budget: about one key per visibility, 2^24 .. 2^27 (measured on config 4: at 4e7 visibilities
        // 2^26 beats 2^25, at 3.8e8 2^27 beats 2^26 — the finer windows save the gridder more than the larger
        // offset table costs the binning)
        int bits = 24;
        while (bits < 27 && ((int64_t)1 << bits) < nvis) ++bits;
        nkeys = (int64_t)1 << (ctx->opt_key_bits ? ctx->opt_key_bits : bits);
        if (nkeys < (int64_t)bp->ncls * d->grid_N) nkeys = (int64_t)bp->ncls * d->grid_N;
    }
    if (nkeys > ((int64_t)1 << 30)) return wpg_fail(ctx, WPG_EINVAL, "sort key space %lld too large", (long long)nkeys);
    bp->nkeys = (uint32_t)nkeys;

    memset(ws, 0, sizeof *ws);
    ws->nkeys = (uint32_t)nkeys;
    ws->nblocks_scan = (uint32_t)((nkeys + 1 + 4095) / 4096);
    size_t rec = prec == WPG_F32 ? sizeof(Rec<float>) : sizeof(Rec<double>);
    size_t o = 0;
    ws->off_counters = o; o += align_up(sizeof(Counters));
    ws->off_hist = o + 12; o += align_up((size_t)(nkeys + 8) * 4);    // bucket_start[0..nkeys]; [1..] is 16-byte aligned
    ws->off_blocksum = o; o += align_up((size_t)ws->nblocks_scan * 4 + 8);
    ws->off_fscale = o;   o += align_up((size_t)nchan * 8);
    ws->off_records = o;  o += align_up((size_t)nvis * rec);
    ws->total = o;
    return WPG_OK;
}

extern "C" size_t wpg_grid_workspace_bytes(const wpg_ctx *ctx, int64_t nrow, int nchan, const wpg_kdesc *desc,
                                           wpg_prec prec) {
    PlaneTab tab; BinParams bp; WorkspaceLayout ws;
    wpg_ctx tmp;
    if (ctx) { tmp.opt_segment = ctx->opt_segment; tmp.opt_key_bits = ctx->opt_key_bits; tmp.opt_chunk_sort = ctx->opt_chunk_sort; }
    if (wpg_make_plan(&tmp, desc, nrow, nchan, prec, &tab, &bp, &ws)) return 0;
    return ws.total;
}

static int read_stats(wpg_ctx *ctx, const Counters *d_c, wpg_stats *out, Counters *h_opt) {
    Counters h;
    WPG_CUDA(ctx, cudaMemcpyAsync(&h, d_c, sizeof h, cudaMemcpyDeviceToHost, ctx->stream));
    WPG_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    if (out) {
        memset(out, 0, sizeof *out);
        for (int s = 0; s < kStatSlots; ++s) {
            out->n_gridded += (int64_t)h.n_gridded[s]; out->n_skipped_oob += (int64_t)h.n_skipped_oob[s];
            out->n_skipped_zero_weight += (int64_t)h.n_skipped_zero_weight[s];
            out->n_clamped_w += (int64_t)h.n_clamped_w[s]; out->n_updates += (int64_t)h.n_updates[s];
        }
    }
    if (h_opt) *h_opt = h;
    return WPG_OK;
}

static int check_ptrs(wpg_ctx *ctx, const void *vis, const void *uvw, const void *wt, const void *freq, int64_t nrow) {
    if (!ctx) return WPG_EINVAL;
    if (nrow > 0 && (!vis || !uvw || !wt)) return wpg_fail(ctx, WPG_EINVAL, "NULL input pointer");
    if (!freq) return wpg_fail(ctx, WPG_EINVAL, "freq is NULL");
    return WPG_OK;
}

extern "C" int64_t wpg_launch_count(const wpg_ctx *ctx) { return ctx ? ctx->n_launches : 0; }

extern "C" int wpg_phase_ms(wpg_ctx *ctx, double *out) {
    if (!ctx || !out) return WPG_EINVAL;
    if (!ctx->ev_used) return wpg_fail(ctx, WPG_EINVAL, "no timed wpg_grid call (set option \"timing\" = 1 first)");
    WPG_CUDA(ctx, cudaEventSynchronize(ctx->ev[3 * ctx->ev_used - 1]));
    double a = 0.0, b = 0.0;
    for (size_t i = 0; i < ctx->ev_used; ++i) {
        float x = 0.f, y = 0.f;
        WPG_CUDA(ctx, cudaEventElapsedTime(&x, ctx->ev[3 * i], ctx->ev[3 * i + 1]));
        WPG_CUDA(ctx, cudaEventElapsedTime(&y, ctx->ev[3 * i + 1], ctx->ev[3 * i + 2]));
        a += x; b += y;
    }
    out[0] = a / (double)ctx->ev_used; out[1] = b / (double)ctx->ev_used;
    ctx->ev_used = 0;
    return WPG_OK;
}

// Event i (0 start, 1 after binning, 2 after gridder) of the current timed call.
int wpg_mark(wpg_ctx *ctx, int i) {
    if (!ctx->opt_timing) return WPG_OK;
    if (i == 0 && ctx->ev_used >= 4096) ctx->ev_used = 0;       // pool bound: start over
    size_t k = 3 * ctx->ev_used + (size_t)i;
    while (ctx->ev.size() <= k) {
        cudaEvent_t e;
        WPG_CUDA(ctx, cudaEventCreate(&e));
        ctx->ev.push_back(e);
    }
    WPG_CUDA(ctx, cudaEventRecord(ctx->ev[k], ctx->stream));
    if (i == 2) ctx->ev_used += 1;
    return WPG_OK;
}

static int bin_common(wpg_ctx *ctx, const void *d_vis, const double *d_uvw, const float *d_weight,
                      const double *d_freq, int64_t nrow, int nchan, const wpg_kdesc *desc, wpg_prec prec,
                      void *d_workspace, size_t workspace_bytes, PlaneTab *tab, BinParams *bp, WorkspaceLayout *ws) {
    int rc = check_ptrs(ctx, d_vis, d_uvw, d_weight, d_freq, nrow);
    if (rc) return rc;
    rc = wpg_make_plan(ctx, desc, nrow, nchan, prec, tab, bp, ws);
    if (rc) return rc;
    if (!d_workspace || workspace_bytes < ws->total)
        return wpg_fail(ctx, WPG_ENOMEM, "workspace of %zu bytes given, %zu needed", workspace_bytes, ws->total);
    if ((rc = wpg_mark(ctx, 0))) return rc;
    char *w = (char *)d_workspace;
    // counters + histogram are contiguous at the head of the workspace
    WPG_CUDA(ctx, cudaMemsetAsync(w, 0, ws->off_blocksum, ctx->stream));
    return wpg_launch_bin(ctx, d_vis, d_uvw, d_weight, d_freq, *tab, *bp, *ws, prec, w);
}

extern "C" int wpg_bin(wpg_ctx *ctx, const void *d_vis, const double *d_uvw, const float *d_weight,
                       const double *d_freq, int64_t nrow, int nchan, const wpg_kdesc *desc, wpg_prec prec,
                       void *d_workspace, size_t workspace_bytes, wpg_bin_info *info, wpg_stats *h_stats) {
    if (!ctx) return WPG_EINVAL;
    WPG_DEVICE(ctx);
    PlaneTab tab; BinParams bp; WorkspaceLayout ws;
    int rc = bin_common(ctx, d_vis, d_uvw, d_weight, d_freq, nrow, nchan, desc, prec, d_workspace, workspace_bytes, &tab, &bp, &ws);
    if (rc) return rc;
    Counters h;
    rc = read_stats(ctx, (const Counters *)((char *)d_workspace + ws.off_counters), h_stats, &h);
    if (rc) return rc;
    if (info) {
        info->n_records = h.n_records; info->n_keys = ws.nkeys;
        info->n_classes = bp.ncls; info->key_shift = bp.dyn_keys ? -1 : bp.kshift;
        info->record_bytes = prec == WPG_F32 ? 16 : 24; info->keys_per_class = (int32_t)bp.keys_per_class;
        info->off_records = (int64_t)ws.off_records; info->off_bucket_start = (int64_t)ws.off_hist;
    }
    return WPG_OK;
}

extern "C" int wpg_grid(wpg_ctx *ctx, const void *d_vis, const double *d_uvw, const float *d_weight,
                        const double *d_freq, int64_t nrow, int nchan, const void *d_kernels,
                        const wpg_kdesc *desc, wpg_prec prec, void *d_grid,
                        void *d_workspace, size_t workspace_bytes, wpg_stats *h_stats) {
    if (!ctx) return WPG_EINVAL;
    if (!d_kernels || !d_grid) return wpg_fail(ctx, WPG_EINVAL, "kernels or grid pointer is NULL");
    WPG_DEVICE(ctx);
    PlaneTab tab; BinParams bp; WorkspaceLayout ws;
    int rc = bin_common(ctx, d_vis, d_uvw, d_weight, d_freq, nrow, nchan, desc, prec, d_workspace, workspace_bytes, &tab, &bp, &ws);
    if (rc) return rc;
    if ((rc = wpg_mark(ctx, 1))) return rc;
    rc = wpg_launch_grid(ctx, tab, bp, ws, prec, d_kernels, d_grid, (char *)d_workspace);
    if (rc) return rc;
    if ((rc = wpg_mark(ctx, 2))) return rc;
    if (h_stats) return read_stats(ctx, (const Counters *)((char *)d_workspace + ws.off_counters), h_stats, nullptr);
    return WPG_OK;
}

// ---- polarised gridder
static int pol_plan(wpg_ctx *ctx, const wpg_kdesc *desc, int64_t nrow, int nchan, int npol, wpg_prec prec, PlaneTab *tab,
                    BinParams *bp, WorkspaceLayout *ws) {
    if (npol != 2 && npol != 4) return wpg_fail(ctx, WPG_EINVAL, "npol = %d: 2 or 4 correlations", npol);
    int rc = wpg_make_plan(ctx, desc, nrow, nchan, prec, tab, bp, ws);
    if (rc) return rc;
    const size_t recb = (prec == WPG_F32 ? 8 : 16) * (size_t)npol + 8;
    ws->total = ws->off_records + align_up((size_t)nrow * nchan * recb);
    return WPG_OK;
}

extern "C" size_t wpg_grid_pol_workspace_bytes(const wpg_ctx *ctx, int64_t nrow, int nchan, int npol, const wpg_kdesc *desc,
                                               wpg_prec prec) {
    PlaneTab tab; BinParams bp; WorkspaceLayout ws;
    wpg_ctx tmp;
    if (ctx) { tmp.opt_key_bits = ctx->opt_key_bits; }
    if (pol_plan(&tmp, desc, nrow, nchan, npol, prec, &tab, &bp, &ws)) return 0;
    return ws.total;
}

extern "C" int wpg_grid_pol(wpg_ctx *ctx, const void *d_vis, const double *d_uvw, const float *d_weight,
                            const double *d_freq, int64_t nrow, int nchan, int npol, const void *d_kernels,
                            const wpg_kdesc *desc, wpg_prec prec, void *d_grid, void *d_workspace, size_t workspace_bytes,
                            wpg_stats *h_stats) {
    int rc = check_ptrs(ctx, d_vis, d_uvw, d_weight, d_freq, nrow);
    if (rc) return rc;
    if (!d_kernels || !d_grid) return wpg_fail(ctx, WPG_EINVAL, "kernels or grid pointer is NULL");
    PlaneTab tab; BinParams bp; WorkspaceLayout ws;
    rc = pol_plan(ctx, desc, nrow, nchan, npol, prec, &tab, &bp, &ws);
    if (rc) return rc;
    if (!d_workspace || workspace_bytes < ws.total)
        return wpg_fail(ctx, WPG_ENOMEM, "workspace of %zu bytes given, %zu needed", workspace_bytes, ws.total);
    WPG_DEVICE(ctx);
    char *w = (char *)d_workspace;
    if ((rc = wpg_mark(ctx, 0))) return rc;
    WPG_CUDA(ctx, cudaMemsetAsync(w, 0, ws.off_blocksum, ctx->stream));
    rc = wpg_launch_bin_pol(ctx, d_vis, d_uvw, d_weight, d_freq, tab, bp, ws, prec, npol, w);
    if (rc) return rc;
    if ((rc = wpg_mark(ctx, 1))) return rc;
    rc = wpg_launch_grid_pol(ctx, tab, bp, ws, prec, npol, d_kernels, d_grid, w);
    if (rc) return rc;
    if ((rc = wpg_mark(ctx, 2))) return rc;
    if (h_stats) return read_stats(ctx, (const Counters *)(w + ws.off_counters), h_stats, nullptr);
    return WPG_OK;
}

extern "C" int wpg_grid_naive(wpg_ctx *ctx, const void *d_vis, const double *d_uvw, const float *d_weight,
                              const double *d_freq, int64_t nrow, int nchan, const void *d_kernels,
                              const wpg_kdesc *desc, wpg_prec prec, void *d_grid, wpg_stats *h_stats) {
    int rc = check_ptrs(ctx, d_vis, d_uvw, d_weight, d_freq, nrow);
    if (rc) return rc;
    if (!d_kernels || !d_grid) return wpg_fail(ctx, WPG_EINVAL, "kernels or grid pointer is NULL");
    PlaneTab tab; BinParams bp; WorkspaceLayout ws;
    rc = wpg_make_plan(ctx, desc, nrow, nchan, prec, &tab, &bp, &ws);
    if (rc) return rc;
    WPG_DEVICE(ctx);
    Counters *d_c = nullptr;
    WPG_CUDA(ctx, cudaMallocAsync((void **)&d_c, sizeof(Counters), ctx->stream));
    WPG_CUDA(ctx, cudaMemsetAsync(d_c, 0, sizeof(Counters), ctx->stream));
    rc = wpg_launch_naive(ctx, d_vis, d_uvw, d_weight, d_freq, tab, bp, prec, d_kernels, d_grid, d_c);
    if (!rc && h_stats) rc = read_stats(ctx, d_c, h_stats, nullptr);
    cudaFreeAsync(d_c, ctx->stream);
    return rc;
}

extern "C" int wpg_grid_host(wpg_ctx *ctx, const void *h_vis, const double *h_uvw, const float *h_weight,
                             const double *h_freq, int64_t nrow, int nchan, const void *d_kernels,
                             const wpg_kdesc *desc, wpg_prec prec, void *h_grid_out, wpg_stats *h_stats,
                             void *h_image_out, double weight_sum) {
    int rc = check_ptrs(ctx, h_vis, h_uvw, h_weight, h_freq, nrow);
    if (rc) return rc;
    if (!d_kernels || !h_grid_out) return wpg_fail(ctx, WPG_EINVAL, "kernels or grid pointer is NULL");
    PlaneTab tab; BinParams bp; WorkspaceLayout ws;
    rc = wpg_make_plan(ctx, desc, nrow, nchan, prec, &tab, &bp, &ws);
    if (rc) return rc;
    WPG_DEVICE(ctx);
    int64_t nvis = nrow * nchan;
    size_t cplx = prec == WPG_F32 ? 8 : 16;
    size_t b_vis = align_up((size_t)nvis * 8), b_uvw = align_up((size_t)nrow * 24), b_wt = align_up((size_t)nvis * 4),
           b_freq = align_up((size_t)nchan * 8), b_grid = align_up((size_t)desc->grid_N * desc->grid_N * cplx);
    size_t b_img = h_image_out ? align_up(wpg_dirty_image_workspace_bytes(desc->grid_N, prec)) +
                                     align_up((size_t)desc->grid_N * desc->grid_N * (cplx / 2)) : 0;
    size_t need = b_vis + b_uvw + b_wt + b_freq + b_grid + std::max(ws.total, b_img);
    if (need > ctx->host_scratch_bytes) {
        WPG_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
        if (ctx->d_host_scratch) cudaFree(ctx->d_host_scratch);
        ctx->d_host_scratch = nullptr; ctx->host_scratch_bytes = 0;
        cudaError_t e = cudaMalloc(&ctx->d_host_scratch, need);
        if (e != cudaSuccess) return wpg_fail(ctx, WPG_ENOMEM, "cannot allocate %zu bytes of device scratch: %s", need, cudaGetErrorString(e));
        ctx->host_scratch_bytes = need;
    }
    char *base = (char *)ctx->d_host_scratch;
    char *dv = base, *du = dv + b_vis, *dw = du + b_uvw, *df = dw + b_wt, *dg = df + b_freq, *dws = dg + b_grid;
    cudaStream_t s = ctx->stream;
    // Pipeline over row chunks: gridding is additive (P12), so chunk k is binned and gridded into the same grid
    // while chunk k + 1 is still crossing PCIe on the copy stream; only the last chunk's compute is exposed.
    if (!ctx->copy_stream) {
        WPG_CUDA(ctx, cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking));
        WPG_CUDA(ctx, cudaEventCreateWithFlags(&ctx->ev_start, cudaEventDisableTiming));
        for (int i = 0; i < 4; ++i) WPG_CUDA(ctx, cudaEventCreateWithFlags(&ctx->ev_chunk[i], cudaEventDisableTiming));
    }
    const int nchunk = nrow >= (1 << 20) ? 4 : 1;
    int64_t rows_per = (nrow + nchunk - 1) / nchunk;
    if (ctx->opt_row_block > 0) rows_per = (rows_per + ctx->opt_row_block - 1) / ctx->opt_row_block * ctx->opt_row_block;
    WPG_CUDA(ctx, cudaEventRecord(ctx->ev_start, s));                       // the previous call has consumed the buffers
    WPG_CUDA(ctx, cudaStreamWaitEvent(ctx->copy_stream, ctx->ev_start, 0));
    WPG_CUDA(ctx, cudaMemcpyAsync(df, h_freq, (size_t)nchan * 8, cudaMemcpyHostToDevice, s));
    WPG_CUDA(ctx, cudaMemsetAsync(dg, 0, (size_t)desc->grid_N * desc->grid_N * cplx, s));
    for (int k = 0; k < nchunk; ++k) {
        const int64_t r0 = std::min(nrow, k * rows_per), r1 = std::min(nrow, r0 + rows_per);
        if (r1 > r0) {
            cudaStream_t c = ctx->copy_stream;
            WPG_CUDA(ctx, cudaMemcpyAsync(dv + r0 * nchan * 8, (const char *)h_vis + r0 * nchan * 8, (size_t)(r1 - r0) * nchan * 8, cudaMemcpyHostToDevice, c));
            WPG_CUDA(ctx, cudaMemcpyAsync(du + r0 * 24, (const char *)h_uvw + r0 * 24, (size_t)(r1 - r0) * 24, cudaMemcpyHostToDevice, c));
            WPG_CUDA(ctx, cudaMemcpyAsync(dw + r0 * nchan * 4, (const char *)h_weight + r0 * nchan * 4, (size_t)(r1 - r0) * nchan * 4, cudaMemcpyHostToDevice, c));
        }
        WPG_CUDA(ctx, cudaEventRecord(ctx->ev_chunk[k], ctx->copy_stream));
    }
    wpg_stats tot; memset(&tot, 0, sizeof tot);
    for (int k = 0; k < nchunk; ++k) {
        const int64_t r0 = std::min(nrow, k * rows_per), r1 = std::min(nrow, r0 + rows_per);
        WPG_CUDA(ctx, cudaStreamWaitEvent(s, ctx->ev_chunk[k], 0));
        if (r1 <= r0 && k > 0) continue;
        wpg_stats part; memset(&part, 0, sizeof part);
        rc = wpg_grid(ctx, dv + r0 * nchan * 8, (const double *)(du + r0 * 24), (const float *)(dw + r0 * nchan * 4),
                      (const double *)df, r1 - r0, nchan, d_kernels, desc, prec, dg, dws, ws.total, h_stats ? &part : nullptr);
        if (rc) return rc;
        tot.n_gridded += part.n_gridded; tot.n_skipped_oob += part.n_skipped_oob;
        tot.n_skipped_zero_weight += part.n_skipped_zero_weight; tot.n_clamped_w += part.n_clamped_w;
        tot.n_updates += part.n_updates;
    }
    if (h_stats) *h_stats = tot;
    WPG_CUDA(ctx, cudaMemcpyAsync(h_grid_out, dg, (size_t)desc->grid_N * desc->grid_N * cplx, cudaMemcpyDeviceToHost, s));
    if (h_image_out) {
        size_t b_fft = align_up(wpg_dirty_image_workspace_bytes(desc->grid_N, prec));
        char *dimg = dws + b_fft;
        rc = wpg_dirty_image(ctx, dg, desc, weight_sum, prec, dimg, dws, b_fft);
        if (rc) return rc;
        WPG_CUDA(ctx, cudaMemcpyAsync(h_image_out, dimg, (size_t)desc->grid_N * desc->grid_N * (cplx / 2), cudaMemcpyDeviceToHost, s));
    }
    WPG_CUDA(ctx, cudaStreamSynchronize(s));
    return WPG_OK;
}

// Row range of one rank (see wpgrid.h): units of row_block rows (or single rows) dealt out as evenly as possible,
// the first (units % world) ranks take one unit more.
extern "C" int wpg_shard_rows(int64_t nrow, int64_t row_block, int world, int rank, int64_t *row0, int64_t *row1) {
    if (!row0 || !row1 || world < 1 || rank < 0 || rank >= world || nrow < 0 || row_block < 0) return WPG_EINVAL;
    const int64_t unit = row_block > 0 ? row_block : 1;
    const int64_t units = (nrow + unit - 1) / unit;
    const int64_t base = units / world, extra = units % world;
    const int64_t u0 = rank * base + std::min<int64_t>(rank, extra);
    const int64_t u1 = u0 + base + (rank < extra ? 1 : 0);
    *row0 = std::min(nrow, u0 * unit);
    *row1 = std::min(nrow, u1 * unit);
    return WPG_OK;
}
