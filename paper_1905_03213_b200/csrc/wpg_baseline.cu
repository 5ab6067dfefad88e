// The paper's own data order: baseline index Eq. (1), count array C, exclusive prefix
// sum Eq. (2), re-order "grouped by baseline and then ordered by time" — done on the device
// instead of on the host — and then the register-accumulating gridder walking each baseline's time series
// (PAPER.md:80, 84).  It reaches the same grid as wpg_grid (the sum is order-independent); it exists to compare
// the paper's ordering with the position sort of wpg_bin.cu on the track-based workloads.
#include <cstring>

#include "wpg_common.h"

namespace {

constexpr int kMaxSeg = 8192;          // rows of one baseline that the shared-memory sort takes

// Eq. (1):  I_B = (-S^2 + 2 S N_ant + S) / 2 + |I_ant1 - I_ant2|,  S = min(I_ant1, I_ant2)
__device__ __forceinline__ unsigned baseline_index(int a1, int a2, int n_ant) {
    const long long S = min(a1, a2);
    return (unsigned)((-S * S + 2 * S * n_ant + S) / 2 + abs(a1 - a2));
}

// Pass 1: I_B of every row and the count array C ("count the number of timestamps under the same
// baseline number ... store them in the array C").  status[0] counts rows with an antenna ID outside [0, N_ant).
__global__ void __launch_bounds__(256)
bl_count_kernel(const int *__restrict__ ant1, const int *__restrict__ ant2, int n_ant, long long nrow,
                unsigned *__restrict__ ib_out, unsigned *__restrict__ C, unsigned *__restrict__ status) {
    const long long r = (long long)blockIdx.x * 256 + threadIdx.x;
    if (r >= nrow) return;
    const int a1 = ant1[r], a2 = ant2[r];
    if (a1 < 0 || a2 < 0 || a1 >= n_ant || a2 >= n_ant) { atomicAdd(&status[0], 1u); ib_out[r] = 0xFFFFFFFFu; return; }
    const unsigned ib = baseline_index(a1, a2, n_ant);
    ib_out[r] = ib;
    atomicAdd(&C[ib], 1u);
}

// Pass 3: every row takes a slot inside its baseline's run [B_start[I_B], B_start[I_B + 1]); the order inside
// the run is whatever the atomics give — pass 4 puts it back into time (= input row) order.
__global__ void __launch_bounds__(256)
bl_scatter_kernel(const unsigned *__restrict__ ib, long long nrow, unsigned *__restrict__ cursor,
                  unsigned *__restrict__ perm) {
    const long long r = (long long)blockIdx.x * 256 + threadIdx.x;
    if (r >= nrow || ib[r] == 0xFFFFFFFFu) return;
    perm[atomicAdd(&cursor[ib[r]], 1u)] = (unsigned)r;
}

// Pass 4: one block per baseline sorts its run of row numbers ascending (bitonic, shared memory): "ordered by
// time".  status[1] counts baselines with more than kMaxSeg rows (left unsorted; the caller reports an error).
__global__ void __launch_bounds__(256)
bl_segment_sort_kernel(const unsigned *__restrict__ B_start, unsigned *__restrict__ perm, unsigned *__restrict__ status) {
    __shared__ unsigned s_key[kMaxSeg];
    const unsigned b0 = B_start[blockIdx.x], b1 = B_start[blockIdx.x + 1];
    const unsigned n = b1 - b0;
    if (n < 2) return;
    if (n > kMaxSeg) { if (threadIdx.x == 0) atomicAdd(&status[1], 1u); return; }
    unsigned m = 2;
    while (m < n) m <<= 1;
    for (unsigned i = threadIdx.x; i < m; i += 256) s_key[i] = i < n ? perm[b0 + i] : 0xFFFFFFFFu;
    __syncthreads();
    for (unsigned k = 2; k <= m; k <<= 1) {
        for (unsigned j = k >> 1; j > 0; j >>= 1) {
            for (unsigned i = threadIdx.x; i < m; i += 256) {
                const unsigned l = i ^ j;
                if (l > i) {
                    const unsigned a = s_key[i], b = s_key[l];
                    const bool up = (i & k) == 0;
                    if ((a > b) == up) { s_key[i] = b; s_key[l] = a; }
                }
            }
            __syncthreads();
        }
    }
    for (unsigned i = threadIdx.x; i < n; i += 256) perm[b0 + i] = s_key[i];
}


__global__ void bl_chan_scale_kernel(const double *__restrict__ freq, int nchan, double *__restrict__ fscale) {
    int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c < nchan) fscale[c] = __ddiv_rn(freq[c], WPG_C0);
}

// Support class of visibility idx of the baseline-then-time order (w -> plane -> class; G1-G2 only).
__device__ __forceinline__ int bl_class_of(long long idx, const BinParams &P, const unsigned *__restrict__ perm,
                                           const double *__restrict__ uvw, const double *__restrict__ fscale, const uint2 *s_tab) {
    const unsigned s = (unsigned)(idx / P.nchan);
    const int ch = (int)(idx - (long long)s * P.nchan);
    const double w = __dmul_rn(__ldg(uvw + 3 * (long long)perm[s] + 2), __ldg(fscale + ch));
    int p = 0;
    if (P.dw > 0.0) {
        const double ws = __dadd_rn(w, P.w_max);
        double qd = wpg_div_const(ws, P.dw, P.rdw);
        if (wpg_near_integer(qd)) qd = __ddiv_rn(ws, P.dw);
        const double fp = floor(qd);
        p = fp < 0.0 ? 0 : (fp > (double)(P.Nw - 1) ? P.Nw - 1 : (int)fp);
    }
    return (int)(s_tab[p].y >> 8);
}

// Ragged stacks, pass 4b: records per (support class, block of 256 consecutive positions of the baseline-then-time
// order): ctab[cls * nblocks + block].  Its exclusive scan (class-major) gives every block the start of its records
// inside each class, so that the classes are contiguous AND each keeps the baseline-then-time order (a stable
// partition): the gridder of a class then walks its baselines' time series as in the uniform case.
__global__ void __launch_bounds__(256)
bl_class_count_kernel(const double *__restrict__ uvw, const double *__restrict__ fscale, const __grid_constant__ PlaneTab T,
                      const __grid_constant__ BinParams P, const unsigned *__restrict__ perm, unsigned *__restrict__ ctab) {
    __shared__ uint2 s_tab[WPG_MAX_NW];
    __shared__ unsigned s_cnt[WPG_MAX_CLS];
    wpg_stage_planetab(s_tab, T, P.Nw);
    if (threadIdx.x < WPG_MAX_CLS) s_cnt[threadIdx.x] = 0;
    __syncthreads();
    const long long nvis = P.nrow * P.nchan;
    const long long idx = (long long)blockIdx.x * 256 + threadIdx.x;
    if (idx < nvis) atomicAdd(&s_cnt[bl_class_of(idx, P, perm, uvw, fscale, s_tab)], 1u);
    __syncthreads();
    if ((int)threadIdx.x < P.ncls) ctab[(size_t)threadIdx.x * gridDim.x + blockIdx.x] = s_cnt[threadIdx.x];
}

// Pass 5: the records, in baseline-then-time order (record s * nchan + ch = row perm[s], channel ch; ragged stacks:
// that order inside each support class, classes one after the other).  A flagged or out-of-grid visibility keeps its
// place in the time series as a zero-valued record at the window start clamped into the grid (it adds zeros; the
// counters do not count it as gridded).  bucket[c] = first record of class c, bucket[ncls] = number of records.
template <typename TT>
__global__ void __launch_bounds__(256)
bl_build_records_kernel(const float2 *__restrict__ vis, const double *__restrict__ uvw, const float *__restrict__ weight,
                        const double *__restrict__ fscale, const __grid_constant__ PlaneTab T,
                        const __grid_constant__ BinParams P, const unsigned *__restrict__ perm, Counters *__restrict__ ctr,
                        Rec<TT> *__restrict__ rec, unsigned *__restrict__ bucket, const unsigned *__restrict__ ctab) {
    __shared__ uint2 s_tab[WPG_MAX_NW];
    __shared__ unsigned s_wcnt[8][WPG_MAX_CLS];
    wpg_stage_planetab(s_tab, T, P.Nw);
    if (P.ncls > 1) for (int i = threadIdx.x; i < 8 * WPG_MAX_CLS; i += 256) (&s_wcnt[0][0])[i] = 0;
    __syncthreads();
    const SmemPlaneTab ST{s_tab, nullptr};
    const long long nvis = P.nrow * P.nchan;
    const long long idx = (long long)blockIdx.x * 256 + threadIdx.x;
    if (P.ncls == 1) { if (idx == 0) { bucket[0] = 0u; bucket[1] = (unsigned)nvis; } }
    else if (blockIdx.x == 0 && (int)threadIdx.x <= P.ncls)
        bucket[threadIdx.x] = (int)threadIdx.x < P.ncls ? ctab[(size_t)threadIdx.x * gridDim.x] : (unsigned)nvis;
    unsigned c_grid = 0, c_oob = 0, c_zero = 0, c_clamp = 0, c_upd = 0;
    bool have = idx < nvis;
    Rec<TT> out; out.re = out.im = (TT)0; out.pos = out.koff = 0;
    int cls = 0;
    if (have) {
        const unsigned s = (unsigned)(idx / P.nchan);
        const int ch = (int)(idx - (long long)s * P.nchan);
        const long long row = perm[s], i = row * P.nchan + ch;
        const float wt = __ldg(weight + i);
        VisPos r = wpg_locate(__ldg(uvw + 3 * row), __ldg(uvw + 3 * row + 1), __ldg(uvw + 3 * row + 2),
                              __ldg(fscale + ch), P, ST);
        cls = ST.cls(r.p);
        const bool ok = wt != 0.0f && r.inside;
        if (wt == 0.0f) c_zero = 1; else if (!r.inside) c_oob = 1;
        else { c_grid = 1; c_clamp = r.clamped; c_upd = r.S * r.S; }
        const int j0u = min(max(r.j0u, 0), P.N - r.S), j0v = min(max(r.j0v, 0), P.N - r.S);
        const float2 v = __ldg(vis + i);
        // literal zeros for a flagged / off-grid sample: its value may be NaN or Inf (RFI), and 0 * NaN = NaN
        out.re = ok ? (TT)wt * (TT)v.x : (TT)0; out.im = ok ? (TT)wt * (TT)v.y : (TT)0;
        out.pos = (unsigned)j0u | ((unsigned)j0v << 16);
        out.koff = ok ? wpg_koff(r, P, ST) : (unsigned)ST.off(r.p);
    }
    unsigned dst = (unsigned)idx;
    if (P.ncls > 1) {
        // stable rank inside the block among the records of the same class: lower lanes of the warp, then lower warps
        const unsigned live = __ballot_sync(0xffffffffu, have);
        unsigned rank = 0, m = 0;
        if (have) {
            m = __match_any_sync(live, cls);
            rank = __popc(m & ((1u << (threadIdx.x & 31)) - 1u));
            if (rank == 0) s_wcnt[threadIdx.x >> 5][cls] = __popc(m);
        }
        __syncthreads();
        if (have) {
            for (unsigned w = 0; w < (threadIdx.x >> 5); ++w) rank += s_wcnt[w][cls];
            dst = ctab[(size_t)cls * gridDim.x + blockIdx.x] + rank;
        }
    }
    if (have) rec[dst] = out;
    // statistics: warp sums, spread over the counter slots
    unsigned v5[5] = {c_grid, c_oob, c_zero, c_clamp, c_upd};
    unsigned long long *dstc[5] = {ctr->n_gridded, ctr->n_skipped_oob, ctr->n_skipped_zero_weight, ctr->n_clamped_w, ctr->n_updates};
#pragma unroll
    for (int k = 0; k < 5; ++k) {
        const unsigned t = __reduce_add_sync(0xffffffffu, v5[k]);
        if ((threadIdx.x & 31) == 0 && t) atomicAdd(dstc[k] + (blockIdx.x * 8 + (threadIdx.x >> 5)) % kStatSlots, (unsigned long long)t);
    }
}

}  // namespace

// ---------------------------------------------------------------------------------------------- host side
namespace {

static size_t al(size_t x) { return (x + 255) & ~(size_t)255; }

struct BlLayout { size_t off_counters, off_bucket2, off_bstart, off_cursor, off_blocksum, off_status, off_ib, off_perm, off_fscale, off_ctab, off_cblocksum, off_records, total; unsigned nb, nvblocks; };

BlLayout bl_layout(int64_t nrow, int nchan, int n_ant, size_t rec_bytes) {
    BlLayout L{};
    L.nb = (unsigned)((int64_t)n_ant * (n_ant + 1) / 2);
    size_t o = 0;
    L.off_counters = o; o += al(sizeof(Counters));
    L.off_bucket2 = o;  o += 256;                       // class starts of the records: up to WPG_MAX_CLS + 1 words
    L.off_status = o;   o += 256;
    L.off_bstart = o;   o += al(((size_t)L.nb + 8) * 4);
    L.off_cursor = o;   o += al(((size_t)L.nb + 8) * 4);
    L.off_blocksum = o; o += al((((size_t)L.nb + 1 + 4095) / 4096) * 4 + 8);
    L.off_ib = o;       o += al((size_t)nrow * 4);
    L.off_perm = o;     o += al((size_t)nrow * 4);
    L.off_fscale = o;   o += al((size_t)nchan * 8);
    // ragged stacks: records per (support class, block of 256 records), scanned class-major
    L.nvblocks = (unsigned)(((size_t)nrow * nchan + 255) / 256);
    const size_t nct = (size_t)WPG_MAX_CLS * L.nvblocks;
    L.off_ctab = o;     o += al((nct + 8) * 4);
    L.off_cblocksum = o; o += al(((nct + 1 + 4095) / 4096) * 4 + 8);
    L.off_records = o;  o += al((size_t)nrow * nchan * rec_bytes);
    L.total = o;
    return L;
}

// Eq. (1) + count + Eq. (2) + stable re-order into w (layout L).  Synchronises to read the status words.
int bl_reorder(wpg_ctx *ctx, const int *d_ant1, const int *d_ant2, int n_ant, int64_t nrow, char *w, const BlLayout &L) {
    cudaStream_t s = ctx->stream;
    unsigned *bstart = (unsigned *)(w + L.off_bstart), *cursor = (unsigned *)(w + L.off_cursor);
    unsigned *status = (unsigned *)(w + L.off_status), *ib = (unsigned *)(w + L.off_ib), *perm = (unsigned *)(w + L.off_perm);
    WPG_CUDA(ctx, cudaMemsetAsync(w, 0, L.off_blocksum, s));                 // counters, bucket2, status, C, cursor
    const unsigned nbk = (unsigned)((nrow + 255) / 256);
    if (nbk) bl_count_kernel<<<nbk, 256, 0, s>>>(d_ant1, d_ant2, n_ant, nrow, ib, bstart, status);
    int rc = wpg_launch_exclusive_scan(ctx, bstart, L.nb, (unsigned *)(w + L.off_blocksum), (Counters *)(w + L.off_counters));
    if (rc) return rc;
    WPG_CUDA(ctx, cudaMemcpyAsync(cursor, bstart, ((size_t)L.nb + 1) * 4, cudaMemcpyDeviceToDevice, s));
    if (nbk) bl_scatter_kernel<<<nbk, 256, 0, s>>>(ib, nrow, cursor, perm);
    bl_segment_sort_kernel<<<L.nb, 256, 0, s>>>(bstart, perm, status);
    ctx->n_launches += nbk ? 3 : 1;
    WPG_CUDA(ctx, cudaGetLastError());
    unsigned h_status[2] = {0, 0};
    WPG_CUDA(ctx, cudaMemcpyAsync(h_status, status, sizeof h_status, cudaMemcpyDeviceToHost, s));
    WPG_CUDA(ctx, cudaStreamSynchronize(s));
    if (h_status[0]) return wpg_fail(ctx, WPG_EINVAL, "%u rows have an antenna ID outside 0..%d", h_status[0], n_ant - 1);
    if (h_status[1]) return wpg_fail(ctx, WPG_EINVAL, "%u baselines have more than %d rows: chunk the input in time", h_status[1], kMaxSeg);
    return WPG_OK;
}

int bl_check(wpg_ctx *ctx, const void *a1, const void *a2, int n_ant, int64_t nrow) {
    if (!ctx) return WPG_EINVAL;
    if (n_ant < 1 || n_ant > 4096) return wpg_fail(ctx, WPG_EINVAL, "n_ant = %d outside 1..4096", n_ant);
    if (nrow < 0 || nrow >= ((int64_t)1 << 32) - 2) return wpg_fail(ctx, WPG_EINVAL, "nrow = %lld", (long long)nrow);
    if (nrow > 0 && (!a1 || !a2)) return wpg_fail(ctx, WPG_EINVAL, "antenna ID pointer is NULL");
    return WPG_OK;
}

}  // namespace

extern "C" size_t wpg_baseline_workspace_bytes(int64_t nrow, int nchan, int n_ant, wpg_prec prec) {
    if (nrow < 0 || nchan < 1 || n_ant < 1 || n_ant > 4096) return 0;
    return bl_layout(nrow, nchan, n_ant, prec == WPG_F32 ? sizeof(Rec<float>) : sizeof(Rec<double>)).total;
}

extern "C" int wpg_baseline_reorder(wpg_ctx *ctx, const int *d_ant1, const int *d_ant2, int n_ant, int64_t nrow,
                                    unsigned *d_bstart_out, unsigned *d_perm_out, void *d_workspace, size_t workspace_bytes) {
    int rc = bl_check(ctx, d_ant1, d_ant2, n_ant, nrow);
    if (rc) return rc;
    const BlLayout L = bl_layout(nrow, 1, n_ant, 0);
    if (!d_workspace || workspace_bytes < L.total)
        return wpg_fail(ctx, WPG_ENOMEM, "workspace of %zu bytes given, %zu needed", workspace_bytes, L.total);
    if (!d_bstart_out || !d_perm_out) return wpg_fail(ctx, WPG_EINVAL, "output pointer is NULL");
    WPG_DEVICE(ctx);
    char *w = (char *)d_workspace;
    rc = bl_reorder(ctx, d_ant1, d_ant2, n_ant, nrow, w, L);
    if (rc) return rc;
    WPG_CUDA(ctx, cudaMemcpyAsync(d_bstart_out, w + L.off_bstart, ((size_t)L.nb + 1) * 4, cudaMemcpyDeviceToDevice, ctx->stream));
    WPG_CUDA(ctx, cudaMemcpyAsync(d_perm_out, w + L.off_perm, (size_t)nrow * 4, cudaMemcpyDeviceToDevice, ctx->stream));
    WPG_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return WPG_OK;
}

extern "C" int wpg_grid_baseline_order(wpg_ctx *ctx, const void *d_vis, const double *d_uvw, const float *d_weight,
                                       const double *d_freq, const int *d_ant1, const int *d_ant2, int n_ant,
                                       int64_t nrow, int nchan, const void *d_kernels, const wpg_kdesc *desc,
                                       wpg_prec prec, void *d_grid, void *d_workspace, size_t workspace_bytes,
                                       wpg_stats *h_stats) {
    int rc = bl_check(ctx, d_ant1, d_ant2, n_ant, nrow);
    if (rc) return rc;
    if (!d_kernels || !d_grid || !d_freq || (nrow > 0 && (!d_vis || !d_uvw || !d_weight)))
        return wpg_fail(ctx, WPG_EINVAL, "NULL pointer argument");
    PlaneTab tab; BinParams bp; WorkspaceLayout ws0;
    rc = wpg_make_plan(ctx, desc, nrow, nchan, prec, &tab, &bp, &ws0);
    if (rc) return rc;
    if ((int64_t)bp.ncls * ((nrow * nchan + 255) / 256) >= ((int64_t)1 << 31))
        return wpg_fail(ctx, WPG_EINVAL, "too many visibilities for the per-class block table; chunk the input");
    const size_t recb = prec == WPG_F32 ? sizeof(Rec<float>) : sizeof(Rec<double>);
    const BlLayout L = bl_layout(nrow, nchan, n_ant, recb);
    if (!d_workspace || workspace_bytes < L.total)
        return wpg_fail(ctx, WPG_ENOMEM, "workspace of %zu bytes given, %zu needed", workspace_bytes, L.total);
    WPG_DEVICE(ctx);
    char *w = (char *)d_workspace;
    cudaStream_t s = ctx->stream;
    if ((rc = wpg_mark(ctx, 0))) return rc;
    rc = bl_reorder(ctx, d_ant1, d_ant2, n_ant, nrow, w, L);             // Eqs. (1)-(2), baseline-then-time order
    if (rc) return rc;
    const long long nvis = (long long)nrow * nchan;
    double *fscale = (double *)(w + L.off_fscale);
    bl_chan_scale_kernel<<<(nchan + 255) / 256, 256, 0, s>>>(d_freq, nchan, fscale);
    Counters *ctr = (Counters *)(w + L.off_counters);
    const unsigned nbk = (unsigned)((nvis + 255) / 256);
    unsigned *ctab = (unsigned *)(w + L.off_ctab);
    if (nbk && bp.ncls > 1) {          // ragged stack: stable partition of the order by support class
        bl_class_count_kernel<<<nbk, 256, 0, s>>>(d_uvw, fscale, tab, bp, (const unsigned *)(w + L.off_perm), ctab);
        ctx->n_launches += 1;
        rc = wpg_launch_exclusive_scan(ctx, ctab, (unsigned)bp.ncls * nbk, (unsigned *)(w + L.off_cblocksum), ctr);
        if (rc) return rc;
    }
    if (nbk) {
        if (prec == WPG_F32)
            bl_build_records_kernel<float><<<nbk, 256, 0, s>>>((const float2 *)d_vis, d_uvw, d_weight, fscale, tab, bp,
                (const unsigned *)(w + L.off_perm), ctr, (Rec<float> *)(w + L.off_records), (unsigned *)(w + L.off_bucket2), ctab);
        else
            bl_build_records_kernel<double><<<nbk, 256, 0, s>>>((const float2 *)d_vis, d_uvw, d_weight, fscale, tab, bp,
                (const unsigned *)(w + L.off_perm), ctr, (Rec<double> *)(w + L.off_records), (unsigned *)(w + L.off_bucket2), ctab);
    }
    ctx->n_launches += nbk ? 2 : 1;
    WPG_CUDA(ctx, cudaGetLastError());
    if ((rc = wpg_mark(ctx, 1))) return rc;
    if (nvis) {
        // the gridder of wpg_grid.cu walks the records in this order: per class, key range [cls, cls + 1) = its records
        WorkspaceLayout ws{};
        ws.off_counters = L.off_counters; ws.off_hist = L.off_bucket2; ws.off_records = L.off_records;
        bp.dyn_keys = 0; bp.keys_per_class = 1; bp.nkeys = 1;
        rc = wpg_launch_grid(ctx, tab, bp, ws, prec, d_kernels, d_grid, w);
        if (rc) return rc;
    }
    if ((rc = wpg_mark(ctx, 2))) return rc;
    if (h_stats) {
        Counters h;
        WPG_CUDA(ctx, cudaMemcpyAsync(&h, ctr, sizeof h, cudaMemcpyDeviceToHost, s));
        WPG_CUDA(ctx, cudaStreamSynchronize(s));
        memset(h_stats, 0, sizeof *h_stats);
        for (int k = 0; k < kStatSlots; ++k) {
            h_stats->n_gridded += (int64_t)h.n_gridded[k]; h_stats->n_skipped_oob += (int64_t)h.n_skipped_oob[k];
            h_stats->n_skipped_zero_weight += (int64_t)h.n_skipped_zero_weight[k];
            h_stats->n_clamped_w += (int64_t)h.n_clamped_w[k]; h_stats->n_updates += (int64_t)h.n_updates[k];
        }
    }
    return WPG_OK;
}
