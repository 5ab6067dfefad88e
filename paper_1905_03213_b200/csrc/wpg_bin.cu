// Step a1 — visibility binning: uvw -> (plane, window start, sub-cell offsets), sort key,
// histogram, exclusive prefix scan, scatter into key-sorted 16/24-byte records.
//
// The paper's analogue is the re-order of PAPER.md:62-78: count array C, exclusive prefix sum
// Eq. (2), scatter — keyed there by baseline (Eq. 1) so that consecutive samples of a baseline hit
// the same grid point.  Here the key is (support class, window start j0u, j0v), i.e.
// the visibilities are ordered by the grid point they hit, whatever baseline they came from: runs
// of equal window start are what the gridder (wpg_grid.cu) accumulates in registers, and between
// runs the window slides down the v axis at a fixed column.
#include "wpg_common.h"

namespace {

constexpr int kScanBlock = 4096;   // keys per scan block (1024 threads x 4)

// Block totals of the five wpg_stats counters: warp sums, shared memory, one reduction per counter and block.
__device__ __forceinline__ void block_count(Counters *ctr, unsigned c_grid, unsigned c_oob, unsigned c_zero,
                                            unsigned c_clamp, unsigned c_upd) {
    __shared__ unsigned s_cnt[5];
    if (threadIdx.x < 5) s_cnt[threadIdx.x] = 0;
    __syncthreads();
    unsigned v[5] = {c_grid, c_oob, c_zero, c_clamp, c_upd};
#pragma unroll
    for (int k = 0; k < 5; ++k) {
        const unsigned t = __reduce_add_sync(0xffffffffu, v[k]);
        if ((threadIdx.x & 31) == 0 && t) atomicAdd(&s_cnt[k], t);
    }
    __syncthreads();
    if (threadIdx.x < 5 && s_cnt[threadIdx.x]) {
        unsigned long long *dst = threadIdx.x == 0 ? ctr->n_gridded : threadIdx.x == 1 ? ctr->n_skipped_oob
                                : threadIdx.x == 2 ? ctr->n_skipped_zero_weight : threadIdx.x == 3 ? ctr->n_clamped_w
                                : ctr->n_updates;
        atomicAdd(dst + blockIdx.x % kStatSlots, (unsigned long long)s_cnt[threadIdx.x]);
    }
}

// Pass 0: f[ch] = freq[ch] / c0 (G1), once per channel instead of once per visibility.  Same IEEE
// division as G1 states, so the products u = uvw * f are bit-identical.  For uniform stacks thread 0 also
// writes the (static) key layout of the classes.
__global__ void chan_scale_kernel(const double *__restrict__ freq, int nchan, double *__restrict__ fscale,
                                  const __grid_constant__ BinParams P, Counters *__restrict__ ctr) {
    int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c < nchan) fscale[c] = __ddiv_rn(freq[c], WPG_C0);
    if (c == 0 && !P.dyn_keys) {
        for (int k = 0; k < P.ncls; ++k) {
            ctr->key_base[k] = (unsigned)k * P.keys_per_class;
            ctr->key_shift[k] = (unsigned)P.kshift;
            ctr->key_nkg[k] = (unsigned)P.nkg;
        }
        ctr->key_base[P.ncls] = (unsigned)P.ncls * P.keys_per_class;
    }
}

// Ragged stacks, pass 0b: census of the support classes (w -> plane -> class; weights and grid edges are
// ignored — the census only steers the key resolution).  One thread per row, all channels.
__global__ void __launch_bounds__(256)
census_kernel(const double *__restrict__ uvw, const double *__restrict__ fscale, const __grid_constant__ PlaneTab T,
              const __grid_constant__ BinParams P, Counters *__restrict__ ctr) {
    __shared__ unsigned s_cnt[8][WPG_MAX_CLS];
    __shared__ uint2 s_tab[WPG_MAX_NW];
    for (int i = threadIdx.x; i < 8 * WPG_MAX_CLS; i += 256) (&s_cnt[0][0])[i] = 0;
    wpg_stage_planetab(s_tab, T, P.Nw);
    __syncthreads();
    unsigned *mine = s_cnt[threadIdx.x >> 5];
    for (long long row = (long long)blockIdx.x * 256 + threadIdx.x; row < P.nrow; row += (long long)gridDim.x * 256) {
        const double wm = __ldg(uvw + 3 * row + 2);
        for (int ch = 0; ch < P.nchan; ++ch) {
            const double w = __dmul_rn(wm, __ldg(fscale + ch));
            int p = 0;
            if (P.dw > 0.0) {
                const double fp = floor(wpg_div_const(__dadd_rn(w, P.w_max), P.dw, P.rdw));
                p = fp < 0.0 ? 0 : (fp > (double)(P.Nw - 1) ? P.Nw - 1 : (int)fp);
            }
            atomicAdd(&mine[s_tab[p].y >> 8], 1u);
        }
    }
    __syncthreads();
    if (threadIdx.x < P.ncls) {
        unsigned t = 0;
        for (int wv = 0; wv < 8; ++wv) t += s_cnt[wv][threadIdx.x];
        if (t) atomicAdd(&ctr->census[threadIdx.x], t);
    }
}

// Ragged stacks, pass 0c (one thread): split the key budget among the classes.  Every class starts with one
// key per grid column; the class with the most visibilities per key is refined (one more bit of j0v) as long
// as the total stays within the budget.
__global__ void plan_keys_kernel(Counters *__restrict__ ctr, int ncls, int N, unsigned budget) {
    if (blockIdx.x || threadIdx.x) return;
    unsigned sh[WPG_MAX_CLS];
    unsigned long long total = 0;
    auto keys = [&](unsigned s_) { return (unsigned long long)N * (unsigned)((N + (1 << s_) - 1) >> s_); };
    for (int c = 0; c < ncls; ++c) { sh[c] = 13; total += keys(13); }
    for (;;) {
        int best = -1; double best_d = -1.0;
        for (int c = 0; c < ncls; ++c) {
            if (sh[c] == 0 || keys(sh[c] - 1) == keys(sh[c])) { if (sh[c] && keys(sh[c] - 1) == keys(sh[c])) { sh[c] -= 1; c -= 1; } continue; }
            if (total - keys(sh[c]) + keys(sh[c] - 1) > budget) continue;
            const double d = ((double)ctr->census[c] + 1.0) / (double)keys(sh[c]);
            if (d > best_d) { best_d = d; best = c; }
        }
        if (best < 0) break;
        total += keys(sh[best] - 1) - keys(sh[best]);
        sh[best] -= 1;
    }
    unsigned base = 0;
    for (int c = 0; c < ncls; ++c) {
        ctr->key_base[c] = base; ctr->key_shift[c] = sh[c];
        ctr->key_nkg[c] = (unsigned)((N + (1 << sh[c]) - 1) >> sh[c]);
        base += (unsigned)keys(sh[c]);
    }
    ctr->key_base[ncls] = base;
}

constexpr int kVpt = 4;            // visibilities per thread: four independent atomics in flight per thread

// The kVpt visibilities of a thread.  Default: a block takes 256 * kVpt consecutive visibilities, thread t the
// ones at t, t + 256, ...  With the "row_block" hint (P.vis_block = visibilities per time step): thread
// (dg, x) takes visibility x of the time steps dg * kVpt + j — the same baseline and channel at consecutive
// times, whose window starts (and so sort keys) mostly coincide, so that the bucket counter is
// touched once per run of equal keys.  Loads stay coalesced either way (consecutive lanes, consecutive x).
__device__ __forceinline__ void vis_indices(const BinParams &P, unsigned (&idx)[kVpt]) {
    const unsigned long long nvis = (unsigned long long)(P.nrow * P.nchan);     // < 2^32 - 1 (wpg_make_plan)
    if (P.vis_block) {
        const unsigned t = blockIdx.x * 256u + threadIdx.x;
        const unsigned dg = t / P.vis_block, x = t - dg * P.vis_block;
#pragma unroll
        for (int j = 0; j < kVpt; ++j) {
            const unsigned long long i = (unsigned long long)(dg * kVpt + j) * P.vis_block + x;
            idx[j] = i < nvis ? (unsigned)i : 0xFFFFFFFFu;
        }
    } else {
#pragma unroll
        for (int j = 0; j < kVpt; ++j) {
            const unsigned long long i = (unsigned long long)blockIdx.x * (256 * kVpt) + j * 256 + threadIdx.x;
            idx[j] = i < nvis ? (unsigned)i : 0xFFFFFFFFu;
        }
    }
}
// run structure of a thread's keys: head[j] = first of a run of equal valid keys, len[j] = length of the run from j
__device__ __forceinline__ void key_runs(const unsigned (&key)[kVpt], bool (&head)[kVpt], unsigned (&len)[kVpt]) {
#pragma unroll
    for (int j = kVpt - 1; j >= 0; --j) {
        len[j] = 1u + ((j + 1 < kVpt && key[j + 1] == key[j]) ? len[j + 1 < kVpt ? j + 1 : j] : 0u);
        head[j] = key[j] != WPG_NO_KEY && (j == 0 || key[j] != key[j - 1]);
    }
}

// Position math (fp64, G1-G3) and validity (G4, R9) of visibility i; returns the sort key or WPG_NO_KEY.
// The two passes below both evaluate it: recomputing is cheaper than a round trip of (key, position,
// coefficient offset) through HBM, and the workspace holds nothing per visibility but the records.
struct Located { unsigned key, pos, koff; int S; bool clamped, zero_weight; };
struct RawVis { double um, vm, wm, f; float wt; bool valid; };

// All global loads of one visibility, issued before any arithmetic so that a thread has the inputs of
// its kVpt visibilities in flight at once (the passes are latency-bound otherwise).
__device__ __forceinline__ RawVis load_vis(long long i, long long nvis, const double *__restrict__ uvw,
                                           const float *__restrict__ weight, const double *__restrict__ fscale,
                                           const BinParams &P) {
    RawVis r; r.valid = i < nvis; r.um = r.vm = r.wm = 0.0; r.f = 0.0; r.wt = 0.f;
    if (r.valid) {
        long long row = i; int ch = 0;
        if (P.nchan > 1) {             // nrow * nchan < 2^32 (wpg_make_plan): 32-bit division
            const unsigned r32 = (unsigned)i / (unsigned)P.nchan;
            row = r32; ch = (int)((unsigned)i - r32 * (unsigned)P.nchan);
        }
        r.wt = __ldg(weight + i);
        r.um = __ldg(uvw + 3 * row); r.vm = __ldg(uvw + 3 * row + 1); r.wm = __ldg(uvw + 3 * row + 2);
        r.f = __ldg(fscale + ch);
    }
    return r;
}
// Keeps the compiler from consuming a loaded value (and so waiting for it) before the loads that
// follow in program order have been issued.
__device__ __forceinline__ void use_after_here(RawVis &r) {
    asm volatile("" : "+f"(r.wt), "+d"(r.um), "+d"(r.vm), "+d"(r.wm));
}

__device__ __forceinline__ Located locate_vis(const RawVis &v, const SmemPlaneTab &T, const BinParams &P) {
    Located L; L.key = WPG_NO_KEY; L.pos = L.koff = 0; L.S = 0; L.clamped = false;
    L.zero_weight = v.valid && v.wt == 0.0f;
    if (!v.valid || L.zero_weight) return L;
    VisPos r = wpg_locate(v.um, v.vm, v.wm, v.f, P, T);
    if (!r.inside) return L;
    L.S = r.S; L.clamped = r.clamped;
    const uint4 ck = T.ck[T.cls(r.p)];
    L.key = ck.x + (unsigned)r.j0u * ck.y + ((unsigned)r.j0v >> ck.z);
    L.pos = (unsigned)r.j0u | ((unsigned)r.j0v << 16);
    L.koff = wpg_koff(r, P, T);
    return L;
}

// Pass 1: histogram of the keys (reductions without return value) and the wpg_stats counters.
__global__ void __launch_bounds__(256, 4)
bin_count_kernel(const double *__restrict__ uvw, const float *__restrict__ weight,
                 const double *__restrict__ fscale, const __grid_constant__ PlaneTab T,
                 const __grid_constant__ BinParams P, Counters *__restrict__ ctr, unsigned *__restrict__ hist) {
    const long long nvis = P.nrow * P.nchan;
    unsigned idx[kVpt];
    vis_indices(P, idx);
    unsigned c_grid = 0, c_oob = 0, c_zero = 0, c_clamp = 0, c_upd = 0;
    __shared__ uint2 s_tab[WPG_MAX_NW];
    __shared__ uint4 s_ck[WPG_MAX_CLS];
    const SmemPlaneTab ST{s_tab, s_ck};
    RawVis raw[kVpt];
#pragma unroll
    for (int j = 0; j < kVpt; ++j) raw[j] = load_vis(idx[j], nvis, uvw, weight, fscale, P);
#pragma unroll
    for (int j = 0; j < kVpt; ++j) use_after_here(raw[j]);
    wpg_stage_planetab(s_tab, T, P.Nw);
    wpg_stage_classkeys(s_ck, ctr, P);
    __syncthreads();
    unsigned key[kVpt], len[kVpt];
    bool head[kVpt];
#pragma unroll
    for (int j = 0; j < kVpt; ++j) {
        key[j] = WPG_NO_KEY;
        if (!raw[j].valid) continue;
        const Located L = locate_vis(raw[j], ST, P);
        if (L.zero_weight) c_zero += 1;
        else if (L.key == WPG_NO_KEY) c_oob += 1;
        else { c_grid += 1; c_clamp += L.clamped; c_upd += L.S * L.S; key[j] = L.key; }
    }
    key_runs(key, head, len);
#pragma unroll
    for (int j = 0; j < kVpt; ++j)
        if (head[j]) asm volatile("red.global.add.u32 [%0], %1;" ::"l"(hist + key[j]), "r"(len[j]) : "memory");
    block_count(ctr, c_grid, c_oob, c_zero, c_clamp, c_upd);
}

// Block-wide inclusive scan of one unsigned per thread (1024 threads); returns the inclusive
// value, *total receives the block total.
__device__ __forceinline__ unsigned block_scan_incl(unsigned v, unsigned *total) {
    __shared__ unsigned wsum[32];
    int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        unsigned a = __shfl_up_sync(0xffffffffu, v, d);
        if (lane >= d) v += a;
    }
    if (lane == 31) wsum[wid] = v;
    __syncthreads();
    if (wid == 0) {
        unsigned w = wsum[lane];
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            unsigned a = __shfl_up_sync(0xffffffffu, w, d);
            if (lane >= d) w += a;
        }
        wsum[lane] = w;
    }
    __syncthreads();
    if (wid > 0) v += wsum[wid - 1];
    *total = wsum[31];
    __syncthreads();
    return v;
}

// Scan phase A: per-block totals of the counts.
__global__ void __launch_bounds__(1024)
scan_reduce_kernel(const unsigned *__restrict__ hist, unsigned nkeys, unsigned *__restrict__ blocksum) {
    unsigned k0 = blockIdx.x * kScanBlock + threadIdx.x * 4;
    unsigned v = 0;
    if (k0 + 3 < nkeys) {
        uint4 q = *reinterpret_cast<const uint4 *>(hist + k0);
        v = q.x + q.y + q.z + q.w;
    } else {
#pragma unroll
        for (int j = 0; j < 4; ++j) v += (k0 + j < nkeys) ? hist[k0 + j] : 0;
    }
    unsigned tot;
    block_scan_incl(v, &tot);
    if (threadIdx.x == 0) blocksum[blockIdx.x] = tot;
}

// Scan phase B: exclusive scan of the block totals (single block), total to the counters.
__global__ void __launch_bounds__(1024)
scan_blocksums_kernel(unsigned *__restrict__ blocksum, unsigned nblocks, Counters *__restrict__ ctr) {
    unsigned carry = 0;
    for (unsigned b0 = 0; b0 < nblocks; b0 += 1024) {
        unsigned b = b0 + threadIdx.x;
        unsigned v = b < nblocks ? blocksum[b] : 0;
        unsigned tot;
        unsigned inc = block_scan_incl(v, &tot);
        if (b < nblocks) blocksum[b] = carry + inc - v;
        carry += tot;
    }
    if (threadIdx.x == 0) ctr->n_records = carry;
}

// Scan phase C: bucket_start, in place over the histogram (bucket_start[nkeys] = total).
__global__ void __launch_bounds__(1024)
scan_apply_kernel(unsigned *__restrict__ hist, unsigned nkeys, const unsigned *__restrict__ blocksum) {
    unsigned k0 = blockIdx.x * kScanBlock + threadIdx.x * 4;
    unsigned c[4];
    unsigned v = 0;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        c[j] = (k0 + j < nkeys) ? hist[k0 + j] : 0;
        v += c[j];
    }
    unsigned tot;
    unsigned inc = block_scan_incl(v, &tot);
    unsigned start = blocksum[blockIdx.x] + inc - v;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        if (k0 + j <= nkeys) hist[k0 + j] = start;
        start += c[j];
    }
}

// One 16-byte store per fp32 record; 8 + 8 + 8 for the 24-byte fp64 record.
__device__ __forceinline__ void store_rec(Rec<float> *dst, float re, float im, uint2 p) {
    *reinterpret_cast<uint4 *>(dst) = make_uint4(__float_as_uint(re), __float_as_uint(im), p.x, p.y);
}
__device__ __forceinline__ void store_rec(Rec<double> *dst, double re, double im, uint2 p) {
    dst->re = re; dst->im = im;
    *reinterpret_cast<uint2 *>(&dst->pos) = p;
}

// Pass 3: scatter into key order.  The slot of a visibility is the running cursor of its bucket
// (bucket_start[key], advanced atomically: after this pass bucket_start[key] is the END of bucket key,
// i.e. the array read one element earlier is the start array again — see wpg_launch_bin).  The record
// carries weight*vis (R9, natural weighting).
template <typename TT>
__global__ void __launch_bounds__(256, 4)
scatter_kernel(const float2 *__restrict__ vis, const double *__restrict__ uvw, const float *__restrict__ weight,
               const double *__restrict__ fscale, const __grid_constant__ PlaneTab T,
               const __grid_constant__ BinParams P, const Counters *__restrict__ ctr, unsigned *__restrict__ cursor,
               Rec<TT> *__restrict__ rec) {
    const long long nvis = P.nrow * P.nchan;
    unsigned idx[kVpt];
    vis_indices(P, idx);
    Located L[kVpt];
    float wt[kVpt];
    unsigned dst[kVpt];
    float2 v[kVpt];
    __shared__ uint2 s_tab[WPG_MAX_NW];
    __shared__ uint4 s_ck[WPG_MAX_CLS];
    const SmemPlaneTab ST{s_tab, s_ck};
    {
        RawVis raw[kVpt];
#pragma unroll
        for (int j = 0; j < kVpt; ++j) {
            const long long i = idx[j];        // 0xFFFFFFFF = none (>= nvis)
            raw[j] = load_vis(i, nvis, uvw, weight, fscale, P);
            v[j] = i < nvis ? __ldg(vis + i) : make_float2(0.f, 0.f);
        }
#pragma unroll
        for (int j = 0; j < kVpt; ++j) use_after_here(raw[j]);
        wpg_stage_planetab(s_tab, T, P.Nw);
        wpg_stage_classkeys(s_ck, ctr, P);
        __syncthreads();
#pragma unroll
        for (int j = 0; j < kVpt; ++j) { L[j] = locate_vis(raw[j], ST, P); wt[j] = raw[j].wt; }
    }
    // one returning atomic per run of equal keys (the slowest instruction of the pass: ~5 cycles per lane)
    unsigned key[kVpt], len[kVpt];
    bool head[kVpt];
#pragma unroll
    for (int j = 0; j < kVpt; ++j) key[j] = L[j].key;
    key_runs(key, head, len);
#pragma unroll
    for (int j = 0; j < kVpt; ++j) dst[j] = head[j] ? atomicAdd(cursor + key[j], len[j]) : 0u;
#pragma unroll
    for (int j = 1; j < kVpt; ++j)
        if (key[j] != WPG_NO_KEY && !head[j]) dst[j] = dst[j - 1] + 1u;
#pragma unroll
    for (int j = 0; j < kVpt; ++j) {
        if (L[j].key == WPG_NO_KEY) continue;
        const TT w = (TT)wt[j];
        store_rec(rec + dst[j], w * (TT)v[j].x, w * (TT)v[j].y, make_uint2(L[j].pos, L[j].koff));
    }
}

// Pass 3 for NPOL correlations per (row, channel): vis[row][chan][pol]; one record carries all of them.
template <int NPOL>
__global__ void __launch_bounds__(256, 3)
scatter_pol_kernel(const float2 *__restrict__ vis, const double *__restrict__ uvw, const float *__restrict__ weight,
                   const double *__restrict__ fscale, const __grid_constant__ PlaneTab T,
                   const __grid_constant__ BinParams P, const Counters *__restrict__ ctr, unsigned *__restrict__ cursor,
                   RecP<NPOL> *__restrict__ rec) {
    const long long nvis = P.nrow * P.nchan;
    unsigned idx[kVpt];
    vis_indices(P, idx);
    Located L[kVpt];
    float wt[kVpt];
    unsigned dst[kVpt];
    __shared__ uint2 s_tab[WPG_MAX_NW];
    __shared__ uint4 s_ck[WPG_MAX_CLS];
    const SmemPlaneTab ST{s_tab, s_ck};
    {
        RawVis raw[kVpt];
#pragma unroll
        for (int j = 0; j < kVpt; ++j) raw[j] = load_vis(idx[j], nvis, uvw, weight, fscale, P);
#pragma unroll
        for (int j = 0; j < kVpt; ++j) use_after_here(raw[j]);
        wpg_stage_planetab(s_tab, T, P.Nw);
        wpg_stage_classkeys(s_ck, ctr, P);
        __syncthreads();
#pragma unroll
        for (int j = 0; j < kVpt; ++j) { L[j] = locate_vis(raw[j], ST, P); wt[j] = raw[j].wt; }
    }
    unsigned key[kVpt], len[kVpt];
    bool head[kVpt];
#pragma unroll
    for (int j = 0; j < kVpt; ++j) key[j] = L[j].key;
    key_runs(key, head, len);
#pragma unroll
    for (int j = 0; j < kVpt; ++j) dst[j] = head[j] ? atomicAdd(cursor + key[j], len[j]) : 0u;
#pragma unroll
    for (int j = 1; j < kVpt; ++j)
        if (key[j] != WPG_NO_KEY && !head[j]) dst[j] = dst[j - 1] + 1u;
#pragma unroll
    for (int j = 0; j < kVpt; ++j) {
        if (key[j] == WPG_NO_KEY) continue;
        const float2 *src = vis + (size_t)idx[j] * NPOL;
        RecP<NPOL> out;
#pragma unroll
        for (int p = 0; p < NPOL; ++p) { const float2 v = __ldg(src + p); out.v[p] = make_float2(wt[j] * v.x, wt[j] * v.y); }
        out.pos = L[j].pos; out.koff = L[j].koff;
        rec[dst[j]] = out;
    }
}

}  // namespace

// Exclusive prefix sum of hist[0 .. n-1] in place, hist[n] = total (also written to ctr->n_records);
// blocksum: ceil((n + 1) / 4096) words of scratch.  Shared with the baseline re-order (wpg_baseline.cu, Eq. 2).
int wpg_launch_exclusive_scan(wpg_ctx *ctx, unsigned *hist, unsigned n, unsigned *blocksum, Counters *ctr) {
    const unsigned nblocks = (n + 1 + kScanBlock - 1) / kScanBlock;
    cudaStream_t s = ctx->stream;
    scan_reduce_kernel<<<nblocks, 1024, 0, s>>>(hist, n, blocksum);
    scan_blocksums_kernel<<<1, 1024, 0, s>>>(blocksum, nblocks, ctr);
    scan_apply_kernel<<<nblocks, 1024, 0, s>>>(hist, n, blocksum);
    ctx->n_launches += 3;
    WPG_CUDA(ctx, cudaGetLastError());
    return WPG_OK;
}

int wpg_launch_bin(wpg_ctx *ctx, const void *d_vis, const double *d_uvw, const float *d_weight,
                   const double *d_freq, const PlaneTab &tab, const BinParams &bp,
                   const WorkspaceLayout &ws, wpg_prec prec, char *w) {
    long long nvis = bp.nrow * bp.nchan;
    Counters *ctr = (Counters *)(w + ws.off_counters);
    // bucket_start[0 .. nkeys] lives at off_hist; the counts of key k are accumulated one element
    // further on, at bucket_start[k + 1] (16-byte aligned for the scan: off_hist is 256-aligned + 12).
    // The exclusive scan then leaves start[k] there, the scatter advances it to end[k] = start[k + 1],
    // and bucket_start[0] stays 0: the array ends up as the start offsets of all nkeys + 1 buckets.
    unsigned *bucket_start = (unsigned *)(w + ws.off_hist);
    unsigned *hist = bucket_start + 1;
    unsigned *blocksum = (unsigned *)(w + ws.off_blocksum);
    cudaStream_t s = ctx->stream;
    double *fscale = (double *)(w + ws.off_fscale);
    unsigned nb = (unsigned)((nvis + 256 * kVpt - 1) / (256 * kVpt));
    if (bp.vis_block) {                // ceil(time steps / kVpt) * vis_block threads
        const long long nd = (nvis + bp.vis_block - 1) / bp.vis_block;
        nb = (unsigned)((((nd + kVpt - 1) / kVpt) * bp.vis_block + 255) / 256);
    }
    chan_scale_kernel<<<(bp.nchan + 255) / 256, 256, 0, s>>>(d_freq, bp.nchan, fscale, bp, ctr);
    if (bp.dyn_keys) {
        census_kernel<<<ctx->sm_count * 8, 256, 0, s>>>(d_uvw, fscale, tab, bp, ctr);
        plan_keys_kernel<<<1, 32, 0, s>>>(ctr, bp.ncls, bp.N, ws.nkeys);
        ctx->n_launches += 2;
    }
    if (nb) bin_count_kernel<<<nb, 256, 0, s>>>(d_uvw, d_weight, fscale, tab, bp, ctr, hist);
    scan_reduce_kernel<<<ws.nblocks_scan, 1024, 0, s>>>(hist, ws.nkeys, blocksum);
    scan_blocksums_kernel<<<1, 1024, 0, s>>>(blocksum, ws.nblocks_scan, ctr);
    scan_apply_kernel<<<ws.nblocks_scan, 1024, 0, s>>>(hist, ws.nkeys, blocksum);
    if (nb) {
        if (prec == WPG_F32)
            scatter_kernel<float><<<nb, 256, 0, s>>>((const float2 *)d_vis, d_uvw, d_weight, fscale, tab, bp, ctr, hist,
                                                      (Rec<float> *)(w + ws.off_records));
        else
            scatter_kernel<double><<<nb, 256, 0, s>>>((const float2 *)d_vis, d_uvw, d_weight, fscale, tab, bp, ctr, hist,
                                                       (Rec<double> *)(w + ws.off_records));
    }
    ctx->n_launches += nb ? 6 : 4;
    WPG_CUDA(ctx, cudaGetLastError());
    return WPG_OK;
}

// Binning for the polarised gridder: the count pass and the scan are those of wpg_launch_bin (positions do not
// depend on the correlation), the scatter writes RecP<npol> records.
int wpg_launch_bin_pol(wpg_ctx *ctx, const void *d_vis, const double *d_uvw, const float *d_weight, const double *d_freq,
                       const PlaneTab &tab, const BinParams &bp, const WorkspaceLayout &ws, int npol, char *w) {
    long long nvis = bp.nrow * bp.nchan;
    Counters *ctr = (Counters *)(w + ws.off_counters);
    unsigned *bucket_start = (unsigned *)(w + ws.off_hist);
    unsigned *hist = bucket_start + 1;
    unsigned *blocksum = (unsigned *)(w + ws.off_blocksum);
    cudaStream_t s = ctx->stream;
    double *fscale = (double *)(w + ws.off_fscale);
    unsigned nb = (unsigned)((nvis + 256 * kVpt - 1) / (256 * kVpt));
    if (bp.vis_block) {
        const long long nd = (nvis + bp.vis_block - 1) / bp.vis_block;
        nb = (unsigned)((((nd + kVpt - 1) / kVpt) * bp.vis_block + 255) / 256);
    }
    chan_scale_kernel<<<(bp.nchan + 255) / 256, 256, 0, s>>>(d_freq, bp.nchan, fscale, bp, ctr);
    if (nb) bin_count_kernel<<<nb, 256, 0, s>>>(d_uvw, d_weight, fscale, tab, bp, ctr, hist);
    scan_reduce_kernel<<<ws.nblocks_scan, 1024, 0, s>>>(hist, ws.nkeys, blocksum);
    scan_blocksums_kernel<<<1, 1024, 0, s>>>(blocksum, ws.nblocks_scan, ctr);
    scan_apply_kernel<<<ws.nblocks_scan, 1024, 0, s>>>(hist, ws.nkeys, blocksum);
    if (nb) {
        if (npol == 4)
            scatter_pol_kernel<4><<<nb, 256, 0, s>>>((const float2 *)d_vis, d_uvw, d_weight, fscale, tab, bp, ctr, hist,
                                                     (RecP<4> *)(w + ws.off_records));
        else
            scatter_pol_kernel<2><<<nb, 256, 0, s>>>((const float2 *)d_vis, d_uvw, d_weight, fscale, tab, bp, ctr, hist,
                                                     (RecP<2> *)(w + ws.off_records));
    }
    ctx->n_launches += nb ? 6 : 4;
    WPG_CUDA(ctx, cudaGetLastError());
    return WPG_OK;
}
