// Step a1 — visibility binning: uvw -> (plane, window start, sub-cell offsets), sort key,
// histogram, exclusive prefix scan, scatter into key-sorted 16/24-byte records, work-item list.
//
// The paper's analogue is the re-order of PAPER.md:62-78: count array C, exclusive prefix sum
// Eq. (2), scatter — keyed there by baseline (Eq. 1), here by (w-plane | support class, uv tile)
// so that the gridder (wpg_grid.cu) can keep a tile's cells in registers.
#include "wpg_common.h"

namespace {

constexpr int kScanBlock = 4096;   // keys per scan block (1024 threads x 4)

__device__ __forceinline__ void warp_count(unsigned long long *dst, unsigned v) {
    unsigned s = __reduce_add_sync(0xffffffffu, v);
    if ((threadIdx.x & 31) == 0 && s) atomicAdd(dst, (unsigned long long)s);
}

// Pass 1: position math (fp64, G1-G3), validity (G4, R9), key, rank inside the key's bucket.
__global__ void __launch_bounds__(256)
bin_count_kernel(const double *__restrict__ uvw, const float *__restrict__ weight,
                 const double *__restrict__ freq, const __grid_constant__ PlaneTab T,
                 const __grid_constant__ BinParams P, Counters *__restrict__ ctr,
                 unsigned *__restrict__ hist, unsigned *__restrict__ key_out,
                 unsigned *__restrict__ rank_out, uint2 *__restrict__ pre_out) {
    long long nvis = P.nrow * P.nchan;
    long long base = (long long)blockIdx.x * blockDim.x;
    long long i = base + threadIdx.x;
    unsigned c_grid = 0, c_oob = 0, c_zero = 0, c_clamp = 0, c_upd = 0;
    if (i < nvis) {
        long long row = i / P.nchan;
        int ch = (int)(i - row * P.nchan);
        unsigned key = WPG_NO_KEY;
        if (weight[i] == 0.0f) {
            c_zero = 1;
        } else {
            double f = __ddiv_rn(freq[ch], WPG_C0);
            VisPos r = wpg_locate(uvw[3 * row], uvw[3 * row + 1], uvw[3 * row + 2], f, P, T);
            if (!r.inside) {
                c_oob = 1;
            } else {
                c_grid = 1; c_clamp = r.clamped; c_upd = r.S * r.S;
                unsigned tid = (unsigned)(r.j0v / P.tile) * P.ntile + (unsigned)(r.j0u / P.tile);
                unsigned cls = T.cls[r.p];
                key = P.order == 1 ? cls * (unsigned)(P.ntile * P.ntile) + tid : tid * (unsigned)P.ncls + cls;
                rank_out[i] = atomicAdd(&hist[key], 1u);
                pre_out[i] = make_uint2((unsigned)r.j0u | ((unsigned)r.j0v << 13) | ((unsigned)(r.S - 1) << 26),
                                        wpg_koff(r, P, T));
            }
        }
        key_out[i] = key;
    }
    warp_count(&ctr->n_gridded, c_grid);
    warp_count(&ctr->n_skipped_oob, c_oob);
    warp_count(&ctr->n_skipped_zero_weight, c_zero);
    warp_count(&ctr->n_clamped_w, c_clamp);
    warp_count(&ctr->n_updates, c_upd);
}

__device__ __forceinline__ unsigned nseg_of(unsigned cnt, unsigned seg) { return (cnt + seg - 1) / seg; }

// Block-wide inclusive scan of one uint2 per thread (1024 threads); returns the inclusive value,
// *total receives the block total.
__device__ __forceinline__ uint2 block_scan_incl(uint2 v, uint2 *total) {
    __shared__ uint2 wsum[32];
    int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        unsigned a = __shfl_up_sync(0xffffffffu, v.x, d), b = __shfl_up_sync(0xffffffffu, v.y, d);
        if (lane >= d) { v.x += a; v.y += b; }
    }
    if (lane == 31) wsum[wid] = v;
    __syncthreads();
    if (wid == 0) {
        uint2 w = wsum[lane];
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            unsigned a = __shfl_up_sync(0xffffffffu, w.x, d), b = __shfl_up_sync(0xffffffffu, w.y, d);
            if (lane >= d) { w.x += a; w.y += b; }
        }
        wsum[lane] = w;
    }
    __syncthreads();
    if (wid > 0) { v.x += wsum[wid - 1].x; v.y += wsum[wid - 1].y; }
    *total = wsum[31];
    __syncthreads();
    return v;
}

// Scan phase A: per-block totals of (count, number of work items).
__global__ void __launch_bounds__(1024)
scan_reduce_kernel(const unsigned *__restrict__ hist, unsigned nkeys, unsigned seg, uint2 *__restrict__ blocksum) {
    unsigned k0 = blockIdx.x * kScanBlock + threadIdx.x * 4;
    uint2 v = make_uint2(0, 0);
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        unsigned k = k0 + j;
        unsigned c = k < nkeys ? hist[k] : 0;
        v.x += c; v.y += nseg_of(c, seg);
    }
    uint2 tot;
    block_scan_incl(v, &tot);
    if (threadIdx.x == 0) blocksum[blockIdx.x] = tot;
}

// Scan phase B: exclusive scan of the block totals (single block), totals to the counters.
__global__ void __launch_bounds__(1024)
scan_blocksums_kernel(uint2 *__restrict__ blocksum, unsigned nblocks, Counters *__restrict__ ctr) {
    uint2 carry = make_uint2(0, 0);
    for (unsigned b0 = 0; b0 < nblocks; b0 += 1024) {
        unsigned b = b0 + threadIdx.x;
        uint2 v = b < nblocks ? blocksum[b] : make_uint2(0, 0);
        uint2 tot;
        uint2 inc = block_scan_incl(v, &tot);
        if (b < nblocks) blocksum[b] = make_uint2(carry.x + inc.x - v.x, carry.y + inc.y - v.y);
        carry.x += tot.x; carry.y += tot.y;
    }
    if (threadIdx.x == 0) { ctr->n_records = carry.x; ctr->n_items = carry.y; }
}

// Scan phase C: bucket_start (in place over the histogram) and the work items of each key.
__global__ void __launch_bounds__(1024)
scan_apply_kernel(unsigned *__restrict__ hist, unsigned nkeys, const uint2 *__restrict__ blocksum,
                  const __grid_constant__ PlaneTab T, const __grid_constant__ BinParams P,
                  Item *__restrict__ items) {
    unsigned k0 = blockIdx.x * kScanBlock + threadIdx.x * 4;
    unsigned c[4];
    uint2 v = make_uint2(0, 0);
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        unsigned k = k0 + j;
        c[j] = k < nkeys ? hist[k] : 0;
        v.x += c[j]; v.y += nseg_of(c[j], P.segment);
    }
    uint2 tot;
    uint2 inc = block_scan_incl(v, &tot);
    uint2 off = blocksum[blockIdx.x];
    unsigned start = off.x + inc.x - v.x, istart = off.y + inc.y - v.y;
    unsigned ntile2 = (unsigned)(P.ntile * P.ntile);
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        unsigned k = k0 + j;
        if (k <= nkeys) hist[k] = start;             // hist[nkeys] = total
        if (k < nkeys && c[j]) {
            unsigned cls, tid;
            if (P.order == 1) { cls = k / ntile2; tid = k - cls * ntile2; }
            else { tid = k / (unsigned)P.ncls; cls = k - tid * (unsigned)P.ncls; }
            unsigned tv = tid / (unsigned)P.ntile, tu = tid - tv * (unsigned)P.ntile;
            unsigned ns = nseg_of(c[j], P.segment);
            unsigned len = (c[j] + ns - 1) / ns;
            for (unsigned s = 0; s < ns; ++s) {
                Item it;
                it.rec_begin = start + s * len;
                it.count = min(len, c[j] - s * len);
                it.origin = (tu * (unsigned)P.tile) | ((tv * (unsigned)P.tile) << 16);
                it.S = T.clsS[cls];
                items[istart + s] = it;
            }
            istart += ns;
        }
        start += c[j];
    }
}

// Pass 3: scatter into key order.  The record carries weight*vis (R9, natural weighting).
template <typename TT>
__global__ void __launch_bounds__(256)
scatter_kernel(const float2 *__restrict__ vis, const float *__restrict__ weight,
               const unsigned *__restrict__ key, const unsigned *__restrict__ rank,
               const uint2 *__restrict__ pre, const unsigned *__restrict__ bucket_start,
               long long nvis, Rec<TT> *__restrict__ rec) {
    long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nvis) return;
    unsigned k = key[i];
    if (k == WPG_NO_KEY) return;
    unsigned dst = bucket_start[k] + rank[i];
    float2 v = vis[i];
    TT w = (TT)weight[i];
    uint2 p = pre[i];
    Rec<TT> r;
    r.re = w * (TT)v.x; r.im = w * (TT)v.y; r.pos = p.x; r.koff = p.y;
    rec[dst] = r;
}

}  // namespace

int wpg_launch_bin(wpg_ctx *ctx, const void *d_vis, const double *d_uvw, const float *d_weight,
                   const double *d_freq, const PlaneTab &tab, const BinParams &bp,
                   const WorkspaceLayout &ws, wpg_prec prec, char *w) {
    long long nvis = bp.nrow * bp.nchan;
    Counters *ctr = (Counters *)(w + ws.off_counters);
    unsigned *hist = (unsigned *)(w + ws.off_hist);
    uint2 *blocksum = (uint2 *)(w + ws.off_blocksum);
    unsigned *key = (unsigned *)(w + ws.off_key), *rank = (unsigned *)(w + ws.off_rank);
    uint2 *pre = (uint2 *)(w + ws.off_pre);
    Item *items = (Item *)(w + ws.off_items);
    cudaStream_t s = ctx->stream;
    unsigned nb = (unsigned)((nvis + 255) / 256);
    if (nb) bin_count_kernel<<<nb, 256, 0, s>>>(d_uvw, d_weight, d_freq, tab, bp, ctr, hist, key, rank, pre);
    scan_reduce_kernel<<<ws.nblocks_scan, 1024, 0, s>>>(hist, ws.nkeys, (unsigned)bp.segment, blocksum);
    scan_blocksums_kernel<<<1, 1024, 0, s>>>(blocksum, ws.nblocks_scan, ctr);
    scan_apply_kernel<<<ws.nblocks_scan, 1024, 0, s>>>(hist, ws.nkeys, blocksum, tab, bp, items);
    if (nb) {
        if (prec == WPG_F32)
            scatter_kernel<float><<<nb, 256, 0, s>>>((const float2 *)d_vis, d_weight, key, rank, pre, hist, nvis,
                                                      (Rec<float> *)(w + ws.off_records));
        else
            scatter_kernel<double><<<nb, 256, 0, s>>>((const float2 *)d_vis, d_weight, key, rank, pre, hist, nvis,
                                                       (Rec<double> *)(w + ws.off_records));
    }
    ctx->n_launches += nb ? 5 : 3;
    WPG_CUDA(ctx, cudaGetLastError());
    return WPG_OK;
}
