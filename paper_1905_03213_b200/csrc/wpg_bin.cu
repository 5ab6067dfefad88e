// Step a1 — visibility binning: uvw -> (plane, window start, sub-cell offsets), sort key,
// histogram, exclusive prefix scan, scatter into key-sorted 16/24-byte records.
//
// The paper's analogue is the re-order of PAPER.md:62-78: count array C, exclusive prefix sum
// Eq. (2), scatter — keyed there by baseline (Eq. 1) so that consecutive samples of a baseline hit
// the same grid point.  Here the key is (support class, window start j0v, parity of
// j0u, j0u >> 1), i.e. the visibilities are ordered by the grid point they hit, whatever baseline
// they came from: runs of equal window start are what the gridder (wpg_grid.cu) accumulates in
// registers, and within a (row, parity) sweep the window start moves by even steps.
#include "wpg_common.h"

namespace {

constexpr int kScanBlock = 4096;   // keys per scan block (1024 threads x 4)

__device__ __forceinline__ void warp_count(unsigned long long *dst, unsigned v) {
    unsigned s = __reduce_add_sync(0xffffffffu, v);
    if ((threadIdx.x & 31) == 0 && s) atomicAdd(dst, (unsigned long long)s);
}

// Pass 0: f[ch] = freq[ch] / c0 (G1), once per channel instead of once per visibility.  Same IEEE
// division as G1 states, so the products u = uvw * f are bit-identical.
__global__ void chan_scale_kernel(const double *__restrict__ freq, int nchan, double *__restrict__ fscale) {
    int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c < nchan) fscale[c] = __ddiv_rn(freq[c], WPG_C0);
}

constexpr int kVpt = 4;            // visibilities per thread: four histogram atomics in flight per thread

// Pass 1: position math (fp64, G1-G3), validity (G4, R9), key, rank inside the key's bucket.
__global__ void __launch_bounds__(256)
bin_count_kernel(const double *__restrict__ uvw, const float *__restrict__ weight,
                 const double *__restrict__ fscale, const __grid_constant__ PlaneTab T,
                 const __grid_constant__ BinParams P, Counters *__restrict__ ctr,
                 unsigned *__restrict__ hist, unsigned *__restrict__ key_out,
                 unsigned *__restrict__ rank_out, uint2 *__restrict__ pre_out) {
    const long long nvis = P.nrow * P.nchan;
    const long long base = (long long)blockIdx.x * (256 * kVpt) + threadIdx.x;
    unsigned c_grid = 0, c_oob = 0, c_zero = 0, c_clamp = 0, c_upd = 0;
    unsigned key[kVpt], rank[kVpt];
#pragma unroll
    for (int j = 0; j < kVpt; ++j) {
        const long long i = base + j * 256;
        key[j] = WPG_NO_KEY;
        if (i < nvis) {
            long long row = i; int ch = 0;
            if (P.nchan > 1) { row = i / P.nchan; ch = (int)(i - row * P.nchan); }
            if (__ldg(weight + i) == 0.0f) {
                c_zero += 1;
            } else {
                VisPos r = wpg_locate(__ldg(uvw + 3 * row), __ldg(uvw + 3 * row + 1), __ldg(uvw + 3 * row + 2),
                                      __ldg(fscale + ch), P, T);
                if (!r.inside) {
                    c_oob += 1;
                } else {
                    c_grid += 1; c_clamp += r.clamped; c_upd += r.S * r.S;
                    key[j] = (unsigned)T.cls[r.p] * P.keys_per_class + (unsigned)r.j0v * (unsigned)P.nug +
                             ((unsigned)r.j0u & 1u) * (unsigned)P.nuh + (((unsigned)r.j0u >> 1) >> P.ushift);
                    pre_out[i] = make_uint2((unsigned)r.j0u | ((unsigned)r.j0v << 16), wpg_koff(r, P, T));
                }
            }
        }
    }
#pragma unroll
    for (int j = 0; j < kVpt; ++j) rank[j] = key[j] != WPG_NO_KEY ? atomicAdd(&hist[key[j]], 1u) : 0u;
#pragma unroll
    for (int j = 0; j < kVpt; ++j) {
        const long long i = base + j * 256;
        if (i < nvis) {
            key_out[i] = key[j];
            if (key[j] != WPG_NO_KEY) rank_out[i] = rank[j];
        }
    }
    warp_count(&ctr->n_gridded, c_grid);
    warp_count(&ctr->n_skipped_oob, c_oob);
    warp_count(&ctr->n_skipped_zero_weight, c_zero);
    warp_count(&ctr->n_clamped_w, c_clamp);
    warp_count(&ctr->n_updates, c_upd);
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

// Pass 3: scatter into key order.  The record carries weight*vis (R9, natural weighting).
template <typename TT>
__global__ void __launch_bounds__(256)
scatter_kernel(const float2 *__restrict__ vis, const float *__restrict__ weight,
               const unsigned *__restrict__ key, const unsigned *__restrict__ rank,
               const uint2 *__restrict__ pre, const unsigned *__restrict__ bucket_start,
               long long nvis, Rec<TT> *__restrict__ rec) {
    const long long base = (long long)blockIdx.x * (256 * kVpt) + threadIdx.x;
    unsigned k[kVpt], dst[kVpt];
#pragma unroll
    for (int j = 0; j < kVpt; ++j) {
        const long long i = base + j * 256;
        k[j] = i < nvis ? __ldg(key + i) : WPG_NO_KEY;
    }
#pragma unroll
    for (int j = 0; j < kVpt; ++j) {
        const long long i = base + j * 256;
        dst[j] = k[j] != WPG_NO_KEY ? __ldg(bucket_start + k[j]) + __ldg(rank + i) : 0u;
    }
#pragma unroll
    for (int j = 0; j < kVpt; ++j) {
        const long long i = base + j * 256;
        if (k[j] == WPG_NO_KEY) continue;
        float2 v = __ldg(vis + i);
        TT w = (TT)__ldg(weight + i);
        uint2 p = __ldg(pre + i);
        store_rec(rec + dst[j], w * (TT)v.x, w * (TT)v.y, p);
    }
}

}  // namespace

int wpg_launch_bin(wpg_ctx *ctx, const void *d_vis, const double *d_uvw, const float *d_weight,
                   const double *d_freq, const PlaneTab &tab, const BinParams &bp,
                   const WorkspaceLayout &ws, wpg_prec prec, char *w) {
    long long nvis = bp.nrow * bp.nchan;
    Counters *ctr = (Counters *)(w + ws.off_counters);
    unsigned *hist = (unsigned *)(w + ws.off_hist);
    unsigned *blocksum = (unsigned *)(w + ws.off_blocksum);
    unsigned *key = (unsigned *)(w + ws.off_key), *rank = (unsigned *)(w + ws.off_rank);
    uint2 *pre = (uint2 *)(w + ws.off_pre);
    cudaStream_t s = ctx->stream;
    double *fscale = (double *)(w + ws.off_fscale);
    unsigned nb = (unsigned)((nvis + 256 * kVpt - 1) / (256 * kVpt));
    chan_scale_kernel<<<(bp.nchan + 255) / 256, 256, 0, s>>>(d_freq, bp.nchan, fscale);
    if (nb) bin_count_kernel<<<nb, 256, 0, s>>>(d_uvw, d_weight, fscale, tab, bp, ctr, hist, key, rank, pre);
    scan_reduce_kernel<<<ws.nblocks_scan, 1024, 0, s>>>(hist, ws.nkeys, blocksum);
    scan_blocksums_kernel<<<1, 1024, 0, s>>>(blocksum, ws.nblocks_scan, ctr);
    scan_apply_kernel<<<ws.nblocks_scan, 1024, 0, s>>>(hist, ws.nkeys, blocksum);
    if (nb) {
        if (prec == WPG_F32)
            scatter_kernel<float><<<nb, 256, 0, s>>>((const float2 *)d_vis, d_weight, key, rank, pre, hist, nvis,
                                                      (Rec<float> *)(w + ws.off_records));
        else
            scatter_kernel<double><<<nb, 256, 0, s>>>((const float2 *)d_vis, d_weight, key, rank, pre, hist, nvis,
                                                       (Rec<double> *)(w + ws.off_records));
    }
    ctx->n_launches += nb ? 6 : 4;
    WPG_CUDA(ctx, cudaGetLastError());
    return WPG_OK;
}
