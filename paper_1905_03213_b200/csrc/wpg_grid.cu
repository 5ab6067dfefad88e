// Step a2 — the gridder: grid[j0v+iv][j0u+iu] += (wt*vis) * K[p][ov][ou][iv][iu]  (O4 G5).
//
// Two kernels:
//  * grid_naive_kernel — one global reduction per update straight from the raw inputs (the design
//    whose ceiling is the atomic roofline; "write access to the global memory ... in an
//    atomic manner").  Independent of the binning pass, so it also cross-checks it.
//  * grid_tiles_kernel — the paper's register accumulator ("accumulated and
//    buffered in a register ... written into the global memory when the processing moves on"),
//    re-cut for key-sorted records: a warp walks the records of one work item (one uv tile, one
//    support S); lane <-> support-cell residue (b, a) = cell position modulo S relative to the tile
//    origin.  Because the window start stays inside a tile of edge <= S, each residue can only land
//    on 2 x 2 grid cells, so 4 register accumulators per residue hold the whole item and the global
//    reductions (red.global.add.v2.f32 / .f64) happen once per item instead of once per update.
#include "wpg_common.h"

namespace {

template <typename T> struct Cplx;
template <> struct Cplx<float> { using type = float2; };
template <> struct Cplx<double> { using type = double2; };

__device__ __forceinline__ void red_add(float2 *addr, float re, float im) {
    asm volatile("red.global.add.v2.f32 [%0], {%1, %2};" ::"l"(addr), "f"(re), "f"(im) : "memory");
}
__device__ __forceinline__ void red_add(double2 *addr, double re, double im) {
    asm volatile("red.global.add.f64 [%0], %1;" ::"l"(&addr->x), "d"(re) : "memory");
    asm volatile("red.global.add.f64 [%0], %1;" ::"l"(&addr->y), "d"(im) : "memory");
}

// ------------------------------------------------------------------------------------ naive
template <typename T>
__global__ void __launch_bounds__(256)
grid_naive_kernel(const float2 *__restrict__ vis, const double *__restrict__ uvw,
                  const float *__restrict__ weight, const double *__restrict__ freq,
                  const __grid_constant__ PlaneTab Tb, const __grid_constant__ BinParams P,
                  const typename Cplx<T>::type *__restrict__ K, typename Cplx<T>::type *__restrict__ grid,
                  Counters *__restrict__ ctr) {
    using C = typename Cplx<T>::type;
    long long nvis = P.nrow * P.nchan;
    long long nwarp = ((long long)gridDim.x * blockDim.x) >> 5;
    int lane = threadIdx.x & 31;
    unsigned long long c_grid = 0, c_oob = 0, c_zero = 0, c_clamp = 0, c_upd = 0;
    for (long long i = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5; i < nvis; i += nwarp) {
        float wt = weight[i];
        if (wt == 0.0f) { c_zero++; continue; }
        long long row = i / P.nchan;
        int ch = (int)(i - row * P.nchan);
        double f = __ddiv_rn(freq[ch], WPG_C0);
        VisPos r = wpg_locate(uvw[3 * row], uvw[3 * row + 1], uvw[3 * row + 2], f, P, Tb);
        if (!r.inside) { c_oob++; continue; }
        c_grid++; c_clamp += r.clamped; c_upd += r.S * r.S;
        float2 v = vis[i];
        T re = (T)wt * (T)v.x, im = (T)wt * (T)v.y;
        const C *Ks = K + wpg_koff(r, P, Tb);
        int S = r.S, S2 = S * S;
        for (int c = lane; c < S2; c += 32) {
            int iv = c / S, iu = c - iv * S;
            C k = Ks[c];
            red_add(grid + (long long)(r.j0v + iv) * P.N + (r.j0u + iu), re * k.x - im * k.y, re * k.y + im * k.x);
        }
    }
    if (lane == 0) {
        if (c_grid) atomicAdd(&ctr->n_gridded, c_grid);
        if (c_oob) atomicAdd(&ctr->n_skipped_oob, c_oob);
        if (c_zero) atomicAdd(&ctr->n_skipped_zero_weight, c_zero);
        if (c_clamp) atomicAdd(&ctr->n_clamped_w, c_clamp);
        if (c_upd) atomicAdd(&ctr->n_updates, c_upd);
    }
}

// ------------------------------------------------------------------------------------ tiled
template <typename T> __device__ __forceinline__ Rec<T> load_rec(const Rec<T> *p);
template <> __device__ __forceinline__ Rec<float> load_rec<float>(const Rec<float> *p) {
    float4 q = __ldg(reinterpret_cast<const float4 *>(p));
    Rec<float> r;
    r.re = q.x; r.im = q.y; r.pos = __float_as_uint(q.z); r.koff = __float_as_uint(q.w);
    return r;
}
template <> __device__ __forceinline__ Rec<double> load_rec<double>(const Rec<double> *p) {
    Rec<double> r;                                              // 24-byte records: 8-byte aligned only
    r.re = __ldg(&p->re); r.im = __ldg(&p->im);
    uint2 t = __ldg(reinterpret_cast<const uint2 *>(&p->pos));
    r.pos = t.x; r.koff = t.y;
    return r;
}

constexpr int kGridThreads = 256;

template <typename T, int RMAX, int MINB>
__global__ void __launch_bounds__(kGridThreads, MINB)
grid_tiles_kernel(const Rec<T> *__restrict__ rec, const Item *__restrict__ items,
                  const Counters *__restrict__ ctr, const typename Cplx<T>::type *__restrict__ K,
                  typename Cplx<T>::type *__restrict__ grid, int N, int nchunk) {
    using C = typename Cplx<T>::type;
    const int lane = threadIdx.x & 31;
    const unsigned nwarp = (gridDim.x * blockDim.x) >> 5;
    const unsigned long long nunits = (unsigned long long)ctr->n_items * (unsigned)nchunk;
    for (unsigned long long unit = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; unit < nunits; unit += nwarp) {
        const unsigned item = (unsigned)(unit / (unsigned)nchunk);
        const int chunk = (int)(unit - (unsigned long long)item * (unsigned)nchunk);
        const uint4 itq = __ldg(reinterpret_cast<const uint4 *>(items + item));
        const int S = (int)itq.w, S2 = S * S;
        const int r0 = chunk * 32 * RMAX;
        if (r0 >= S2) continue;
        const int u0 = (int)(itq.z & 0xFFFFu), v0 = (int)(itq.z >> 16);
        const int kmax = min(RMAX, (S2 - r0 + 31) >> 5);
        int a[RMAX], b[RMAX];
        T acc[RMAX][4][2];
#pragma unroll
        for (int k = 0; k < RMAX; ++k) {
            int r = r0 + k * 32 + lane;
            bool valid = r < S2;
            b[k] = valid ? r / S : -1;               // b = -1 marks an idle slot
            a[k] = valid ? r - b[k] * S : 0;
#pragma unroll
            for (int s = 0; s < 4; ++s) acc[k][s][0] = acc[k][s][1] = (T)0;
        }
        const Rec<T> *rp = rec + itq.x;
        const unsigned cnt = itq.y;
        Rec<T> cur = load_rec<T>(rp);
        for (unsigned i = 0; i < cnt; ++i) {
            Rec<T> nxt = cur;
            if (i + 1 < cnt) nxt = load_rec<T>(rp + i + 1);
            const int du = (int)(cur.pos & 0x1FFFu) - u0, dv = (int)((cur.pos >> 13) & 0x1FFFu) - v0;
            const C *Ks = K + cur.koff;
#pragma unroll
            for (int k = 0; k < RMAX; ++k) {
                if (k < kmax && b[k] >= 0) {
                    const bool hu = a[k] < du, hv = b[k] < dv;
                    const int iu = a[k] - du + (hu ? S : 0), iv = b[k] - dv + (hv ? S : 0);
                    const C c = __ldg(Ks + iv * S + iu);
                    const T pr = cur.re * c.x - cur.im * c.y, pi = cur.re * c.y + cur.im * c.x;
                    const int sel = (hv ? 2 : 0) + (hu ? 1 : 0);
#pragma unroll
                    for (int s = 0; s < 4; ++s)
                        if (sel == s) { acc[k][s][0] += pr; acc[k][s][1] += pi; }
                }
            }
            cur = nxt;
        }
        // flush: one reduction per touched cell of the 2S x 2S neighbourhood
#pragma unroll
        for (int k = 0; k < RMAX; ++k) {
            if (k < kmax && b[k] >= 0) {
#pragma unroll
                for (int s = 0; s < 4; ++s) {
                    if (acc[k][s][0] != (T)0 || acc[k][s][1] != (T)0) {
                        int cu = u0 + a[k] + ((s & 1) ? S : 0), cv = v0 + b[k] + ((s & 2) ? S : 0);
                        red_add(grid + (long long)cv * N + cu, acc[k][s][0], acc[k][s][1]);
                    }
                }
            }
        }
    }
}

template <typename T, int RMAX, int MINB>
int launch_tiles(wpg_ctx *ctx, const BinParams &bp, const WorkspaceLayout &ws, const void *K, void *grid,
                 char *w, int maxS) {
    using C = typename Cplx<T>::type;
    int nchunk = (maxS * maxS + 32 * RMAX - 1) / (32 * RMAX);
    int per_sm = ctx->opt_ctas_per_sm ? ctx->opt_ctas_per_sm : MINB;
    int blocks = ctx->sm_count * per_sm;
    grid_tiles_kernel<T, RMAX, MINB><<<blocks, kGridThreads, 0, ctx->stream>>>(
        (const Rec<T> *)(w + ws.off_records), (const Item *)(w + ws.off_items),
        (const Counters *)(w + ws.off_counters), (const C *)K, (C *)grid, bp.N, nchunk);
    ctx->n_launches += 1;
    WPG_CUDA(ctx, cudaGetLastError());
    return WPG_OK;
}

}  // namespace

int wpg_launch_grid(wpg_ctx *ctx, const PlaneTab &, const BinParams &bp, const WorkspaceLayout &ws,
                    wpg_prec prec, const void *K, void *grid, char *w, int maxS) {
    if (bp.nrow == 0) return WPG_OK;
    int S2 = maxS * maxS;
    if (prec == WPG_F32) {
        if (S2 <= 32) return launch_tiles<float, 1, 6>(ctx, bp, ws, K, grid, w, maxS);
        if (S2 <= 64) return launch_tiles<float, 2, 4>(ctx, bp, ws, K, grid, w, maxS);
        if (S2 <= 128) return launch_tiles<float, 4, 3>(ctx, bp, ws, K, grid, w, maxS);
        return launch_tiles<float, 8, 2>(ctx, bp, ws, K, grid, w, maxS);
    }
    if (S2 <= 32) return launch_tiles<double, 1, 4>(ctx, bp, ws, K, grid, w, maxS);
    if (S2 <= 64) return launch_tiles<double, 2, 3>(ctx, bp, ws, K, grid, w, maxS);
    return launch_tiles<double, 4, 2>(ctx, bp, ws, K, grid, w, maxS);
}

int wpg_launch_naive(wpg_ctx *ctx, const void *d_vis, const double *d_uvw, const float *d_weight,
                     const double *d_freq, const PlaneTab &tab, const BinParams &bp, wpg_prec prec,
                     const void *K, void *grid, Counters *d_c) {
    if (bp.nrow == 0) return WPG_OK;
    int blocks = ctx->sm_count * 8;
    if (prec == WPG_F32)
        grid_naive_kernel<float><<<blocks, 256, 0, ctx->stream>>>((const float2 *)d_vis, d_uvw, d_weight, d_freq, tab, bp,
                                                                   (const float2 *)K, (float2 *)grid, d_c);
    else
        grid_naive_kernel<double><<<blocks, 256, 0, ctx->stream>>>((const float2 *)d_vis, d_uvw, d_weight, d_freq, tab, bp,
                                                                    (const double2 *)K, (double2 *)grid, d_c);
    ctx->n_launches += 1;
    WPG_CUDA(ctx, cudaGetLastError());
    return WPG_OK;
}
