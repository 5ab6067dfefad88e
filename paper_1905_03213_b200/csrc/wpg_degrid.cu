// Degridding (PAPER.md:36 names it as gridding's companion): the adjoint of the gridder
// with unit weights, vis[r][c] = sum over the S x S window of grid * conj(K[p][ov][ou]) — a gather, no atomics.
// A warp takes 32 visibilities: every lane does the fp64 position math (G1-G4, identical to the binning) of one of
// them, then the warp walks the 32 windows together, lane <-> window cell, and sums across lanes.
#include "wpg_common.h"

namespace {

template <typename T> struct Cx;
template <> struct Cx<float> { using type = float2; };
template <> struct Cx<double> { using type = double2; };

template <typename T>
__device__ __forceinline__ T warp_sum(T v) {
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
    return v;
}

__global__ void dg_chan_scale_kernel(const double *__restrict__ freq, int nchan, double *__restrict__ fscale) {
    int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c < nchan) fscale[c] = __ddiv_rn(freq[c], WPG_C0);
}

// SCT: compile-time support of a uniform stack (lane -> cell arithmetic folds to shifts and masks), 0 = per-visibility
// S.  LPV lanes work on one visibility, 32 / LPV visibilities side by side in the warp (S = 8: two half-warps, four
// cells per lane, a 4-step sum): the loads stay coalesced (a group covers whole window rows), the cross-lane sum
// and the per-visibility broadcasts are shared.
template <typename T, int SCT, int LPV>
__global__ void __launch_bounds__(256)
degrid_kernel(const typename Cx<T>::type *__restrict__ grid, const double *__restrict__ uvw,
              const double *__restrict__ fscale, const __grid_constant__ PlaneTab Tb, const __grid_constant__ BinParams P,
              const typename Cx<T>::type *__restrict__ K, typename Cx<T>::type *__restrict__ vis_out,
              unsigned long long *__restrict__ counts) {
    using C = typename Cx<T>::type;
    constexpr int VPW = 32 / LPV;
    __shared__ uint2 s_tab[WPG_MAX_NW];
    wpg_stage_planetab(s_tab, Tb, P.Nw);
    __syncthreads();
    const SmemPlaneTab ST{s_tab, nullptr};
    const long long nvis = P.nrow * P.nchan;
    const int lane = threadIdx.x & 31;
    const int gl = lane % LPV, sub = lane / LPV;                    // lane inside its group, group = visibility slot
    const long long nwarp = ((long long)gridDim.x * 256) >> 5;
    unsigned n_pred = 0, n_out = 0;
    for (long long base = (((long long)blockIdx.x * 256 + threadIdx.x) >> 5) * 32; base < nvis; base += nwarp * 32) {
        // one visibility per lane: window start, coefficient slice, support
        const long long i = base + lane;
        unsigned pos = 0, koff = 0; int S = 0;
        if (i < nvis) {
            long long row = i; int ch = 0;
            if (P.nchan > 1) { const unsigned r32 = (unsigned)i / (unsigned)P.nchan; row = r32; ch = (int)((unsigned)i - r32 * (unsigned)P.nchan); }
            const VisPos r = wpg_locate(__ldg(uvw + 3 * row), __ldg(uvw + 3 * row + 1), __ldg(uvw + 3 * row + 2),
                                        __ldg(fscale + ch), P, ST);
            if (r.inside) { S = r.S; pos = (unsigned)r.j0u | ((unsigned)r.j0v << 16); koff = wpg_koff(r, P, ST); n_pred++; }
            else n_out++;
        }
        C mine; mine.x = mine.y = (T)0;
        const int cnt = (int)min((long long)32, nvis - base);
        for (int it = 0; it * VPW < cnt; ++it) {
            const int j = it * VPW + sub;                           // the visibility this lane's group works on (S = 0 past the end)
            const int Sq = __shfl_sync(0xffffffffu, S, j);
            const unsigned pj = __shfl_sync(0xffffffffu, pos, j), kj = __shfl_sync(0xffffffffu, koff, j);
            T sr = (T)0, si = (T)0;
            if (Sq) {                                               // 0: outside the grid, predicted as 0
                const int Sj = SCT ? SCT : Sq;
                const C *g0 = grid + (size_t)(pj >> 16) * P.N + (pj & 0xFFFFu);
                const C *k0 = K + kj;
                int iv = gl / Sj, iu = gl - iv * Sj;
                const int dv = LPV / Sj, du_ = LPV - dv * Sj;
                for (int c = gl; c < Sj * Sj; c += LPV) {
                    const C g = __ldg(g0 + (size_t)iv * P.N + iu), k = __ldg(k0 + c);
                    sr = fma(g.x, k.x, sr); sr = fma(g.y, k.y, sr);    // g * conj(k)
                    si = fma(g.y, k.x, si); si = fma(-g.x, k.y, si);
                    iu += du_; iv += dv;
                    if (iu >= Sj) { iu -= Sj; iv += 1; }
                }
            }
#pragma unroll
            for (int d = LPV / 2; d > 0; d >>= 1) {
                sr += __shfl_xor_sync(0xffffffffu, sr, d);
                si += __shfl_xor_sync(0xffffffffu, si, d);
            }
            // visibility L of the batch was summed in trip L / VPW by group L % VPW (every lane of the group has the sum)
            const T vr = __shfl_sync(0xffffffffu, sr, (lane % VPW) * LPV), vi = __shfl_sync(0xffffffffu, si, (lane % VPW) * LPV);
            if (lane / VPW == it) { mine.x = vr; mine.y = vi; }
        }
        if (i < nvis) vis_out[i] = mine;                            // one coalesced store of the 32 results
    }
    n_pred = __reduce_add_sync(0xffffffffu, n_pred); n_out = __reduce_add_sync(0xffffffffu, n_out);
    if (lane == 0) {
        if (n_pred) atomicAdd(&counts[2 * (blockIdx.x % kStatSlots)], (unsigned long long)n_pred);
        if (n_out) atomicAdd(&counts[2 * (blockIdx.x % kStatSlots) + 1], (unsigned long long)n_out);
    }
}

// ---------------------------------------------------------------------------------------------
// The fast degridder for uniform power-of-two supports 4, 8, 16 and power-of-two oversampling (configs 2, 3, 5).
// Same gather, input order and lane <-> cell mapping as degrid_kernel (a group of LPV lanes covers whole window rows
// with every load: 12 L1 wavefronts per visibility at S = 8, the minimum without reuse), but:
//  * positions by the lean straight-line math of the binning pass (wpg_locate_lean);
//  * the 32 window starts / slice offsets of a batch go through shared memory (one broadcast LDS per visibility instead of
//    three shuffles);
//  * the cell loop is unrolled at compile time (pointer + constant offsets, no index arithmetic);
//  * the cross-lane sums of R = 16 visibilities are taken together: each lane keeps its R partial sums and one butterfly
//    of R - 1 exchanges leaves every lane with one finished visibility, instead of R reductions of log2(LPV) steps.
template <typename T, int S>
__global__ void __launch_bounds__(256)
degrid_fast_kernel(const typename Cx<T>::type *__restrict__ grid, const double *__restrict__ uvw,
                   const double *__restrict__ fscale, const __grid_constant__ BinParams P,
                   const typename Cx<T>::type *__restrict__ K, typename Cx<T>::type *__restrict__ vis_out,
                   unsigned long long *__restrict__ counts) {
    using C = typename Cx<T>::type;
    constexpr int LPV = S == 4 ? 8 : (S == 8 ? 16 : 32);       // lanes per visibility
    constexpr int VPW = 32 / LPV;                               // visibilities side by side in the warp
    constexpr int CPL = S * S / LPV;                            // cells per lane
    constexpr int RPT = LPV / S;                                // window rows covered by one load of the group
    constexpr int NIT = 32 / VPW;                               // trips per batch of 32 visibilities
    constexpr int R = NIT < 16 ? NIT : 16;                      // partial sums reduced together
    __shared__ uint2 s_pk[8][32];                               // per warp: {pos | 0xFFFFFFFF, koff} of the batch
    const int lane = threadIdx.x & 31;
    const int gl = lane % LPV, sub = lane / LPV;
    uint2 *pk = s_pk[threadIdx.x >> 5];
    const long long nvis = P.nrow * P.nchan;
    const long long nwarp = ((long long)gridDim.x * 256) >> 5;
    const int c_row = gl / S, c_col = gl % S;
    unsigned n_pred = 0, n_out = 0;
    for (long long base = (((long long)blockIdx.x * 256 + threadIdx.x) >> 5) * 32; base < nvis; base += nwarp * 32) {
        const long long i = base + lane;
        uint2 mine_pk = make_uint2(0xFFFFFFFFu, 0u);
        if (i < nvis) {
            long long row = i; int ch = 0;
            if (P.nchan > 1) {
                const unsigned r32 = P.chan_shift >= 0 ? (unsigned)i >> P.chan_shift : (unsigned)i / (unsigned)P.nchan;
                row = r32; ch = (int)((unsigned)i - r32 * (unsigned)P.nchan);
            }
            const LeanPos r = wpg_locate_lean<true>(__ldg(uvw + 3 * row), __ldg(uvw + 3 * row + 1), __ldg(uvw + 3 * row + 2),
                                                    __ldg(fscale + ch), P, nullptr);
            if (r.inside) {
                mine_pk = make_uint2((unsigned)r.j0u | ((unsigned)r.j0v << 16), (unsigned)(((r.p * P.Q + r.ov) * P.Q + r.ou) * S * S));
                n_pred++;
            } else n_out++;
        }
        __syncwarp();
        pk[lane] = mine_pk;
        __syncwarp();
        C result; result.x = result.y = (T)0;
#pragma unroll
        for (int half = 0; half < NIT / R; ++half) {
            T pr[R], pi[R];
#pragma unroll
            for (int t = 0; t < R; ++t) {
                const uint2 q = pk[(half * R + t) * VPW + sub];          // broadcast inside the group
                T sr = (T)0, si = (T)0;
                if (q.x != 0xFFFFFFFFu) {
                    const C *g = grid + (size_t)((q.x >> 16) + c_row) * P.N + ((q.x & 0xFFFFu) + c_col);
                    const C *k = K + q.y + gl;
                    C gv[CPL], kv[CPL];
#pragma unroll
                    for (int c = 0; c < CPL; ++c) { gv[c] = __ldg(g + (size_t)c * RPT * P.N); kv[c] = __ldg(k + c * LPV); }
#pragma unroll
                    for (int c = 0; c < CPL; ++c) {                           // g * conj(k)
                        sr = fma(gv[c].x, kv[c].x, sr); sr = fma(gv[c].y, kv[c].y, sr);
                        si = fma(gv[c].y, kv[c].x, si); si = fma(-gv[c].x, kv[c].y, si);
                    }
                }
                pr[t] = sr; pi[t] = si;
            }
            // butterfly over the group's lanes: lane gl ends with the sum of partial index (gl * R / LPV)
            int d = LPV / 2;
#pragma unroll
            for (int h = R / 2; h >= 1; h /= 2, d /= 2) {
                const bool up = (gl & d) != 0;
#pragma unroll
                for (int j = 0; j < h; ++j) {
                    const T sr = up ? pr[j] : pr[j + h], si = up ? pi[j] : pi[j + h];
                    const T kr = up ? pr[j + h] : pr[j], ki = up ? pi[j + h] : pi[j];
                    pr[j] = kr + __shfl_xor_sync(0xffffffffu, sr, d);
                    pi[j] = ki + __shfl_xor_sync(0xffffffffu, si, d);
                }
            }
            for (; d >= 1; d /= 2) {                                          // R < LPV: the remaining lanes hold the same index
                pr[0] += __shfl_xor_sync(0xffffffffu, pr[0], d);
                pi[0] += __shfl_xor_sync(0xffffffffu, pi[0], d);
            }
            // lane gl now holds trip t = gl * R / LPV of this half, i.e. visibility (half * R + t) * VPW + sub of the batch
            if (NIT / R == 1) { result.x = pr[0]; result.y = pi[0]; }
            else if ((lane & 1) == half) { result.x = pr[0]; result.y = pi[0]; }    // S = 16: even lanes keep half 0, odd lanes half 1
        }
        // which visibility of the batch this lane holds
        int jv;
        if (NIT / R == 1) jv = (gl * R / LPV) * VPW + sub;                    // S = 4, 8: one finished visibility per lane
        else jv = ((lane & 1) * R + (lane >> 1)) * VPW + sub;                 // S = 16: lane pair (2t, 2t+1) holds trips t and 16 + t
        if (base + jv < nvis) vis_out[base + jv] = result;
    }
    n_pred = __reduce_add_sync(0xffffffffu, n_pred); n_out = __reduce_add_sync(0xffffffffu, n_out);
    if (lane == 0) {
        if (n_pred) atomicAdd(&counts[2 * (blockIdx.x % kStatSlots)], (unsigned long long)n_pred);
        if (n_out) atomicAdd(&counts[2 * (blockIdx.x % kStatSlots) + 1], (unsigned long long)n_out);
    }
}

}  // namespace

extern "C" size_t wpg_degrid_workspace_bytes(int nchan) {
    return nchan < 1 ? 0 : (size_t)((nchan * 8 + 255) & ~255) + 256;
}

extern "C" int wpg_degrid(wpg_ctx *ctx, const void *d_grid, const double *d_uvw, const double *d_freq, int64_t nrow,
                          int nchan, const void *d_kernels, const wpg_kdesc *desc, wpg_prec prec, void *d_vis_out,
                          void *d_workspace, size_t workspace_bytes, int64_t *h_counts2) {
    if (!ctx) return WPG_EINVAL;
    if (!d_grid || !d_kernels || !d_freq || (nrow > 0 && (!d_uvw || !d_vis_out)))
        return wpg_fail(ctx, WPG_EINVAL, "NULL pointer argument");
    PlaneTab tab; BinParams bp; WorkspaceLayout ws0;
    int rc = wpg_make_plan(ctx, desc, nrow, nchan, prec, &tab, &bp, &ws0);
    if (rc) return rc;
    const size_t need = wpg_degrid_workspace_bytes(nchan);
    if (!d_workspace || workspace_bytes < need)
        return wpg_fail(ctx, WPG_ENOMEM, "workspace of %zu bytes given, %zu needed", workspace_bytes, need);
    WPG_DEVICE(ctx);
    cudaStream_t s = ctx->stream;
    char *w = (char *)d_workspace;
    unsigned long long *counts = (unsigned long long *)w;             // kStatSlots x {predicted, outside}
    double *fscale = (double *)(w + 256);
    WPG_CUDA(ctx, cudaMemsetAsync(counts, 0, 256, s));
    dg_chan_scale_kernel<<<(nchan + 255) / 256, 256, 0, s>>>(d_freq, nchan, fscale);
    const long long nvis = (long long)nrow * nchan;
    if (nvis) {
        const int blocks = (int)min((long long)ctx->sm_count * 8, (nvis + 255) / 256);
        const int S1 = bp.ncls == 1 ? tab.clsS[0] : 0;
#define WPG_DG(TT, CC, SS, LL) degrid_kernel<TT, SS, LL><<<blocks, 256, 0, s>>>((const CC *)d_grid, d_uvw, fscale, tab, bp, (const CC *)d_kernels, (CC *)d_vis_out, counts)
#define WPG_DGF(TT, CC, SS) degrid_fast_kernel<TT, SS><<<blocks, 256, 0, s>>>((const CC *)d_grid, d_uvw, fscale, bp, (const CC *)d_kernels, (CC *)d_vis_out, counts)
        const bool fast = !ctx->opt_no_pairs && bp.qshift >= 0 && (S1 == 4 || S1 == 8 || S1 == 16);
        if (fast && prec == WPG_F32) { if (S1 == 8) WPG_DGF(float, float2, 8); else if (S1 == 16) WPG_DGF(float, float2, 16); else WPG_DGF(float, float2, 4); }
        else if (fast) { if (S1 == 8) WPG_DGF(double, double2, 8); else if (S1 == 16) WPG_DGF(double, double2, 16); else WPG_DGF(double, double2, 4); }
        else if (prec == WPG_F32) { if (S1 == 8) WPG_DG(float, float2, 8, 16); else if (S1 == 16) WPG_DG(float, float2, 16, 32); else if (S1 == 4) WPG_DG(float, float2, 4, 8); else WPG_DG(float, float2, 0, 32); }
        else { if (S1 == 8) WPG_DG(double, double2, 8, 16); else if (S1 == 16) WPG_DG(double, double2, 16, 32); else if (S1 == 4) WPG_DG(double, double2, 4, 8); else WPG_DG(double, double2, 0, 32); }
#undef WPG_DG
#undef WPG_DGF
    }
    ctx->n_launches += nvis ? 2 : 1;
    WPG_CUDA(ctx, cudaGetLastError());
    if (h_counts2) {
        unsigned long long h[2 * kStatSlots];
        WPG_CUDA(ctx, cudaMemcpyAsync(h, counts, sizeof h, cudaMemcpyDeviceToHost, s));
        WPG_CUDA(ctx, cudaStreamSynchronize(s));
        h_counts2[0] = h_counts2[1] = 0;
        for (int k = 0; k < kStatSlots; ++k) { h_counts2[0] += (int64_t)h[2 * k]; h_counts2[1] += (int64_t)h[2 * k + 1]; }
    }
    return WPG_OK;
}
