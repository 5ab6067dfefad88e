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

// Block totals of the wpg_stats counters.  The four per-visibility flags travel as 8-bit fields of one word (a
// warp holds 32 * kVpt = 128 visibilities), the update count on its own: two warp reductions per block.
constexpr unsigned kFlagGridded = 1u, kFlagOob = 1u << 8, kFlagZero = 1u << 16, kFlagClamped = 1u << 24;
__device__ __forceinline__ void block_count(Counters *ctr, unsigned flags, unsigned c_upd) {
    __shared__ unsigned s_cnt[5];
    if (threadIdx.x < 5) s_cnt[threadIdx.x] = 0;
    __syncthreads();
    const unsigned f = __reduce_add_sync(0xffffffffu, flags), u = __reduce_add_sync(0xffffffffu, c_upd);
    if ((threadIdx.x & 31) == 0) {
        if (f & 0xFFu) atomicAdd(&s_cnt[0], f & 0xFFu);
        if ((f >> 8) & 0xFFu) atomicAdd(&s_cnt[1], (f >> 8) & 0xFFu);
        if ((f >> 16) & 0xFFu) atomicAdd(&s_cnt[2], (f >> 16) & 0xFFu);
        if (f >> 24) atomicAdd(&s_cnt[3], f >> 24);
        if (u) atomicAdd(&s_cnt[4], u);
    }
    __syncthreads();
    if (threadIdx.x < 5 && s_cnt[threadIdx.x]) {
        unsigned long long *dst = threadIdx.x == 0 ? ctr->n_gridded : threadIdx.x == 1 ? ctr->n_skipped_oob
                                : threadIdx.x == 2 ? ctr->n_skipped_zero_weight : threadIdx.x == 3 ? ctr->n_clamped_w
                                : ctr->n_updates;
        atomicAdd(dst + (blockIdx.x + blockIdx.y) % kStatSlots, (unsigned long long)s_cnt[threadIdx.x]);
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
// ignored — the census only steers the key resolution, the result of the binning does not depend on it, so every
// kCensusStride-th row is enough).  One thread per sampled row, all channels.
constexpr int kCensusStride = 16;
__global__ void __launch_bounds__(256)
census_kernel(const double *__restrict__ uvw, const double *__restrict__ fscale, const __grid_constant__ PlaneTab T,
              const __grid_constant__ BinParams P, Counters *__restrict__ ctr) {
    __shared__ unsigned s_cnt[8][WPG_MAX_CLS];
    __shared__ uint2 s_tab[WPG_MAX_NW];
    for (int i = threadIdx.x; i < 8 * WPG_MAX_CLS; i += 256) (&s_cnt[0][0])[i] = 0;
    wpg_stage_planetab(s_tab, T, P.Nw);
    __syncthreads();
    unsigned *mine = s_cnt[threadIdx.x >> 5];
    const long long stride = P.nrow >= 65536 ? kCensusStride : 1;
    for (long long row = ((long long)blockIdx.x * 256 + threadIdx.x) * stride; row < P.nrow; row += (long long)gridDim.x * 256 * stride) {
        const double wm = __ldg(uvw + 3 * row + 2);
        for (int ch = 0; ch < P.nchan; ++ch) {
            const double w = __dmul_rn(wm, __ldg(fscale + ch));
            int p = 0;
            if (P.dw > 0.0) {
                const double fp = floor(wpg_div_const(__dadd_rn(w, P.w_max), P.dw, P.rdw));
                p = fp < 0.0 ? 0 : (fp > (double)(P.Nw - 1) ? P.Nw - 1 : (int)fp);
            }
            atomicAdd(&mine[s_tab[p].y >> 8], (unsigned)stride);
        }
    }
    __syncthreads();
    if (threadIdx.x < P.ncls) {
        unsigned t = 0;
        for (int wv = 0; wv < 8; ++wv) t += s_cnt[wv][threadIdx.x];
        if (t) atomicAdd(&ctr->census[threadIdx.x], t);
    }
}

// Ragged stacks, pass 0c (one warp, lane = support class): split the key budget among the classes.  Every class
// starts with one key per grid column; the class with the most visibilities per key is refined (one more bit of
// j0v) as long as the total stays within the budget.
__global__ void plan_keys_kernel(Counters *__restrict__ ctr, int ncls, int N, unsigned budget) {
    static_assert(WPG_MAX_CLS <= 32, "one lane per support class");
    if (blockIdx.x) return;
    const int c = threadIdx.x;                       // 32 threads
    const bool have = c < ncls;
    auto keys = [&](unsigned s_) { return (unsigned long long)N * (unsigned)((N + (1 << s_) - 1) >> s_); };
    const float census = have ? (float)ctr->census[c] + 1.0f : 0.0f;
    unsigned sh = 13;
    while (have && sh && keys(sh - 1) == keys(sh)) sh -= 1;          // bits that do not add keys (N < 2^13)
    unsigned long long total = 0;
    {
        unsigned long long mine = have ? keys(sh) : 0ull;
        for (int d = 16; d > 0; d >>= 1) mine += __shfl_xor_sync(0xffffffffu, mine, d);
        total = mine;
    }
    for (;;) {
        // this lane's candidate: one more bit, if it adds keys and fits
        const unsigned long long grow = have && sh ? keys(sh - 1) - keys(sh) : 0ull;
        const bool can = have && sh && grow > 0 && total + grow <= budget;
        float d = can ? census / (float)keys(sh) : -1.0f;
        // argmax over the lanes (lowest class wins ties)
        float best = d; int who = c;
        for (int o = 16; o > 0; o >>= 1) {
            const float ob = __shfl_xor_sync(0xffffffffu, best, o);
            const int ow = __shfl_xor_sync(0xffffffffu, who, o);
            if (ob > best || (ob == best && ow < who)) { best = ob; who = ow; }
        }
        if (best < 0.0f) break;
        const unsigned long long g = __shfl_sync(0xffffffffu, grow, who);
        if (c == who) { sh -= 1; while (sh && keys(sh - 1) == keys(sh)) sh -= 1; }
        total += g;
    }
    // bases: exclusive prefix sum of the classes' key counts
    unsigned long long mine = have ? keys(sh) : 0ull, incl = mine;
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned long long t = __shfl_up_sync(0xffffffffu, incl, o);
        if (c >= o) incl += t;
    }
    if (have) {
        ctr->key_base[c] = (unsigned)(incl - mine); ctr->key_shift[c] = sh;
        ctr->key_nkg[c] = (unsigned)((N + (1 << sh) - 1) >> sh);
        if (c == ncls - 1) ctr->key_base[ncls] = (unsigned)incl;
    }
}

constexpr int kVpt = 4;            // visibilities per thread: four independent atomics in flight per thread

// The kVpt visibilities of a thread.  Default: a block takes 256 * kVpt consecutive visibilities, thread t the
// ones at t, t + 256, ...  With the "row_block" hint (P.vis_block = visibilities per time step; the blocks of a group
// of kVpt time steps are consecutive): thread x of group dg takes visibility x of the time steps dg * kVpt + j — the same baseline and
// channel at consecutive times, whose window starts (and so sort keys) mostly coincide, so that the
// bucket counter is touched once per run of equal keys, and equal records are merged (compression).  Loads stay
// coalesced either way (consecutive lanes, consecutive x).  idx = 0xFFFFFFFF: no visibility.
struct VisIdx { unsigned i[kVpt], row[kVpt]; int ch[kVpt]; };
__device__ __forceinline__ VisIdx vis_indices(const BinParams &P) {
    VisIdx V;
    const unsigned nvis = (unsigned)(P.nrow * P.nchan);             // < 2^32 - 2 (wpg_make_plan)
    if (P.vis_block) {
        // Block order: tiles of vis_tile groups of time steps; inside a tile consecutive blocks — the ones resident
        // together — take the SAME 256 baselines / channels at successive time groups.  A baseline's track crosses a
        // window in ~10 samples, so these blocks hit the same bucket counters and append to the same stretches of the
        // sorted records while those are still in L2; across tiles the inputs are still read front to back.
        // (grid.y = tile, grid.x = (block of 256 baselines / channels) * vis_tile + group inside the tile; vis_tile = 2^k)
        const unsigned bx = blockIdx.x >> P.vis_tile_shift;
        const unsigned dg = blockIdx.y * P.vis_tile + (blockIdx.x & (P.vis_tile - 1u));
        const unsigned x = bx * 256u + threadIdx.x;
        // one division per thread, not per visibility — a shift for a power-of-two channel count
        const unsigned xr = P.chan_shift >= 0 ? x >> P.chan_shift : x / (unsigned)P.nchan;
        const int ch = (int)(x - xr * (unsigned)P.nchan);
        const unsigned rows_per_step = P.row_block;
#pragma unroll
        for (int j = 0; j < kVpt; ++j) {
            const unsigned long long step = (unsigned long long)dg * kVpt + j;
            const unsigned long long i = step * P.vis_block + x;
            const bool ok = x < P.vis_block && i < nvis;
            V.i[j] = ok ? (unsigned)i : 0xFFFFFFFFu;
            V.row[j] = (unsigned)(step * rows_per_step) + xr;
            V.ch[j] = ch;
        }
    } else {
#pragma unroll
        for (int j = 0; j < kVpt; ++j) {
            const unsigned long long i = (unsigned long long)blockIdx.x * (256 * kVpt) + j * 256 + threadIdx.x;
            const bool ok = i < nvis;
            V.i[j] = ok ? (unsigned)i : 0xFFFFFFFFu;
            const unsigned r = P.chan_shift >= 0 ? (unsigned)i >> P.chan_shift : (unsigned)i / (unsigned)P.nchan;
            V.row[j] = r; V.ch[j] = (int)((unsigned)i - r * (unsigned)P.nchan);
        }
    }
    return V;
}

// Run structure of a thread's visibilities.  head[j]: first of a run of equal valid keys; rhead[j]: starts a
// record — with record compression ("compression": samples that fall on the
// same point are merged before gridding) a visibility whose window start AND coefficient slice equal its
// predecessor's is summed into the predecessor's record instead of getting its own; nrec[j]: records in the key
// run that starts at j.  Without compression every valid visibility is its own record.
__device__ __forceinline__ void key_runs(const unsigned (&key)[kVpt], const unsigned (&pos)[kVpt], const unsigned (&koff)[kVpt],
                                         bool compress, bool (&head)[kVpt], bool (&rhead)[kVpt], unsigned (&nrec)[kVpt]) {
#pragma unroll
    for (int j = 0; j < kVpt; ++j) {
        const bool valid = key[j] != WPG_NO_KEY;
        const bool same_key = j > 0 && key[j] == key[j - 1];
        head[j] = valid && !same_key;
        rhead[j] = valid && !(compress && same_key && pos[j] == pos[j > 0 ? j - 1 : 0] && koff[j] == koff[j > 0 ? j - 1 : 0]);
    }
#pragma unroll
    for (int j = kVpt - 1; j >= 0; --j)
        nrec[j] = (rhead[j] ? 1u : 0u) + ((j + 1 < kVpt && key[j + 1] == key[j]) ? nrec[j + 1 < kVpt ? j + 1 : j] : 0u);
}

// ---------------------------------------------------------------------------------------------
// Position math (fp64, G1-G3) and validity (G4, R9).  Both passes evaluate it: recomputing is cheaper than a round
// trip of (key, position, coefficient offset) through HBM (measured in round 2: an 8-byte intermediate per visibility
// made the pair of passes slower on every workload), and the workspace holds nothing per visibility but the records.
//
// The fast path is straight-line code: quotients by Markstein's sequence (wpg_div_const), floor() through the
// 2^52 + 2^51 rounding constant instead of the conversion pipe, and ONE flag that says whether any of the three
// values whose floor is taken lies within 1e-6 of an integer (or outside the range where the trick is valid).  Only
// then — a few visibilities in a million — the written form with IEEE divisions is evaluated out of line
// (wpg_locate), so that G6 holds whatever the constant-divisor sequence does in its last bit.
struct RawVis { double um, vm, wm, f; float wt; };
struct Located { unsigned key, pos, koff; int S; bool clamped; };

// QP2: the oversampling factor is a power of two (else the general form is used throughout)
template <bool QP2>
__device__ __forceinline__ Located locate_vis(const RawVis &v, const uint2 *s_tab, const uint4 *s_ck, const BinParams &P) {
    Located L; L.key = WPG_NO_KEY; L.pos = L.koff = 0; L.S = 0; L.clamped = false;
    const LeanPos r = wpg_locate_lean<QP2>(v.um, v.vm, v.wm, v.f, P, s_tab);
    const int p = r.p, j0u = r.j0u, j0v = r.j0v, ou = r.ou, ov = r.ov, S = r.S;
    const bool inside = r.inside, clamped = r.clamped;
    if (!inside) return L;
    L.S = S; L.clamped = clamped;
    if (P.ncls == 1) {
        L.key = (unsigned)j0u * (unsigned)P.nkg + ((unsigned)j0v >> P.kshift);
        L.koff = (unsigned)(((p * P.Q + ov) * P.Q + ou) * S * S);
    } else {
        const uint2 e = s_tab[p];
        const uint4 ck = s_ck[e.y >> 8];
        L.key = ck.x + (unsigned)j0u * ck.y + ((unsigned)j0v >> ck.z);
        L.koff = e.x + (unsigned)((ov * P.Q + ou) * S * S);
    }
    L.pos = (unsigned)j0u | ((unsigned)j0v << 16);
    return L;
}

// The loads of a thread's kVpt visibilities, all issued before any arithmetic (the passes are latency-bound
// otherwise).  wt = 0 for "no visibility".
__device__ __forceinline__ void load_raw(const VisIdx &V, const double *__restrict__ uvw, const float *__restrict__ weight,
                                         const double *__restrict__ fscale, RawVis (&raw)[kVpt]) {
#pragma unroll
    for (int j = 0; j < kVpt; ++j) {
        const bool ok = V.i[j] != 0xFFFFFFFFu;
        // the inputs stream through once per pass: evict-first, so that they do not push the bucket table out of L2
        raw[j].wt = ok ? __ldcs(weight + V.i[j]) : 0.f;
        const double *q = uvw + 3ull * (ok ? V.row[j] : 0u);
        raw[j].um = ok ? __ldcs(q) : 0.0; raw[j].vm = ok ? __ldcs(q + 1) : 0.0; raw[j].wm = ok ? __ldcs(q + 2) : 0.0;
        raw[j].f = __ldg(fscale + (ok ? V.ch[j] : 0));
    }
    // keeps the compiler from consuming a loaded value (and so waiting for it) before the loads that follow in
    // program order have been issued
#pragma unroll
    for (int j = 0; j < kVpt; ++j) asm volatile("" : "+f"(raw[j].wt), "+d"(raw[j].um), "+d"(raw[j].vm), "+d"(raw[j].wm));
}

// Pass 1: histogram of the keys (reductions without return value) and the wpg_stats counters.
template <bool QP2>
__global__ void __launch_bounds__(256, 4)
bin_count_kernel(const double *__restrict__ uvw, const float *__restrict__ weight,
                 const double *__restrict__ fscale, const __grid_constant__ PlaneTab T,
                 const __grid_constant__ BinParams P, Counters *__restrict__ ctr, unsigned *__restrict__ hist) {
    const VisIdx V = vis_indices(P);
    __shared__ uint2 s_tab[WPG_MAX_NW];
    __shared__ uint4 s_ck[WPG_MAX_CLS];
    RawVis raw[kVpt];
    load_raw(V, uvw, weight, fscale, raw);
    wpg_stage_planetab(s_tab, T, P.Nw);
    wpg_stage_classkeys(s_ck, ctr, P);
    __syncthreads();
    unsigned key[kVpt], pos[kVpt], koff[kVpt], nrec[kVpt], flags = 0, c_upd = 0;
    bool head[kVpt], rhead[kVpt];
#pragma unroll
    for (int j = 0; j < kVpt; ++j) {
        key[j] = WPG_NO_KEY; pos[j] = koff[j] = 0;
        if (V.i[j] == 0xFFFFFFFFu) continue;
        if (raw[j].wt == 0.0f) { flags += kFlagZero; continue; }                  // R19: zero weight is tested first
        const Located L = locate_vis<QP2>(raw[j], s_tab, s_ck, P);
        if (L.key == WPG_NO_KEY) { flags += kFlagOob; continue; }
        flags += kFlagGridded + (L.clamped ? kFlagClamped : 0u); c_upd += L.S * L.S;
        key[j] = L.key; pos[j] = L.pos; koff[j] = L.koff;
    }
    key_runs(key, pos, koff, P.compress != 0, head, rhead, nrec);
#pragma unroll
    for (int j = 0; j < kVpt; ++j)
        if (head[j]) asm volatile("red.global.add.u32 [%0], %1;" ::"l"(hist + key[j]), "r"(nrec[j]) : "memory");
    block_count(ctr, flags, c_upd);
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
// (pol: the L2 evict-last policy of the scatter pass; the fp64 record's plain stores ignore it)
__device__ __forceinline__ void store_rec(Rec<float> *dst, float re, float im, uint2 p, unsigned long long pol) {
    asm volatile("st.global.L2::cache_hint.v4.b32 [%0], {%1, %2, %3, %4}, %5;" ::"l"(dst), "r"(__float_as_uint(re)), "r"(__float_as_uint(im)),
                 "r"(p.x), "r"(p.y), "l"(pol) : "memory");
}
__device__ __forceinline__ void store_rec(Rec<double> *dst, double re, double im, uint2 p, unsigned long long) {
    dst->re = re; dst->im = im;
    *reinterpret_cast<uint2 *>(&dst->pos) = p;
}

// Pass 3: scatter into key order.  The slot of a record is the running cursor of its bucket (bucket_start[key],
// advanced atomically once per run of equal keys: after this pass bucket_start[key] is the END of bucket key, i.e.
// the array read one element earlier is the start array again — see wpg_launch_bin).  The record carries
// weight * vis (R9, natural weighting), summed over the visibilities merged into it (compression).
// NPOL = 1: Rec<TT>;  NPOL = 2 | 4: vis[row][chan][pol], one RecP<NPOL> (fp32) / RecPD<NPOL> (fp64) record carries
// all correlations.
template <typename TT, int NPOL, bool QP2>
__global__ void __launch_bounds__(256, NPOL == 1 ? 4 : 3)
scatter_kernel(const float2 *__restrict__ vis, const double *__restrict__ uvw, const float *__restrict__ weight,
               const double *__restrict__ fscale, const __grid_constant__ PlaneTab T,
               const __grid_constant__ BinParams P, const Counters *__restrict__ ctr, unsigned *__restrict__ cursor,
               void *__restrict__ rec_out) {
    const VisIdx V = vis_indices(P);
    __shared__ uint2 s_tab[WPG_MAX_NW];
    __shared__ uint4 s_ck[WPG_MAX_CLS];
    unsigned key[kVpt], pos[kVpt], koff[kVpt], nrec[kVpt], dst[kVpt];
    bool head[kVpt], rhead[kVpt];
    float wt[kVpt];
    float2 v[kVpt];
    {
        RawVis raw[kVpt];
#pragma unroll
        for (int j = 0; j < kVpt; ++j) v[j] = NPOL == 1 && V.i[j] != 0xFFFFFFFFu ? __ldcs(vis + V.i[j]) : make_float2(0.f, 0.f);
        load_raw(V, uvw, weight, fscale, raw);
        wpg_stage_planetab(s_tab, T, P.Nw);
        wpg_stage_classkeys(s_ck, ctr, P);
        __syncthreads();
#pragma unroll
        for (int j = 0; j < kVpt; ++j) {
            key[j] = WPG_NO_KEY; pos[j] = koff[j] = 0; wt[j] = raw[j].wt;
            if (V.i[j] == 0xFFFFFFFFu || raw[j].wt == 0.0f) continue;
            const Located L = locate_vis<QP2>(raw[j], s_tab, s_ck, P);
            key[j] = L.key; pos[j] = L.pos; koff[j] = L.koff;
        }
    }
    // one returning atomic per run of equal keys (the slowest instruction of the pass: ~2 cycles per lane)
    key_runs(key, pos, koff, P.compress != 0, head, rhead, nrec);
    // The bucket cursors and the half-written sectors of the records are what this pass wants to find in L2 again
    // (the inputs stream through evict-first): both carry an evict-last hint.  Measured: binning -0.2 ms on config 4.
    unsigned long long pol;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
#pragma unroll
    for (int j = 0; j < kVpt; ++j) {
        dst[j] = 0u;
        if (head[j])
            asm volatile("atom.global.add.L2::cache_hint.u32 %0, [%1], %2, %3;" : "=r"(dst[j]) : "l"(cursor + key[j]), "r"(nrec[j]), "l"(pol) : "memory");
    }
#pragma unroll
    for (int j = 1; j < kVpt; ++j)
        if (key[j] != WPG_NO_KEY && !head[j]) dst[j] = dst[j - 1] + (rhead[j] ? 1u : 0u);
    if (NPOL == 1) {
        TT re[kVpt], im[kVpt];
#pragma unroll
        for (int j = 0; j < kVpt; ++j) { const TT w = (TT)wt[j]; re[j] = w * (TT)v[j].x; im[j] = w * (TT)v[j].y; }
#pragma unroll
        for (int j = kVpt - 1; j > 0; --j)
            if (key[j] != WPG_NO_KEY && !rhead[j]) { re[j - 1] += re[j]; im[j - 1] += im[j]; }
#pragma unroll
        for (int j = 0; j < kVpt; ++j)
            if (rhead[j]) store_rec(reinterpret_cast<Rec<TT> *>(rec_out) + dst[j], re[j], im[j], make_uint2(pos[j], koff[j]), pol);
    } else {
        // walk the thread's visibilities in order; a record is written when the next one starts a new record
        constexpr int NP = NPOL > 1 ? NPOL : 2;
        using RP = typename RecPOf<TT, NP>::type;
        RP out;
#pragma unroll
        for (int j = 0; j < kVpt; ++j) {
            if (key[j] == WPG_NO_KEY) continue;
            const float2 *src = vis + (size_t)V.i[j] * NP;
            const TT w = (TT)wt[j];
#pragma unroll
            for (int p = 0; p < NP; ++p) {
                const float2 q = __ldg(src + p);
                if (rhead[j]) { out.v[p].x = w * (TT)q.x; out.v[p].y = w * (TT)q.y; }
                else { out.v[p].x += w * (TT)q.x; out.v[p].y += w * (TT)q.y; }
            }
            out.pos = pos[j]; out.koff = koff[j];
            const bool last = j + 1 == kVpt || key[j + 1 < kVpt ? j + 1 : j] == WPG_NO_KEY || rhead[j + 1 < kVpt ? j + 1 : j];
            if (last) reinterpret_cast<RP *>(rec_out)[dst[j]] = out;
        }
    }
}

// Pass 4 (only where the sort key drops low bits of j0v: large grids, the sparse support classes of a ragged stack):
// inside a bucket the records stand in the order the atomics gave them, so the gridder's window would jump back and
// forth over the bucket's rows and write its sums out at every jump.  Every warp sorts chunks of 32 consecutive records
// of the class by the full window start (j0u, then j0v) — a bitonic network over the lanes on (key, source lane), then
// one gather of the records.
// Buckets are contiguous and ordered, so sorting a chunk by the full key restores the column-major sweep inside it
// (a bucket cut by a chunk boundary becomes two sorted runs).  W = 32-bit words per record (4: fp32, 6: fp64).
template <int W>
__global__ void __launch_bounds__(256)
chunk_sort_kernel(unsigned *__restrict__ rec, const unsigned *__restrict__ bucket_start, const Counters *__restrict__ ctr,
                  int cls, unsigned key_lo, unsigned key_hi, int uniform_shift) {
    unsigned shift = (unsigned)uniform_shift;
    if (uniform_shift < 0) { key_lo = ctr->key_base[cls]; key_hi = ctr->key_base[cls + 1]; shift = ctr->key_shift[cls]; }
    if (shift == 0) return;                                    // full resolution already
    const unsigned r0 = __ldg(bucket_start + key_lo), r1 = __ldg(bucket_start + key_hi);
    // dense classes (more than two records per window position on average) are left alone: their windows repeat,
    // a chunk of 32 records does not span a bucket, and the pass would cost more than the gridder gains
    if ((unsigned long long)(r1 - r0) > 2ull * ((unsigned long long)(key_hi - key_lo) << shift)) return;
    const unsigned lane = threadIdx.x & 31u;
    const unsigned nwarp = (gridDim.x * 256u) >> 5;
    for (unsigned c0 = r0 + 32u * ((blockIdx.x * 256u + threadIdx.x) >> 5); c0 < r1; c0 += 32u * nwarp) {
        const unsigned i = c0 + lane;
        const bool have = i < r1;
        unsigned v[W];
#pragma unroll
        for (int k = 0; k < W; k += 2) {
            const uint2 t = have ? *reinterpret_cast<const uint2 *>(rec + (size_t)i * W + k) : make_uint2(0u, 0u);
            v[k] = t.x; v[k + 1] = t.y;
        }
        const unsigned pos = v[W - 2];
        unsigned key = have ? ((pos << 16) | (pos >> 16)) : 0xFFFFFFFFu;       // j0u major, j0v minor; empty lanes last
        // already sorted (runs of equal windows, monotone sweeps): nothing to do
        const unsigned prev = __shfl_up_sync(0xffffffffu, key, 1);
        if (!__any_sync(0xffffffffu, lane > 0 && prev > key)) continue;
        // sort (key, source lane) pairs, then fetch the record of the source lane: two words per exchange instead of W
        unsigned src = lane;
#pragma unroll
        for (unsigned k = 2; k <= 32; k <<= 1) {
#pragma unroll
            for (unsigned j = k >> 1; j > 0; j >>= 1) {
                const unsigned pk = __shfl_xor_sync(0xffffffffu, key, j), ps = __shfl_xor_sync(0xffffffffu, src, j);
                const bool lower = (lane & j) == 0, asc = (lane & k) == 0;
                const bool take = (lower == asc) ? key > pk : key < pk;
                if (take) { key = pk; src = ps; }
            }
        }
#pragma unroll
        for (int q = 0; q < W; ++q) v[q] = __shfl_sync(0xffffffffu, v[q], src);
        if (have) {
#pragma unroll
            for (int k = 0; k < W; k += 2) *reinterpret_cast<uint2 *>(rec + (size_t)i * W + k) = make_uint2(v[k], v[k + 1]);
        }
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

// The binning passes (npol = 1: Rec<float | double> records; npol = 2 | 4: RecP<npol> / RecPD<npol> — positions do not
// depend on the correlation, so only the scatter differs).
static int launch_bin_passes(wpg_ctx *ctx, const void *d_vis, const double *d_uvw, const float *d_weight,
                             const double *d_freq, const PlaneTab &tab, const BinParams &bp,
                             const WorkspaceLayout &ws, wpg_prec prec, int npol, char *w) {
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
    dim3 nb((unsigned)((nvis + 256 * kVpt - 1) / (256 * kVpt)), 1, 1);
    if (bp.vis_block) {                // ceil(vis_block / 256) blocks per group of kVpt time steps
        const long long nd = (nvis + bp.vis_block - 1) / bp.vis_block;
        const long long ngr = (nd + kVpt - 1) / kVpt, ntile = (ngr + bp.vis_tile - 1) / bp.vis_tile;
        if (ntile > 65535 || (long long)bp.vis_nbx * bp.vis_tile >= (1ll << 31))
            return wpg_fail(ctx, WPG_EINVAL, "row_block = %u gives too many binning blocks", bp.vis_block / bp.nchan);
        nb = dim3(bp.vis_nbx * bp.vis_tile, (unsigned)ntile, 1);                    // (groups past the end find no visibility)
    }
    const bool any = nvis > 0;
    const bool qp2 = bp.qshift >= 0;
    chan_scale_kernel<<<(bp.nchan + 255) / 256, 256, 0, s>>>(d_freq, bp.nchan, fscale, bp, ctr);
    if (bp.dyn_keys) {
        census_kernel<<<ctx->sm_count * 4, 256, 0, s>>>(d_uvw, fscale, tab, bp, ctr);
        plan_keys_kernel<<<1, 32, 0, s>>>(ctr, bp.ncls, bp.N, ws.nkeys);
        ctx->n_launches += 2;
    }
    if (any) {
        if (qp2) bin_count_kernel<true><<<nb, 256, 0, s>>>(d_uvw, d_weight, fscale, tab, bp, ctr, hist);
        else bin_count_kernel<false><<<nb, 256, 0, s>>>(d_uvw, d_weight, fscale, tab, bp, ctr, hist);
    }
    scan_reduce_kernel<<<ws.nblocks_scan, 1024, 0, s>>>(hist, ws.nkeys, blocksum);
    scan_blocksums_kernel<<<1, 1024, 0, s>>>(blocksum, ws.nblocks_scan, ctr);
    scan_apply_kernel<<<ws.nblocks_scan, 1024, 0, s>>>(hist, ws.nkeys, blocksum);
    if (any) {
        const float2 *v = (const float2 *)d_vis;
        void *rec = w + ws.off_records;
#define WPG_SCATTER(TT, NP)                                                                                              \
        do {                                                                                                             \
            if (qp2) scatter_kernel<TT, NP, true><<<nb, 256, 0, s>>>(v, d_uvw, d_weight, fscale, tab, bp, ctr, hist, rec);  \
            else scatter_kernel<TT, NP, false><<<nb, 256, 0, s>>>(v, d_uvw, d_weight, fscale, tab, bp, ctr, hist, rec);     \
        } while (0)
        if (npol == 4 && prec == WPG_F32) WPG_SCATTER(float, 4);
        else if (npol == 4) WPG_SCATTER(double, 4);
        else if (npol == 2 && prec == WPG_F32) WPG_SCATTER(float, 2);
        else if (npol == 2) WPG_SCATTER(double, 2);
        else if (prec == WPG_F32) WPG_SCATTER(float, 1);
        else WPG_SCATTER(double, 1);
#undef WPG_SCATTER
        // fine order inside the buckets of keys that dropped bits of j0v (single-correlation records)
        if (npol == 1 && ctx->opt_chunk_sort && (bp.dyn_keys || bp.kshift > 0)) {
            unsigned *r32 = (unsigned *)rec;
            const unsigned *bs = (const unsigned *)(w + ws.off_hist);
            const int blocks = ctx->sm_count * 8;
            for (int cls = 0; cls < bp.ncls; ++cls) {
                const unsigned lo = (unsigned)cls * bp.keys_per_class, hi = (unsigned)(cls + 1) * bp.keys_per_class;
                const int ush = bp.dyn_keys ? -1 : bp.kshift;
                if (prec == WPG_F32) chunk_sort_kernel<4><<<blocks, 256, 0, s>>>(r32, bs, ctr, cls, lo, hi, ush);
                else chunk_sort_kernel<6><<<blocks, 256, 0, s>>>(r32, bs, ctr, cls, lo, hi, ush);
                ctx->n_launches += 1;
            }
        }
    }
    ctx->n_launches += any ? 6 : 4;
    WPG_CUDA(ctx, cudaGetLastError());
    return WPG_OK;
}

int wpg_launch_bin(wpg_ctx *ctx, const void *d_vis, const double *d_uvw, const float *d_weight,
                   const double *d_freq, const PlaneTab &tab, const BinParams &bp,
                   const WorkspaceLayout &ws, wpg_prec prec, char *w) {
    return launch_bin_passes(ctx, d_vis, d_uvw, d_weight, d_freq, tab, bp, ws, prec, 1, w);
}

int wpg_launch_bin_pol(wpg_ctx *ctx, const void *d_vis, const double *d_uvw, const float *d_weight, const double *d_freq,
                       const PlaneTab &tab, const BinParams &bp, const WorkspaceLayout &ws, wpg_prec prec, int npol, char *w) {
    return launch_bin_passes(ctx, d_vis, d_uvw, d_weight, d_freq, tab, bp, ws, prec, npol, w);
}
