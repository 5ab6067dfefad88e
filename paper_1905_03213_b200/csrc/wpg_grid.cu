// Step a2 — the gridder: grid[j0v+iv][j0u+iu] += (wt*vis) * K[p][ov][ou][iv][iu]  (O4 G5).
//
// Two kernels:
//  * grid_naive_kernel — one global reduction per update straight from the raw inputs (the design
//    whose ceiling is the atomic roofline; "write access to the global memory ... in an
//    atomic manner").  Independent of the binning pass, so it also cross-checks it.
//  * grid_runs_kernel — the paper's register accumulator (one thread per support
//    cell; contributions "accumulated and buffered in a register" while consecutive samples hit the
//    same grid point, "written into the global memory when the processing moves on"), fed with the
//    position-sorted records of wpg_bin.cu instead of per-baseline time series.  A warp walks a
//    fixed-length segment of the sorted records; lane-slot <-> support-cell residue (b, a): the one
//    cell of the S x S window whose grid coordinates are congruent to (b, a) modulo S.  While the
//    window start does not change the cell and the coefficient offset of every lane stay put, so a
//    run of visibilities costs one coefficient load and two packed FMAs per update; when the window
//    moves, only the lanes whose cell changed flush (red.global.add.v2.f32 / .f64).
//    Coefficients are read through L1 from the L2-resident stack, one record ahead of their use.
#include <type_traits>

#include "wpg_common.h"

namespace {

template <typename T> struct Cplx;
template <> struct Cplx<float> { using type = float2; };
template <> struct Cplx<double> { using type = double2; };

__device__ __forceinline__ void red_add(float2 *addr, float2 v) {
    asm volatile("red.global.add.v2.f32 [%0], {%1, %2};" ::"l"(addr), "f"(v.x), "f"(v.y) : "memory");
}
__device__ __forceinline__ void red_add(double2 *addr, double2 v) {
    asm volatile("red.global.add.f64 [%0], %1;" ::"l"(&addr->x), "d"(v.x) : "memory");
    asm volatile("red.global.add.f64 [%0], %1;" ::"l"(&addr->y), "d"(v.y) : "memory");
}

// acc += (re + i im) * c
__device__ __forceinline__ void cmac(float2 &acc, float re, float im, float2 c) {
    // two packed FMAs (FFMA2): (acc.x, acc.y) += c.x * (re, im);  += c.y * (-im, re)
    unsigned long long A, V1, V2, CX, CY;
    asm("mov.b64 %0, {%1, %2};" : "=l"(A) : "f"(acc.x), "f"(acc.y));
    asm("mov.b64 %0, {%1, %2};" : "=l"(V1) : "f"(re), "f"(im));
    asm("mov.b64 %0, {%1, %2};" : "=l"(V2) : "f"(-im), "f"(re));
    asm("mov.b64 %0, {%1, %1};" : "=l"(CX) : "f"(c.x));
    asm("mov.b64 %0, {%1, %1};" : "=l"(CY) : "f"(c.y));
    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(A) : "l"(V1), "l"(CX));
    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(A) : "l"(V2), "l"(CY));
    asm("mov.b64 {%0, %1}, %2;" : "=f"(acc.x), "=f"(acc.y) : "l"(A));
}
__device__ __forceinline__ void cmac(double2 &acc, double re, double im, double2 c) {
    acc.x = fma(re, c.x, acc.x); acc.x = fma(-im, c.y, acc.x);
    acc.y = fma(re, c.y, acc.y); acc.y = fma(im, c.x, acc.y);
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
        const ParamPlaneTab PT{Tb};
        VisPos r = wpg_locate(uvw[3 * row], uvw[3 * row + 1], uvw[3 * row + 2], f, P, PT);
        if (!r.inside) { c_oob++; continue; }
        c_grid++; c_clamp += r.clamped; c_upd += r.S * r.S;
        float2 v = vis[i];
        T re = (T)wt * (T)v.x, im = (T)wt * (T)v.y;
        const C *Ks = K + wpg_koff(r, P, PT);
        int S = r.S, S2 = S * S;
        for (int c = lane; c < S2; c += 32) {
            int iv = c / S, iu = c - iv * S;
            C k = Ks[c];
            C p;
            p.x = re * k.x - im * k.y; p.y = re * k.y + im * k.x;
            red_add(grid + (long long)(r.j0v + iv) * P.N + (r.j0u + iu), p);
        }
    }
    if (lane == 0) {
        if (c_grid) atomicAdd(&ctr->n_gridded[blockIdx.x % kStatSlots], c_grid);
        if (c_oob) atomicAdd(&ctr->n_skipped_oob[blockIdx.x % kStatSlots], c_oob);
        if (c_zero) atomicAdd(&ctr->n_skipped_zero_weight[blockIdx.x % kStatSlots], c_zero);
        if (c_clamp) atomicAdd(&ctr->n_clamped_w[blockIdx.x % kStatSlots], c_clamp);
        if (c_upd) atomicAdd(&ctr->n_updates[blockIdx.x % kStatSlots], c_upd);
    }
}

// ------------------------------------------------------------------------------------ runs
// Per-warp ring of sorted records in shared memory, filled with cp.async (LDGSTS) two chunks ahead
// of their use; a record is then one broadcast LDS away from every lane.
constexpr int kRunThreads = 256;
constexpr int kChunk = 16;                       // records per chunk
constexpr int kRing = 4;                         // chunks in the ring
constexpr unsigned kRingMask = kChunk * kRing - 1;

__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// Copy chunk c of the item [i0, i1) into its ring slot (only the records that exist).
__device__ __forceinline__ void ring_fill(Rec<float> *ring, const Rec<float> *rec, unsigned i0, unsigned i1, unsigned c, int lane) {
    const unsigned i = i0 + c * kChunk + lane;
    if (lane < kChunk && i < i1)
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(ring + ((c * kChunk + lane) & kRingMask))), "l"(rec + i) : "memory");
}
__device__ __forceinline__ void ring_fill(Rec<double> *ring, const Rec<double> *rec, unsigned i0, unsigned i1, unsigned c, int lane) {
    // 24-byte records are 8-byte aligned only: three 8-byte pieces per record
    const unsigned long long *g = reinterpret_cast<const unsigned long long *>(rec + i0 + c * kChunk);
    unsigned long long *sm = reinterpret_cast<unsigned long long *>(ring + ((c * kChunk) & kRingMask));
    const unsigned first = i0 + c * kChunk;
    const unsigned npiece = first < i1 ? 3u * min((unsigned)kChunk, i1 - first) : 0u;
    for (unsigned q = lane; q < npiece; q += 32)
        asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(smem_u32(sm + q)), "l"(g + q) : "memory");
}
__device__ __forceinline__ void ring_get(const Rec<float> *ring, unsigned slot, float &re, float &im, unsigned &pos, unsigned &koff) {
    const uint4 q = *reinterpret_cast<const uint4 *>(ring + slot);
    re = __uint_as_float(q.x); im = __uint_as_float(q.y); pos = q.z; koff = q.w;
}
__device__ __forceinline__ void ring_get(const Rec<double> *ring, unsigned slot, double &re, double &im, unsigned &pos, unsigned &koff) {
    re = ring[slot].re; im = ring[slot].im;
    const uint2 t = *reinterpret_cast<const uint2 *>(&ring[slot].pos);
    pos = t.x; koff = t.y;
}

// SCT: compile-time support (a power of two) or 0 = S_rt.  NSLOT >= ceil(S^2 / 32).
template <typename T, int SCT, int NSLOT, int MINB>
__global__ void __launch_bounds__(kRunThreads, MINB)
grid_runs_kernel(const Rec<T> *__restrict__ rec, const unsigned *__restrict__ bucket_start,
                 const unsigned *__restrict__ key_base, int cls, unsigned key_lo, unsigned key_hi, int S_rt, unsigned *__restrict__ cursor,
                 const typename Cplx<T>::type *__restrict__ K, typename Cplx<T>::type *__restrict__ grid,
                 int N, unsigned seg) {
    using C = typename Cplx<T>::type;
    constexpr bool PIPE = NSLOT <= 8;          // coefficients of record i+1 are requested before record i is added
    constexpr bool FULL = SCT * SCT == NSLOT * 32;   // every lane-slot owns a cell
    const int S = SCT ? SCT : S_rt;
    const int S2 = S * S;
    const int lane = threadIdx.x & 31;
    // key range of this support class: from the device table (ragged stacks) or by value (key_base == nullptr)
    if (key_base) { key_lo = __ldg(key_base + cls); key_hi = __ldg(key_base + cls + 1); }
    const unsigned r_begin = __ldg(bucket_start + key_lo), r_end = __ldg(bucket_start + key_hi);
    const unsigned nitems = (r_end - r_begin + seg - 1) / seg;

    __shared__ __align__(16) Rec<T> ring_all[kRunThreads / 32][kChunk * kRing];
    Rec<T> *ring = ring_all[threadIdx.x >> 5];

    int ra[NSLOT], rb[NSLOT];                  // this lane-slot's residue (b, a); rb = -1: idle slot
#pragma unroll
    for (int k = 0; k < NSLOT; ++k) {
        int r = k * 32 + lane;
        rb[k] = r < S2 ? r / S : -1;
        ra[k] = r < S2 ? r - rb[k] * S : 0;
    }

    for (;;) {
        unsigned item = 0;
        if (lane == 0) item = atomicAdd(cursor, 1u);
        item = __shfl_sync(0xffffffffu, item, 0);
        if (item >= nitems) break;
        const unsigned i0 = r_begin + item * seg, i1 = min(i0 + seg, r_end);

        __syncwarp();                          // the previous item's ring reads are done
#pragma unroll
        for (unsigned c = 0; c < 3; ++c) { ring_fill(ring, rec, i0, i1, c, lane); cp_async_commit(); }

        C acc[NSLOT];
        unsigned cell[NSLOT], coff[NSLOT];
#pragma unroll
        for (int k = 0; k < NSLOT; ++k) { acc[k].x = acc[k].y = (T)0; cell[k] = 0; coff[k] = 0; }
        unsigned pos_cur = 0;

        // the window moves to `pos`: lane-slots whose cell changes write their sum out (FLUSH) and
        // every lane-slot gets the offset of its cell inside the S x S coefficient slice
        auto place = [&](unsigned pos, auto flush_tag) {
            constexpr bool FLUSH = decltype(flush_tag)::value;
            const int j0u = (int)(pos & 0xFFFFu), j0v = (int)(pos >> 16);
            const int ju = SCT ? (j0u & (S - 1)) : j0u % S, jv = SCT ? (j0v & (S - 1)) : j0v % S;
#pragma unroll
            for (int k = 0; k < NSLOT; ++k) {
                int iu = ra[k] - ju; iu += iu < 0 ? S : 0;
                int iv = rb[k] - jv; iv += iv < 0 ? S : 0;
                coff[k] = (unsigned)(iv * S + iu);
                const unsigned nc = (unsigned)((j0v + iv) * N + j0u + iu);
                if (FLUSH) {
                    if ((FULL || rb[k] >= 0) && nc != cell[k]) {
                        red_add(grid + cell[k], acc[k]);
                        acc[k].x = acc[k].y = (T)0;
                    }
                }
                cell[k] = nc;
            }
            pos_cur = pos;
        };
        auto fetch = [&](C(&c)[NSLOT], unsigned koff, bool pred) {
#pragma unroll
            for (int k = 0; k < NSLOT; ++k)
                if (pred && (FULL || rb[k] >= 0)) c[k] = __ldg(K + (koff + coff[k]));     // 32-bit index, one widening multiply-add
        };
        auto add = [&](T re, T im, const C(&c)[NSLOT]) {
#pragma unroll
            for (int k = 0; k < NSLOT; ++k)
                if (FULL || rb[k] >= 0) cmac(acc[k], re, im, c[k]);
        };
        // entering chunk c: request chunk c + 3 (its slot held chunk c - 1), make chunks <= c + 1 visible
        auto enter_chunk = [&](unsigned c) {
            __syncwarp();
            ring_fill(ring, rec, i0, i1, c + 3, lane);
            cp_async_commit();
            cp_async_wait<2>();
            __syncwarp();
        };

        T reA, imA, reB, imB; unsigned posA, koffA, posB, koffB;
        C cA[NSLOT], cB[PIPE ? NSLOT : 1];
        enter_chunk(0);
        ring_get(ring, 0, reA, imA, posA, koffA);
        place(posA, std::false_type());
        if (PIPE) fetch(cA, koffA, true);

        // one record: `cur` is added, `nxt` is looked at (and its coefficients requested) first.
        // Returns false after the last record of the item.
        auto half = [&](unsigned i, T re, T im, unsigned koff, C(&cc)[NSLOT], T &nre, T &nim, unsigned &npos,
                        unsigned &nkoff, C(&cn)[PIPE ? NSLOT : 1]) -> bool {
            const bool has_next = i + 1 < i1;
            ring_get(ring, (i + 1 - i0) & kRingMask, nre, nim, npos, nkoff);
            const bool same = has_next && npos == pos_cur;
            if (PIPE) {
                fetch(reinterpret_cast<C(&)[NSLOT]>(cn), nkoff, same);
            } else {
                fetch(cc, koff, true);
            }
            add(re, im, cc);
            if (!has_next) return false;
            if (!same) {
                place(npos, std::true_type());
                if (PIPE) fetch(reinterpret_cast<C(&)[NSLOT]>(cn), nkoff, true);
            }
            return true;
        };

        for (unsigned i = i0;; i += 2) {
            if (i != i0 && ((i - i0) & (kChunk - 1)) == 0) enter_chunk((i - i0) / kChunk);
            if (PIPE) {
                if (!half(i, reA, imA, koffA, cA, reB, imB, posB, koffB, cB)) break;
                if (!half(i + 1, reB, imB, koffB, reinterpret_cast<C(&)[NSLOT]>(cB), reA, imA, posA, koffA,
                          reinterpret_cast<C(&)[PIPE ? NSLOT : 1]>(cA))) break;
            } else {
                if (!half(i, reA, imA, koffA, cA, reB, imB, posB, koffB, cB)) break;
                if (!half(i + 1, reB, imB, koffB, cA, reA, imA, posA, koffA, cB)) break;
            }
        }
#pragma unroll
        for (int k = 0; k < NSLOT; ++k)
            if (FULL || rb[k] >= 0) red_add(grid + cell[k], acc[k]);
        cp_async_wait<0>();
    }
}

// ------------------------------------------------------------------------------------ pairs
// fp32, even support.  A lane-slot owns a PAIR of horizontally adjacent cells: the cells of the window
// whose row is congruent to rb and whose columns are congruent to (ra2 + par, ra2 + par + 1) modulo S,
// par = parity of the window start j0u (the records come sorted by (column j0u, row j0v), so within a
// sweep down the v axis the ownership never changes, and the cells a window leaves behind are whole
// row segments: one contiguous 16-byte reduction per lane, 8 S bytes per row).  The two coefficients of a pair are adjacent and 16-byte aligned
// in K[p][ov][ou][iv][:], so one LDG.128 feeds two updates.
//
// v*c = (re, im)*c.x + (-im, re)*c.y: two packed FMAs per update; (re, im) and (-im, re) are formed once per
// record and the coefficient components enter as broadcast scalars, so the accumulators are the cell
// sums themselves and a pair is written out as one 16-byte reduction.
//
// The coefficient loads run DEPTH records ahead of their use in a register ring (statically indexed,
// the record loop is unrolled by DEPTH): the slice of a record is picked at random from a stack that
// is several times the L1, so most loads are L2 hits (~300 cycles).  The look-ahead is "stateless":
// the lane's offset inside the slice, (iv, iu0), is computed from the record's window start alone.
__device__ __forceinline__ unsigned long long pack2(float lo, float hi) {
    unsigned long long r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void fma2(unsigned long long &acc, unsigned long long a, unsigned long long b) {
    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(acc) : "l"(a), "l"(b));
}
__device__ __forceinline__ float2 unpack2(unsigned long long v) {
    float2 r;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(r.x), "=f"(r.y) : "l"(v));
    return r;
}
__device__ __forceinline__ void ldg128(const float2 *p, unsigned long long &c0, unsigned long long &c1) {
    asm volatile("ld.global.nc.v2.b64 {%0, %1}, [%2];" : "=l"(c0), "=l"(c1) : "l"(p));
}

// G > 1: the warp is split into G groups of 32/G lanes and every group takes its own record, G records per step
// (group g walks the g-th contiguous part of the item); a group's NSLOT * 32/G lane-slots hold the S*S/2 pairs of
// its window.  For
// S = 4 (8 pairs) this fills the warp; for S = 8 (two half-warps, two pairs per lane) it halves the per-record
// share of everything that is not a coefficient load or an FMA — record fetch, window test, loop control.
// RPS > 0: a slot holds RPS whole window rows (RPS * S/2 <= 32 lanes, the rest idle) instead of 32 consecutive
// pairs: for S = 12 four rows are 384 bytes = three whole 128-byte lines of the slice, where 32 consecutive pairs
// (5 1/3 rows) straddle five, and the coefficient loads are bound by the lines they touch.
// ST: the producer keeps the lane-slots' offsets of the current window and re-derives them only when the window
// start changes (supports that are not a power of two pay ~25 instructions per slot for the modulo arithmetic;
// for powers of two the two-instruction stateless form is cheaper than the test).
// WS > 1: the window is split over WS work items (each takes all records of its segment but only NSLOT of the
// WS * NSLOT lane-slot sets): a 16 x 16 window as two items of two slots needs half the registers of one item of
// four, so twice as many warps are resident.
template <int SCT, int NSLOT, int DEPTH, int MINB, int G = 1, int RPS = 0, bool ST = false, int WS = 1>
__global__ void __launch_bounds__(kRunThreads, MINB)
grid_pairs_kernel(const Rec<float> *__restrict__ rec, const unsigned *__restrict__ bucket_start,
                  const unsigned *__restrict__ key_base, int cls, unsigned key_lo, unsigned key_hi, int S_rt, unsigned magicS, unsigned *__restrict__ cursor,
                  const float2 *__restrict__ K, float2 *__restrict__ grid, int N, unsigned seg) {
    static_assert((kChunk / G) % DEPTH == 0, "a look-ahead step divides a group's share of a chunk");
    constexpr unsigned CL = kChunk / G;                  // records of one group in a chunk of the ring
    static_assert(G == 1 || RPS == 0, "lane groups use the packed pair -> lane-slot mapping");
    static_assert(!ST || G == 1, "window tracking in the producer needs one window per warp");
    constexpr int LPG = 32 / G;                          // lanes per group
    using U64 = unsigned long long;
    const int S = SCT ? SCT : S_rt;
    const int H = S >> 1;                                // pairs per window row
    const int NP = S * H;                                // pairs per window
    const int lane = threadIdx.x & 31;
    const int grp = G > 1 ? lane / LPG : 0;              // this lane's group: takes the grp-th contiguous part of an item
    // key range of this support class: from the device table (ragged stacks) or by value (key_base == nullptr)
    if (key_base) { key_lo = __ldg(key_base + cls); key_hi = __ldg(key_base + cls + 1); }
    const unsigned r_begin = __ldg(bucket_start + key_lo), r_end = __ldg(bucket_start + key_hi);
    const unsigned nitems = WS * ((r_end - r_begin + seg - 1) / seg);

    __shared__ __align__(16) Rec<float> ring_all[kRunThreads / 32][kChunk * kRing];
    Rec<float> *ring = ring_all[threadIdx.x >> 5];

    // lane-slot constants.  Power-of-two S: RG packs (ra2 + 1, rb) with a guard bit so that
    // (RG - pos) & M is (iu0 | iv << 16) in two instructions: iu0 = (ra2 + par - j0u) mod S equals
    // ((ra2 + 1 - j0u) mod S) & ~1 because S and ra2 are even.
    static_assert(WS == 1 || (G == 1 && RPS == 0), "window splitting only for the plain one-group mapping");
    unsigned RG[NSLOT];
    int ra2p1[NSLOT], rb[NSLOT];
    bool act[NSLOT];
    auto set_slots = [&](int part) {                     // part: which NSLOT of the WS * NSLOT slot sets (0 if WS = 1)
#pragma unroll
    for (int k = 0; k < NSLOT; ++k) {
        int r = (part * NSLOT + k) * LPG + lane % LPG;   // (G = 1: slot * 32 + lane)
        act[k] = r < NP;
        if (RPS) {                                       // RPS rows per slot
            const int row = k * RPS + lane / H;
            act[k] = lane < RPS * H && row < S;
            r = row * H + lane % H;
        }
        r = act[k] ? r : 0;
        rb[k] = r / H;
        ra2p1[k] = 2 * (r - rb[k] * H) + 1;
        RG[k] = (0x8000u + (unsigned)ra2p1[k]) | ((0x8000u + (unsigned)rb[k]) << 16);
    }
    };
    set_slots(0);
    constexpr bool POW2 = SCT > 0 && (SCT & (SCT - 1)) == 0;       // compile-time S that is not a power of two: generic formula, constant folded
    constexpr unsigned M = POW2 ? ((unsigned)(SCT - 2) | ((unsigned)(SCT - 1) << 16)) : 0u;

    // (iu0 | iv << 16) of this lane-slot for a window starting at pos = j0u | j0v << 16
    auto offset_in_window = [&](unsigned pos, int k) -> unsigned {
        if (POW2) return (RG[k] - pos) & M;
        const unsigned j0u = pos & 0xFFFFu, j0v = pos >> 16;
        const unsigned mg = SCT ? (1u << 20) / (unsigned)(SCT ? SCT : 1) + 1u : magicS;
        const int ju = (int)(j0u - ((j0u * mg) >> 20) * (unsigned)S);     // j0u mod S
        const int jv = (int)(j0v - ((j0v * mg) >> 20) * (unsigned)S);
        int x = ra2p1[k] - ju; x += x < 0 ? S : 0;
        int y = rb[k] - jv;    y += y < 0 ? S : 0;
        return (unsigned)(x & ~1) | ((unsigned)y << 16);
    };

    U64 zero64;
    asm volatile("mov.b64 %0, 0;" : "=l"(zero64));      // volatile: stays a register, not re-materialised at each use

    for (;;) {
        unsigned item = 0;
        if (lane == 0) item = atomicAdd(cursor, 1u);
        item = __shfl_sync(0xffffffffu, item, 0);
        if (item >= nitems) break;
        if (WS > 1) { set_slots((int)(item % WS)); item /= WS; }
        const unsigned i0 = r_begin + item * seg, i1 = min(i0 + seg, r_end);
        const unsigned cnt = i1 - i0;

        // group g walks records [g * glen, g * glen + cnt_g) of the item (contiguous parts, so that a run of equal
        // windows stays with one group); chunk c of the ring holds local records [c * CL, (c + 1) * CL) of every group
        const unsigned glen = G == 1 ? cnt : (cnt + G - 1) / G;
        auto part_len = [&](unsigned g) { return G == 1 ? cnt : (g * glen < cnt ? min(glen, cnt - g * glen) : 0u); };
        const unsigned my_cnt = part_len((unsigned)grp), min_cnt = part_len(G - 1);
        auto fill = [&](unsigned c) {
            if (G == 1) { ring_fill(ring, rec, i0, i1, c, lane); return; }
            const unsigned g = (unsigned)lane / CL, t = c * CL + (unsigned)lane % CL;
            if (lane < kChunk && t < part_len(g))
                asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(ring + ((c * kChunk + lane) & kRingMask))),
                             "l"(rec + (i0 + g * glen + t)) : "memory");
        };
        auto slot_of = [&](unsigned t) {
            return G == 1 ? ring + (t & kRingMask) : ring + (((t / CL) * kChunk + (unsigned)grp * CL + t % CL) & kRingMask);
        };

        __syncwarp();                          // the previous item's ring reads are done
#pragma unroll
        for (unsigned c = 0; c < 2; ++c) { fill(c); cp_async_commit(); }

        constexpr unsigned kNoCell = 0xFFFFFFFFu;
        U64 acc0[NSLOT], acc1[NSLOT];                       // (re, im) sums of the pair's two cells
        unsigned qcur[NSLOT] = {};                          // (column | row << 16) of the pair's first cell
#pragma unroll
        for (int k = 0; k < NSLOT; ++k) { acc0[k] = acc1[k] = 0ull; qcur[k] = kNoCell; }

        // look-ahead ring (registers): coefficients, visibility and the lane-slot's cell of the DEPTH
        // records in flight
        U64 c0[DEPTH][NSLOT], c1[DEPTH][NSLOT];
        U64 vis[DEPTH];
        unsigned qn[DEPTH][NSLOT];

        // Write the pair out and clear its sums.  One asm statement with the accumulators as read-write
        // operands: the cleared value then lives in the SAME register as the sum (a separate "acc = 0"
        // makes the compiler keep two copies alive and pay moves for it on every record).
        unsigned posP = 0xFFFFFFFFu, dP[NSLOT], cP[NSLOT];  // ST: window of the last record produced, offsets in it
#pragma unroll
        for (int k = 0; k < NSLOT; ++k) dP[k] = cP[k] = 0;
        auto flush = [&](int k) {
            const unsigned q = qcur[k];
            float2 *g = grid + ((q >> 16) * (unsigned)N + (q & 0xFFFFu));
            // (two 8-byte reductions rather than one 16-byte red.v4: the latter wants both sums in one aligned
            // register quad, which costs register moves on every record)
            // (the zero comes from a register: an immediate 64-bit zero costs four instructions per sum)
            asm volatile("{ .reg .f32 a, b, c, d;\n\t"
                         "mov.b64 {a, b}, %0; mov.b64 {c, d}, %1;\n\t"
                         "red.global.add.v2.f32 [%2], {a, b};\n\t"
                         "red.global.add.v2.f32 [%2 + 8], {c, d};\n\t"
                         "mov.b64 %0, %3; mov.b64 %1, %3; }"
                         : "+l"(acc0[k]), "+l"(acc1[k]) : "l"(g), "l"(zero64) : "memory");
        };
        // stage s <- record rp[0]: coefficient loads; the lane's offset inside the slice changes only
        // with the window (warp-uniform branch, taken once per run of equal window starts)
        // `valid` (per lane, only ever false for G > 1 at the ragged end of an item): a lane without a record
        // loads coefficient 0 of the stack, adds 0 * c and reports "no cell" (which writes its sums out early)
        auto produce = [&](int s, const Rec<float> *rp, bool valid) {
            // two 8-byte reads: (re, im) stays in its register pair until the record is consumed,
            // (pos, koff) is used up at once
            vis[s] = valid ? *reinterpret_cast<const U64 *>(rp) : 0ull;
            const uint2 pk = valid ? *reinterpret_cast<const uint2 *>(&rp->pos) : make_uint2(0u, 0u);
            const unsigned pos = pk.x, koff = pk.y;
            if (ST) {
                if (__any_sync(0xffffffffu, pos != posP)) {
#pragma unroll
                    for (int k = 0; k < NSLOT; ++k) {
                        dP[k] = offset_in_window(pos, k);
                        cP[k] = act[k] ? (dP[k] >> 16) * (unsigned)S + (dP[k] & 0xFFFFu) : 0u;
                    }
                    posP = pos;
                }
#pragma unroll
                for (int k = 0; k < NSLOT; ++k) {
                    qn[s][k] = act[k] && valid ? pos + dP[k] : kNoCell;
                    ldg128(K + (koff + cP[k]), c0[s][k], c1[s][k]);
                }
            } else {
#pragma unroll
                for (int k = 0; k < NSLOT; ++k) {
                    const unsigned d = offset_in_window(pos, k);
                    qn[s][k] = act[k] && valid ? pos + d : kNoCell;
                    const unsigned coff = (d >> 16) * (unsigned)S + (d & 0xFFFFu);
                    ldg128(K + (koff + (act[k] ? coff : 0u)), c0[s][k], c1[s][k]);
                }
            }
        };
        auto consume = [&](int s) {
            bool any = false;
#pragma unroll
            for (int k = 0; k < NSLOT; ++k) any |= qn[s][k] != qcur[k];
            if (__any_sync(0xffffffffu, any)) {      // the window moved: lane-slots whose cells changed write out
#pragma unroll
                for (int k = 0; k < NSLOT; ++k) {
                    if (qn[s][k] != qcur[k]) {
                        if (qcur[k] != kNoCell) flush(k);      // (the sums are zero before the first window)
                        asm volatile("mov.b32 %0, %1;" : "+r"(qcur[k]) : "r"(qn[s][k]));    // tied: no second copy of qcur
                    }
                }
            }
            // acc += v * c = (re, im) * c.x + (-im, re) * c.y: the visibility pairs are formed once per record,
            // the coefficient components enter as broadcast scalars
            const float2 vv = unpack2(vis[s]);
            const U64 v1 = vis[s], v2 = pack2(-vv.y, vv.x);
#pragma unroll
            for (int k = 0; k < NSLOT; ++k) {
                const float2 k0 = unpack2(c0[s][k]), k1 = unpack2(c1[s][k]);
                fma2(acc0[k], v1, pack2(k0.x, k0.x)); fma2(acc0[k], v2, pack2(k0.y, k0.y));
                fma2(acc1[k], v1, pack2(k1.x, k1.x)); fma2(acc1[k], v2, pack2(k1.y, k1.y));
            }
        };
        // entering chunk c of the PRODUCER: request chunk c + 2 (its slot held chunk c - 2; the consumer, DEPTH
        // records behind, may still re-read window starts of chunk c - 1), make chunks <= c visible
        auto enter_chunk = [&](unsigned c) {
            __syncwarp();
            fill(c + 2);
            cp_async_commit();
            cp_async_wait<2>();
            __syncwarp();
        };

        // prologue: local records 0 .. DEPTH-1 of every group into the look-ahead ring
        enter_chunk(0);
#pragma unroll
        for (int s = 0; s < DEPTH; ++s)
            if ((unsigned)s < glen) produce(s, slot_of((unsigned)s), (unsigned)s < my_cnt);

        for (unsigned t = 0; t < glen; t += DEPTH) {
            // the producer is at local records t + DEPTH .. t + 2 DEPTH - 1: all in one chunk (DEPTH divides CL)
            const unsigned tp = t + DEPTH;
            if (tp % CL == 0 && tp < glen) enter_chunk(tp / CL);
            const Rec<float> *rp = slot_of(tp);
            if (tp + DEPTH <= min_cnt) {             // every group has all of them
#pragma unroll
                for (int s = 0; s < DEPTH; ++s) { consume(s); produce(s, rp + s, true); }
            } else {
#pragma unroll
                for (int s = 0; s < DEPTH; ++s) {
                    if (t + s < glen) consume(s);
                    if (tp + s < glen) produce(s, rp + s, tp + s < my_cnt);
                }
            }
        }
#pragma unroll
        for (int k = 0; k < NSLOT; ++k)
            if (act[k] && qcur[k] != kNoCell) flush(k);
        cp_async_wait<0>();
    }
}

template <int SCT, int NSLOT, int DEPTH, int MINB, int G = 1, int RPS = 0, bool ST = false, int WS = 1>
int launch_pairs(wpg_ctx *ctx, cudaStream_t strm, const BinParams &bp, const WorkspaceLayout &ws, const void *K, void *grid, char *w,
                 int cls, int S) {
    int per_sm = ctx->opt_ctas_per_sm ? ctx->opt_ctas_per_sm : MINB;
    int blocks = ctx->sm_count * per_sm;
    unsigned seg = ctx->opt_segment ? (unsigned)ctx->opt_segment : 256u;
    Counters *ctr = (Counters *)(w + ws.off_counters);
    unsigned magicS = (1u << 20) / (unsigned)S + 1u;         // (x * magicS) >> 20 == x / S for x < 2^13, S <= 32
    grid_pairs_kernel<SCT, NSLOT, DEPTH, MINB, G, RPS, ST, WS><<<blocks, kRunThreads, 0, strm>>>(
        (const Rec<float> *)(w + ws.off_records), (const unsigned *)(w + ws.off_hist),
        bp.dyn_keys ? ctr->key_base : nullptr, cls, (unsigned)cls * bp.keys_per_class, (unsigned)(cls + 1) * bp.keys_per_class, S, magicS, &ctr->cursor[cls],
        (const float2 *)K, (float2 *)grid, bp.N, seg);
    ctx->n_launches += 1;
    WPG_CUDA(ctx, cudaGetLastError());
    return WPG_OK;
}

// ------------------------------------------------------------------------------------ pairs, NPOL correlations
// SURVEY.md §8(f) item 4 (data are row x channel x polarisation): the NPOL correlations of a
// (row, channel) share window and coefficient slice, so one LDG.128 feeds 2 * NPOL updates — the one change that
// lifts the L1 coefficient-feed bound of the single-correlation gridder.  Same structure as grid_pairs_kernel
// (power-of-two S, one record per warp step); grid[pol][N][N].
template <int NPOL>
__device__ __forceinline__ void ring_fill_pol(RecP<NPOL> *ring, const RecP<NPOL> *rec, unsigned i0, unsigned i1, unsigned c, int lane) {
    constexpr unsigned PIECES = sizeof(RecP<NPOL>) / 8;           // 8-byte pieces per record
    const unsigned long long *g = reinterpret_cast<const unsigned long long *>(rec + i0 + c * kChunk);
    unsigned long long *sm = reinterpret_cast<unsigned long long *>(ring + ((c * kChunk) & kRingMask));
    const unsigned first = i0 + c * kChunk;
    const unsigned npiece = first < i1 ? PIECES * min((unsigned)kChunk, i1 - first) : 0u;
    for (unsigned q = lane; q < npiece; q += 32)
        asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(smem_u32(sm + q)), "l"(g + q) : "memory");
}

template <int SCT, int NSLOT, int DEPTH, int MINB, int NPOL, int WS = 1>
__global__ void __launch_bounds__(kRunThreads, MINB)
grid_pairs_pol_kernel(const RecP<NPOL> *__restrict__ rec, const unsigned *__restrict__ bucket_start, unsigned key_lo,
                      unsigned key_hi, unsigned *__restrict__ cursor, const float2 *__restrict__ K,
                      float2 *__restrict__ grid, int N, unsigned seg) {
    static_assert(kChunk % DEPTH == 0 && SCT > 0 && (SCT & (SCT - 1)) == 0 && SCT * SCT / 2 == WS * NSLOT * 32, "power-of-two support, full warps");
    using U64 = unsigned long long;
    constexpr int S = SCT, H = S >> 1;
    const int lane = threadIdx.x & 31;
    const unsigned r_begin = __ldg(bucket_start + key_lo), r_end = __ldg(bucket_start + key_hi);
    const unsigned nitems = WS * ((r_end - r_begin + seg - 1) / seg);   // WS > 1: the window split over WS work items
    const size_t plane = (size_t)N * N;

    __shared__ __align__(16) RecP<NPOL> ring_all[kRunThreads / 32][kChunk * kRing];
    RecP<NPOL> *ring = ring_all[threadIdx.x >> 5];

    unsigned RG[NSLOT];
    auto set_slots = [&](int part) {
#pragma unroll
        for (int k = 0; k < NSLOT; ++k) {
            const int r = (part * NSLOT + k) * 32 + lane, rb = r / H, ra2p1 = 2 * (r - rb * H) + 1;
            RG[k] = (0x8000u + (unsigned)ra2p1) | ((0x8000u + (unsigned)rb) << 16);
        }
    };
    set_slots(0);
    constexpr unsigned M = (unsigned)(S - 2) | ((unsigned)(S - 1) << 16);

    for (;;) {
        unsigned item = 0;
        if (lane == 0) item = atomicAdd(cursor, 1u);
        item = __shfl_sync(0xffffffffu, item, 0);
        if (item >= nitems) break;
        if (WS > 1) { set_slots((int)(item % WS)); item /= WS; }
        const unsigned i0 = r_begin + item * seg, i1 = min(i0 + seg, r_end);
        const unsigned cnt = i1 - i0;

        __syncwarp();
#pragma unroll
        for (unsigned c = 0; c < 2; ++c) { ring_fill_pol<NPOL>(ring, rec, i0, i1, c, lane); cp_async_commit(); }

        U64 acc0[NSLOT][NPOL], acc1[NSLOT][NPOL];
        unsigned qcur[NSLOT] = {};
#pragma unroll
        for (int k = 0; k < NSLOT; ++k) {
            qcur[k] = 0xFFFFFFFFu;
#pragma unroll
            for (int p = 0; p < NPOL; ++p) acc0[k][p] = acc1[k][p] = 0ull;
        }
        U64 c0[DEPTH][NSLOT], c1[DEPTH][NSLOT], vis[DEPTH][NPOL];
        unsigned qn[DEPTH][NSLOT];

        auto flush = [&](int k) {
            const unsigned q = qcur[k];
            float2 *g = grid + ((q >> 16) * (unsigned)N + (q & 0xFFFFu));
#pragma unroll
            for (int p = 0; p < NPOL; ++p)
                asm volatile("{ .reg .f32 a, b, c, d;\n\t"
                             "mov.b64 {a, b}, %0; mov.b64 {c, d}, %1;\n\t"
                             "red.global.add.v2.f32 [%2], {a, b};\n\t"
                             "red.global.add.v2.f32 [%2 + 8], {c, d};\n\t"
                             "mov.b64 %0, 0; mov.b64 %1, 0; }"
                             : "+l"(acc0[k][p]), "+l"(acc1[k][p]) : "l"(g + p * plane) : "memory");
        };
        auto produce = [&](int s, const RecP<NPOL> *rp) {
#pragma unroll
            for (int p = 0; p < NPOL; ++p) vis[s][p] = *reinterpret_cast<const U64 *>(&rp->v[p]);
            const uint2 pk = *reinterpret_cast<const uint2 *>(&rp->pos);
            const unsigned pos = pk.x, koff = pk.y;
#pragma unroll
            for (int k = 0; k < NSLOT; ++k) {
                const unsigned d = (RG[k] - pos) & M;
                qn[s][k] = pos + d;
                ldg128(K + (koff + (d >> 16) * (unsigned)S + (d & 0xFFFFu)), c0[s][k], c1[s][k]);
            }
        };
        auto consume = [&](int s) {
            bool any = false;
#pragma unroll
            for (int k = 0; k < NSLOT; ++k) any |= qn[s][k] != qcur[k];
            if (__any_sync(0xffffffffu, any)) {
#pragma unroll
                for (int k = 0; k < NSLOT; ++k) {
                    if (qn[s][k] != qcur[k]) {
                        if (qcur[k] != 0xFFFFFFFFu) flush(k);
                        asm volatile("mov.b32 %0, %1;" : "+r"(qcur[k]) : "r"(qn[s][k]));
                    }
                }
            }
#pragma unroll
            for (int p = 0; p < NPOL; ++p) {
                const float2 vv = unpack2(vis[s][p]);
                const U64 v1 = vis[s][p], v2 = pack2(-vv.y, vv.x);
#pragma unroll
                for (int k = 0; k < NSLOT; ++k) {
                    const float2 k0 = unpack2(c0[s][k]), k1 = unpack2(c1[s][k]);
                    fma2(acc0[k][p], v1, pack2(k0.x, k0.x)); fma2(acc0[k][p], v2, pack2(k0.y, k0.y));
                    fma2(acc1[k][p], v1, pack2(k1.x, k1.x)); fma2(acc1[k][p], v2, pack2(k1.y, k1.y));
                }
            }
        };
        auto enter_chunk = [&](unsigned c) {
            __syncwarp();
            ring_fill_pol<NPOL>(ring, rec, i0, i1, c + 2, lane);
            cp_async_commit();
            cp_async_wait<2>();
            __syncwarp();
        };

        enter_chunk(0);
#pragma unroll
        for (int s = 0; s < DEPTH; ++s)
            if ((unsigned)s < cnt) produce(s, ring + s);
        for (unsigned j = 0; j < cnt; j += DEPTH) {
            const unsigned jp = j + DEPTH;
            if ((jp & (kChunk - 1)) == 0 && jp < cnt) enter_chunk(jp / kChunk);
            const RecP<NPOL> *rp = ring + (jp & kRingMask);
            if (jp + DEPTH <= cnt) {
#pragma unroll
                for (int s = 0; s < DEPTH; ++s) { consume(s); produce(s, rp + s); }
            } else {
#pragma unroll
                for (int s = 0; s < DEPTH; ++s) {
                    if (j + s < cnt) consume(s);
                    if (jp + s < cnt) produce(s, rp + s);
                }
            }
        }
#pragma unroll
        for (int k = 0; k < NSLOT; ++k)
            if (qcur[k] != 0xFFFFFFFFu) flush(k);
        cp_async_wait<0>();
    }
}

// ------------------------------------------------------------------------------------ cells (fp64)
// The fp64 counterpart of the pair gridder: a c128 coefficient is 16 bytes, so a lane-slot owns ONE cell
// (residue (rb, ra) of the window, any S) and one LDG.128 feeds one update of four DFMA.  Same structure
// otherwise: cp.async record ring (24-byte records), stateless look-ahead DEPTH records deep, write-out
// (two red.global.add.f64) as one asm with the sums as read-write operands.
// Write one cell out and clear its sums (one asm statement with the sums as read-write operands, see the pair gridder).
__device__ __forceinline__ void flush_cell(double2 *g, double &x, double &y) {
    asm volatile("red.global.add.f64 [%2], %0;\n\t"
                 "red.global.add.f64 [%2 + 8], %1;\n\t"
                 "mov.f64 %0, 0d0000000000000000; mov.f64 %1, 0d0000000000000000;"
                 : "+d"(x), "+d"(y) : "l"(g) : "memory");
}
__device__ __forceinline__ void flush_cell(float2 *g, float &x, float &y) {
    asm volatile("red.global.add.v2.f32 [%2], {%0, %1};\n\t"
                 "mov.f32 %0, 0f00000000; mov.f32 %1, 0f00000000;"
                 : "+f"(x), "+f"(y) : "l"(g) : "memory");
}

// WS > 1: the window is split over WS work items (NSLOT of the WS * NSLOT lane-slot sets each), as in grid_pairs_kernel.
template <typename T, int SCT, int NSLOT, int DEPTH, int MINB, int WS = 1>
__global__ void __launch_bounds__(kRunThreads, MINB)
grid_cells_kernel(const Rec<T> *__restrict__ rec, const unsigned *__restrict__ bucket_start,
                    const unsigned *__restrict__ key_base, int cls, unsigned key_lo, unsigned key_hi, int S_rt, unsigned magicS, unsigned *__restrict__ cursor,
                    const typename Cplx<T>::type *__restrict__ K, typename Cplx<T>::type *__restrict__ grid, int N, unsigned seg) {
    using C = typename Cplx<T>::type;
    static_assert(kChunk % DEPTH == 0, "the look-ahead depth divides the chunk");
    const int S = SCT ? SCT : S_rt;
    const int NC = S * S;
    const int lane = threadIdx.x & 31;
    // key range of this support class: from the device table (ragged stacks) or by value (key_base == nullptr)
    if (key_base) { key_lo = __ldg(key_base + cls); key_hi = __ldg(key_base + cls + 1); }
    const unsigned r_begin = __ldg(bucket_start + key_lo), r_end = __ldg(bucket_start + key_hi);
    const unsigned nitems = WS * ((r_end - r_begin + seg - 1) / seg);

    __shared__ __align__(16) Rec<T> ring_all[kRunThreads / 32][kChunk * kRing];
    Rec<T> *ring = ring_all[threadIdx.x >> 5];

    unsigned RG[NSLOT];
    int ra[NSLOT], rb[NSLOT];
    bool act[NSLOT];
    auto set_slots = [&](int part) {
#pragma unroll
    for (int k = 0; k < NSLOT; ++k) {
        int r = (part * NSLOT + k) * 32 + lane;
        act[k] = r < NC;
        r = act[k] ? r : 0;
        rb[k] = r / S;
        ra[k] = r - rb[k] * S;
        RG[k] = (0x8000u + (unsigned)ra[k]) | ((0x8000u + (unsigned)rb[k]) << 16);
    }
    };
    set_slots(0);
    constexpr unsigned M = SCT ? ((unsigned)(SCT - 1) | ((unsigned)(SCT - 1) << 16)) : 0u;
    // (iu | iv << 16) of this lane-slot's cell for a window starting at pos = j0u | j0v << 16
    auto offset_in_window = [&](unsigned pos, int k) -> unsigned {
        if (SCT) return (RG[k] - pos) & M;
        const unsigned j0u = pos & 0xFFFFu, j0v = pos >> 16;
        const int ju = (int)(j0u - ((j0u * magicS) >> 20) * (unsigned)S);
        const int jv = (int)(j0v - ((j0v * magicS) >> 20) * (unsigned)S);
        int x = ra[k] - ju; x += x < 0 ? S : 0;
        int y = rb[k] - jv; y += y < 0 ? S : 0;
        return (unsigned)x | ((unsigned)y << 16);
    };

    for (;;) {
        unsigned item = 0;
        if (lane == 0) item = atomicAdd(cursor, 1u);
        item = __shfl_sync(0xffffffffu, item, 0);
        if (item >= nitems) break;
        if (WS > 1) { set_slots((int)(item % WS)); item /= WS; }
        const unsigned i0 = r_begin + item * seg, i1 = min(i0 + seg, r_end);
        const unsigned cnt = i1 - i0;

        __syncwarp();
#pragma unroll
        for (unsigned c = 0; c < 2; ++c) { ring_fill(ring, rec, i0, i1, c, lane); cp_async_commit(); }

        T accx[NSLOT], accy[NSLOT];
        unsigned qcur[NSLOT] = {};
#pragma unroll
        for (int k = 0; k < NSLOT; ++k) { accx[k] = accy[k] = (T)0; qcur[k] = 0xFFFFFFFFu; }
        C cf[DEPTH][NSLOT];
        T vre[DEPTH], vim[DEPTH];
        unsigned qn[DEPTH][NSLOT];

        unsigned posP = 0xFFFFFFFFu, dP[NSLOT], cP[NSLOT];     // window of the last record produced, offsets in it
#pragma unroll
        for (int k = 0; k < NSLOT; ++k) dP[k] = cP[k] = 0;
        auto flush = [&](int k) {
            const unsigned q = qcur[k];
            flush_cell(grid + ((q >> 16) * (unsigned)N + (q & 0xFFFFu)), accx[k], accy[k]);
        };
        auto produce = [&](int s, const Rec<T> *rp) {
            vre[s] = rp->re; vim[s] = rp->im;
            const uint2 pk = *reinterpret_cast<const uint2 *>(&rp->pos);
            const unsigned pos = pk.x, koff = pk.y;
            if (SCT == 0) {            // runtime support: offsets re-derived only when the window start changes
                if (__any_sync(0xffffffffu, pos != posP)) {
#pragma unroll
                    for (int k = 0; k < NSLOT; ++k) {
                        dP[k] = offset_in_window(pos, k);
                        cP[k] = act[k] ? (dP[k] >> 16) * (unsigned)S + (dP[k] & 0xFFFFu) : 0u;
                    }
                    posP = pos;
                }
#pragma unroll
                for (int k = 0; k < NSLOT; ++k) {
                    qn[s][k] = act[k] ? pos + dP[k] : 0xFFFFFFFFu;
                    cf[s][k] = __ldg(K + (koff + cP[k]));
                }
            } else {
#pragma unroll
                for (int k = 0; k < NSLOT; ++k) {
                    const unsigned d = offset_in_window(pos, k);
                    qn[s][k] = act[k] ? pos + d : 0xFFFFFFFFu;
                    const unsigned coff = (d >> 16) * (unsigned)S + (d & 0xFFFFu);
                    cf[s][k] = __ldg(K + (koff + (act[k] ? coff : 0u)));
                }
            }
        };
        auto consume = [&](int s) {
            bool any = false;
#pragma unroll
            for (int k = 0; k < NSLOT; ++k) any |= qn[s][k] != qcur[k];
            if (__any_sync(0xffffffffu, any)) {
#pragma unroll
                for (int k = 0; k < NSLOT; ++k) {
                    if (qn[s][k] != qcur[k]) {
                        if (qcur[k] != 0xFFFFFFFFu) flush(k);
                        asm volatile("mov.b32 %0, %1;" : "+r"(qcur[k]) : "r"(qn[s][k]));
                    }
                }
            }
            const T re = vre[s], im = vim[s];
#pragma unroll
            for (int k = 0; k < NSLOT; ++k) {
                accx[k] = fma(re, cf[s][k].x, accx[k]); accx[k] = fma(-im, cf[s][k].y, accx[k]);
                accy[k] = fma(re, cf[s][k].y, accy[k]); accy[k] = fma(im, cf[s][k].x, accy[k]);
            }
        };
        auto enter_chunk = [&](unsigned c) {
            __syncwarp();
            ring_fill(ring, rec, i0, i1, c + 2, lane);
            cp_async_commit();
            cp_async_wait<2>();
            __syncwarp();
        };

        enter_chunk(0);
#pragma unroll
        for (int s = 0; s < DEPTH; ++s)
            if ((unsigned)s < cnt) produce(s, ring + s);

        for (unsigned j = 0; j < cnt; j += DEPTH) {
            const unsigned jp = j + DEPTH;
            if ((jp & (kChunk - 1)) == 0 && jp < cnt) enter_chunk(jp / kChunk);
            const Rec<T> *rp = ring + (jp & kRingMask);
            if (jp + DEPTH <= cnt) {
#pragma unroll
                for (int s = 0; s < DEPTH; ++s) { consume(s); produce(s, rp + s); }
            } else {
#pragma unroll
                for (int s = 0; s < DEPTH; ++s) {
                    if (j + s < cnt) consume(s);
                    if (jp + s < cnt) produce(s, rp + s);
                }
            }
        }
#pragma unroll
        for (int k = 0; k < NSLOT; ++k)
            if (act[k] && qcur[k] != 0xFFFFFFFFu) flush(k);
        cp_async_wait<0>();
    }
}

// ------------------------------------------------------------------------------------ cells, NPOL correlations
// The general polarised gridder (data are row x channel x polarisation): any
// support (even or odd, ragged stacks through the class loop), fp32 and fp64 (the paper runs both precisions
// everywhere).  Structure of grid_cells_kernel with a runtime support: one cell per lane-slot, the
// window's lane offsets tracked in the producer, the window split over `ws` work items of NSLOT lane-slot sets; the
// NPOL correlations of a record share the coefficient load and the window bookkeeping.  grid[pol][N][N].
template <typename T, int NPOL, int NSLOT, int DEPTH, int MINB>
__global__ void __launch_bounds__(kRunThreads, MINB)
grid_cells_pol_kernel(const typename RecPOf<T, NPOL>::type *__restrict__ rec, const unsigned *__restrict__ bucket_start,
                      const unsigned *__restrict__ key_base, int cls, unsigned key_lo, unsigned key_hi, int S, unsigned magicS,
                      unsigned ws, unsigned *__restrict__ cursor, const typename Cplx<T>::type *__restrict__ K,
                      typename Cplx<T>::type *__restrict__ grid, int N, unsigned seg) {
    using C = typename Cplx<T>::type;
    using RP = typename RecPOf<T, NPOL>::type;
    static_assert(kChunk % DEPTH == 0, "the look-ahead depth divides the chunk");
    constexpr unsigned PIECES = sizeof(RP) / 8;
    const int NC = S * S;
    const int lane = threadIdx.x & 31;
    if (key_base) { key_lo = __ldg(key_base + cls); key_hi = __ldg(key_base + cls + 1); }
    const unsigned r_begin = __ldg(bucket_start + key_lo), r_end = __ldg(bucket_start + key_hi);
    const unsigned nitems = ws * ((r_end - r_begin + seg - 1) / seg);
    const size_t plane = (size_t)N * N;

    __shared__ __align__(16) RP ring_all[kRunThreads / 32][kChunk * kRing];
    RP *ring = ring_all[threadIdx.x >> 5];

    int ra[NSLOT], rb[NSLOT];
    bool act[NSLOT];
    auto set_slots = [&](int part) {
#pragma unroll
        for (int k = 0; k < NSLOT; ++k) {
            int r = (part * NSLOT + k) * 32 + lane;
            act[k] = r < NC;
            r = act[k] ? r : 0;
            rb[k] = r / S;
            ra[k] = r - rb[k] * S;
        }
    };
    auto fill = [&](unsigned i0, unsigned i1, unsigned c) {        // chunk c of the item into its ring slot, 8-byte pieces
        const unsigned long long *g = reinterpret_cast<const unsigned long long *>(rec + i0 + c * kChunk);
        unsigned long long *sm = reinterpret_cast<unsigned long long *>(ring + ((c * kChunk) & kRingMask));
        const unsigned first = i0 + c * kChunk;
        const unsigned npiece = first < i1 ? PIECES * min((unsigned)kChunk, i1 - first) : 0u;
        for (unsigned q = lane; q < npiece; q += 32)
            asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(smem_u32(sm + q)), "l"(g + q) : "memory");
    };

    for (;;) {
        unsigned item = 0;
        if (lane == 0) item = atomicAdd(cursor, 1u);
        item = __shfl_sync(0xffffffffu, item, 0);
        if (item >= nitems) break;
        set_slots((int)(item % ws)); item /= ws;
        const unsigned i0 = r_begin + item * seg, i1 = min(i0 + seg, r_end);
        const unsigned cnt = i1 - i0;

        __syncwarp();
#pragma unroll
        for (unsigned c = 0; c < 2; ++c) { fill(i0, i1, c); cp_async_commit(); }

        T accx[NSLOT][NPOL], accy[NSLOT][NPOL];
        unsigned qcur[NSLOT];
#pragma unroll
        for (int k = 0; k < NSLOT; ++k) {
            qcur[k] = 0xFFFFFFFFu;
#pragma unroll
            for (int p = 0; p < NPOL; ++p) accx[k][p] = accy[k][p] = (T)0;
        }
        C cf[DEPTH][NSLOT];
        T vre[DEPTH][NPOL], vim[DEPTH][NPOL];
        unsigned qn[DEPTH][NSLOT];
        unsigned posP = 0xFFFFFFFFu, dP[NSLOT], cP[NSLOT];
#pragma unroll
        for (int k = 0; k < NSLOT; ++k) dP[k] = cP[k] = 0;

        auto flush = [&](int k) {
            const unsigned q = qcur[k];
            C *g = grid + ((q >> 16) * (unsigned)N + (q & 0xFFFFu));
#pragma unroll
            for (int p = 0; p < NPOL; ++p) flush_cell(g + p * plane, accx[k][p], accy[k][p]);
        };
        auto produce = [&](int s, const RP *rp) {
#pragma unroll
            for (int p = 0; p < NPOL; ++p) { vre[s][p] = rp->v[p].x; vim[s][p] = rp->v[p].y; }
            const uint2 pk = *reinterpret_cast<const uint2 *>(&rp->pos);
            const unsigned pos = pk.x, koff = pk.y;
            if (__any_sync(0xffffffffu, pos != posP)) {      // offsets re-derived only when the window start changes
                const unsigned j0u = pos & 0xFFFFu, j0v = pos >> 16;
                const int ju = (int)(j0u - ((j0u * magicS) >> 20) * (unsigned)S);
                const int jv = (int)(j0v - ((j0v * magicS) >> 20) * (unsigned)S);
#pragma unroll
                for (int k = 0; k < NSLOT; ++k) {
                    int x = ra[k] - ju; x += x < 0 ? S : 0;
                    int y = rb[k] - jv; y += y < 0 ? S : 0;
                    dP[k] = (unsigned)x | ((unsigned)y << 16);
                    cP[k] = act[k] ? (unsigned)(y * S + x) : 0u;
                }
                posP = pos;
            }
#pragma unroll
            for (int k = 0; k < NSLOT; ++k) {
                qn[s][k] = act[k] ? pos + dP[k] : 0xFFFFFFFFu;
                cf[s][k] = __ldg(K + (koff + cP[k]));
            }
        };
        auto consume = [&](int s) {
            bool any = false;
#pragma unroll
            for (int k = 0; k < NSLOT; ++k) any |= qn[s][k] != qcur[k];
            if (__any_sync(0xffffffffu, any)) {
#pragma unroll
                for (int k = 0; k < NSLOT; ++k) {
                    if (qn[s][k] != qcur[k]) {
                        if (qcur[k] != 0xFFFFFFFFu) flush(k);
                        asm volatile("mov.b32 %0, %1;" : "+r"(qcur[k]) : "r"(qn[s][k]));
                    }
                }
            }
#pragma unroll
            for (int p = 0; p < NPOL; ++p) {
                const T re = vre[s][p], im = vim[s][p];
#pragma unroll
                for (int k = 0; k < NSLOT; ++k) {
                    accx[k][p] = fma(re, cf[s][k].x, accx[k][p]); accx[k][p] = fma(-im, cf[s][k].y, accx[k][p]);
                    accy[k][p] = fma(re, cf[s][k].y, accy[k][p]); accy[k][p] = fma(im, cf[s][k].x, accy[k][p]);
                }
            }
        };
        auto enter_chunk = [&](unsigned c) {
            __syncwarp();
            fill(i0, i1, c + 2);
            cp_async_commit();
            cp_async_wait<2>();
            __syncwarp();
        };

        enter_chunk(0);
#pragma unroll
        for (int s = 0; s < DEPTH; ++s)
            if ((unsigned)s < cnt) produce(s, ring + s);
        for (unsigned j = 0; j < cnt; j += DEPTH) {
            const unsigned jp = j + DEPTH;
            if ((jp & (kChunk - 1)) == 0 && jp < cnt) enter_chunk(jp / kChunk);
            const RP *rp = ring + (jp & kRingMask);
#pragma unroll
            for (int s = 0; s < DEPTH; ++s) {
                if (j + s < cnt) consume(s);
                if (jp + s < cnt) produce(s, rp + s);
            }
        }
#pragma unroll
        for (int k = 0; k < NSLOT; ++k)
            if (act[k] && qcur[k] != 0xFFFFFFFFu) flush(k);
        cp_async_wait<0>();
    }
}

template <typename T, int SCT, int NSLOT, int DEPTH, int MINB, int WS = 1>
int launch_cells(wpg_ctx *ctx, cudaStream_t strm, const BinParams &bp, const WorkspaceLayout &ws, const void *K, void *grid, char *w,
                   int cls, int S) {
    int per_sm = ctx->opt_ctas_per_sm ? ctx->opt_ctas_per_sm : MINB;
    int blocks = ctx->sm_count * per_sm;
    unsigned seg = ctx->opt_segment ? (unsigned)ctx->opt_segment : 256u;
    Counters *ctr = (Counters *)(w + ws.off_counters);
    unsigned magicS = (1u << 20) / (unsigned)S + 1u;
    grid_cells_kernel<T, SCT, NSLOT, DEPTH, MINB, WS><<<blocks, kRunThreads, 0, strm>>>(
        (const Rec<T> *)(w + ws.off_records), (const unsigned *)(w + ws.off_hist),
        bp.dyn_keys ? ctr->key_base : nullptr, cls, (unsigned)cls * bp.keys_per_class, (unsigned)(cls + 1) * bp.keys_per_class, S, magicS, &ctr->cursor[cls],
        (const typename Cplx<T>::type *)K, (typename Cplx<T>::type *)grid, bp.N, seg);
    ctx->n_launches += 1;
    WPG_CUDA(ctx, cudaGetLastError());
    return WPG_OK;
}

template <typename T, int SCT, int NSLOT, int MINB>
int launch_runs(wpg_ctx *ctx, cudaStream_t strm, const BinParams &bp, const WorkspaceLayout &ws, const void *K, void *grid, char *w,
                int cls, int S) {
    using C = typename Cplx<T>::type;
    int per_sm = ctx->opt_ctas_per_sm ? ctx->opt_ctas_per_sm : MINB;
    int blocks = ctx->sm_count * per_sm;
    unsigned seg = ctx->opt_segment ? (unsigned)ctx->opt_segment : 256u;
    Counters *ctr = (Counters *)(w + ws.off_counters);
    grid_runs_kernel<T, SCT, NSLOT, MINB><<<blocks, kRunThreads, 0, strm>>>(
        (const Rec<T> *)(w + ws.off_records), (const unsigned *)(w + ws.off_hist),
        bp.dyn_keys ? ctr->key_base : nullptr, cls, (unsigned)cls * bp.keys_per_class, (unsigned)(cls + 1) * bp.keys_per_class, S, &ctr->cursor[cls],
        (const C *)K, (C *)grid, bp.N, seg);
    ctx->n_launches += 1;
    WPG_CUDA(ctx, cudaGetLastError());
    return WPG_OK;
}

template <typename T>
int launch_class(wpg_ctx *ctx, cudaStream_t strm, const BinParams &bp, const WorkspaceLayout &ws, const void *K, void *grid, char *w,
                 int cls, int S) {
    constexpr bool F = sizeof(T) == 4;
    if (F && S % 2 == 0 && !ctx->opt_no_pairs && ((uintptr_t)K & 15) == 0) {
        // fp32, even support: the pair gridder (S*S/2 pairs over 32 lanes)
        const int np = S * S / 2, nslot = (np + 31) / 32;
        if (S == 8) return launch_pairs<8, 2, 4, 3, 2>(ctx, strm, bp, ws, K, grid, w, cls, S);        // two half-warps, two pairs per lane
        if (S == 16) return launch_pairs<16, 2, 4, 3, 1, 0, false, 2>(ctx, strm, bp, ws, K, grid, w, cls, S);   // window split over two work items
        if (S == 4) return launch_pairs<4, 1, 4, 4, 4>(ctx, strm, bp, ws, K, grid, w, cls, S);        // 8 pairs: 4 records per step
        if (S == 12) return launch_pairs<12, 3, 2, 3, 1, 4, true>(ctx, strm, bp, ws, K, grid, w, cls, S);     // 4 rows per slot
        if (S == 10) return launch_pairs<10, 2, 4, 3, 1, 0, true>(ctx, strm, bp, ws, K, grid, w, cls, S);     // (config 4's second and
        if (S == 14) return launch_pairs<14, 4, 2, 2, 1, 0, true>(ctx, strm, bp, ws, K, grid, w, cls, S);     //  fourth largest classes)
        if (nslot <= 1) return launch_pairs<0, 1, 4, 4, 1, 0, true>(ctx, strm, bp, ws, K, grid, w, cls, S);
        if (nslot <= 2) return launch_pairs<0, 2, 4, 3, 1, 0, true>(ctx, strm, bp, ws, K, grid, w, cls, S);
        if (nslot <= 3) return launch_pairs<0, 3, 2, 3, 1, 0, true>(ctx, strm, bp, ws, K, grid, w, cls, S);
        if (nslot <= 4) return launch_pairs<0, 4, 2, 2, 1, 0, true>(ctx, strm, bp, ws, K, grid, w, cls, S);
        if (nslot <= 6) return launch_pairs<0, 3, 2, 3, 1, 0, true, 2>(ctx, strm, bp, ws, K, grid, w, cls, S);    // two work items of 3 slot sets
        if (nslot <= 8) return launch_pairs<0, 4, 2, 2, 1, 0, true, 2>(ctx, strm, bp, ws, K, grid, w, cls, S);    // two work items of 4 slot sets
        if (nslot <= 12) return launch_pairs<0, 4, 2, 2, 1, 0, true, 3>(ctx, strm, bp, ws, K, grid, w, cls, S);   // three (S = 24)
        if (nslot <= 16) return launch_pairs<0, 4, 2, 2, 1, 0, true, 4>(ctx, strm, bp, ws, K, grid, w, cls, S);   // four (S = 26 .. 32)
    }
    if (!F && !ctx->opt_no_pairs && ((uintptr_t)K & 15) == 0) {
        // fp64: one cell per lane-slot, S*S cells over 32 lanes
        const int nslot = (S * S + 31) / 32;
        if (S == 8) return launch_cells<double, 8, 2, 4, 3>(ctx, strm, bp, ws, K, grid, w, cls, S);
        if (S == 16) return launch_cells<double, 16, 4, 2, 2, 2>(ctx, strm, bp, ws, K, grid, w, cls, S);       // window split over two work items
        if (S == 4) return launch_cells<double, 4, 1, 4, 4>(ctx, strm, bp, ws, K, grid, w, cls, S);
        if (nslot <= 2) return launch_cells<double, 0, 2, 4, 3>(ctx, strm, bp, ws, K, grid, w, cls, S);
        if (nslot <= 5) return launch_cells<double, 0, 5, 2, 2>(ctx, strm, bp, ws, K, grid, w, cls, S);
        if (nslot <= 8) return launch_cells<double, 0, 4, 2, 2, 2>(ctx, strm, bp, ws, K, grid, w, cls, S);    // two work items of 4 slot sets
        if (nslot <= 12) return launch_cells<double, 0, 4, 2, 2, 3>(ctx, strm, bp, ws, K, grid, w, cls, S);
        if (nslot <= 16) return launch_cells<double, 0, 4, 2, 2, 4>(ctx, strm, bp, ws, K, grid, w, cls, S);
        if (nslot <= 20) return launch_cells<double, 0, 4, 2, 2, 5>(ctx, strm, bp, ws, K, grid, w, cls, S);
        if (nslot <= 24) return launch_cells<double, 0, 4, 2, 2, 6>(ctx, strm, bp, ws, K, grid, w, cls, S);
        if (nslot <= 28) return launch_cells<double, 0, 4, 2, 2, 7>(ctx, strm, bp, ws, K, grid, w, cls, S);
        if (nslot <= 32) return launch_cells<double, 0, 4, 2, 2, 8>(ctx, strm, bp, ws, K, grid, w, cls, S);    // S = 32: eight work items
    }
    if (F && !ctx->opt_no_pairs) {
        // fp32, odd support (the paper's own experiments use full support 9): one cell per lane-slot
        const int nslot = (S * S + 31) / 32;
        if (nslot <= 2) return launch_cells<float, 0, 2, 4, 4>(ctx, strm, bp, ws, K, grid, w, cls, S);            // S <= 7
        if (nslot <= 4) return launch_cells<float, 0, 4, 2, 3>(ctx, strm, bp, ws, K, grid, w, cls, S);            // S = 9, 11
        if (nslot <= 8) return launch_cells<float, 0, 4, 2, 3, 2>(ctx, strm, bp, ws, K, grid, w, cls, S);         // S = 13, 15
        if (nslot <= 16) return launch_cells<float, 0, 4, 2, 3, 4>(ctx, strm, bp, ws, K, grid, w, cls, S);        // S = 17 .. 21
        if (nslot <= 32) return launch_cells<float, 0, 4, 2, 3, 8>(ctx, strm, bp, ws, K, grid, w, cls, S);        // S = 23 .. 31
    }
    if (S == 8) return launch_runs<T, 8, 2, F ? 4 : 3>(ctx, strm, bp, ws, K, grid, w, cls, S);
    if (S == 16) return launch_runs<T, 16, 8, F ? 2 : 1>(ctx, strm, bp, ws, K, grid, w, cls, S);
    if (S == 4) return launch_runs<T, 4, 1, F ? 6 : 4>(ctx, strm, bp, ws, K, grid, w, cls, S);
    int nslot = (S * S + 31) / 32;
    if (nslot <= 2) return launch_runs<T, 0, 2, F ? 4 : 3>(ctx, strm, bp, ws, K, grid, w, cls, S);
    if (nslot <= 5) return launch_runs<T, 0, 5, F ? 3 : 2>(ctx, strm, bp, ws, K, grid, w, cls, S);
    if (nslot <= 8) return launch_runs<T, 0, 8, F ? 2 : 1>(ctx, strm, bp, ws, K, grid, w, cls, S);
    if (nslot <= 18) return launch_runs<T, 0, 18, F ? 2 : 1>(ctx, strm, bp, ws, K, grid, w, cls, S);
    return launch_runs<T, 0, 32, 1>(ctx, strm, bp, ws, K, grid, w, cls, S);
}

}  // namespace

int wpg_launch_grid(wpg_ctx *ctx, const PlaneTab &tab, const BinParams &bp, const WorkspaceLayout &ws,
                    wpg_prec prec, const void *K, void *grid, char *w) {
    if (bp.nrow == 0) return WPG_OK;
    if (bp.ncls == 1) {
        return prec == WPG_F32 ? launch_class<float>(ctx, ctx->stream, bp, ws, K, grid, w, 0, tab.clsS[0])
                               : launch_class<double>(ctx, ctx->stream, bp, ws, K, grid, w, 0, tab.clsS[0]);
    }
    // Ragged stack: one launch per support class, independent of each other (they only meet in the grid's
    // reductions).  Most classes hold few visibilities and cannot fill the machine on their own, so the
    // launches are spread over the context's stream and three side streams, large supports first.
    cudaStream_t main_stream = ctx->stream;
    if (!ctx->side_ready) {             // all or nothing: a partial failure leaves no half-built set behind
        cudaError_t e = cudaEventCreateWithFlags(&ctx->ev_fork, cudaEventDisableTiming);
        for (int i = 0; i < 3 && e == cudaSuccess; ++i) {
            e = cudaStreamCreateWithFlags(&ctx->side[i], cudaStreamNonBlocking);
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->ev_join[i], cudaEventDisableTiming);
        }
        if (e != cudaSuccess) {
            for (int i = 0; i < 3; ++i) {
                if (ctx->side[i]) cudaStreamDestroy(ctx->side[i]);
                if (ctx->ev_join[i]) cudaEventDestroy(ctx->ev_join[i]);
                ctx->side[i] = nullptr; ctx->ev_join[i] = nullptr;
            }
            if (ctx->ev_fork) cudaEventDestroy(ctx->ev_fork);
            ctx->ev_fork = nullptr;
            return wpg_fail(ctx, WPG_ECUDA, "cannot create the side streams of the ragged-stack gridder: %s", cudaGetErrorString(e));
        }
        ctx->side_ready = true;
    }
    WPG_CUDA(ctx, cudaEventRecord(ctx->ev_fork, main_stream));
    for (int i = 0; i < 3; ++i) WPG_CUDA(ctx, cudaStreamWaitEvent(ctx->side[i], ctx->ev_fork, 0));
    int rc = WPG_OK;
    for (int cls = bp.ncls - 1; cls >= 0 && rc == WPG_OK; --cls) {
        const int S = tab.clsS[cls];
        cudaStream_t strm = cls % 4 == 0 ? main_stream : ctx->side[cls % 4 - 1];
        rc = prec == WPG_F32 ? launch_class<float>(ctx, strm, bp, ws, K, grid, w, cls, S)
                             : launch_class<double>(ctx, strm, bp, ws, K, grid, w, cls, S);
    }
    for (int i = 0; i < 3; ++i) {
        WPG_CUDA(ctx, cudaEventRecord(ctx->ev_join[i], ctx->side[i]));
        WPG_CUDA(ctx, cudaStreamWaitEvent(main_stream, ctx->ev_join[i], 0));
    }
    return rc;
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

int wpg_launch_grid_pol(wpg_ctx *ctx, const PlaneTab &tab, const BinParams &bp, const WorkspaceLayout &ws, wpg_prec prec,
                        int npol, const void *K, void *grid, char *w) {
    if (bp.nrow == 0) return WPG_OK;
    Counters *ctr = (Counters *)(w + ws.off_counters);
    const unsigned seg = ctx->opt_segment ? (unsigned)ctx->opt_segment : 256u;
    const unsigned *bs = (const unsigned *)(w + ws.off_hist);
    cudaStream_t s = ctx->stream;
    const bool aligned = ((uintptr_t)K & 15) == 0;
    // the fp32 pair gridders for uniform supports 8 and 16 (one LDG.128 feeds 2 * npol updates)
    if (prec == WPG_F32 && bp.ncls == 1 && aligned && !ctx->opt_no_pairs && (tab.clsS[0] == 8 || tab.clsS[0] == 16)) {
        const int S = tab.clsS[0];
#define WPG_POL(SS, NS, DD, MB, NP, WW)                                                                                 \
        grid_pairs_pol_kernel<SS, NS, DD, MB, NP, WW><<<ctx->sm_count * (ctx->opt_ctas_per_sm ? ctx->opt_ctas_per_sm : MB), \
            kRunThreads, 0, s>>>((const RecP<NP> *)(w + ws.off_records), bs, 0u, bp.keys_per_class, &ctr->cursor[0],        \
                                 (const float2 *)K, (float2 *)grid, bp.N, seg)
        if (S == 8 && npol == 4) WPG_POL(8, 1, 4, 3, 4, 1);
        else if (S == 8 && npol == 2) WPG_POL(8, 1, 4, 3, 2, 1);
        else if (S == 16 && npol == 4) WPG_POL(16, 1, 4, 3, 4, 4);      // window split over four work items
        else WPG_POL(16, 2, 2, 2, 2, 2);
#undef WPG_POL
        ctx->n_launches += 1;
        WPG_CUDA(ctx, cudaGetLastError());
        return WPG_OK;
    }
    // everything else — other supports, ragged stacks (one launch per support class), fp64 — through the cell gridder
    for (int cls = bp.ncls - 1; cls >= 0; --cls) {
        const int S = tab.clsS[cls];
        const unsigned magicS = (1u << 20) / (unsigned)S + 1u;
        const unsigned nslot = (unsigned)(S * S + 31) / 32;
#define WPG_POLC(TT, NP, NS, DD, MB)                                                                                    \
        grid_cells_pol_kernel<TT, NP, NS, DD, MB><<<ctx->sm_count * (ctx->opt_ctas_per_sm ? ctx->opt_ctas_per_sm : MB),     \
            kRunThreads, 0, s>>>((const typename RecPOf<TT, NP>::type *)(w + ws.off_records), bs,                          \
                                 bp.dyn_keys ? ctr->key_base : nullptr, cls, (unsigned)cls * bp.keys_per_class,            \
                                 (unsigned)(cls + 1) * bp.keys_per_class, S, magicS, (nslot + NS - 1) / NS, &ctr->cursor[cls], \
                                 (const typename Cplx<TT>::type *)K, (typename Cplx<TT>::type *)grid, bp.N, seg)
        if (prec == WPG_F32 && npol == 4) WPG_POLC(float, 4, 2, 2, 2);
        else if (prec == WPG_F32) WPG_POLC(float, 2, 2, 2, 3);
        else if (npol == 4) WPG_POLC(double, 4, 1, 2, 2);
        else WPG_POLC(double, 2, 2, 2, 2);
#undef WPG_POLC
        ctx->n_launches += 1;
    }
    WPG_CUDA(ctx, cudaGetLastError());
    return WPG_OK;
}
