// Internal declarations shared by the translation units of libwpgrid.so (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <cufft.h>
#include <stdint.h>
#include <string>
#include <vector>

#include "../../include/wpgrid.h"

#define WPG_C0 299792458.0
#define WPG_MAX_NW 256
#define WPG_MAX_N 8192
#define WPG_MAX_S 32
#define WPG_MAX_CLS 32
#define WPG_NO_KEY 0xFFFFFFFFu

// Per-plane table, passed to kernels by value (__grid_constant__): element offset of the plane in
// the stack, its full support S_p and its sort class (planes of equal support share a class).
struct PlaneTab {
    int32_t off[WPG_MAX_NW + 1];
    uint8_t S[WPG_MAX_NW];
    uint8_t cls[WPG_MAX_NW];
    uint8_t clsS[WPG_MAX_CLS];     // support of each sort class, ascending
};

// Everything the position math (G1-G3) and the sort key need.
struct BinParams {
    int64_t nrow;
    int nchan;
    uint32_t row_block, vis_nbx;   // with vis_block: rows per time step; ceil(vis_block / 256) (host-computed: no divisions in the kernels)
    uint32_t vis_ngroups;          // with vis_block: groups of kVpt time steps
    uint32_t vis_tile_shift;       // log2 vis_tile
    uint32_t vis_tile;             // (a power of two) with vis_block: consecutive blocks take vis_tile successive time groups of the same 256 baselines / channels
    int chan_shift;                // log2 nchan if nchan is a power of two, else -1
    uint32_t vis_block;            // 0, or visibilities per time step (row_block * nchan): a binning thread then takes
                                   // the SAME baseline/channel at consecutive time steps (see wpg_vis_index)
    int N, Q, Nw;
    double w_max, dw, du, halfN;   // dw = 2 w_max / Nw, du = 1/(N cell), halfN = N/2
    double rdu, rdw, invQ;         // RN(1/du), RN(1/dw), 1/Q (wpg_div_const, floor division by Q)
    int qshift;                    // log2 Q if Q is a power of two, else -1
    int kshift;                    // the key drops this many low bits of j0v (0 unless the key space is capped)
    int nkg;                       // ceil(N / 2^kshift): keys per grid column
    int ncls;                      // number of sort classes (distinct supports)
    uint32_t keys_per_class;       // N * nkg; key = (cls * N + j0u) * nkg + (j0v >> kshift)
    uint32_t nkeys;                // size of the key space (ncls * keys_per_class, or the key budget if dynamic)
    int dyn_keys;                  // 1: per-class key layout chosen on the device (ragged stacks)
    int S0;                        // support of class 0 (uniform stacks: THE support, no table lookup)
    int compress;                  // 1: record compression (visibilities with equal window start and coefficient slice share a record)
};

// Sorted record.  pos = j0u | j0v << 16 (window start, cells); koff = element offset
// of the S x S coefficient slice K[p][ov][ou] inside the stack.
template <typename T> struct Rec { T re, im; uint32_t pos, koff; };
static_assert(sizeof(Rec<float>) == 16, "fp32 record is 16 B");
static_assert(sizeof(Rec<double>) == 24, "fp64 record is 24 B");

// Record of the polarised gridder: NPOL correlations of one (row, channel) share the
// window and the coefficient slice.
template <int NPOL> struct RecP { float2 v[NPOL]; uint32_t pos, koff; };
static_assert(sizeof(RecP<4>) == 40 && sizeof(RecP<2>) == 24, "polarised records are 8 NPOL + 8 bytes");
struct Dpair { double x, y; };                                                    // (8-byte aligned, unlike double2)
template <int NPOL> struct RecPD { Dpair v[NPOL]; uint32_t pos, koff; };        // fp64: 16 NPOL + 8 bytes
static_assert(sizeof(RecPD<4>) == 72 && sizeof(RecPD<2>) == 40, "fp64 polarised records are 16 NPOL + 8 bytes");
template <typename T, int NPOL> struct RecPOf;
template <int NPOL> struct RecPOf<float, NPOL> { using type = RecP<NPOL>; };
template <int NPOL> struct RecPOf<double, NPOL> { using type = RecPD<NPOL>; };

// Device counters block at the head of the workspace.
struct Counters {
    // wpg_stats counters, each spread over kStatSlots addresses (blocks add to slot blockIdx % kStatSlots:
    // tens of thousands of reductions on ONE address serialise in L2); the host sums the slots
    unsigned long long n_gridded[16], n_skipped_oob[16], n_skipped_zero_weight[16], n_clamped_w[16], n_updates[16];
    unsigned int n_records, pad0, pad1, pad2;
    unsigned int cursor[WPG_MAX_CLS];   // work-item cursors of the gridder launches (one per sort class)
    // key layout of each sort class: key = key_base[cls] + j0u * key_nkg[cls] + (j0v >> key_shift[cls]).
    // Uniform stacks: filled from the host plan.  Ragged stacks: chosen on the device from a census of the
    // classes (the key budget goes to the classes that hold the visibilities).
    unsigned int key_base[WPG_MAX_CLS + 1], key_shift[WPG_MAX_CLS], key_nkg[WPG_MAX_CLS], census[WPG_MAX_CLS];
};

constexpr int kStatSlots = 16;
struct WorkspaceLayout {
    size_t off_counters, off_records, off_hist, off_blocksum, off_fscale;
    size_t total;
    uint32_t nkeys, nblocks_scan;
};

struct wpg_ctx {
    int device = 0;
    cudaStream_t stream = nullptr;
    int sm_count = 148;
    std::string err;
    // options
    int opt_segment = 0;      // records per gridder work item, 0 = default
    int opt_ctas_per_sm = 0;  // gridder CTAs per SM, 0 = default
    int opt_key_bits = 0;     // cap of the sort key space (log2), 0 = default 24
    int opt_timing = 0;       // 1: wpg_grid brackets its phases with CUDA events
    int64_t opt_row_block = 0; // rows per time step (0 = unknown), see wpg_set_option
    int opt_no_pairs = 0;     // 1: fp32 even supports also go through the run gridder (A/B comparison)
    int opt_compress = 1;     // record compression in the binning pass (0: one record per gridded visibility)
    int opt_bin_tile = 0;     // time groups per block tile of the binning passes, 0 = default
    int opt_chunk_sort = 1;   // fine order inside coarse buckets (chunk_sort_kernel); 0: off
    // instrumentation
    int64_t n_launches = 0;   // kernels of this library launched so far
    std::vector<cudaEvent_t> ev;   // triplets: start, after binning, after gridder (pool, reused)
    size_t ev_used = 0;            // triplets recorded since the last wpg_phase_ms
    // side streams for the gridder launches of ragged stacks (one launch per support class; created lazily)
    cudaStream_t side[3] = {nullptr, nullptr, nullptr};
    cudaEvent_t ev_fork = nullptr, ev_join[3] = {nullptr, nullptr, nullptr};
    bool side_ready = false;
    // copy stream and events of the host-buffer pipeline (wpg_grid_host; created lazily)
    cudaStream_t copy_stream = nullptr;
    cudaEvent_t ev_start = nullptr, ev_chunk[4] = {nullptr, nullptr, nullptr, nullptr};
    // cuFFT plan cache
    cufftHandle plan = 0; int plan_N = 0; int plan_prec = -1;
    // device scratch of the host-buffer variant (grow-only)
    void *d_host_scratch = nullptr; size_t host_scratch_bytes = 0;
};

int wpg_fail(wpg_ctx *ctx, int code, const char *fmt, ...);

// Selects the context's device for the duration of an entry point and restores the caller's current device on
// return (the caller may drive several GPUs from one thread; torch's current device must not change under it).
struct DeviceGuard {
    int prev = -1; cudaError_t err;
    explicit DeviceGuard(int device) {
        err = cudaGetDevice(&prev);
        if (err == cudaSuccess && prev != device) err = cudaSetDevice(device); else if (err == cudaSuccess) prev = -1;
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
    DeviceGuard(const DeviceGuard &) = delete;
    DeviceGuard &operator=(const DeviceGuard &) = delete;
};
#define WPG_DEVICE(ctx)                                                                          \
    DeviceGuard dev_guard_((ctx)->device);                                                       \
    if (dev_guard_.err != cudaSuccess)                                                           \
        return wpg_fail(ctx, WPG_ECUDA, "cannot select device %d: %s", (ctx)->device, cudaGetErrorString(dev_guard_.err))
#define WPG_CUDA(ctx, call)                                                                   \
    do {                                                                                      \
        cudaError_t e_ = (call);                                                              \
        if (e_ != cudaSuccess)                                                                \
            return wpg_fail(ctx, WPG_ECUDA, "%s failed: %s (%s:%d)", #call,                   \
                            cudaGetErrorString(e_), __FILE__, __LINE__);                      \
    } while (0)

// host helpers (wpg_api.cu)
int wpg_check_desc(wpg_ctx *ctx, const wpg_kdesc *d);
int wpg_make_plan(wpg_ctx *ctx, const wpg_kdesc *d, int64_t nrow, int nchan, wpg_prec prec,
                  PlaneTab *tab, BinParams *bp, WorkspaceLayout *ws);
void wpg_pswf_eval(const double *nu, int64_t n, double *out);     // wpg_wkernel.cu (host)
int wpg_launch_taper(wpg_ctx *ctx, double *d_out, int n, double step);   // psi(2 (j - n/2) step), j < n, on the device

int wpg_mark(wpg_ctx *ctx, int i);      // timing event i (0 start, 1 after binning / re-order, 2 after gridder) if option "timing"
// launchers
int wpg_launch_bin_pol(wpg_ctx *ctx, const void *d_vis, const double *d_uvw, const float *d_weight, const double *d_freq,
                       const PlaneTab &tab, const BinParams &bp, const WorkspaceLayout &ws, wpg_prec prec, int npol, char *d_ws);
int wpg_launch_grid_pol(wpg_ctx *ctx, const PlaneTab &tab, const BinParams &bp, const WorkspaceLayout &ws, wpg_prec prec, int npol,
                        const void *d_kernels, void *d_grid, char *d_ws);
int wpg_launch_exclusive_scan(wpg_ctx *ctx, unsigned *hist, unsigned n, unsigned *blocksum, Counters *ctr);
int wpg_launch_bin(wpg_ctx *ctx, const void *d_vis, const double *d_uvw, const float *d_weight,
                   const double *d_freq, const PlaneTab &tab, const BinParams &bp,
                   const WorkspaceLayout &ws, wpg_prec prec, char *d_ws);
int wpg_launch_grid(wpg_ctx *ctx, const PlaneTab &tab, const BinParams &bp, const WorkspaceLayout &ws,
                    wpg_prec prec, const void *d_kernels, void *d_grid, char *d_ws);
int wpg_launch_naive(wpg_ctx *ctx, const void *d_vis, const double *d_uvw, const float *d_weight,
                     const double *d_freq, const PlaneTab &tab, const BinParams &bp, wpg_prec prec,
                     const void *d_kernels, void *d_grid, Counters *d_counters);

// ---------------------------------------------------------------------------------------------
// Position math G1-G3 (exactness rule G6): IEEE fp64, written order, no FMA
// contraction — every operation is an explicit round-to-nearest intrinsic.
#ifdef __CUDACC__
struct VisPos { int p, S, j0u, j0v, ou, ov; bool inside, clamped; };

// a / b for a divisor that is a launch constant, rb = RN(1 / b) computed on the host: the product, one exact
// residual and one correction (Markstein's sequence) give the correctly rounded quotient, i.e. the value
// of __ddiv_rn(a, b), in three instructions instead of the division's reciprocal iteration.  *t_guard: the
// callers take floor() of a value derived from the quotient; if that value sits within a few ulps of an
// integer they recompute with the IEEE division (never observed to differ; keeps G6 unconditional).
__device__ __forceinline__ double wpg_div_const(double a, double b, double rb) {
    const double q0 = __dmul_rn(a, rb);
    const double rem = __fma_rn(-b, q0, a);
    return __fma_rn(rem, rb, q0);
}
// For |t| < 2^30 (everything that can land on a grid) one ulp of t is below 2.4e-7, so an absolute guard band of
// 1e-6 covers a quotient that is off by a few ulps; it sends 2e-6 of the visibilities through the IEEE division
// for nothing.  Larger |t| are integers or nearly so: the guard fires, harmlessly.
__device__ __forceinline__ bool wpg_near_integer(double t) {
    const double fr = t - floor(t);
    return !(fr >= 1e-6 && fr <= 1.0 - 1e-6);         // also true for NaN
}

__device__ __forceinline__ void wpg_axis(double x_lambda, const BinParams &P, int S, int &j0, int &o) {
    double x = __dadd_rn(wpg_div_const(x_lambda, P.du, P.rdu), P.halfN);
    double t = __dadd_rn(__dmul_rn(x, (double)P.Q), 0.5);
    if (wpg_near_integer(t)) {                                   // practically never
        x = __dadd_rn(__ddiv_rn(x_lambda, P.du), P.halfN);
        t = __dadd_rn(__dmul_rn(x, (double)P.Q), 0.5);
    }
    if (!(fabs(t) < 1073741824.0)) { j0 = -(1 << 20); o = 0; return; }      // far outside any grid (also NaN)
    const int X = __double2int_rd(t);                            // floor
    const int Y = X - (S - 2) * P.Q / 2;
    int q;
    if (P.qshift >= 0) {                                         // Q = 2^qshift: floor division is a shift
        q = Y >> P.qshift;
    } else {
        q = __double2int_rd((double)Y * P.invQ);                 // within 1 of floor(Y / Q); fixed up below
        int r = Y - q * P.Q;
        q += r >= P.Q ? 1 : (r < 0 ? -1 : 0);
    }
    j0 = max(min(q, 1 << 20), -(1 << 20));
    o = Y - q * P.Q;
}

// Plane lookup: `tab` is either the PlaneTab itself (kernel parameter, constant bank — fine when the
// index is warp-uniform or rarely used) or its packed copy in shared memory (SmemPlaneTab: the binning
// passes index it with a different plane in every lane, which the constant cache would serialise).
struct SmemPlaneTab {
    const uint2 *e;        // e[p] = {element offset of plane p, S_p | class << 8}
    const uint4 *ck;       // ck[cls] = {key_base, key_nkg, key_shift, -}
    __device__ __forceinline__ int S(int p) const { return (int)(e[p].y & 0xFFu); }
    __device__ __forceinline__ int cls(int p) const { return (int)(e[p].y >> 8); }
    __device__ __forceinline__ int off(int p) const { return (int)e[p].x; }
};
struct ParamPlaneTab {
    const PlaneTab &t;
    __device__ __forceinline__ int S(int p) const { return t.S[p]; }
    __device__ __forceinline__ int cls(int p) const { return t.cls[p]; }
    __device__ __forceinline__ int off(int p) const { return t.off[p]; }
};
// fills the shared copy (call from every thread of the block, then __syncthreads)
__device__ __forceinline__ void wpg_stage_planetab(uint2 *dst, const PlaneTab &T, int Nw) {
    for (int p = threadIdx.x; p < Nw; p += blockDim.x) dst[p] = make_uint2((unsigned)T.off[p], (unsigned)T.S[p] | ((unsigned)T.cls[p] << 8));
}
__device__ __forceinline__ void wpg_stage_classkeys(uint4 *dst, const Counters *ctr, const BinParams &P) {
    for (int c = threadIdx.x; c < P.ncls; c += blockDim.x)
        dst[c] = P.dyn_keys ? make_uint4(ctr->key_base[c], ctr->key_nkg[c], ctr->key_shift[c], 0u)
                            : make_uint4((unsigned)c * P.keys_per_class, (unsigned)P.nkg, (unsigned)P.kshift, 0u);   // no load
}

template <typename Tab>
__device__ __forceinline__ VisPos wpg_locate(double um, double vm, double wm, double f,
                                             const BinParams &P, const Tab &T) {
    VisPos r;
    double u = __dmul_rn(um, f), v = __dmul_rn(vm, f), w = __dmul_rn(wm, f);     // G1
    r.clamped = fabs(w) > P.w_max;                                               // G2
    int p = 0;
    if (P.dw > 0.0) {
        const double ws = __dadd_rn(w, P.w_max);
        double qd = wpg_div_const(ws, P.dw, P.rdw);
        if (wpg_near_integer(qd)) qd = __ddiv_rn(ws, P.dw);
        double fp = floor(qd);
        p = fp < 0.0 ? 0 : (fp > (double)(P.Nw - 1) ? P.Nw - 1 : (int)fp);
    }
    r.p = p;
    r.S = T.S(p);
    wpg_axis(u, P, r.S, r.j0u, r.ou);                                            // G3
    wpg_axis(v, P, r.S, r.j0v, r.ov);
    r.inside = r.j0u >= 0 && r.j0v >= 0 && r.j0u + r.S <= P.N && r.j0v + r.S <= P.N;   // G4
    return r;
}

// ---------------------------------------------------------------------------------------------
// The lean form of wpg_locate used by the hot passes (binning, degridding).  Straight-line code: quotients by
// Markstein's sequence (wpg_div_const), floor() through the 2^52 + 2^51 rounding constant instead of the conversion
// pipe, and ONE flag that says whether any of the three values whose floor is taken lies within 1e-6 of an integer (or
// outside the range where the trick is valid).  Only then — a few visibilities in a million — the written form with
// IEEE divisions is evaluated out of line (wpg_locate), so that G6 holds whatever the constant-divisor sequence does
// in its last bit.
__device__ __forceinline__ int wpg_floor_magic(double t, double lim, bool &risk) {
    // |t| < lim <= 2^30: t + M holds rint(t) in its low word; t - rint(t) is exact.  One ulp of t is below 2.4e-7 there.
    // Outside the range (also NaN) the flag is raised and the value returned is not used.
    const double M = 6755399441055744.0;
    const double tm = __dadd_rn(t, M);
    const double d = __dadd_rn(t, -__dadd_rn(tm, -M));           // in [-0.5, 0.5]
    risk |= !(fabs(d) >= 1e-6) | !(fabs(t) < lim);
    return __double2loint(tm) - (d < 0.0 ? 1 : 0);
}

// the rare exact path, out of line so that the fast path stays compact;
// returns {p | S << 16 | inside << 24 | clamped << 25, j0u, j0v, ou | ov << 8}
static __device__ __noinline__ int4 wpg_locate_exact(double um, double vm, double wm, double f, const BinParams &P, const uint2 *s_tab) {
    const SmemPlaneTab T{s_tab, nullptr};
    VisPos r;
    if (P.ncls == 1) {                    // uniform stack: no table in shared memory
        struct OneS { int s; __device__ int S(int) const { return s; } };
        r = wpg_locate(um, vm, wm, f, P, OneS{P.S0});
    } else {
        r = wpg_locate(um, vm, wm, f, P, T);
    }
    return make_int4(r.p | (r.S << 16) | (r.inside ? 1 << 24 : 0) | (r.clamped ? 1 << 25 : 0), r.j0u, r.j0v, r.ou | (r.ov << 8));
}

// s_tab: the packed per-plane table in shared memory (ragged stacks; not read for uniform stacks).  QP2: the oversampling factor is a power of two (else the general form throughout).
struct LeanPos { int p, S, j0u, j0v, ou, ov; bool inside, clamped; };
template <bool QP2>
__device__ __forceinline__ LeanPos wpg_locate_lean(double um, double vm, double wm, double f, const BinParams &P, const uint2 *s_tab) {
    LeanPos r; r.p = 0; r.S = 0; r.j0u = r.j0v = r.ou = r.ov = 0; r.inside = false; r.clamped = false;
    bool risk = !QP2;
    if (QP2) {
        const double u = __dmul_rn(um, f), vv = __dmul_rn(vm, f), w = __dmul_rn(wm, f);                  // G1
        r.clamped = fabs(w) > P.w_max;                                                                    // G2
        if (P.dw > 0.0) {               // (uniform branch)
            // (far outside [-w_max, w_max], and for NaN, the flag is raised: the exact path clamps)
            const double qd = wpg_div_const(__dadd_rn(w, P.w_max), P.dw, P.rdw);
            r.p = min(max(wpg_floor_magic(qd, 1048576.0, risk), 0), P.Nw - 1);
        }
        r.S = P.ncls == 1 ? P.S0 : (int)(s_tab[r.p].y & 0xFFu);      // {plane offset, S | class << 8}
        const int c = (r.S - 2) * P.Q / 2;
        const double Qd = (double)P.Q, lim = 1073741824.0;
        // G3.  x * Q is exact for Q = 2^k, so the fused form rounds once, like the written two-step form.  Far outside
        // any grid (also NaN) the flag is raised and the exact path reports "outside".
        const double tu = __fma_rn(__dadd_rn(wpg_div_const(u, P.du, P.rdu), P.halfN), Qd, 0.5);
        const double tv = __fma_rn(__dadd_rn(wpg_div_const(vv, P.du, P.rdu), P.halfN), Qd, 0.5);
        const int Yu = wpg_floor_magic(tu, lim, risk) - c;
        const int Yv = wpg_floor_magic(tv, lim, risk) - c;
        r.j0u = Yu >> P.qshift; r.ou = Yu & (P.Q - 1);
        r.j0v = Yv >> P.qshift; r.ov = Yv & (P.Q - 1);
        const unsigned lim_j = (unsigned)(P.N - r.S);
        r.inside = (unsigned)r.j0u <= lim_j && (unsigned)r.j0v <= lim_j;                                 // G4
    }
    if (risk) {
        const int4 o = wpg_locate_exact(um, vm, wm, f, P, s_tab);
        r.p = o.x & 0xFFFF; r.S = (o.x >> 16) & 0xFF; r.inside = (o.x >> 24) & 1; r.clamped = (o.x >> 25) & 1;
        r.j0u = o.y; r.j0v = o.z; r.ou = o.w & 0xFF; r.ov = o.w >> 8;
    }
    return r;
}

template <typename Tab>
__device__ __forceinline__ uint32_t wpg_koff(const VisPos &r, const BinParams &P, const Tab &T) {
    return (uint32_t)(T.off(r.p) + (r.ov * P.Q + r.ou) * r.S * r.S);
}
#endif
