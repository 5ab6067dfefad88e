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
    int N, Q, Nw;
    double w_max, dw, du, halfN;   // dw = 2 w_max / Nw, du = 1/(N cell), halfN = N/2
    int kshift;                    // the key drops this many low bits of j0v (0 unless the key space is capped)
    int nkg;                       // ceil(N / 2^kshift): keys per grid column
    int ncls;                      // number of sort classes (distinct supports)
    uint32_t keys_per_class;       // N * nkg; key = (cls * N + j0u) * nkg + (j0v >> kshift)
    uint32_t nkeys;                // ncls * keys_per_class
};

// Sorted record.  pos = j0u | j0v << 16 (window start, cells); koff = element offset
// of the S x S coefficient slice K[p][ov][ou] inside the stack.
template <typename T> struct Rec { T re, im; uint32_t pos, koff; };
static_assert(sizeof(Rec<float>) == 16, "fp32 record is 16 B");
static_assert(sizeof(Rec<double>) == 24, "fp64 record is 24 B");

// Device counters block at the head of the workspace.
struct Counters {
    unsigned long long n_gridded, n_skipped_oob, n_skipped_zero_weight, n_clamped_w, n_updates;
    unsigned int n_records, pad0, pad1, pad2;
    unsigned int cursor[WPG_MAX_CLS];   // work-item cursors of the gridder launches (one per sort class)
};

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
    int opt_key_bits = 0;     // cap of the sort key space (log2), 0 = default 26
    int opt_timing = 0;       // 1: wpg_grid brackets its phases with CUDA events
    int opt_variant = 0;      // experimental kernel variant selector
    int opt_no_pairs = 0;     // 1: fp32 even supports also go through the run gridder (A/B comparison)
    // instrumentation
    int64_t n_launches = 0;   // kernels of this library launched so far
    std::vector<cudaEvent_t> ev;   // triplets: start, after binning, after gridder (pool, reused)
    size_t ev_used = 0;            // triplets recorded since the last wpg_phase_ms
    // cuFFT plan cache
    cufftHandle plan = 0; int plan_N = 0; int plan_prec = -1;
    // taper table cache for dirty_image
    double *d_taper = nullptr; int taper_N = 0;
    // device scratch of the host-buffer variant (grow-only)
    void *d_host_scratch = nullptr; size_t host_scratch_bytes = 0;
};

int wpg_fail(wpg_ctx *ctx, int code, const char *fmt, ...);
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
void wpg_pswf_eval(const double *nu, int64_t n, double *out);     // wpg_pswf.cu (host)

// launchers
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

__device__ __forceinline__ void wpg_axis(double x_lambda, const BinParams &P, int S, int &j0, int &o) {
    double x = __dadd_rn(__ddiv_rn(x_lambda, P.du), P.halfN);
    long long X = (long long)floor(__dadd_rn(__dmul_rn(x, (double)P.Q), 0.5));
    long long Y = X - (long long)((S - 2) * P.Q / 2);
    long long q = Y / P.Q;
    if ((Y % P.Q != 0) && (Y < 0)) q -= 1;           // floor division
    j0 = (int)max(min(q, (long long)(1 << 20)), (long long)(-(1 << 20)));
    o = (int)(Y - q * P.Q);
}

__device__ __forceinline__ VisPos wpg_locate(double um, double vm, double wm, double f,
                                             const BinParams &P, const PlaneTab &T) {
    VisPos r;
    double u = __dmul_rn(um, f), v = __dmul_rn(vm, f), w = __dmul_rn(wm, f);     // G1
    r.clamped = fabs(w) > P.w_max;                                               // G2
    int p = 0;
    if (P.dw > 0.0) {
        double fp = floor(__ddiv_rn(__dadd_rn(w, P.w_max), P.dw));
        p = fp < 0.0 ? 0 : (fp > (double)(P.Nw - 1) ? P.Nw - 1 : (int)fp);
    }
    r.p = p;
    r.S = T.S[p];
    wpg_axis(u, P, r.S, r.j0u, r.ou);                                            // G3
    wpg_axis(v, P, r.S, r.j0v, r.ov);
    r.inside = r.j0u >= 0 && r.j0v >= 0 && r.j0u + r.S <= P.N && r.j0v + r.S <= P.N;   // G4
    return r;
}

__device__ __forceinline__ uint32_t wpg_koff(const VisPos &r, const BinParams &P, const PlaneTab &T) {
    return (uint32_t)(T.off[r.p] + (r.ov * P.Q + r.ou) * r.S * r.S);
}
#endif
