// Step a0 — oversampled W-kernel stack (setup, untimed), DESIGN.md §2 R1-R3, R5-R7, R20, steps K1-K6.
// The paper only names it ("a new convolution kernel function"; 23 planes, support 9,
// PAPER.md:108); the construction is w-projection's (ref [9]):
//   F_p(l, m) = T(l, m) exp(+2 pi i w_p (n - 1))   sampled on Nk x Nk points across the field of view,
//   C_p(t_v, t_u) = sum_b sum_a F_p[b][a] exp(-2 pi i (t_u (a - Nk/2) + t_v (b - Nk/2)) / (Q Nk)),
//   K[p][ov][ou][iv][iu] = C_p[t(iv, ov)][t(iu, ou)] / s,   t(i, o) = (i + 1) Q - S Q / 2 - o.
// All fp64.  The taper is an independent Legendre-series evaluation of the order-0 prolate
// spheroidal wave function (the oracle uses scipy's routine).
#include <algorithm>
#include <cmath>
#include <map>

#include "wpg_common.h"

// ------------------------------------------------------------------------------------ taper (host)
namespace {

struct Pswf {
    static constexpr int kTerms = 48;
    double coef[kTerms];   // psi(x) = sum_j coef[j] P_{2j}(x) / norm
    double norm;
    Pswf() {
        const double c = 3.0 * M_PI;           // c = pi m_t / 2, m_t = 6 (R2)
        double d[kTerms], e[kTerms];
        for (int j = 0; j < kTerms; ++j) {
            double k = 2.0 * j;
            d[j] = k * (k + 1) + c * c * (2 * k * (k + 1) - 1) / ((2 * k + 3) * (2 * k - 1));
            e[j] = c * c * (k + 2) * (k + 1) / ((2 * k + 3) * std::sqrt((2 * k + 1) * (2 * k + 5)));
        }
        // smallest eigenvalue's eigenvector by inverse iteration (the matrix is SPD; shift 0)
        double x[kTerms], cp[kTerms], dp[kTerms];
        for (int j = 0; j < kTerms; ++j) x[j] = 1.0 / (1 + j);
        for (int it = 0; it < 200; ++it) {
            cp[0] = e[0] / d[0]; dp[0] = x[0] / d[0];                       // Thomas algorithm
            for (int j = 1; j < kTerms; ++j) {
                double m = d[j] - e[j - 1] * cp[j - 1];
                cp[j] = e[j] / m;
                dp[j] = (x[j] - e[j - 1] * dp[j - 1]) / m;
            }
            x[kTerms - 1] = dp[kTerms - 1];
            for (int j = kTerms - 2; j >= 0; --j) x[j] = dp[j] - cp[j] * x[j + 1];
            double nrm = 0;
            for (int j = 0; j < kTerms; ++j) nrm += x[j] * x[j];
            nrm = std::sqrt(nrm);
            for (int j = 0; j < kTerms; ++j) x[j] /= nrm;
        }
        for (int j = 0; j < kTerms; ++j) coef[j] = x[j] * std::sqrt(2.0 * j + 0.5);
        norm = 1.0;
        norm = raw(0.0);
    }
    double raw(double x) const {
        // Legendre recurrence (k+1) P_{k+1} = (2k+1) x P_k - k P_{k-1}; even orders are summed
        double pkm1 = 1.0, pk = x, s = coef[0];
        for (int k = 1; k < 2 * kTerms - 1; ++k) {
            double pkp1 = ((2 * k + 1) * x * pk - k * pkm1) / (k + 1);
            pkm1 = pk; pk = pkp1;
            if (((k + 1) & 1) == 0) s += coef[(k + 1) / 2] * pk;
        }
        return s / norm;
    }
    double operator()(double nu) const { return std::fabs(nu) < 1.0 ? raw(nu) : 0.0; }
};

const Pswf &pswf() { static Pswf p; return p; }

}  // namespace

void wpg_pswf_eval(const double *nu, int64_t n, double *out) {
    const Pswf &p = pswf();
    for (int64_t i = 0; i < n; ++i) out[i] = p(nu[i]);
}

extern "C" int wpg_taper(const double *h_nu, int64_t n, double *h_out) {
    if (n < 0 || (n > 0 && (!h_nu || !h_out))) return WPG_EINVAL;
    wpg_pswf_eval(h_nu, n, h_out);
    return WPG_OK;
}

static int nk_of(int S) { int nk = 32; while (nk < 4 * S) nk <<= 1; return nk; }

extern "C" int64_t wpg_wkernel_elems(int Nw, int support, int oversample) {
    if (Nw < 1 || support < 1 || oversample < 1) return 0;
    return (int64_t)Nw * oversample * oversample * support * support;
}

extern "C" int wpg_ragged_support(int Nw, double w_max, int grid_N, double cell, int oversample,
                                  int S_min, int S_max, int *sup, int64_t *off) {
    if (Nw < 1 || Nw > WPG_MAX_NW || !sup || !off || S_min < 1 || S_max < S_min || S_max > WPG_MAX_S ||
        oversample < 1 || !(cell > 0) || !(w_max >= 0) || grid_N < 2)
        return WPG_EINVAL;
    double fov = (double)grid_N * cell, dw = 2.0 * w_max / Nw;
    int64_t o = 0;
    for (int p = 0; p < Nw; ++p) {
        double wp = -w_max + (p + 0.5) * dw;                                 // K1
        double s = 2.0 * std::ceil(std::sqrt(9.0 + std::pow(std::fabs(wp) * fov * fov / 2.0, 2)));  // K6, m_t/2 = 3
        int S = (int)std::min<double>(std::max<double>(s, S_min), S_max);
        sup[p] = S;
        off[p] = o;
        o += (int64_t)oversample * oversample * S * S;
    }
    off[Nw] = o;
    return WPG_OK;
}

// ------------------------------------------------------------------------------------ device
namespace {

// K2: F[pl][b][a] = psi_b psi_a exp(2 pi i w (n - 1))
__global__ void fill_image_plane(double2 *__restrict__ F, const double *__restrict__ psi, int Nk, double fov,
                                 const double *__restrict__ wlist) {
    int a = blockIdx.x * blockDim.x + threadIdx.x, b = blockIdx.y, pl = blockIdx.z;
    if (a >= Nk) return;
    double l = (a - Nk / 2) * fov / Nk, m = (b - Nk / 2) * fov / Nk;
    double r2 = l * l + m * m;
    double2 v = make_double2(0.0, 0.0);
    if (r2 < 1.0) {
        double nm1 = -r2 / (1.0 + sqrt(1.0 - r2));
        double s, c;
        sincos(2.0 * M_PI * wlist[pl] * nm1, &s, &c);
        double t = psi[a] * psi[b];
        v = make_double2(t * c, t * s);
    }
    F[((size_t)pl * Nk + b) * Nk + a] = v;
}

// K3 twiddles: E[ti][a] = exp(-2 pi i t (a - Nk/2) / (Q Nk)), t = ti - S Q / 2 + 1 (exact integer phase)
__global__ void fill_twiddles(double2 *__restrict__ E, int SQ, int Nk, int Q) {
    int a = blockIdx.x * blockDim.x + threadIdx.x, ti = blockIdx.y;
    if (a >= Nk) return;
    long long t = ti - SQ / 2 + 1, period = (long long)Q * Nk;
    long long m = (t * (a - Nk / 2)) % period;
    double s, c;
    sincospi(-2.0 * (double)m / (double)period, &s, &c);
    E[(size_t)ti * Nk + a] = make_double2(c, s);
}

__device__ __forceinline__ double2 cmadd(double2 acc, double2 x, double2 y) {
    acc.x += x.x * y.x - x.y * y.y;
    acc.y += x.x * y.y + x.y * y.x;
    return acc;
}

// K3 stage 1: G[pl][b][tu] = sum_a F[pl][b][a] E[tu][a]
__global__ void dft_rows(const double2 *__restrict__ F, const double2 *__restrict__ E, double2 *__restrict__ G,
                         int Nk, int SQ) {
    int tu = blockIdx.x * blockDim.x + threadIdx.x, b = blockIdx.y, pl = blockIdx.z;
    if (tu >= SQ) return;
    const double2 *f = F + ((size_t)pl * Nk + b) * Nk, *e = E + (size_t)tu * Nk;
    double2 acc = make_double2(0.0, 0.0);
    for (int a = 0; a < Nk; ++a) acc = cmadd(acc, f[a], e[a]);
    G[((size_t)pl * Nk + b) * SQ + tu] = acc;
}

// K3 stage 2: Ct[pl][tv][tu] = sum_b E[tv][b] G[pl][b][tu]
__global__ void dft_cols(const double2 *__restrict__ G, const double2 *__restrict__ E, double2 *__restrict__ Ct,
                         int Nk, int SQ) {
    int tu = blockIdx.x * blockDim.x + threadIdx.x, tv = blockIdx.y, pl = blockIdx.z;
    if (tu >= SQ) return;
    const double2 *e = E + (size_t)tv * Nk;
    double2 acc = make_double2(0.0, 0.0);
    for (int b = 0; b < Nk; ++b) acc = cmadd(acc, e[b], G[((size_t)pl * Nk + b) * SQ + tu]);
    Ct[((size_t)pl * SQ + tv) * SQ + tu] = acc;
}

// K4 + K5: slice the table into K[p][ov][ou][iv][iu] and divide by s
template <typename C, typename T>
__global__ void slice_kernel(const double2 *__restrict__ Ct, C *__restrict__ K, const int *__restrict__ plane_off,
                             int S, int Q, double inv_s) {
    int SQ = S * Q, pl = blockIdx.y;
    int n = Q * Q * S * S;
    int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= n) return;
    int iu = idx % S, iv = (idx / S) % S, ou = (idx / (S * S)) % Q, ov = idx / (S * S * Q);
    int tvi = (iv + 1) * Q - ov - 1, tui = (iu + 1) * Q - ou - 1;        // t + S Q / 2 - 1
    double2 v = Ct[((size_t)pl * SQ + tvi) * SQ + tui];
    C o;
    o.x = (T)(v.x * inv_s); o.y = (T)(v.y * inv_s);
    K[(size_t)plane_off[pl] + idx] = o;
}

struct DevBuf {
    void *p = nullptr;
    ~DevBuf() { if (p) cudaFree(p); }
    cudaError_t alloc(size_t n) { return cudaMalloc(&p, n ? n : 1); }
};

}  // namespace

// Runs K2-K3 for `npl` w values with support S; leaves the tables in Ct (device, [npl][SQ][SQ]).
static int build_tables(wpg_ctx *ctx, int S, int Q, double fov, const std::vector<double> &wl, DevBuf &Ct) {
    int Nk = nk_of(S), SQ = S * Q, npl = (int)wl.size();
    std::vector<double> nu(Nk), psi(Nk);
    for (int a = 0; a < Nk; ++a) nu[a] = 2.0 * ((a - Nk / 2) * fov / Nk) / fov;
    wpg_pswf_eval(nu.data(), Nk, psi.data());
    DevBuf dpsi, dw, F, E, G;
    WPG_CUDA(ctx, dpsi.alloc(Nk * 8));
    WPG_CUDA(ctx, dw.alloc(npl * 8));
    WPG_CUDA(ctx, F.alloc((size_t)npl * Nk * Nk * 16));
    WPG_CUDA(ctx, E.alloc((size_t)SQ * Nk * 16));
    WPG_CUDA(ctx, G.alloc((size_t)npl * Nk * SQ * 16));
    WPG_CUDA(ctx, Ct.alloc((size_t)npl * SQ * SQ * 16));
    cudaStream_t s = ctx->stream;
    WPG_CUDA(ctx, cudaMemcpyAsync(dpsi.p, psi.data(), Nk * 8, cudaMemcpyHostToDevice, s));
    WPG_CUDA(ctx, cudaMemcpyAsync(dw.p, wl.data(), npl * 8, cudaMemcpyHostToDevice, s));
    fill_image_plane<<<dim3((Nk + 63) / 64, Nk, npl), 64, 0, s>>>((double2 *)F.p, (const double *)dpsi.p, Nk, fov, (const double *)dw.p);
    fill_twiddles<<<dim3((Nk + 63) / 64, SQ), 64, 0, s>>>((double2 *)E.p, SQ, Nk, Q);
    dft_rows<<<dim3((SQ + 127) / 128, Nk, npl), 128, 0, s>>>((const double2 *)F.p, (const double2 *)E.p, (double2 *)G.p, Nk, SQ);
    dft_cols<<<dim3((SQ + 127) / 128, SQ, npl), 128, 0, s>>>((const double2 *)G.p, (const double2 *)E.p, (double2 *)Ct.p, Nk, SQ);
    ctx->n_launches += 4;
    WPG_CUDA(ctx, cudaGetLastError());
    WPG_CUDA(ctx, cudaStreamSynchronize(s));      // the temporaries die with this scope
    return WPG_OK;
}

extern "C" int wpg_wkernel_build(wpg_ctx *ctx, const wpg_kdesc *desc, wpg_prec prec, void *d_out) {
    if (!ctx) return WPG_EINVAL;
    int rc = wpg_check_desc(ctx, desc);
    if (rc) return rc;
    if (!d_out) return wpg_fail(ctx, WPG_EINVAL, "output pointer is NULL");
    if (prec != WPG_F32 && prec != WPG_F64) return wpg_fail(ctx, WPG_EINVAL, "bad precision");
    WPG_DEVICE(ctx);
    const int Nw = desc->Nw, Q = desc->oversample;
    const double fov = (double)desc->grid_N * desc->cell, dw = 2.0 * desc->w_max / Nw;
    std::map<int, std::vector<int>> groups;                 // support -> planes
    int Smin = WPG_MAX_S + 1;
    std::vector<int64_t> off(Nw + 1, 0);
    for (int p = 0; p < Nw; ++p) {
        int S = desc->support ? desc->support[p] : desc->support_max;
        groups[S].push_back(p);
        Smin = std::min(Smin, S);
        off[p + 1] = off[p] + (int64_t)Q * Q * S * S;
    }
    // K5: s = Re(sum of the on-cell slice of the w = 0 table), support S_min
    double s_norm;
    {
        DevBuf Ct;
        rc = build_tables(ctx, Smin, Q, fov, std::vector<double>(1, 0.0), Ct);
        if (rc) return rc;
        int SQ = Smin * Q;
        std::vector<double> h((size_t)SQ * SQ * 2);
        WPG_CUDA(ctx, cudaMemcpy(h.data(), Ct.p, h.size() * 8, cudaMemcpyDeviceToHost));
        int o = (Smin % 2 == 0) ? 0 : Q / 2;
        double acc = 0.0;
        for (int iv = 0; iv < Smin; ++iv)
            for (int iu = 0; iu < Smin; ++iu)
                acc += h[2 * ((size_t)((iv + 1) * Q - o - 1) * SQ + ((iu + 1) * Q - o - 1))];
        s_norm = acc;
    }
    if (!(std::fabs(s_norm) > 0)) return wpg_fail(ctx, WPG_EINVAL, "kernel normalisation is zero");
    for (auto &g : groups) {
        int S = g.first, npl = (int)g.second.size();
        std::vector<double> wl(npl);
        std::vector<int> poff(npl);
        for (int i = 0; i < npl; ++i) {
            wl[i] = -desc->w_max + (g.second[i] + 0.5) * dw;                     // K1
            poff[i] = (int)off[g.second[i]];
        }
        DevBuf Ct, dpo;
        rc = build_tables(ctx, S, Q, fov, wl, Ct);
        if (rc) return rc;
        WPG_CUDA(ctx, dpo.alloc(npl * 4));
        WPG_CUDA(ctx, cudaMemcpyAsync(dpo.p, poff.data(), npl * 4, cudaMemcpyHostToDevice, ctx->stream));
        int n = Q * Q * S * S;
        dim3 gr((n + 255) / 256, npl);
        if (prec == WPG_F32)
            slice_kernel<float2, float><<<gr, 256, 0, ctx->stream>>>((const double2 *)Ct.p, (float2 *)d_out, (const int *)dpo.p, S, Q, 1.0 / s_norm);
        else
            slice_kernel<double2, double><<<gr, 256, 0, ctx->stream>>>((const double2 *)Ct.p, (double2 *)d_out, (const int *)dpo.p, S, Q, 1.0 / s_norm);
        ctx->n_launches += 1;
        WPG_CUDA(ctx, cudaGetLastError());
        WPG_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    }
    return WPG_OK;
}
