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

// psi(nu_j), nu_j = 2 (j - n/2) step, j = 0 .. n-1, on the device: the same Legendre series (coefficients by value),
// so that neither the kernel stack nor the dirty image needs a host table, a copy or a synchronisation.
namespace {
struct PswfCoef { double coef[Pswf::kTerms]; double norm; };
__global__ void pswf_kernel(double *__restrict__ out, int n, double step, const __grid_constant__ PswfCoef P) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n) return;
    const double x = 2.0 * ((double)(j - n / 2) * step);
    double v = 0.0;
    if (fabs(x) < 1.0) {
        double pkm1 = 1.0, pk = x, s = P.coef[0];
        for (int k = 1; k < 2 * Pswf::kTerms - 1; ++k) {
            const double pkp1 = ((2 * k + 1) * x * pk - k * pkm1) / (k + 1);
            pkm1 = pk; pk = pkp1;
            if (((k + 1) & 1) == 0) s += P.coef[(k + 1) / 2] * pk;
        }
        v = s / P.norm;
    }
    out[j] = v;
}
}  // namespace

int wpg_launch_taper(wpg_ctx *ctx, double *d_out, int n, double step) {
    PswfCoef c;
    const Pswf &p = pswf();
    for (int j = 0; j < Pswf::kTerms; ++j) c.coef[j] = p.coef[j];
    c.norm = p.norm;
    pswf_kernel<<<(n + 127) / 128, 128, 0, ctx->stream>>>(d_out, n, step, c);
    ctx->n_launches += 1;
    WPG_CUDA(ctx, cudaGetLastError());
    return WPG_OK;
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

// planes of one support group: index of the plane in the stack and element offset of its slices
struct GroupTab { int npl; int plane[WPG_MAX_NW]; int poff[WPG_MAX_NW]; };

// K1 + K2: F[pl][b][a] = psi_b psi_a exp(2 pi i w_p (n - 1)),  w_p = -w_max + (plane + 1/2) dw  (plane < 0: w = 0)
__global__ void fill_image_plane(double2 *__restrict__ F, const double *__restrict__ psi, int Nk, double fov,
                                 double w_max, double dw, const __grid_constant__ GroupTab G) {
    int a = blockIdx.x * blockDim.x + threadIdx.x, b = blockIdx.y, pl = blockIdx.z;
    if (a >= Nk) return;
    const int plane = G.plane[pl];
    const double wp = plane < 0 ? 0.0 : -w_max + (plane + 0.5) * dw;
    double l = (a - Nk / 2) * fov / Nk, m = (b - Nk / 2) * fov / Nk;
    double r2 = l * l + m * m;
    double2 v = make_double2(0.0, 0.0);
    if (r2 < 1.0) {
        double nm1 = -r2 / (1.0 + sqrt(1.0 - r2));
        double s, c;
        sincos(2.0 * M_PI * wp * nm1, &s, &c);
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

// K5: 1 / s, s = Re(sum of the on-cell slice of the w = 0 table, support S) — one block, on the device, so that the
// build needs no read-back.
__global__ void __launch_bounds__(256)
norm_kernel(const double2 *__restrict__ Ct, int S, int Q, double *__restrict__ inv_s) {
    __shared__ double part[256];
    const int SQ = S * Q, o = (S % 2 == 0) ? 0 : Q / 2;
    double acc = 0.0;
    for (int c = threadIdx.x; c < S * S; c += 256) {
        const int iv = c / S, iu = c - iv * S;
        acc += Ct[(size_t)((iv + 1) * Q - o - 1) * SQ + ((iu + 1) * Q - o - 1)].x;
    }
    part[threadIdx.x] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {              // fixed order: the scalar is reproducible
        double s = 0.0;
        for (int i = 0; i < 256; ++i) s += part[i];
        *inv_s = 1.0 / s;
    }
}

// K4 + K5: slice the table into K[p][ov][ou][iv][iu] and divide by s
template <typename C, typename T>
__global__ void slice_kernel(const double2 *__restrict__ Ct, C *__restrict__ K, const __grid_constant__ GroupTab G,
                             int S, int Q, const double *__restrict__ inv_s_ptr) {
    int SQ = S * Q, pl = blockIdx.y;
    int n = Q * Q * S * S;
    int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= n) return;
    const double inv_s = *inv_s_ptr;
    int iu = idx % S, iv = (idx / S) % S, ou = (idx / (S * S)) % Q, ov = idx / (S * S * Q);
    int tvi = (iv + 1) * Q - ov - 1, tui = (iu + 1) * Q - ou - 1;        // t + S Q / 2 - 1
    double2 v = Ct[((size_t)pl * SQ + tvi) * SQ + tui];
    C o;
    o.x = (T)(v.x * inv_s); o.y = (T)(v.y * inv_s);
    K[(size_t)G.poff[pl] + idx] = o;
}

static size_t al256(size_t x) { return (x + 255) & ~(size_t)255; }

// workspace of one table build: psi[Nk], F[npl][Nk][Nk], E[SQ][Nk], G[npl][Nk][SQ], Ct[npl][SQ][SQ]
struct TableLayout { size_t psi, F, E, G, Ct, total; int Nk, SQ; };
static TableLayout table_layout(int S, int Q, int npl) {
    TableLayout L{};
    L.Nk = nk_of(S); L.SQ = S * Q;
    size_t o = 0;
    L.psi = o; o += al256((size_t)L.Nk * 8);
    L.F = o;   o += al256((size_t)npl * L.Nk * L.Nk * 16);
    L.E = o;   o += al256((size_t)L.SQ * L.Nk * 16);
    L.G = o;   o += al256((size_t)npl * L.Nk * L.SQ * 16);
    L.Ct = o;  o += al256((size_t)npl * L.SQ * L.SQ * 16);
    L.total = o;
    return L;
}

}  // namespace

// Runs K1-K3 for the planes of G with support S in the workspace region w; the tables end up at w + L.Ct.
static int build_tables(wpg_ctx *ctx, int S, int Q, double fov, double w_max, double dw, const GroupTab &G, char *w,
                        const TableLayout &L) {
    const int Nk = L.Nk, SQ = L.SQ, npl = G.npl;
    cudaStream_t s = ctx->stream;
    int rc = wpg_launch_taper(ctx, (double *)(w + L.psi), Nk, 1.0 / Nk);          // nu_a = 2 (a - Nk/2) / Nk
    if (rc) return rc;
    fill_image_plane<<<dim3((Nk + 63) / 64, Nk, npl), 64, 0, s>>>((double2 *)(w + L.F), (const double *)(w + L.psi), Nk, fov, w_max, dw, G);
    fill_twiddles<<<dim3((Nk + 63) / 64, SQ), 64, 0, s>>>((double2 *)(w + L.E), SQ, Nk, Q);
    dft_rows<<<dim3((SQ + 127) / 128, Nk, npl), 128, 0, s>>>((const double2 *)(w + L.F), (const double2 *)(w + L.E), (double2 *)(w + L.G), Nk, SQ);
    dft_cols<<<dim3((SQ + 127) / 128, SQ, npl), 128, 0, s>>>((const double2 *)(w + L.G), (const double2 *)(w + L.E), (double2 *)(w + L.Ct), Nk, SQ);
    ctx->n_launches += 4;
    WPG_CUDA(ctx, cudaGetLastError());
    return WPG_OK;
}

// support groups of a stack: support -> planes (ascending support)
static void support_groups(const wpg_kdesc *desc, std::map<int, std::vector<int>> &groups, std::vector<int64_t> &off, int &Smin) {
    const int Nw = desc->Nw, Q = desc->oversample;
    Smin = WPG_MAX_S + 1;
    off.assign(Nw + 1, 0);
    for (int p = 0; p < Nw; ++p) {
        int S = desc->support ? desc->support[p] : desc->support_max;
        groups[S].push_back(p);
        Smin = std::min(Smin, S);
        off[p + 1] = off[p] + (int64_t)Q * Q * S * S;
    }
}

extern "C" size_t wpg_wkernel_workspace_bytes(const wpg_kdesc *desc) {
    wpg_ctx tmp;
    if (wpg_check_desc(&tmp, desc)) return 0;
    std::map<int, std::vector<int>> groups; std::vector<int64_t> off; int Smin;
    support_groups(desc, groups, off, Smin);
    size_t need = table_layout(Smin, desc->oversample, 1).total;
    for (auto &g : groups) need = std::max(need, table_layout(g.first, desc->oversample, (int)g.second.size()).total);
    return 256 + need;
}

extern "C" int wpg_wkernel_build(wpg_ctx *ctx, const wpg_kdesc *desc, wpg_prec prec, void *d_out, void *d_workspace,
                                 size_t workspace_bytes) {
    if (!ctx) return WPG_EINVAL;
    int rc = wpg_check_desc(ctx, desc);
    if (rc) return rc;
    if (!d_out) return wpg_fail(ctx, WPG_EINVAL, "output pointer is NULL");
    if (prec != WPG_F32 && prec != WPG_F64) return wpg_fail(ctx, WPG_EINVAL, "bad precision");
    const size_t need = wpg_wkernel_workspace_bytes(desc);
    if (!d_workspace || workspace_bytes < need)
        return wpg_fail(ctx, WPG_ENOMEM, "workspace of %zu bytes given, %zu needed", workspace_bytes, need);
    WPG_DEVICE(ctx);
    const int Nw = desc->Nw, Q = desc->oversample;
    const double fov = (double)desc->grid_N * desc->cell, dw = 2.0 * desc->w_max / Nw;
    std::map<int, std::vector<int>> groups; std::vector<int64_t> off; int Smin;
    support_groups(desc, groups, off, Smin);
    // The workspace is used by one table build after the other; the stream orders them.
    double *inv_s = (double *)d_workspace;
    char *w = (char *)d_workspace + 256;
    {   // K5: s from the w = 0 table of support S_min
        GroupTab G{}; G.npl = 1; G.plane[0] = -1;
        const TableLayout L = table_layout(Smin, Q, 1);
        rc = build_tables(ctx, Smin, Q, fov, desc->w_max, dw, G, w, L);
        if (rc) return rc;
        norm_kernel<<<1, 256, 0, ctx->stream>>>((const double2 *)(w + L.Ct), Smin, Q, inv_s);
        ctx->n_launches += 1;
    }
    for (auto &g : groups) {
        const int S = g.first, npl = (int)g.second.size();
        GroupTab G{}; G.npl = npl;
        for (int i = 0; i < npl; ++i) { G.plane[i] = g.second[i]; G.poff[i] = (int)off[g.second[i]]; }
        const TableLayout L = table_layout(S, Q, npl);
        rc = build_tables(ctx, S, Q, fov, desc->w_max, dw, G, w, L);
        if (rc) return rc;
        const int n = Q * Q * S * S;
        dim3 gr((n + 255) / 256, npl);
        if (prec == WPG_F32)
            slice_kernel<float2, float><<<gr, 256, 0, ctx->stream>>>((const double2 *)(w + L.Ct), (float2 *)d_out, G, S, Q, inv_s);
        else
            slice_kernel<double2, double><<<gr, 256, 0, ctx->stream>>>((const double2 *)(w + L.Ct), (double2 *)d_out, G, S, Q, inv_s);
        ctx->n_launches += 1;
        WPG_CUDA(ctx, cudaGetLastError());
    }
    return WPG_OK;
}
