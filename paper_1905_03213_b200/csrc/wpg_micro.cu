// Microbenchmarks of the machine limits the gridder is read against ("fractions of
// MEASURED peaks"): the global reduction rate (the ceiling of the naive one-atomic-per-update design and of the
// paper's own kernel), the L1 coefficient feed (one LDG.128 per two fp32 updates), and the packed
// FP32 / FP64 FMA issue rates.  Instrumentation only: nothing on the gridding path calls these.
#include "wpg_common.h"

namespace {

// which = 0: red.global.add.v2.f32, consecutive lanes -> consecutive cells, every warp its own 256-byte segment
//            picked pseudo-randomly in the buffer (the naive gridder's pattern: a window row per 8 lanes);
// which = 1: the same instruction, every LANE its own pseudo-random cell (worst case);
__global__ void __launch_bounds__(256)
micro_red_kernel(float2 *__restrict__ buf, unsigned ncell_mask, int iters, int scattered) {
    const unsigned gtid = blockIdx.x * 256u + threadIdx.x;
    const unsigned lane = threadIdx.x & 31u, gwarp = gtid >> 5;
    unsigned x = (scattered ? gtid : gwarp) * 2654435761u + 12345u;
    for (int i = 0; i < iters; ++i) {
        x = x * 1664525u + 1013904223u;
        const unsigned cell = scattered ? ((x >> 4) & ncell_mask) : ((((x >> 4) & ncell_mask) & ~31u) + lane);
        asm volatile("red.global.add.v2.f32 [%0], {%1, %2};" ::"l"(buf + cell), "f"(1.0f), "f"(0.5f) : "memory");
    }
}

// which = 2: L1-resident LDG.128: every warp re-reads its own eight 512-byte slices (32 lanes x 16 B each; 4 KB per
// warp, 16 warps per SM), 8 loads in flight; the slice order rotates with the trip count so that the read-only
// loads can be neither merged nor hoisted
__global__ void __launch_bounds__(256)
micro_l1_kernel(const float4 *src, float *sink, int iters) {
    const unsigned gwarp = (blockIdx.x * 256u + threadIdx.x) >> 5, lane = threadIdx.x & 31u;
    const float4 *p = src + (size_t)(gwarp & 4095u) * 256u + lane;
    float acc = 0.f;
    for (int i = 0; i < iters; ++i) {
        float4 v[8];
#pragma unroll
        for (int k = 0; k < 8; ++k)
            asm volatile("ld.global.nc.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v[k].x), "=f"(v[k].y), "=f"(v[k].z), "=f"(v[k].w) : "l"(p + ((i + k) & 7) * 32));
#pragma unroll
        for (int k = 0; k < 8; ++k) acc += v[k].x + v[k].w;
    }
    if (acc == 123.456f) sink[0] = acc;
}

// which = 3: fma.rn.f32x2 issue rate, 8 independent accumulator pairs per thread
__global__ void __launch_bounds__(256)
micro_ffma2_kernel(float *__restrict__ sink, int iters, float seed) {
    unsigned long long a[8], b, c;
    asm("mov.b64 %0, {%1, %2};" : "=l"(b) : "f"(seed), "f"(seed + 1.f));
    asm("mov.b64 %0, {%1, %1};" : "=l"(c) : "f"(0.999f));
#pragma unroll
    for (int k = 0; k < 8; ++k) asm("mov.b64 %0, {%1, %2};" : "=l"(a[k]) : "f"((float)k), "f"(seed));
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int k = 0; k < 8; ++k) asm volatile("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(a[k]) : "l"(b), "l"(c));
    }
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < 8; ++k) { float x, y; asm("mov.b64 {%0, %1}, %2;" : "=f"(x), "=f"(y) : "l"(a[k])); s += x + y; }
    if (s == 123.456f) sink[0] = s;
}

// which = 4: fma.rn.f64 issue rate, 8 independent accumulators per thread
__global__ void __launch_bounds__(256)
micro_dfma_kernel(double *__restrict__ sink, int iters, double seed) {
    double a[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) a[k] = seed + k;
    const double b = seed * 0.5, c = 0.999;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int k = 0; k < 8; ++k) a[k] = fma(a[k], c, b);
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < 8; ++k) s += a[k];
    if (s == 123.456) sink[0] = s;
}

// which = 5 / 6: the same row-segment reductions as which = 0, issued as ONE bulk reduction per segment by the copy
// engine (cp.reduce.async.bulk.global.shared::cta.add.f32): the lanes stage the sums in shared memory, one lane issues.
// 5: 256-byte segments (32 cells, like which = 0); 6: 64-byte segments (8 cells: one window row at S = 8).
__global__ void __launch_bounds__(256)
micro_bulkred_kernel(float2 *__restrict__ buf, unsigned ncell_mask, int iters, int cells) {
    __shared__ __align__(128) float2 stage[8][4][32];              // per warp: ring of four staging rows
    const unsigned gtid = blockIdx.x * 256u + threadIdx.x;
    const unsigned lane = threadIdx.x & 31u, gwarp = gtid >> 5, w = threadIdx.x >> 5;
    unsigned x = gwarp * 2654435761u + 12345u;
    for (int i = 0; i < iters; ++i) {
        x = x * 1664525u + 1013904223u;
        const unsigned cell = ((x >> 4) & ncell_mask) & ~31u;
        float2 *row = stage[w][i & 3];
        if ((i & 3) == 0 && i) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");   // the ring's rows are free again
        __syncwarp();
        if ((int)lane < cells) row[lane] = make_float2(1.0f, 0.5f);
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncwarp();
        if (lane == 0) {
            asm volatile("cp.reduce.async.bulk.global.shared::cta.bulk_group.add.f32 [%0], [%1], %2;"
                         ::"l"(buf + cell), "r"((unsigned)__cvta_generic_to_shared(row)), "r"(cells * 8) : "memory");
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        }
    }
    asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
}

// which = 7 / 8: the inner loop of a shared-memory-staged subgrid accumulator (SURVEY.md §8 north_star's alternative
// to register accumulation): a CTA owns a 64 x 64-cell tile plus the S - 1 = 7 halo in shared memory (72-cell rows);
// per trip every warp takes one "record" - an L1-resident 512-byte coefficient slice as in which = 2, a window start
// picked pseudo-randomly in the tile - and adds its 64 products into the tile, lane <-> (window row, cell pair).
// 7: red.shared.add.f32 (correct whoever else touches the cells); 8: plain 8-byte load / FFMA2 / store, i.e. the
// ceiling of a scheme that needs no atomics because one warp owns the tile (the write races here are deliberate).
__global__ void __launch_bounds__(256)
micro_subgrid_kernel(const float4 *src, float2 *sink, int iters, int atomic) {
    constexpr int kRow = 72, kCells = 71 * kRow;
    extern __shared__ float2 tile[];
    for (int i = threadIdx.x; i < kCells; i += 256) tile[i] = make_float2(0.f, 0.f);
    __syncthreads();
    const unsigned gwarp = (blockIdx.x * 256u + threadIdx.x) >> 5, lane = threadIdx.x & 31u;
    const float4 *p = src + (size_t)(gwarp & 4095u) * 256u + lane;
    const unsigned r = lane >> 2, c = (lane & 3u) * 2u;
    unsigned x = gwarp * 2654435761u + 12345u;
    const float vr = 1.0f + (float)lane, vi = 0.5f;
    for (int i = 0; i < iters; ++i) {
        x = x * 1664525u + 1013904223u;
        float4 k;
        asm volatile("ld.global.nc.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(k.x), "=f"(k.y), "=f"(k.z), "=f"(k.w) : "l"(p + (i & 7) * 32));
        float2 *cell = tile + (((x >> 8) & 63u) + r) * kRow + ((x >> 16) & 63u) + c;
        const float a0 = vr * k.x - vi * k.y, b0 = vr * k.y + vi * k.x, a1 = vr * k.z - vi * k.w, b1 = vr * k.w + vi * k.z;
        if (atomic) {
            atomicAdd(&cell[0].x, a0); atomicAdd(&cell[0].y, b0);
            atomicAdd(&cell[1].x, a1); atomicAdd(&cell[1].y, b1);
        } else {
            float2 t0 = cell[0], t1 = cell[1];
            t0.x += a0; t0.y += b0; t1.x += a1; t1.y += b1;
            cell[0] = t0; cell[1] = t1;
        }
    }
    __syncthreads();
    float2 acc = make_float2(0.f, 0.f);
    for (int i = threadIdx.x; i < kCells; i += 256) { acc.x += tile[i].x; acc.y += tile[i].y; }
    if (acc.x == 123.456f) sink[0] = acc;
}

// which = 9: the same 16-byte loads as which = 2, but every trip a warp reads a 512-byte slice (32 lanes x 16 B, four
// whole 128-byte lines) at a pseudo-random place of a buffer that fits the L2 and not the L1 (32 MiB), 8 loads in
// flight: the coefficient feed when the slices do NOT stay in L1 — what the gridder sees, ncu: 8 % L1 hit rate at
// S = 12 (a 2.4 MB stack streamed through a 200 KB cache), each missing line costing a second data-pipe wavefront.
__global__ void __launch_bounds__(256)
micro_l2_kernel(const float4 *src, float *sink, int iters, unsigned slice_mask) {
    const unsigned gwarp = (blockIdx.x * 256u + threadIdx.x) >> 5, lane = threadIdx.x & 31u;
    unsigned x = gwarp * 2654435761u + 12345u;
    float acc = 0.f;
    for (int i = 0; i < iters; ++i) {
        float4 v[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            x = x * 1664525u + 1013904223u;
            const float4 *p = src + (size_t)((x >> 8) & slice_mask) * 32u + lane;
            asm volatile("ld.global.nc.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v[k].x), "=f"(v[k].y), "=f"(v[k].z), "=f"(v[k].w) : "l"(p));
        }
#pragma unroll
        for (int k = 0; k < 8; ++k) acc += v[k].x + v[k].w;
    }
    if (acc == 123.456f) sink[0] = acc;
}

}  // namespace

// h_out[0] = operations per second (reductions of one cell, 16-byte loads, packed FMAs = 2 FMA, FMAs, grid updates),
// h_out[1] = kernel milliseconds.  d_buf: device scratch of at least buf_bytes >= 1 MiB (power of two used).
extern "C" int wpg_microbench(wpg_ctx *ctx, int which, int iters, void *d_buf, size_t buf_bytes, double *h_out) {
    if (!ctx || !h_out || !d_buf) return WPG_EINVAL;
    if (which < 0 || which > 9 || iters < 1 || buf_bytes < ((size_t)1 << 20))
        return wpg_fail(ctx, WPG_EINVAL, "wpg_microbench: which 0..9, iters >= 1, buffer >= 1 MiB");
    WPG_DEVICE(ctx);
    size_t ncell = 1;
    while (ncell * 2 * sizeof(float2) <= buf_bytes) ncell *= 2;
    if ((which == 2 || which >= 7) && buf_bytes < ((size_t)16 << 20))
        return wpg_fail(ctx, WPG_EINVAL, "wpg_microbench: which = 2, 7, 8, 9 need a 16 MiB buffer");
    const int blocks = ctx->sm_count * (which == 2 ? 2 : which == 9 ? 6 : which >= 7 ? 4 : 8);
    constexpr int kSubgridBytes = 71 * 72 * (int)sizeof(float2);
    if (which >= 7) WPG_CUDA(ctx, cudaFuncSetAttribute(micro_subgrid_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kSubgridBytes));
    cudaEvent_t e0, e1;
    WPG_CUDA(ctx, cudaEventCreate(&e0));
    WPG_CUDA(ctx, cudaEventCreate(&e1));
    cudaStream_t s = ctx->stream;
    for (int rep = 0; rep < 2; ++rep) {            // the first repetition warms up
        WPG_CUDA(ctx, cudaEventRecord(e0, s));
        if (which <= 1) micro_red_kernel<<<blocks, 256, 0, s>>>((float2 *)d_buf, (unsigned)(ncell - 1), iters, which);
        else if (which == 2) micro_l1_kernel<<<blocks, 256, 0, s>>>((const float4 *)d_buf, (float *)d_buf, iters);
        else if (which == 3) micro_ffma2_kernel<<<blocks, 256, 0, s>>>((float *)d_buf, iters, 1.0f);
        else if (which == 9) {                       // slices of 512 bytes in the largest power of two <= min(buffer, 32 MiB)
            size_t nsl = 1;
            while (nsl * 2 * 512 <= buf_bytes && nsl * 2 * 512 <= ((size_t)32 << 20)) nsl *= 2;
            micro_l2_kernel<<<blocks, 256, 0, s>>>((const float4 *)d_buf, (float *)d_buf, iters, (unsigned)(nsl - 1));
        }
        else if (which >= 7) micro_subgrid_kernel<<<blocks, 256, kSubgridBytes, s>>>((const float4 *)d_buf, (float2 *)d_buf, iters, which == 7);
        else if (which >= 5) micro_bulkred_kernel<<<blocks, 256, 0, s>>>((float2 *)d_buf, (unsigned)(ncell - 1), iters, which == 5 ? 32 : 8);
        else micro_dfma_kernel<<<blocks, 256, 0, s>>>((double *)d_buf, iters, 1.0);
        WPG_CUDA(ctx, cudaEventRecord(e1, s));
        ctx->n_launches += 1;
    }
    WPG_CUDA(ctx, cudaEventSynchronize(e1));
    float ms = 0.f;
    WPG_CUDA(ctx, cudaEventElapsedTime(&ms, e0, e1));
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    WPG_CUDA(ctx, cudaGetLastError());
    const double threads = (double)blocks * 256.0;
    // reductions of one cell (0, 1: one per lane; 5, 6: 32 or 8 per warp), else 8 operations per thread and trip
    const double ops = which == 9 ? threads * (double)iters * 8.0                   // 9: 16-byte loads
                     : which >= 7 ? threads / 32.0 * (double)iters * 64.0           // 7, 8: grid updates (64 per record)
                     : which >= 5 ? threads / 32.0 * (double)iters * (which == 5 ? 32.0 : 8.0)
                                  : threads * (double)iters * (which == 0 || which == 1 ? 1.0 : 8.0);
    h_out[0] = ops / (ms * 1e-3);
    h_out[1] = ms;
    return WPG_OK;
}
