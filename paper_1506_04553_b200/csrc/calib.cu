// calib.cu -- calibration of the ALU roofline denominator:
// a pure-FFMA kernel with enough independent chains per thread to keep the FP32 pipe full.
// mode 0: scalar FFMA, mode 1: packed FFMA2 (two fp32 FMAs per issue slot), both with one vector
// register operand.  Modes 2-4 vary the operands of the FFMA2 (profiles/ffma2_operand_bandwidth_r1.md):
//   2: three distinct register pairs        v = w * u + v     (measured 2/3 of the rate of mode 1)
//   3: pair * scalar-broadcast + pair       v = w * s + v     (SASS operand Rs.F32)
//   4: two distinct register pairs          v = w * w + v
//   5: mode 2 as two scalar FFMAs            v.x = w.x * u.x + v.x, v.y likewise (three distinct registers each)
//   6: mode 3 as two scalar FFMAs            v.x = w.x * s + v.x,   v.y likewise
//   7: mode 2 with the first source shared by eight consecutive instructions (operand reuse cache: SASS .reuse)
// which is what decides the layout of the interaction lists in walk.cu.
// Not part of the hot path; bench.py quotes modes 0 and 1 beside the nominal peak.
#include "p3t_internal.cuh"

#define CALIB_CHAINS 16
#define CALIB_INNER 64

__device__ __forceinline__ u64 calib_ffma2(u64 a, u64 b, u64 c)
{
    u64 d;
    asm volatile("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ float calib_ffma(float a, float b, float c)
{
    float d;
    asm volatile("fma.rn.f32 %0, %1, %2, %3;" : "=f"(d) : "f"(a), "f"(b), "f"(c));
    return d;
}
__device__ __forceinline__ u64 calib_pack(float x, float y)
{
    u64 d;
    asm volatile("mov.b64 %0, {%1, %2};" : "=l"(d) : "f"(x), "f"(y));
    return d;
}

// operand-pattern variants: 8 independent chains, every source a distinct live register (pair)
template <int MODE>
__global__ void __launch_bounds__(128, 4) ffma2_operand_kernel(float *out, int iters, float a, float b)
{
    u64 v[8], w[8], u[8];
    float sc[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        v[k] = calib_pack(threadIdx.x * b + k, 1.f + k);
        w[k] = calib_pack(a + k * b, a - b * threadIdx.x * (k + 1));
        u[k] = calib_pack(b * (k + 1), b * threadIdx.x + k);
        sc[k] = a - b * (k + threadIdx.x);
    }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < CALIB_INNER * 2; ++r) {
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                if (MODE == 2) v[k] = calib_ffma2(w[k], u[k], v[k]);
                if (MODE == 3) v[k] = calib_ffma2(w[k], calib_pack(sc[k], sc[k]), v[k]);
                if (MODE == 4) v[k] = calib_ffma2(w[k], w[k], v[k]);
                if (MODE == 7) v[k] = calib_ffma2(w[r & 7], u[k], v[k]);
            }
        }
    }
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < 8; ++k) s += __uint_as_float((u32)v[k]) + __uint_as_float((u32)(v[k] >> 32));
    if (s == 123.456f) out[0] = s;
}

// the same operand patterns issued as scalar FFMAs (two per packed operation)
template <int MODE>
__global__ void __launch_bounds__(128, 4) ffma_operand_kernel(float *out, int iters, float a, float b)
{
    float vx[8], vy[8], wx[8], wy[8], ux[8], uy[8], sc[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        vx[k] = threadIdx.x * b + k, vy[k] = 1.f + k;
        wx[k] = a + k * b, wy[k] = a - b * threadIdx.x * (k + 1);
        ux[k] = b * (k + 1), uy[k] = b * threadIdx.x + k;
        sc[k] = a - b * (k + threadIdx.x);
    }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < CALIB_INNER * 2; ++r) {
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                if (MODE == 5) { vx[k] = calib_ffma(wx[k], ux[k], vx[k]); vy[k] = calib_ffma(wy[k], uy[k], vy[k]); }
                if (MODE == 6) { vx[k] = calib_ffma(wx[k], sc[k], vx[k]); vy[k] = calib_ffma(wy[k], sc[k], vy[k]); }
            }
        }
    }
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < 8; ++k) s += vx[k] + vy[k];
    if (s == 123.456f) out[0] = s;
}

template <int PACKED>
__global__ void __launch_bounds__(256) ffma_peak_kernel(float *out, int iters, float a, float b)
{
    float2 v[CALIB_CHAINS];
#pragma unroll
    for (int k = 0; k < CALIB_CHAINS; ++k) v[k] = make_float2(threadIdx.x * 1e-3f + k, blockIdx.x * 1e-3f - k);
    const float2 a2 = make_float2(a, a), b2 = make_float2(b, b);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < CALIB_INNER; ++r) {
#pragma unroll
            for (int k = 0; k < CALIB_CHAINS; ++k) {
                if (PACKED) v[k] = __ffma2_rn(v[k], a2, b2);
                else { v[k].x = fmaf(v[k].x, a, b); v[k].y = fmaf(v[k].y, a, b); }
            }
        }
    }
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < CALIB_CHAINS; ++k) s += v[k].x + v[k].y;
    if (s == 123.456f) out[0] = s;   // keeps the chains alive; practically never true
}

extern "C" p3t_status p3t_measure_fp32_peak(p3t_ctx *ctx, int packed, int iters, double *tflops, float *ms_out)
{
    if (!ctx || !tflops || iters <= 0) return p3t_fail(ctx, P3T_EINVAL, "p3t_measure_fp32_peak: bad argument");
    cudaStream_t s = ctx->stream;
    if (packed < 0 || packed > 7) return p3t_fail(ctx, P3T_EINVAL, "p3t_measure_fp32_peak: mode must be 0..7");
    const int grid = packed >= 2 ? ctx->sm_count * 16 : ctx->sm_count * 8, block = packed >= 2 ? 128 : 256;
    cudaEvent_t e0, e1;
    P3T_CUDA(ctx, cudaEventCreate(&e0));
    P3T_CUDA(ctx, cudaEventCreate(&e1));
    float *out = (float *)ctx->ws.scan_tmp;   // never written in practice
    float best = 1e30f;
    for (int rep = 0; rep < 5; ++rep) {       // rep 0 warms up
        P3T_CUDA(ctx, cudaEventRecord(e0, s));
        if (packed == 1) ffma_peak_kernel<1><<<grid, block, 0, s>>>(out, iters, 0.999f, 1e-3f);
        else if (packed == 0) ffma_peak_kernel<0><<<grid, block, 0, s>>>(out, iters, 0.999f, 1e-3f);
        else if (packed == 2) ffma2_operand_kernel<2><<<grid, block, 0, s>>>(out, iters, 0.999f, 1e-3f);
        else if (packed == 3) ffma2_operand_kernel<3><<<grid, block, 0, s>>>(out, iters, 0.999f, 1e-3f);
        else if (packed == 4) ffma2_operand_kernel<4><<<grid, block, 0, s>>>(out, iters, 0.999f, 1e-3f);
        else if (packed == 5) ffma_operand_kernel<5><<<grid, block, 0, s>>>(out, iters, 0.999f, 1e-3f);
        else if (packed == 6) ffma_operand_kernel<6><<<grid, block, 0, s>>>(out, iters, 0.999f, 1e-3f);
        else ffma2_operand_kernel<7><<<grid, block, 0, s>>>(out, iters, 0.999f, 1e-3f);
        P3T_CUDA(ctx, cudaEventRecord(e1, s));
        P3T_CUDA(ctx, cudaEventSynchronize(e1));
        float ms = 0.f;
        P3T_CUDA(ctx, cudaEventElapsedTime(&ms, e0, e1));
        if (rep > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    P3T_CUDA(ctx, cudaGetLastError());
    // modes 0/1: 16 chains x 64 packed ops; modes 2-6: 8 chains x 128 packed ops (or pairs of scalar ops) per outer iteration
    double flop = 2.0 * 2.0 * CALIB_CHAINS * CALIB_INNER * (double)iters * (double)grid * block;
    *tflops = flop / (best * 1e-3) / 1e12;
    if (ms_out) *ms_out = best;
    return P3T_OK;
}

// ------------------------------------------------------------------------------------------------
// Latency probes for the floor table of the a1-a6 chain (profiles/tree_latency_floor_r2.md): what one dependent round
// trip of the kind the look-back, climb and launch chains are made of costs on this device.
//   0  dependent loads that hit L2 (ld.global.cg through a strided cycle over 32 MiB of the workspace), one thread
//   1  dependent global atomics (atomicAdd whose result addresses the next one), one thread
//   2  back-to-back launches of an empty kernel on the stream (ns per launch)
//   3  the same with programmatic dependent launch (the attribute the a1-a6 chain uses)
//   4  release fence + relaxed atomic + dependent L2 load: one level of the moments climb
// ------------------------------------------------------------------------------------------------
#define LAT_LINES (1u << 18)          // 128-byte lines in the probe buffer (32 MiB)
#define LAT_STRIDE 40503u             // odd: i -> i + stride (mod 2^18) is one cycle through all lines

__global__ void lat_init_kernel(u32 *buf)
{
    const u32 i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < LAT_LINES) buf[(size_t)i * 32] = ((i + LAT_STRIDE) & (LAT_LINES - 1u)) * 32u;
}
template <int WHAT>
__global__ void lat_chase_kernel(u32 *buf, u32 steps, u32 *out)
{
    u32 p = 0;
    for (u32 k = 0; k < steps; ++k) {
        if (WHAT == 0) p = __ldcg(buf + p);
        if (WHAT == 1) p = atomicAdd(buf + p, 0u);
        if (WHAT == 4) { __threadfence(); atomicAdd(buf + p + 1, 1u); p = __ldcg(buf + p); }
    }
    out[0] = p;
}
__global__ void lat_empty_kernel(u32 *out)
{
    P3T_GRID_TRIGGER();
    P3T_GRID_WAIT();
    if (out == nullptr) printf("never\n");
}

extern "C" p3t_status p3t_measure_latency(p3t_ctx *ctx, int what, int iters, double *ns)
{
    if (!ctx || !ns || iters <= 0 || what < 0 || what > 4) return p3t_fail(ctx, P3T_EINVAL, "p3t_measure_latency: bad argument");
    if (ctx->ws.total_bytes < ((size_t)LAT_LINES * 128 + 4096)) return p3t_fail(ctx, P3T_ENOMEM, "p3t_measure_latency needs a workspace of 32 MiB (max_n >= 65536)");
    cudaStream_t s = ctx->stream;
    u32 *buf = reinterpret_cast<u32 *>(ctx->base);          // scratch use of the workspace: the context must be reloaded afterwards
    u32 *out = buf + (size_t)LAT_LINES * 32;
    ctx->loaded = ctx->built = ctx->evaluated = ctx->topo_valid = false;
    ctx->status_clean = ctx->tiles_ready = false;
    ctx->cells_dirty = true;
    cudaEvent_t e0, e1;
    P3T_CUDA(ctx, cudaEventCreate(&e0));
    P3T_CUDA(ctx, cudaEventCreate(&e1));
    float best = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {
        if (what == 0 || what == 1 || what == 4) {
            P3T_CUDA(ctx, cudaMemsetAsync(buf, 0, (size_t)LAT_LINES * 128, s));
            lat_init_kernel<<<LAT_LINES / 256, 256, 0, s>>>(buf);
        }
        P3T_CUDA(ctx, cudaEventRecord(e0, s));
        if (what == 0) lat_chase_kernel<0><<<1, 1, 0, s>>>(buf, (u32)iters, out);
        else if (what == 1) lat_chase_kernel<1><<<1, 1, 0, s>>>(buf, (u32)iters, out);
        else if (what == 4) lat_chase_kernel<4><<<1, 1, 0, s>>>(buf, (u32)iters, out);
        else
            for (int k = 0; k < iters; ++k) {
                if (what == 2) lat_empty_kernel<<<148, 128, 0, s>>>(out);
                else P3T_CUDA(ctx, p3t_launch_pdl(lat_empty_kernel, dim3(148), dim3(128), 0, s, out));
            }
        P3T_CUDA(ctx, cudaEventRecord(e1, s));
        P3T_CUDA(ctx, cudaEventSynchronize(e1));
        float ms = 0.f;
        P3T_CUDA(ctx, cudaEventElapsedTime(&ms, e0, e1));
        if (rep > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    P3T_CUDA(ctx, cudaGetLastError());
    // the hilbert tables live in the workspace the probe has scribbled over
    {
        static u32 tab[P3T_HILBERT_TAB_WORDS];
        if (!p3t_hilbert_tables(tab)) return p3t_fail(ctx, P3T_ECUDA, "hilbert tables");
        P3T_CUDA(ctx, cudaMemcpyAsync(ctx->ws.hilbert_tab, tab, sizeof(tab), cudaMemcpyHostToDevice, s));
        P3T_CUDA(ctx, cudaMemsetAsync(ctx->ws.order_meta, 0, 4 * sizeof(u32), s));
        P3T_CUDA(ctx, cudaMemsetAsync(ctx->ws.body_class, 0, ctx->max_n * sizeof(u32), s));
        P3T_CUDA(ctx, cudaMemsetAsync(ctx->ws.counters, 0, CNT_WORDS * sizeof(u64), s));
        P3T_CUDA(ctx, cudaStreamSynchronize(s));
    }
    *ns = (double)best * 1e6 / (double)iters;
    return P3T_OK;
}
