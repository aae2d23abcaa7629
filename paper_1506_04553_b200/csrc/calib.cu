// calib.cu -- calibration of the ALU roofline denominator:
// a pure-FFMA kernel with enough independent chains per thread to keep the FP32 pipe full.
// mode 0: scalar FFMA, mode 1: packed FFMA2 (two fp32 FMAs per issue slot), both with one vector
// register operand.  Modes 2-4 vary the operands of the FFMA2 (profiles/ffma2_operand_bandwidth_r1.md):
//   2: three distinct register pairs        v = w * u + v     (measured 2/3 of the rate of mode 1)
//   3: pair * scalar-broadcast + pair       v = w * s + v     (SASS operand Rs.F32)
//   4: two distinct register pairs          v = w * w + v
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
            }
        }
    }
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < 8; ++k) s += __uint_as_float((u32)v[k]) + __uint_as_float((u32)(v[k] >> 32));
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
    if (packed < 0 || packed > 4) return p3t_fail(ctx, P3T_EINVAL, "p3t_measure_fp32_peak: mode must be 0..4");
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
        else ffma2_operand_kernel<4><<<grid, block, 0, s>>>(out, iters, 0.999f, 1e-3f);
        P3T_CUDA(ctx, cudaEventRecord(e1, s));
        P3T_CUDA(ctx, cudaEventSynchronize(e1));
        float ms = 0.f;
        P3T_CUDA(ctx, cudaEventElapsedTime(&ms, e0, e1));
        if (rep > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    P3T_CUDA(ctx, cudaGetLastError());
    // modes 0/1: 16 chains x 64 packed ops; modes 2-4: 8 chains x 128 packed ops per outer iteration
    double flop = 2.0 * 2.0 * CALIB_CHAINS * CALIB_INNER * (double)iters * (double)grid * block;
    *tflops = flop / (best * 1e-3) / 1e12;
    if (ms_out) *ms_out = best;
    return P3T_OK;
}
