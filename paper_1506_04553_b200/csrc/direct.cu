// direct.cu -- verification entry p3t_eval_direct: brute-force O(N n_subset) soft force with the
// same pair terms as the tree path's slow loop (Eq. 6, 8 of PAPER.md, K of Eq. 12, W of Eq. 16-17)
// and the same neighbour rule (s_ij < h, j != i by index).  fp32 pair arithmetic, one fp64 add per
// tile of 128 sources.  Not on the timed hot path.
#include "p3t_internal.cuh"

#define DIRECT_THREADS 128

__global__ void __launch_bounds__(DIRECT_THREADS) direct_kernel(const float4 *__restrict__ body_user, u32 n,
                                                                const u32 *__restrict__ subset, u32 ns, P3TParams prm,
                                                                float4 *__restrict__ accpot, u32 *__restrict__ nbr_count,
                                                                uint2 *pairs, u64 pair_cap, u64 *counters,
                                                                const u8 *__restrict__ cls_user)
{
    __shared__ float4 s_b[DIRECT_THREADS];
    __shared__ u8 s_c[DIRECT_THREADS];
    const u32 k = blockIdx.x * DIRECT_THREADS + threadIdx.x;
    const bool active = k < ns;
    const u32 i = active ? (subset ? subset[k] : k) : 0u;
    const float4 bi = body_user[i];
    const u32 ci = cls_user ? (cls_user[i] & 1u) : 0u;    // pair classes: kind of a pair = ci + cj
    double ax = 0.0, ay = 0.0, az = 0.0, ph = 0.0;
    u32 cnt = 0;
    u64 npairs = 0;
    for (u32 j0 = 0; j0 < n; j0 += DIRECT_THREADS) {
        u32 jl = j0 + threadIdx.x;
        s_b[threadIdx.x] = jl < n ? body_user[jl] : make_float4(0.f, 0.f, 0.f, 0.f);
        s_c[threadIdx.x] = (cls_user && jl < n) ? (cls_user[jl] & 1u) : 0u;
        __syncthreads();
        u32 lim = min((u32)DIRECT_THREADS, n - j0);
        float fx = 0.f, fy = 0.f, fz = 0.f, fp = 0.f;
        if (active) {
            for (u32 jj = 0; jj < lim; ++jj) {
                u32 j = j0 + jj;
                if (j == i) continue;
                float4 bj = s_b[jj];
                float dx = bj.x - bi.x, dy = bj.y - bi.y, dz = bj.z - bi.z;
                float s2 = fmaf(dx, dx, fmaf(dy, dy, fmaf(dz, dz, prm.eps2)));
                float rinv = rsqrtf(s2);
                float mrinv = bj.w * rinv;
                float mr3 = mrinv * (rinv * rinv);
                float K = 1.f, W = 1.f;
                const u32 kind = ci + s_c[jj];
                if (kind == 2u) { K = 0.f; W = 0.f; }                   // two black holes: not split, all of it hard
                if (kind == 2u || s2 < prm.h2_k[kind & 1u]) {
                    if (kind < 2u && s2 < prm.rout2_k[kind]) p3t_pair_weights(prm.cs[kind], s2, K, W);
                    u64 pos = atomicAdd(&counters[CNT_PAIRS], 1ull);
                    if (pos < pair_cap) pairs[pos] = make_uint2(i, j);
                    ++cnt;
                }
                mr3 *= K;
                fx = fmaf(mr3, dx, fx); fy = fmaf(mr3, dy, fy); fz = fmaf(mr3, dz, fz);
                fp = fmaf(W, mrinv, fp);
                ++npairs;
            }
        }
        ax += (double)fx; ay += (double)fy; az += (double)fz; ph += (double)fp;
        __syncthreads();
    }
    if (active) {
        accpot[i] = make_float4((float)ax, (float)ay, (float)az, (float)(-ph));
        nbr_count[i] = cnt;
        atomicAdd(&counters[CNT_NPP], npairs);
    }
}

p3t_status p3t_stage_direct(p3t_ctx *ctx, const u32 *d_subset, size_t n_subset)
{
    Workspace &w = ctx->ws;
    cudaStream_t s = ctx->stream;
    u32 n = (u32)ctx->n;
    P3T_CUDA(ctx, cudaMemsetAsync(w.counters + CNT_NPP, 0, 8 * sizeof(u64), s));
    P3T_CUDA(ctx, cudaMemsetAsync(w.accpot, 0, (size_t)n * sizeof(float4), s));
    P3T_CUDA(ctx, cudaMemsetAsync(w.nbr_count, 0, (size_t)n * sizeof(u32), s));
    P3T_CUDA(ctx, cudaMemsetAsync(w.nbr_cursor, 0, (size_t)n * sizeof(u32), s));   // scatter cursors of the neighbour stage
    direct_kernel<<<div_up(n_subset, DIRECT_THREADS), DIRECT_THREADS, 0, s>>>(w.body_user, n, d_subset, (u32)n_subset, ctx->prm,
                                                                              w.accpot, w.nbr_count, w.pairs,
                                                                              (u64)ctx->nbr_capacity, w.counters,
                                                                              ctx->cls_n ? w.cls_user : nullptr);
    P3T_CUDA(ctx, cudaGetLastError());
    return P3T_OK;
}
