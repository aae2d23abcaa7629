// walk.cu -- rows a7-a8: group tree walk and interaction kernel (the FP32-bound hot loop).
//
// One warp owns one i-group of up to 32*NI Morton-consecutive bodies (NI per lane, in registers)
// and walks the octree depth-first, 32 cells at a time (one per lane):
//   - cell accepted by R-MAC (d(B, c)^2 > rcrit^2, moments.cu)      -> p-c list (shared memory ring)
//   - else internal                                                  -> children pushed on the warp's stack
//   - else leaf: its bodies are fetched (coalesced) and split by their distance to the group box B:
//         >= h (1+1e-5): plain softened Newtonian term, K = W = 1     -> far ring  (no test in the loop)
//         <  h (1+1e-5): K/W weights (Eq. 8, 6), j != i, neighbour test -> near ring (rare slow path)
// Whenever a ring holds 32 entries the warp evaluates them against its bodies: each entry is read
// from shared memory as a broadcast LDS.128 and feeds NI interactions per lane.  Partial sums of
// one batch are fp32; batches are added into fp64 accumulators.
// Pair terms:  Eq. 8 (L65) and Eq. 6 (L55) of PAPER.md; cell terms: rule R-QUAD of DESIGN.md.
#include "p3t_internal.cuh"

struct WarpShared {
    u32 stack[WALK_STACK_SMEM];
    float4 far_buf[64];
    float4 near_buf[64];
    u32 near_idx[64];
    u32 pc_idx[64];
    float4 pc_a[32], pc_b[32], pc_c[32];
};

template <int NI> struct Acc {
    float ax[NI], ay[NI], az[NI], ph[NI];      // current batch (fp32)
    double dax[NI], day[NI], daz[NI], dph[NI]; // running totals (fp64)
    __device__ __forceinline__ void zero()
    {
#pragma unroll
        for (int b = 0; b < NI; ++b) { ax[b] = ay[b] = az[b] = ph[b] = 0.f; dax[b] = day[b] = daz[b] = dph[b] = 0.0; }
    }
    __device__ __forceinline__ void flush()
    {
#pragma unroll
        for (int b = 0; b < NI; ++b) {
            dax[b] += (double)ax[b]; day[b] += (double)ay[b]; daz[b] += (double)az[b]; dph[b] += (double)ph[b];
            ax[b] = ay[b] = az[b] = ph[b] = 0.f;
        }
    }
};

__device__ __forceinline__ u32 stack_read(const WarpShared &ws, const u32 *gstack, u32 pos)
{
    return pos < WALK_STACK_SMEM ? ws.stack[pos] : gstack[pos - WALK_STACK_SMEM];
}
__device__ __forceinline__ void stack_write(WarpShared &ws, u32 *gstack, u32 pos, u32 v)
{
    if (pos < WALK_STACK_SMEM) ws.stack[pos] = v;
    else gstack[pos - WALK_STACK_SMEM] = v;
}

// ---- p-p, plain softened Newtonian (K = W = 1): 23 flop by the convention of DESIGN.md ---------
template <int NI>
__device__ __forceinline__ void eval_far(const float4 *buf, u32 head, u32 cnt, const float (&xi)[NI], const float (&yi)[NI],
                                         const float (&zi)[NI], float eps2, Acc<NI> &acc)
{
    if (cnt == 32) {
#pragma unroll 8
        for (u32 j = 0; j < 32; ++j) {
            float4 bj = buf[head + j];
#pragma unroll
            for (int b = 0; b < NI; ++b) {
                float dx = bj.x - xi[b], dy = bj.y - yi[b], dz = bj.z - zi[b];
                float r2 = fmaf(dx, dx, fmaf(dy, dy, fmaf(dz, dz, eps2)));
                float rinv = rsqrtf(r2);
                float mrinv = bj.w * rinv;
                float mr3 = mrinv * (rinv * rinv);
                acc.ax[b] = fmaf(mr3, dx, acc.ax[b]);
                acc.ay[b] = fmaf(mr3, dy, acc.ay[b]);
                acc.az[b] = fmaf(mr3, dz, acc.az[b]);
                acc.ph[b] += mrinv;
            }
        }
    } else {
        for (u32 j = 0; j < cnt; ++j) {
            float4 bj = buf[head + j];
#pragma unroll
            for (int b = 0; b < NI; ++b) {
                float dx = bj.x - xi[b], dy = bj.y - yi[b], dz = bj.z - zi[b];
                float r2 = fmaf(dx, dx, fmaf(dy, dy, fmaf(dz, dz, eps2)));
                float rinv = rsqrtf(r2);
                float mrinv = bj.w * rinv;
                float mr3 = mrinv * (rinv * rinv);
                acc.ax[b] = fmaf(mr3, dx, acc.ax[b]);
                acc.ay[b] = fmaf(mr3, dy, acc.ay[b]);
                acc.az[b] = fmaf(mr3, dz, acc.az[b]);
                acc.ph[b] += mrinv;
            }
        }
    }
    acc.flush();
}

// ---- p-c, softened monopole + traceful quadrupole about the COM (R-QUAD), K = W = 1 -------------
//   with d = c - q_i, s^2 = |d|^2 + eps^2:
//   a   += d (M/s^3 + 7.5 dQd/s^7 - 1.5 trQ/s^5) - 3 Qd/s^5
//   -phi += M/s + 1.5 dQd/s^5 - 0.5 trQ/s^3
template <int NI>
__device__ __forceinline__ void eval_pc(WarpShared &ws, u32 head, u32 cnt, const float4 *__restrict__ cell_mac,
                                        const float4 *__restrict__ cell_mom0, const float4 *__restrict__ cell_mom1,
                                        const float (&xi)[NI], const float (&yi)[NI], const float (&zi)[NI], float eps2,
                                        Acc<NI> &acc, u32 lane)
{
    if (lane < cnt) {
        u32 c = ws.pc_idx[head + lane];   // head is 0 or 32 and cnt <= 32: no wrap
        float4 a = cell_mac[c], q0 = cell_mom0[c], q1 = cell_mom1[c];
        ws.pc_a[lane] = make_float4(a.x, a.y, a.z, q0.x);                               // c, M
        ws.pc_b[lane] = make_float4(q0.y, q0.z, q0.w, q0.y + q0.z + q0.w);              // Qxx Qyy Qzz trQ
        ws.pc_c[lane] = make_float4(q1.x, q1.y, q1.z, 0.f);                             // Qxy Qxz Qyz
    }
    __syncwarp();
#pragma unroll 4
    for (u32 j = 0; j < cnt; ++j) {
        float4 A = ws.pc_a[j], B = ws.pc_b[j], C = ws.pc_c[j];
#pragma unroll
        for (int b = 0; b < NI; ++b) {
            float dx = A.x - xi[b], dy = A.y - yi[b], dz = A.z - zi[b];
            float r2 = fmaf(dx, dx, fmaf(dy, dy, fmaf(dz, dz, eps2)));
            float rinv = rsqrtf(r2);
            float r2i = rinv * rinv;
            float r3i = rinv * r2i;
            float r5i = r3i * r2i;
            float r7i = r5i * r2i;
            float qdx = fmaf(B.x, dx, fmaf(C.x, dy, C.y * dz));
            float qdy = fmaf(C.x, dx, fmaf(B.y, dy, C.z * dz));
            float qdz = fmaf(C.y, dx, fmaf(C.z, dy, B.z * dz));
            float dqd = fmaf(dx, qdx, fmaf(dy, qdy, dz * qdz));
            float coef = fmaf(A.w, r3i, fmaf(7.5f * dqd, r7i, -1.5f * B.w * r5i));
            float m3r5 = -3.f * r5i;
            acc.ax[b] += fmaf(coef, dx, m3r5 * qdx);
            acc.ay[b] += fmaf(coef, dy, m3r5 * qdy);
            acc.az[b] += fmaf(coef, dz, m3r5 * qdz);
            acc.ph[b] += fmaf(A.w, rinv, fmaf(1.5f * dqd, r5i, -0.5f * B.w * r3i));
        }
    }
    __syncwarp();
    acc.flush();
}

// ---- p-p slow path: K (Eq. 12) on the force, W (Eq. 16-17) on the potential, j != i by index,
//      neighbour emission for s_ij < h (reading A4) -------------------------------------------------
template <int NI>
__device__ __forceinline__ void eval_near(const WarpShared &ws, u32 head, u32 cnt, const float (&xi)[NI], const float (&yi)[NI],
                                          const float (&zi)[NI], const u32 (&isorted)[NI], const u32 (&iuser)[NI],
                                          const P3TParams &prm, const u32 *__restrict__ sorted_idx, uint2 *pairs, u64 pair_cap,
                                          u64 *counters, u32 (&nnb)[NI], Acc<NI> &acc, u32 lane)
{
    for (u32 j = 0; j < cnt; ++j) {
        float4 bj = ws.near_buf[head + j];
        u32 js = ws.near_idx[head + j];
#pragma unroll
        for (int b = 0; b < NI; ++b) {
            float dx = bj.x - xi[b], dy = bj.y - yi[b], dz = bj.z - zi[b];
            float s2 = fmaf(dx, dx, fmaf(dy, dy, fmaf(dz, dz, prm.eps2)));
            bool live = isorted[b] != 0xffffffffu && isorted[b] != js;
            bool hit = live && s2 < prm.h2;
            if (live) {
                float rinv = rsqrtf(s2);
                float mrinv = bj.w * rinv;
                float mr3 = mrinv * (rinv * rinv);
                float K = 1.f, W = 1.f;
                if (s2 < prm.rout2) p3t_pair_weights(prm, s2, K, W);
                mr3 *= K;
                acc.ax[b] = fmaf(mr3, dx, acc.ax[b]);
                acc.ay[b] = fmaf(mr3, dy, acc.ay[b]);
                acc.az[b] = fmaf(mr3, dz, acc.az[b]);
                acc.ph[b] = fmaf(W, mrinv, acc.ph[b]);
            }
            u32 hb = __ballot_sync(0xffffffffu, hit);
            if (hb) {
                u64 base = 0;
                if (lane == 0) base = atomicAdd(&counters[CNT_PAIRS], (u64)__popc(hb));
                base = __shfl_sync(0xffffffffu, base, 0);
                if (hit) {
                    u64 pos = base + __popc(hb & lanemask_lt());
                    if (pos < pair_cap) pairs[pos] = make_uint2(iuser[b], sorted_idx[js]);
                    ++nnb[b];
                }
            }
        }
    }
    acc.flush();
}

template <int NI>
__global__ void __launch_bounds__(WALK_WARPS * 32, 16 / WALK_WARPS)
walk_kernel(const float4 *__restrict__ body, const u32 *__restrict__ sorted_idx, const u32 *__restrict__ group_start,
            const float4 *__restrict__ cell_mac, const float4 *__restrict__ cell_mom0, const float4 *__restrict__ cell_mom1,
            const uint2 *__restrict__ cell_meta, P3TParams prm, float4 *__restrict__ accpot, u32 *__restrict__ nbr_count,
            uint2 *pairs, u64 pair_cap, u32 *walk_stack, u64 *counters)
{
    __shared__ WarpShared s_ws[WALK_WARPS];
    const u32 lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    WarpShared &ws = s_ws[warp];
    u32 *gstack = walk_stack + (size_t)(blockIdx.x * WALK_WARPS + warp) * WALK_STACK_GMEM;
    const u32 ngroups = (u32)counters[CNT_NGROUPS];
    u64 tot_pp = 0, tot_pc = 0, tot_near = 0;

    while (true) {
        u32 g = 0;
        if (lane == 0) g = (u32)atomicAdd(&counters[CNT_GROUP_TICKET], 1ull);
        g = __shfl_sync(0xffffffffu, g, 0);
        if (g >= ngroups) break;
        const u32 gs = group_start[g], ge = group_start[g + 1];
        const u32 gcount = ge - gs;

        // ---- my bodies; empty slots replicate the group's first body and are flagged dead
        float xi[NI], yi[NI], zi[NI];
        u32 isorted[NI], iuser[NI], nnb[NI];
        float lo[3] = {INFINITY, INFINITY, INFINITY}, hi[3] = {-INFINITY, -INFINITY, -INFINITY};
#pragma unroll
        for (int b = 0; b < NI; ++b) {
            u32 k = gs + b * 32 + lane;
            bool ok = k < ge;
            float4 p = body[ok ? k : gs];
            xi[b] = p.x; yi[b] = p.y; zi[b] = p.z;
            isorted[b] = ok ? k : 0xffffffffu;
            iuser[b] = ok ? sorted_idx[k] : 0u;
            nnb[b] = 0;
            lo[0] = fminf(lo[0], p.x); hi[0] = fmaxf(hi[0], p.x);
            lo[1] = fminf(lo[1], p.y); hi[1] = fmaxf(hi[1], p.y);
            lo[2] = fminf(lo[2], p.z); hi[2] = fmaxf(hi[2], p.z);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                lo[d] = fminf(lo[d], __shfl_xor_sync(0xffffffffu, lo[d], o));
                hi[d] = fmaxf(hi[d], __shfl_xor_sync(0xffffffffu, hi[d], o));
            }
        }
        Acc<NI> acc;
        acc.zero();

        u32 top = 1;
        if (lane == 0) ws.stack[0] = 0;   // root
        u32 far_head = 0, far_cnt = 0, near_head = 0, near_cnt = 0, pc_head = 0, pc_cnt = 0;
        u32 n_far = 0, n_near = 0, n_pc = 0;
        bool overflow = false;
        __syncwarp();

        while (top > 0) {
            const u32 take = min(32u, top);
            top -= take;
            bool have = lane < take;
            u32 cell = have ? stack_read(ws, gstack, top + lane) : 0u;
            __syncwarp();
            bool accept = false;
            u32 nch = 0, first = 0, lcount = 0, lstart = 0;
            if (have) {
                float4 a = cell_mac[cell];
                float ex = fmaxf(0.f, fmaxf(lo[0] - a.x, a.x - hi[0]));
                float ey = fmaxf(0.f, fmaxf(lo[1] - a.y, a.y - hi[1]));
                float ez = fmaxf(0.f, fmaxf(lo[2] - a.z, a.z - hi[2]));
                float d2 = fmaf(ex, ex, fmaf(ey, ey, ez * ez));
                accept = d2 > a.w;
                if (!accept) {
                    uint2 meta = cell_meta[cell];
                    if (meta.y & P3T_LEAF_FLAG) { lstart = meta.x; lcount = meta.y & ~P3T_LEAF_FLAG; }
                    else { first = meta.x; nch = meta.y; }
                }
            }
            // ---- children of opened internal cells -> stack
            {
                u32 inc = nch;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    u32 t = __shfl_up_sync(0xffffffffu, inc, o);
                    if (lane >= o) inc += t;
                }
                u32 total = __shfl_sync(0xffffffffu, inc, 31);
                if (top + total > WALK_STACK_SMEM + WALK_STACK_GMEM) { overflow = true; break; }
                u32 pos = top + inc - nch;
                for (u32 c = 0; c < nch; ++c) stack_write(ws, gstack, pos + c, first + c);
                top += total;
            }
            // ---- accepted cells -> p-c ring
            {
                u32 ab = __ballot_sync(0xffffffffu, accept);
                if (accept) ws.pc_idx[(pc_head + pc_cnt + __popc(ab & lanemask_lt())) & 63u] = cell;
                pc_cnt += __popc(ab);
                __syncwarp();
                if (pc_cnt >= 32) {
                    eval_pc<NI>(ws, pc_head, 32, cell_mac, cell_mom0, cell_mom1, xi, yi, zi, prm.eps2, acc, lane);
                    pc_head = (pc_head + 32) & 63u; pc_cnt -= 32; n_pc += 32;
                }
            }
            // ---- bodies of opened leaves -> near / far rings
            {
                u32 inc = lcount;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    u32 t = __shfl_up_sync(0xffffffffu, inc, o);
                    if (lane >= o) inc += t;
                }
                const u32 total = __shfl_sync(0xffffffffu, inc, 31);
                const u32 excl = inc - lcount;
                for (u32 v0 = 0; v0 < total; v0 += 32) {
                    u32 v = v0 + lane;
                    // owner lane: largest s with excl[s] <= v
                    u32 s = 0;
#pragma unroll
                    for (int step = 16; step > 0; step >>= 1) {
                        u32 cand = s + step;
                        u32 t = __shfl_sync(0xffffffffu, inc, cand - 1);   // = excl[cand]
                        if (t <= v) s = cand;
                    }
                    u32 s_start = __shfl_sync(0xffffffffu, lstart, s);
                    u32 s_excl = __shfl_sync(0xffffffffu, excl, s);
                    bool hv = v < total;
                    u32 bidx = s_start + (v - s_excl);
                    float4 bj = body[hv ? bidx : gs];
                    float ex = fmaxf(0.f, fmaxf(lo[0] - bj.x, bj.x - hi[0]));
                    float ey = fmaxf(0.f, fmaxf(lo[1] - bj.y, bj.y - hi[1]));
                    float ez = fmaxf(0.f, fmaxf(lo[2] - bj.z, bj.z - hi[2]));
                    float d2 = fmaf(ex, ex, fmaf(ey, ey, ez * ez));
                    bool isnear = hv && d2 < prm.hnear2;
                    bool isfar = hv && !isnear;
                    u32 fb = __ballot_sync(0xffffffffu, isfar), nb = __ballot_sync(0xffffffffu, isnear);
                    if (isfar) ws.far_buf[(far_head + far_cnt + __popc(fb & lanemask_lt())) & 63u] = bj;
                    if (isnear) {
                        u32 slot = (near_head + near_cnt + __popc(nb & lanemask_lt())) & 63u;
                        ws.near_buf[slot] = bj;
                        ws.near_idx[slot] = bidx;
                    }
                    far_cnt += __popc(fb);
                    near_cnt += __popc(nb);
                    __syncwarp();
                    if (far_cnt >= 32) {
                        eval_far<NI>(ws.far_buf, far_head, 32, xi, yi, zi, prm.eps2, acc);
                        far_head = (far_head + 32) & 63u; far_cnt -= 32; n_far += 32;
                    }
                    if (near_cnt >= 32) {
                        eval_near<NI>(ws, near_head, 32, xi, yi, zi, isorted, iuser, prm, sorted_idx, pairs, pair_cap, counters,
                                      nnb, acc, lane);
                        near_head = (near_head + 32) & 63u; near_cnt -= 32; n_near += 32;
                    }
                    __syncwarp();
                }
            }
        }
        if (overflow) {
            if (lane == 0) atomicOr(&counters[CNT_ERR_EVAL], (u64)ERR_STACK_OVERFLOW);
        }
        // ---- flush what is left in the rings
        if (pc_cnt) { eval_pc<NI>(ws, pc_head, pc_cnt, cell_mac, cell_mom0, cell_mom1, xi, yi, zi, prm.eps2, acc, lane); n_pc += pc_cnt; }
        if (far_cnt) { eval_far<NI>(ws.far_buf, far_head, far_cnt, xi, yi, zi, prm.eps2, acc); n_far += far_cnt; }
        if (near_cnt) {
            eval_near<NI>(ws, near_head, near_cnt, xi, yi, zi, isorted, iuser, prm, sorted_idx, pairs, pair_cap, counters, nnb,
                          acc, lane);
            n_near += near_cnt;
        }
        __syncwarp();
        // ---- results, user order
#pragma unroll
        for (int b = 0; b < NI; ++b) {
            if (isorted[b] != 0xffffffffu) {
                accpot[iuser[b]] = make_float4((float)acc.dax[b], (float)acc.day[b], (float)acc.daz[b], (float)(-acc.dph[b]));
                nbr_count[iuser[b]] = nnb[b];
            }
        }
        // each live body met itself once on the near path (distance 0 to its own group's box)
        tot_pp += (u64)(n_far + n_near) * gcount - gcount;
        tot_near += (u64)n_near * gcount - gcount;
        tot_pc += (u64)n_pc * gcount;
    }
    if (lane == 0) {
        atomicAdd(&counters[CNT_NPP], tot_pp);
        atomicAdd(&counters[CNT_NPC], tot_pc);
        atomicAdd(&counters[CNT_NNEAR], tot_near);
    }
}

p3t_status p3t_stage_walk(p3t_ctx *ctx)
{
    Workspace &w = ctx->ws;
    cudaStream_t s = ctx->stream;
    P3T_CUDA(ctx, cudaMemsetAsync(w.counters, 0, 8 * sizeof(u64), s));   // eval counters
    u32 grid = (u32)ctx->sm_count * (16 / WALK_WARPS);
    if ((size_t)grid * WALK_WARPS > w.walk_warps_max) grid = (u32)(w.walk_warps_max / WALK_WARPS);
    if (ctx->ngroup == 64)
        walk_kernel<2><<<grid, WALK_WARPS * 32, 0, s>>>(w.body, w.idx[ctx->cur], w.group_start, w.cell_mac, w.cell_mom0, w.cell_mom1,
                                                        w.cell_meta, ctx->prm, w.accpot, w.nbr_count, w.pairs,
                                                        (u64)ctx->nbr_capacity, w.walk_stack, w.counters);
    else
        walk_kernel<1><<<grid, WALK_WARPS * 32, 0, s>>>(w.body, w.idx[ctx->cur], w.group_start, w.cell_mac, w.cell_mom0, w.cell_mom1,
                                                        w.cell_meta, ctx->prm, w.accpot, w.nbr_count, w.pairs,
                                                        (u64)ctx->nbr_capacity, w.walk_stack, w.counters);
    P3T_CUDA(ctx, cudaGetLastError());
    return P3T_OK;
}
