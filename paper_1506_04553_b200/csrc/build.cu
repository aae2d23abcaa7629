// build.cu -- row a5: octree and i-groups from the sorted Morton keys, with no level loop.
//
// Let c[i] be the number of leading octree levels on which key[i-1] and key[i] agree (c[0] = -1).
// The level-L cell containing body i extends left/right while the running minimum of c stays >= L,
// so its population is decidable from a window of c around i:
//   D(i)  = smallest L whose cell holds <= NLEAF bodies   (leaf level of body i, capped at max_level)
//   Dg(i) = the same with NGROUP                          (natural group level)
// and (L, i) is a tree node, starting at body i, exactly for c[i] < L <= D(i).  Nodes are numbered
// level-major (all level-0 nodes, then level 1, ...), each level in body order, so the children of
// a node are contiguous.  Checked against a recursive construction in tests (CPU prototype) and
// against the invariants of SURVEY.md 7.3 on the GPU (tests/test_gpu_tree.py).
#include "p3t_internal.cuh"

#define HALO 72   // >= max(NLEAF, NGROUP) + 2

// ------------------------------------------------------------------------------------------------
// B1: per body leaf level D and group level Dg; per block node counts per level
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(BUILD_THREADS) levels_kernel(const signed char *__restrict__ clev, u8 *__restrict__ dlev,
                                                               u8 *__restrict__ glev, u32 *__restrict__ blk_cnt, u32 n,
                                                               int max_level, int nleaf, int ngroup)
{
    __shared__ signed char s_c[BUILD_THREADS + 2 * HALO];
    __shared__ u32 s_cnt[32];
    const int tid = threadIdx.x;
    const long long base = (long long)blockIdx.x * BUILD_THREADS - HALO;
    for (int t = tid; t < BUILD_THREADS + 2 * HALO; t += BUILD_THREADS) {
        long long j = base + t;
        s_c[t] = (j >= 0 && j <= (long long)n) ? clev[j] : (signed char)-1;
    }
    if (tid < 32) s_cnt[tid] = 0;
    __syncthreads();
    const u32 i = blockIdx.x * BUILD_THREADS + tid;
    const bool ok = i < n;
    int c = 127, D = 0, Dg = 0;
    if (ok) {
        const int t0 = tid + HALO;
        c = s_c[t0];
        // merge the two non-increasing sequences of running minima, largest first
        int a = 0, b = 1;
        int la = s_c[t0], ra = s_c[t0 + 1], v = -1;
        int steps = max(nleaf, ngroup);
        for (int s = 1; s <= steps; ++s) {
            if (la >= ra) { v = la; ++a; la = min(la, (int)s_c[t0 - a]); }
            else          { v = ra; ++b; ra = min(ra, (int)s_c[t0 + b]); }
            if (s == nleaf) D = min(max_level, max(0, v + 1));
            if (s == ngroup) Dg = min(max_level, max(0, v + 1));
        }
        dlev[i] = (u8)D;
        glev[i] = (u8)Dg;
    }
    // nodes starting at i: levels c < L <= D
    for (int L = 0; L <= max_level; ++L) {
        u32 b = __ballot_sync(0xffffffffu, ok && c < L && L <= D);
        if ((tid & 31) == 0 && b) atomicAdd(&s_cnt[L], __popc(b));
    }
    __syncthreads();
    if (tid < 32) blk_cnt[(size_t)blockIdx.x * 32 + tid] = s_cnt[tid];
}

// ------------------------------------------------------------------------------------------------
// B2: exclusive scan over blocks of each level's node count (one CTA per level)
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(1024) level_scan_kernel(const u32 *__restrict__ blk_cnt, u32 *__restrict__ blk_off,
                                                          u32 *level_total, u32 nblk, u64 *counters)
{
    __shared__ u32 s_w[32];
    __shared__ u32 s_carry;
    const int L = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_carry = 0;
    __syncthreads();
    for (u32 b0 = 0; b0 < nblk; b0 += 1024) {
        u32 b = b0 + tid;
        u32 v = b < nblk ? blk_cnt[(size_t)b * 32 + L] : 0;
        u32 inc = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            u32 t = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += t;
        }
        if (lane == 31) s_w[warp] = inc;
        __syncthreads();
        if (warp == 0) {
            u32 w = s_w[lane], wi = w;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                u32 t = __shfl_up_sync(0xffffffffu, wi, o);
                if (lane >= o) wi += t;
            }
            s_w[lane] = wi - w;
        }
        __syncthreads();
        u32 carry = s_carry;
        if (b < nblk) blk_off[(size_t)b * 32 + L] = carry + s_w[warp] + inc - v;
        __syncthreads();
        if (tid == 1023) s_carry = carry + s_w[warp] + inc;
        __syncthreads();
    }
    if (tid == 0) {
        level_total[L] = s_carry;
        if (s_carry) {
            atomicAdd(&counters[CNT_NCELLS], (u64)s_carry);
            atomicMax(&counters[CNT_DEPTH], (u64)L);
        }
    }
}

// ------------------------------------------------------------------------------------------------
// B3: emit the nodes, their parents, first children, leaf ranges; segment cut flags for groups
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(BUILD_THREADS) emit_nodes_kernel(
    const signed char *__restrict__ clev, const u8 *__restrict__ dlev, const u8 *__restrict__ glev,
    const u32 *__restrict__ blk_off, const u32 *__restrict__ level_total, u32 n, int max_level, int merge_levels,
    u32 cell_cap, u32 *__restrict__ cell_start, u8 *__restrict__ cell_level, u32 *__restrict__ cell_parent,
    u32 *__restrict__ cell_first, u32 *cell_nchild, uint2 *__restrict__ cell_meta, u8 *__restrict__ cutflag, u64 *counters)
{
    __shared__ u32 s_wcnt[BUILD_THREADS / 32][32];
    __shared__ u32 s_lvloff[32];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const u32 i = blockIdx.x * BUILD_THREADS + tid;
    const bool ok = i < n;
    int c = 127, D = 0;
    if (ok) { c = clev[i]; D = dlev[i]; }
    for (int L = 0; L <= max_level; ++L) {
        u32 b = __ballot_sync(0xffffffffu, ok && c < L && L <= D);
        if (lane == 0) s_wcnt[warp][L] = __popc(b);
    }
    if (tid == 0) {
        u32 off = 0;
        for (int L = 0; L < 32; ++L) { s_lvloff[L] = off; off += (L <= max_level) ? level_total[L] : 0; }
    }
    __syncthreads();
    if (tid <= max_level) {
        u32 sum = s_lvloff[tid] + blk_off[(size_t)blockIdx.x * 32 + tid];
        for (int w = 0; w < BUILD_THREADS / 32; ++w) {
            u32 t = s_wcnt[w][tid];
            s_wcnt[w][tid] = sum;
            sum += t;
        }
    }
    __syncthreads();
    u32 prev_rank = 0;
    bool prev_flag = false;
    u32 nleaf_here = 0;
    for (int L = 0; L <= max_level; ++L) {
        bool flag = ok && c < L && L <= D;
        u32 b = __ballot_sync(0xffffffffu, flag);
        u32 rank = s_wcnt[warp][L] + __popc(b & lanemask_lt());
        if (flag) {
            if (rank < cell_cap) {
                cell_start[rank] = i;
                cell_level[rank] = (u8)L;
                u32 parent = P3T_NO_PARENT;
                if (L > 0) {
                    parent = prev_flag ? prev_rank : prev_rank - 1;
                    atomicAdd(&cell_nchild[parent], 1u);
                }
                cell_parent[rank] = parent;
                if (prev_flag) cell_first[prev_rank] = rank;
                if (L == D) {   // leaf: bodies i .. while c[j] >= L
                    u32 cnt = 1;
                    while (i + cnt < n && clev[i + cnt] >= L) ++cnt;
                    cell_meta[rank] = make_uint2(i, cnt | P3T_LEAF_FLAG);
                    ++nleaf_here;
                }
            } else {
                atomicOr(&counters[CNT_ERR_BUILD], (u64)ERR_CELL_CAPACITY);
            }
        }
        prev_rank = rank;
        prev_flag = flag;
    }
    // segment cuts: a group may not straddle a boundary more than merge_levels above the natural
    // group level of the bodies on either side
    if (ok) {
        int g = glev[i];
        int gp = i > 0 ? (int)glev[i - 1] : 0;
        cutflag[i] = (i == 0 || c < max(g, gp) - merge_levels) ? 1 : 0;
    }
    u32 nl = __reduce_add_sync(0xffffffffu, nleaf_here);
    if (lane == 0 && nl) atomicAdd(&counters[CNT_NLEAVES], (u64)nl);
}

// ------------------------------------------------------------------------------------------------
// B4: group heads (every ngroup-th body of a segment) compacted to group_start[] in body order
//     (single pass, decoupled look-back over blocks)
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(BUILD_THREADS) group_heads_kernel(const u8 *__restrict__ cutflag, u32 n, int ngroup,
                                                                    u32 *__restrict__ group_start, volatile u32 *status,
                                                                    u64 *counters)
{
    __shared__ u32 s_blk;
    __shared__ int s_carry;       // last cut position before this block
    __shared__ int s_wmax[BUILD_THREADS / 32];
    __shared__ u32 s_wcnt[BUILD_THREADS / 32];
    __shared__ u32 s_excl;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_blk = (u32)atomicAdd(&counters[CNT_HEAD_TICKET], 1ull);
    __syncthreads();
    const u32 blk = s_blk;
    const u32 i = blk * BUILD_THREADS + tid;
    const bool ok = i < n;
    // warp 0 finds the last cut before the block start (cutflag[0] = 1, so the search ends)
    if (warp == 0) {
        int found = -1;
        for (long long top = (long long)blk * BUILD_THREADS - 1; top >= 0 && found < 0; top -= 32) {
            long long pos = top - lane;
            bool hit = pos >= 0 && cutflag[pos];
            u32 b = __ballot_sync(0xffffffffu, hit);
            if (b) found = (int)(top - (__ffs(b) - 1));   // lowest lane = nearest position
        }
        if (lane == 0) s_carry = found;
    }
    int mycut = (ok && cutflag[i]) ? (int)i : -1;
    int run = mycut;   // inclusive max-scan inside the warp
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        int t = __shfl_up_sync(0xffffffffu, run, o);
        if (lane >= o) run = max(run, t);
    }
    if (lane == 31) s_wmax[warp] = run;
    __syncthreads();
    int seg = max(run, s_carry);
    for (int w = 0; w < warp; ++w) seg = max(seg, s_wmax[w]);
    bool head = ok && ((i - (u32)seg) % (u32)ngroup == 0);
    u32 hb = __ballot_sync(0xffffffffu, head);
    if (lane == 0) s_wcnt[warp] = __popc(hb);
    __syncthreads();
    if (tid == 0) {
        u32 total = 0;
        for (int w = 0; w < BUILD_THREADS / 32; ++w) { u32 t = s_wcnt[w]; s_wcnt[w] = total; total += t; }
        // decoupled look-back on one word per block: value | flag (30-bit value)
        status[blk] = total | (blk == 0 ? 0x80000000u : 0x40000000u);
        u32 excl = 0;
        if (blk > 0) {
            int t = (int)blk - 1;
            while (true) {
                u32 v = status[t];
                if ((v & 0xc0000000u) == 0) continue;
                excl += v & 0x3fffffffu;
                if (v & 0x80000000u) break;
                --t;
            }
            status[blk] = (excl + total) | 0x80000000u;
        }
        s_excl = excl;
        if ((blk + 1) * (u32)BUILD_THREADS >= n) {   // last block: total number of groups, terminator
            counters[CNT_NGROUPS] = (u64)(excl + total);
            group_start[excl + total] = n;
        }
    }
    __syncthreads();
    if (head) group_start[s_excl + s_wcnt[warp] + __popc(hb & lanemask_lt())] = i;
}

p3t_status p3t_stage_build(p3t_ctx *ctx)
{
    Workspace &w = ctx->ws;
    u32 n = (u32)ctx->n;
    cudaStream_t s = ctx->stream;
    u32 nblk = div_up(n, BUILD_THREADS);
    // cell_nchild and cell_ready are adjacent in the workspace: one memset zeroes both
    P3T_CUDA(ctx, cudaMemsetAsync(w.cell_nchild, 0, (size_t)((char *)(w.cell_ready + w.cell_cap) - (char *)w.cell_nchild), s));
    P3T_CUDA(ctx, cudaMemsetAsync(w.head_status, 0, (size_t)nblk * sizeof(u32), s));
    levels_kernel<<<nblk, BUILD_THREADS, 0, s>>>(w.clev, w.dlev, w.glev, w.blk_level_cnt, n, ctx->max_level, ctx->nleaf,
                                                 ctx->ngroup);
    level_scan_kernel<<<ctx->max_level + 1, 1024, 0, s>>>(w.blk_level_cnt, w.blk_level_off, w.level_total, nblk, w.counters);
    emit_nodes_kernel<<<nblk, BUILD_THREADS, 0, s>>>(w.clev, w.dlev, w.glev, w.blk_level_off, w.level_total, n, ctx->max_level,
                                                     ctx->merge_levels, (u32)w.cell_cap, w.cell_start, w.cell_level,
                                                     w.cell_parent, w.cell_first, w.cell_nchild, w.cell_meta, w.cutflag,
                                                     w.counters);
    group_heads_kernel<<<nblk, BUILD_THREADS, 0, s>>>(w.cutflag, n, ctx->ngroup, w.group_start, w.head_status, w.counters);
    P3T_CUDA(ctx, cudaGetLastError());
    return P3T_OK;
}
