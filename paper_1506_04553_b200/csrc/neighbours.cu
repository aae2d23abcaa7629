// neighbours.cu -- row a9: per-particle neighbour lists as CSR in user ids ("the
// library also returns, for each particle, the list of particles within the distance h").
//   1. exclusive scan of the per-particle counts (written by the walk) -> offset[n+1] (u64)
//   2. scatter the (i, j) pairs emitted by the walk into their lists
//   3. sort every list ascending in j, so the output is canonical
#include "p3t_internal.cuh"

#define SCAN_THREADS 256
#define SCAN_ITEMS 4
#define SCAN_TILE (SCAN_THREADS * SCAN_ITEMS)

__device__ __forceinline__ u32 block_exclusive_scan(u32 v, u32 *s_w, u32 &total)
{
    const u32 lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    u32 inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        u32 t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) s_w[warp] = inc;
    __syncthreads();
    u32 base = 0, tot = 0;
    for (u32 w = 0; w < SCAN_THREADS / 32; ++w) {
        u32 t = s_w[w];
        if (w < warp) base += t;
        tot += t;
    }
    total = tot;
    __syncthreads();
    return base + inc - v;
}

__global__ void __launch_bounds__(SCAN_THREADS) scan_tile_sums_kernel(const u32 *__restrict__ count, u32 n, u64 *tile_sum)
{
    P3T_GRID_TRIGGER();
    P3T_GRID_WAIT();
    __shared__ u32 s_w[SCAN_THREADS / 32];
    u32 base = blockIdx.x * SCAN_TILE + threadIdx.x * SCAN_ITEMS;
    u32 v = 0;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k)
        if (base + k < n) v += count[base + k];
    u32 total;
    block_exclusive_scan(v, s_w, total);
    if (threadIdx.x == 0) tile_sum[blockIdx.x] = total;
}

// single block: exclusive scan of the tile sums in place (64-bit)
__global__ void __launch_bounds__(1024) scan_tile_prefix_kernel(u64 *tile_sum, u32 ntiles)
{
    P3T_GRID_TRIGGER();
    P3T_GRID_WAIT();
    __shared__ u64 s_w[32];
    __shared__ u64 s_carry;
    const u32 tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_carry = 0;
    __syncthreads();
    for (u32 t0 = 0; t0 < ntiles; t0 += 1024) {
        u32 t = t0 + tid;
        u64 v = t < ntiles ? tile_sum[t] : 0ull;
        u64 inc = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            u64 x = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += x;
        }
        if (lane == 31) s_w[warp] = inc;
        __syncthreads();
        u64 base = s_carry;
        for (u32 w = 0; w < warp; ++w) base += s_w[w];
        if (t < ntiles) tile_sum[t] = base + inc - v;
        __syncthreads();
        if (tid == 1023) s_carry = base + inc;
        __syncthreads();
    }
}

__global__ void __launch_bounds__(SCAN_THREADS) scan_apply_kernel(const u32 *__restrict__ count, u32 n,
                                                                  const u64 *__restrict__ tile_sum, u64 *__restrict__ offset,
                                                                  u64 *counters)
{
    P3T_GRID_TRIGGER();
    P3T_GRID_WAIT();
    __shared__ u32 s_w[SCAN_THREADS / 32];
    u32 base = blockIdx.x * SCAN_TILE + threadIdx.x * SCAN_ITEMS;
    u32 c[SCAN_ITEMS], v = 0, mx = 0;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        c[k] = base + k < n ? count[base + k] : 0u;
        v += c[k];
        mx = max(mx, c[k]);
    }
    u32 total;
    u32 ex = block_exclusive_scan(v, s_w, total);
    u64 run = tile_sum[blockIdx.x] + ex;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        if (base + k < n) offset[base + k] = run;
        run += c[k];
        if (base + k == n - 1) offset[n] = run;
    }
    mx = __reduce_max_sync(0xffffffffu, mx);
    if ((threadIdx.x & 31) == 0 && mx) atomicMax(&counters[CNT_MAXLIST], (u64)mx);
}

__global__ void __launch_bounds__(256) fill_lists_kernel(const uint2 *__restrict__ pairs, u64 pair_cap,
                                                         const u64 *__restrict__ offset, u32 *cursor, u32 *__restrict__ nbr,
                                                         const u64 *__restrict__ counters)
{
    P3T_GRID_TRIGGER();
    P3T_GRID_WAIT();
    u64 total = counters[CNT_PAIRS];
    if (total > pair_cap) return;   // over capacity: lists are not materialised (P3T_ECAPACITY at fetch)
    for (u64 p = (u64)blockIdx.x * blockDim.x + threadIdx.x; p < total; p += (u64)gridDim.x * blockDim.x) {
        uint2 pr = pairs[p];
        u32 slot = atomicAdd(&cursor[pr.x], 1u);
        P3T_DEV_ASSERT(offset[pr.x] + slot < offset[pr.x + 1] && offset[pr.x + 1] <= total);
        nbr[offset[pr.x] + slot] = pr.y;
    }
}

#define SORT_LIST_SERIAL 16   // lists up to this length are sorted by their own thread

// ascending order inside every list: one thread per list, insertion sort for the short ones (the usual case: a
// fraction of an entry per particle); the long ones (dense cores, large h) are queued for sort_long_lists_kernel
__global__ void __launch_bounds__(256) sort_lists_kernel(const u32 *__restrict__ count, const u64 *__restrict__ offset, u32 n,
                                                         u32 *nbr, u64 pair_cap, u64 *counters, u32 *worklist)
{
    P3T_GRID_TRIGGER();
    P3T_GRID_WAIT();
    if (counters[CNT_PAIRS] > pair_cap) return;
    u32 i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    u32 c = count[i];
    if (c < 2) return;
    if (c > SORT_LIST_SERIAL) {
        const u64 wslot = atomicAdd(&counters[CNT_EVAL_SPARE], 1ull);
        P3T_DEV_ASSERT(wslot < n);
        worklist[wslot] = i;
        return;
    }
    u32 *l = nbr + offset[i];
    for (u32 a = 1; a < c; ++a) {
        u32 v = l[a];
        u32 b = a;
        while (b > 0 && l[b - 1] > v) { l[b] = l[b - 1]; --b; }
        l[b] = v;
    }
}

// one warp per long list: rank sort (entries of a list are distinct) through a scratch copy
__global__ void __launch_bounds__(256) sort_long_lists_kernel(const u32 *__restrict__ count, const u64 *__restrict__ offset,
                                                              u32 *nbr, u32 *scratch, const u64 *__restrict__ counters,
                                                              const u32 *__restrict__ worklist)
{
    P3T_GRID_TRIGGER();
    P3T_GRID_WAIT();
    const u32 nlong = (u32)counters[CNT_EVAL_SPARE];
    const u32 lane = threadIdx.x & 31, nwarps = gridDim.x * (blockDim.x >> 5);
    for (u32 wk = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); wk < nlong; wk += nwarps) {
        const u32 i = worklist[wk], c = count[i];
        u32 *l = nbr + offset[i];
        u32 *t = scratch + offset[i];
        for (u32 e = lane; e < c; e += 32) t[e] = l[e];
        __syncwarp();
        for (u32 e = lane; e < c; e += 32) {
            const u32 v = t[e];
            u32 rank = 0;
            for (u32 k = 0; k < c; ++k) rank += t[k] < v ? 1u : 0u;
            l[rank] = v;
        }
        __syncwarp();
    }
}

p3t_status p3t_stage_neighbours(p3t_ctx *ctx)
{
    Workspace &w = ctx->ws;
    cudaStream_t s = ctx->stream;
    u32 n = (u32)ctx->n;
    u32 ntiles = div_up(n, SCAN_TILE);
    // (programmatic dependent launch along the stage; the scatter cursors were zeroed by p3t_stage_walk / p3t_stage_direct, in
    //  front of the evaluation, so that no memset breaks the chain)
    P3T_CUDA(ctx, p3t_launch_pdl(scan_tile_sums_kernel, dim3(ntiles), dim3(SCAN_THREADS), 0, s, (const u32 *)w.nbr_count, n, w.scan_tmp));
    P3T_CUDA(ctx, p3t_launch_pdl(scan_tile_prefix_kernel, dim3(1), dim3(1024), 0, s, w.scan_tmp, ntiles));
    P3T_CUDA(ctx, p3t_launch_pdl(scan_apply_kernel, dim3(ntiles), dim3(SCAN_THREADS), 0, s, (const u32 *)w.nbr_count, n, (const u64 *)w.scan_tmp,
                                 w.nbr_offset, w.counters));
    if (ctx->nbr_capacity) {
        u32 grid = (u32)ctx->sm_count * 4;
        P3T_CUDA(ctx, p3t_launch_pdl(fill_lists_kernel, dim3(grid), dim3(256), 0, s, (const uint2 *)w.pairs, (u64)ctx->nbr_capacity,
                                     (const u64 *)w.nbr_offset, w.nbr_cursor, w.nbr, (const u64 *)w.counters));
        // the scatter cursors are dead after the fill: they hold the queue of long lists; the pair buffer is the scratch copy
        P3T_CUDA(ctx, p3t_launch_pdl(sort_lists_kernel, dim3(div_up(n, 256)), dim3(256), 0, s, (const u32 *)w.nbr_count, (const u64 *)w.nbr_offset, n,
                                     w.nbr, (u64)ctx->nbr_capacity, w.counters, w.nbr_cursor));
        P3T_CUDA(ctx, p3t_launch_pdl(sort_long_lists_kernel, dim3((u32)ctx->sm_count * 2), dim3(256), 0, s, (const u32 *)w.nbr_count,
                                     (const u64 *)w.nbr_offset, w.nbr, reinterpret_cast<u32 *>(w.pairs), (const u64 *)w.counters,
                                     (const u32 *)w.nbr_cursor));
    }
    P3T_CUDA(ctx, cudaGetLastError());
    return P3T_OK;
}
