// build.cu -- row a5: octree and i-groups from the sorted Morton keys, with no level loop.
//
// Let c[i] be the number of leading octree levels on which key[i-1] and key[i] agree (c[0] = c[n] = -1).
// A window of W+1 consecutive bodies j..j+W lies in one level-L cell iff min(c[j+1..j+W]) >= L, so
//   D(i)  = 1 + max over the windows of NLEAF+1 bodies that contain i of that minimum
// is the smallest level at which the cell of body i holds <= NLEAF bodies: the leaf level of body i
// (clamped to [0, max_level]); Dg(i), with NGROUP, is the natural group level.  Both are a sliding
// minimum followed by a sliding maximum, computed here by doubling on packed 16-bit lanes
// (VIMNMX.U16x2) in shared memory.  (L, i) is a tree node, starting at body i, exactly for
// c[i] < L <= D(i).  Nodes are numbered level-major (all level-0 nodes, then level 1, ...), each
// level in body order, so the children of a node are contiguous.
//
// Two launches:
//   levels_kernel  per tile of BUILD_TILE bodies: D, Dg -> dlev, cut flags; node counts per level and
//                  the group-head bookkeeping of the tile; the LAST tile to finish scans these over
//                  all tiles (exclusive prefixes per level, carried cut position, group offsets)
//   emit_kernel    node records (start, level, parent, first child, leaf range) and group_start[]
// Checked against a recursive construction (oracle/keytree.py) in tests/test_gpu_tree.py.
#include "p3t_internal.cuh"

#define GROUP_MERGE_MIN_LEVEL 4                        // see the cut rule in levels_kernel
#define BUILD_HALO 64                                  // >= max(NLEAF, NGROUP)
#define BUILD_WIN (BUILD_TILE + 2 * BUILD_HALO + 16)   // window of c values held per tile (16-bit lanes)
#define BUILD_WORDS (BUILD_WIN / 2)
#define BUILD_PER_THREAD (BUILD_TILE / BUILD_THREADS)  // consecutive bodies per thread

// Per-tile look-back words (flag | value, as in the radix sort) and the resulting exclusive prefixes.
// status[0..23]: nodes per level starting in the tile (levels_kernel); status[24]: group heads in the
// tile (emit_kernel).  BUILD_LOOKBACK sentinel records in front of record 0 hold INC | 0.
struct TileRec {
    u32 status[32];
    u32 excl[32];       // [0..23] exclusive prefix over tiles of the node counts per level
};
static_assert(sizeof(TileRec) == 256, "TileRec is two 128-byte lines");
#define BUILD_LOOKBACK 8
#define TL_FLAG_AGG 0x40000000u
#define TL_FLAG_INC 0x80000000u
#define TL_VAL_MASK 0x3fffffffu

__device__ __forceinline__ u32 ld_tile_status(const u32 *p)
{
    u32 v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_tile_status(u32 *p, u32 v)
{
    asm volatile("st.relaxed.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
// Decoupled look-back of one column.  tile_publish makes `own` of `tile` visible (as early as it is known);
// tile_resolve returns the sum over all tiles before it and publishes the inclusive prefix.
// p0 points at status word `col` of record `tile`; records are sizeof(TileRec) apart.
__device__ __forceinline__ void tile_publish(u32 *p0, u32 tile, u32 own)
{
    st_tile_status(p0, own | (tile == 0 ? TL_FLAG_INC : TL_FLAG_AGG));
}
__device__ __forceinline__ u32 tile_resolve(u32 *p0, u32 tile, u32 own)
{
    const int stride = (int)(sizeof(TileRec) / sizeof(u32));
    u32 excl = 0;
    if (tile > 0) {
        const u32 *p = p0 - stride;
        bool done = false;
        while (!done) {
            u32 v[BUILD_LOOKBACK];
#pragma unroll
            for (int k = 0; k < BUILD_LOOKBACK; ++k) v[k] = ld_tile_status(p - k * stride);
            bool go = true;
            u32 used = 0;
#pragma unroll
            for (int k = 0; k < BUILD_LOOKBACK; ++k) {
                const bool ready = v[k] >= TL_FLAG_AGG, isinc = v[k] >= TL_FLAG_INC;
                if (go && ready) { excl += v[k] & TL_VAL_MASK; ++used; }
                done = done || (go && isinc);
                go = go && ready && !isinc;
            }
            p -= used * stride;
        }
        st_tile_status(p0, (excl + own) | TL_FLAG_INC);
    }
    return excl;
}
// The same for "the last marked position before this tile": own = position + 1 of the tile's last mark, 0 if it has
// none; going backwards the first non-zero word decides (tile 0 always has a mark: body 0 starts a segment).
__device__ __forceinline__ u32 tile_lookback_last(u32 *p0, u32 tile, u32 own)
{
    const int stride = (int)(sizeof(TileRec) / sizeof(u32));
    st_tile_status(p0, own | ((tile == 0 || own) ? TL_FLAG_INC : TL_FLAG_AGG));   // a tile with a mark needs no look-back by others
    u32 last = 0;
    if (tile > 0) {
        const u32 *p = p0 - stride;
        while (!last) {
            const u32 v = ld_tile_status(p);
            if (v < TL_FLAG_AGG) continue;            // not published yet
            last = v & TL_VAL_MASK;
            if (v >= TL_FLAG_INC) break;              // inclusive word: final even if zero (cannot be: tile 0 has a mark)
            p -= stride;
        }
        if (!own) st_tile_status(p0, last | TL_FLAG_INC);
    }
    return last;
}
__device__ __forceinline__ u32 tile_lookback(u32 *p0, u32 tile, u32 own)
{
    tile_publish(p0, tile, own);
    return tile_resolve(p0, tile, own);
}

#define BUILD_PAD 40   // zero words behind every window: shifted reads never leave the array
struct Window { u32 w[BUILD_WORDS + BUILD_PAD]; };

// out[t] = min|max(in[t], in[t + off]) on every 16-bit lane of the window
template <bool MIN, bool ODD> __device__ __forceinline__ void win_step_t(const Window &in, Window &out, int woff)
{
#pragma unroll
    for (int r = 0; r < (BUILD_WORDS + BUILD_THREADS - 1) / BUILD_THREADS; ++r) {
        const int w = threadIdx.x + r * BUILD_THREADS;
        if ((r + 1) * BUILD_THREADS <= BUILD_WORDS || w < BUILD_WORDS) {
            const u32 a = in.w[w];
            u32 b = in.w[w + woff];
            if (ODD) b = __funnelshift_r(b, in.w[w + woff + 1], 16);
            out.w[w] = MIN ? __vminu2(a, b) : __vmaxu2(a, b);
        }
    }
    __syncthreads();
}
template <bool MIN> __device__ __forceinline__ void win_step(const Window &in, Window &out, int off)
{
    if (off & 1) win_step_t<MIN, true>(in, out, off >> 1);
    else win_step_t<MIN, false>(in, out, off >> 1);
}
// Sliding minimum over W entries starting at t, continued from a window `cur` that already holds the
// minimum over p0 entries (p0 a power of two <= W).  Returns the window holding the result.
__device__ const Window *sliding_min(const Window *cur, Window *a, Window *b, int p0, int W)
{
    int p = p0;
    Window *nxt = (cur == a) ? b : a;
    while (2 * p <= W) {
        win_step<true>(*cur, *nxt, p);
        cur = nxt;
        nxt = (nxt == a) ? b : a;
        p *= 2;
    }
    if (p < W) { win_step<true>(*cur, *nxt, W - p); cur = nxt; }
    return cur;
}
// res[t] = max_{u = t-W+1 .. t+1} m[u]: sliding maximum over W+1 entries, re-based to the body index
__device__ void sliding_max_to(const Window *m, Window *a, Window *b, Window &res, int W)
{
    const int V = W + 1;
    int p = 1;
    const Window *cur = m;
    Window *nxt = (m == a) ? b : a;
    while (2 * p <= V) {
        win_step<false>(*cur, *nxt, p);
        cur = nxt;
        nxt = (nxt == a) ? b : a;
        p *= 2;
    }
    if (p < V) { win_step<false>(*cur, *nxt, V - p); cur = nxt; }
    for (int w = threadIdx.x; w < BUILD_WORDS; w += BUILD_THREADS) {
        const int q = 2 * w - (W - 1);   // first lane of the source word
        u32 v = 0;
        if (q >= 0) {
            v = cur->w[q >> 1];
            if (q & 1) v = __funnelshift_r(v, cur->w[(q >> 1) + 1], 16);
        } else if (q == -1) {
            v = cur->w[0] << 16;
        }
        res.w[w] = v;
    }
    __syncthreads();
}

__device__ __forceinline__ int win_get(const Window &win, int t) { return (int)((win.w[t >> 1] >> ((t & 1) * 16)) & 0xffffu); }

// ------------------------------------------------------------------------------------------------
// B1: leaf level and cut flag of every body; per-tile node counts and group bookkeeping; the last
//     tile to finish turns them into prefixes over tiles
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(BUILD_THREADS) levels_kernel(const signed char *__restrict__ clev, u8 *__restrict__ dlev,
                                                               u8 *__restrict__ cutflag, TileRec *tiles, u32 *level_total,
                                                               u32 *prev_ncells, u32 n, u32 ntiles, int max_level, int nleaf, int ngroup,
                                                               int merge_levels, u64 *counters)
{
    // windows: c, leaf level, group level, minimum over NLEAF entries, two scratch
    __shared__ Window s_c, s_d, s_g, s_m, s_a, s_b;
    __shared__ int s_cnt[32];
    __shared__ u32 s_tile, s_lastcut;
    const int tid = threadIdx.x, lane = tid & 31;
    P3T_GRID_TRIGGER();
    if (tid == 0) { s_tile = (u32)atomicAdd(&counters[CNT_HEAD_TICKET], 1ull); s_lastcut = 0; }   // tiles in scheduling order (look-back)
    __syncthreads();
    P3T_GRID_WAIT();
    const u32 tile = s_tile;
    const long long base = (long long)tile * BUILD_TILE;
    // ---- window of biased c values (c + 1 in 0..22; 0 outside the array), two per word
    for (int q = tid; q < BUILD_WORDS / 2; q += BUILD_THREADS) {   // four c values (one 32-bit load) -> two words
        const long long g = base - BUILD_HALO + 4 * q;
        u32 raw = 0xffffffffu;   // c = -1 outside the array
        if (g >= 0 && g <= (long long)n) raw = *reinterpret_cast<const u32 *>(clev + g);
        u32 cb[4];
#pragma unroll
        for (int h = 0; h < 4; ++h) cb[h] = (g + h <= (long long)n) ? (u32)((int)(signed char)(raw >> (8 * h)) + 1) : 0u;
        s_c.w[2 * q] = cb[0] | (cb[1] << 16);
        s_c.w[2 * q + 1] = cb[2] | (cb[3] << 16);
    }
    if (tid < BUILD_PAD) {
        s_c.w[BUILD_WORDS + tid] = 0; s_m.w[BUILD_WORDS + tid] = 0;
        s_a.w[BUILD_WORDS + tid] = 0; s_b.w[BUILD_WORDS + tid] = 0;
    }
    if (tid < 32) s_cnt[tid] = 0;
    __syncthreads();
    {
        // minimum over min(NLEAF, NGROUP) entries first (kept in s_m), continued to the larger width
        const int w1 = min(nleaf, ngroup), w2 = max(nleaf, ngroup);
        const Window *m1 = sliding_min(&s_c, &s_a, &s_b, 1, w1);
        for (int w = tid; w < BUILD_WORDS; w += BUILD_THREADS) s_m.w[w] = m1->w[w];
        __syncthreads();
        int p1 = 1;
        while (2 * p1 <= w1) p1 *= 2;
        // the chain can only be continued from a power-of-two width: restart from there if w1 is not one
        const Window *m2;
        if (p1 == w1) m2 = sliding_min(&s_m, &s_a, &s_b, w1, w2);
        else m2 = sliding_min(&s_c, &s_a, &s_b, 1, w2);
        Window &res2 = (w2 == ngroup) ? s_g : s_d, &res1 = (w2 == ngroup) ? s_d : s_g;
        sliding_max_to(m2, &s_a, &s_b, res2, w2);
        sliding_max_to(&s_m, &s_a, &s_b, res1, w1);
    }
    // ---- my bodies: leaf level, cut flag, node counts per level (difference array)
    {
        const long long i0 = base + tid * BUILD_PER_THREAD;
        u32 dl = 0, cf = 0;
#pragma unroll
        for (int s = 0; s < BUILD_PER_THREAD; ++s) {
            const int t = BUILD_HALO + tid * BUILD_PER_THREAD + s;
            const long long i = i0 + s;
            if (i < (long long)n) {
                const int c = win_get(s_c, t) - 1;
                const int D = min(max_level, win_get(s_d, t));
                const int g = min(max_level, win_get(s_g, t)), gp = i > 0 ? min(max_level, win_get(s_g, t - 1)) : 0;
                // a group may straddle cells up to merge_levels above the natural group level, but only where that
                // level is at least GROUP_MERGE_MIN_LEVEL: in the sparse outskirts the parent cell is so large that a
                // group of consecutive bodies spans an octant, its box reaches the core and it opens the whole tree
                // (one such group took 4.9 ms at N = 256K, 2.2x the rest of the launch)
                const int gm = max(g, gp);
                // (merge_levels >= P3T_MAX_LEVELS: no cuts at all, groups are plain runs of ngroup consecutive bodies --
                //  what a Peano-Hilbert order allows, whose consecutive bodies are neighbours in space everywhere)
                const int minlev = merge_levels >= P3T_MAX_LEVELS ? 0 : GROUP_MERGE_MIN_LEVEL;
                const bool cut = (i == 0) || c < max(gm - merge_levels, min(gm, minlev));
                dl |= (u32)D << (8 * s);
                cf |= (cut ? 1u : 0u) << (8 * s);
                if (D > c) { atomicAdd(&s_cnt[c + 1], 1); atomicAdd(&s_cnt[D + 1], -1); }
            }
        }
        if (i0 < (long long)n) {   // dlev / cutflag are padded to a multiple of four bytes
            *reinterpret_cast<u32 *>(dlev + i0) = dl;
            *reinterpret_cast<u32 *>(cutflag + i0) = cf;
        }
        if (cf) atomicMax(&s_lastcut, (u32)i0 + (31u - __clz(cf)) / 8u + 1u);   // position + 1 of my last cut
    }
    __syncthreads();
    // ---- warp 0: nodes per level -> look-back over the tiles before -> exclusive prefixes
    if (tid < 32) {
        int v = lane < 24 ? s_cnt[lane] : 0;   // difference array -> counts per level
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            int t = __shfl_up_sync(0xffffffffu, v, o);
            if (lane >= o) v += t;
        }
        u32 tot = 0;
        if (lane < 24) {
            const u32 own = (u32)v;
            const u32 excl = tile_lookback(&tiles[tile].status[lane], tile, own);
            tiles[tile].excl[lane] = excl;
            tot = excl + own;
        } else if (lane == 25) {   // the last cut before this tile: emit_kernel's segments start there
            tiles[tile].excl[25] = tile_lookback_last(&tiles[tile].status[25], tile, s_lastcut);
        }
        if (tile == ntiles - 1) {   // the last tile holds the totals: nodes per level, cells, deepest level in use
            if (lane < 24) level_total[lane] = tot;
            const u32 cells = __reduce_add_sync(0xffffffffu, tot);
            const u32 dep = __reduce_max_sync(0xffffffffu, tot ? (u32)lane : 0u);
            if (lane == 0) { counters[CNT_NCELLS] = (u64)cells; counters[CNT_DEPTH] = (u64)dep; *prev_ncells = cells; }
        }
    }
}

// ------------------------------------------------------------------------------------------------
// B2: emit the nodes (start, level, parent, first child, leaf range) and the group heads
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(BUILD_THREADS) emit_kernel(
    const signed char *__restrict__ clev, const u8 *__restrict__ dlev, const u8 *__restrict__ cutflag,
    TileRec *tiles, const u32 *__restrict__ level_total, u32 n, u32 ntiles, int max_level, int ngroup, u32 cell_cap,
    u32 *__restrict__ cell_start, u8 *__restrict__ cell_level, u32 *__restrict__ cell_parent, u32 *__restrict__ cell_first,
    u32 *cell_nchild, uint2 *__restrict__ cell_meta, u32 *__restrict__ group_start, u64 *counters)
{
    __shared__ __align__(16) signed char s_c[BUILD_TILE + BUILD_HALO + 4];   // c[base .. base + TILE + HALO]
    __shared__ u32 s_wcnt[BUILD_THREADS / 32][24];
    __shared__ u32 s_lvloff[24];
    __shared__ int s_lo, s_hi;
    __shared__ int s_wmax[BUILD_THREADS / 32];
    __shared__ u32 s_whead[BUILD_THREADS / 32];
    __shared__ u32 s_tile, s_headbase;
    __shared__ int s_carry;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    P3T_GRID_TRIGGER();
    if (tid == 0) { s_tile = (u32)atomicAdd(&counters[CNT_HEAD_SPARE0], 1ull); s_lo = 99; s_hi = -1; }
    __syncthreads();
    P3T_GRID_WAIT();
    const u32 tile = s_tile;
    const u32 base = tile * BUILD_TILE;
    for (int q = tid; q < (BUILD_TILE + BUILD_HALO + 4) / 4; q += BUILD_THREADS) {   // c[base ..] four at a time
        const u32 g = base + 4 * q;
        u32 raw = 0xffffffffu;
        if (g <= n) raw = *reinterpret_cast<const u32 *>(clev + g);
#pragma unroll
        for (int h = 0; h < 4; ++h)
            if (g + h > n) raw |= 0xffu << (8 * h);
        *reinterpret_cast<u32 *>(&s_c[4 * q]) = raw;
    }
    if (tid < 24) {
        u32 off = 0;
        for (int L = 0; L < tid; ++L) off += level_total[L];
        s_lvloff[tid] = off + tiles[tile].excl[tid];
    }
    // the last cut before the tile: left by levels_kernel (a look-back column of its own; a backward search over the
    // cut flags here cost 0.2 ms at N = 1M once groups were allowed to span several cells)
    if (tid == 0) s_carry = (int)tiles[tile].excl[25] - 1;
    __syncthreads();
    int c[BUILD_PER_THREAD], D[BUILD_PER_THREAD];
    int lo = 99, hi = -1;
    const u32 i0 = base + tid * BUILD_PER_THREAD;
    {
        u32 dl = 0;
        if (i0 + BUILD_PER_THREAD <= n) dl = *reinterpret_cast<const u32 *>(dlev + i0);   // BUILD_PER_THREAD == 4
        else for (int s = 0; s < BUILD_PER_THREAD; ++s) if (i0 + s < n) dl |= (u32)dlev[i0 + s] << (8 * s);
#pragma unroll
        for (int s = 0; s < BUILD_PER_THREAD; ++s) {
            c[s] = 127; D[s] = 0;
            if (i0 + s < n) {
                c[s] = s_c[tid * BUILD_PER_THREAD + s];
                D[s] = (int)((dl >> (8 * s)) & 255u);
                if (D[s] > c[s]) { lo = min(lo, c[s] + 1); hi = max(hi, D[s]); }
            }
        }
    }
    lo = __reduce_min_sync(0xffffffffu, lo);   // levels with nodes starting in this warp's 128 bodies
    hi = __reduce_max_sync(0xffffffffu, hi);
    const int wlo = lo, whi = hi;
    if (lane == 0 && hi >= 0) { atomicMin(&s_lo, lo); atomicMax(&s_hi, hi); }
    __syncthreads();
    const int Llo = s_lo, Lhi = s_hi;   // levels with nodes starting in this tile
    // per-warp node counts per level
    u32 wmask = 0;                      // levels at which this warp has nodes
    for (int L = Llo; L <= Lhi; ++L) {
        u32 cnt = 0;
        if (L >= wlo && L <= whi) {
#pragma unroll
            for (int s = 0; s < BUILD_PER_THREAD; ++s) cnt += (c[s] < L && L <= D[s]) ? 1u : 0u;
            cnt = __reduce_add_sync(0xffffffffu, cnt);
        }
        if (cnt) wmask |= 1u << L;
        if (lane == 0) s_wcnt[warp][L] = cnt;
    }
    __syncthreads();
    if (tid >= Llo && tid <= Lhi) {
        u32 sum = s_lvloff[tid];
        for (int w = 0; w < BUILD_THREADS / 32; ++w) { u32 t = s_wcnt[w][tid]; s_wcnt[w][tid] = sum; sum += t; }
    }
    __syncthreads();
    // ---- group heads: every ngroup-th body of a segment (segments start at cut flags).  Counted first, so that
    //      the tile's count is visible to its successors while the nodes are emitted; resolved at the end.
    u32 head_mask = 0, head_inc = 0, head_mine = 0, head_total = 0;
    {
        u32 cf = 0;
        if (i0 + BUILD_PER_THREAD <= n) cf = *reinterpret_cast<const u32 *>(cutflag + i0);
        else for (int s = 0; s < BUILD_PER_THREAD; ++s) if (i0 + s < n) cf |= (u32)cutflag[i0 + s] << (8 * s);
        int last = -1;
#pragma unroll
        for (int s = 0; s < BUILD_PER_THREAD; ++s) if ((cf >> (8 * s)) & 1u) last = (int)(i0 + s);
        int run = last;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            int t = __shfl_up_sync(0xffffffffu, run, o);
            if (lane >= o) run = max(run, t);
        }
        if (lane == 31) s_wmax[warp] = run;
        __syncthreads();
        int seg = __shfl_up_sync(0xffffffffu, run, 1);
        if (lane == 0) seg = -1;
        seg = max(seg, s_carry);   // cut carried in from the tiles before
        for (int w = 0; w < warp; ++w) seg = max(seg, s_wmax[w]);
        u32 mine = 0;
#pragma unroll
        for (int s = 0; s < BUILD_PER_THREAD; ++s) {
            const u32 i = i0 + s;
            if ((cf >> (8 * s)) & 1u) seg = (int)i;
            const bool hd = i < n && ((i - (u32)seg) % (u32)ngroup) == 0;
            head_mask |= hd ? 1u << s : 0u;
            mine += hd ? 1u : 0u;
        }
        u32 inc = mine;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            u32 t = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += t;
        }
        if (lane == 31) s_whead[warp] = inc;
        head_inc = inc; head_mine = mine;
        __syncthreads();
        for (int w = 0; w < BUILD_THREADS / 32; ++w) head_total += s_whead[w];
        if (tid == 0) tile_publish(&tiles[tile].status[24], tile, head_total);
    }
    // ---- nodes.  rank_L(i) = number of level-L nodes starting before body i; a node's parent is the
    //      level-(L-1) node starting at the same body if there is one, else the last one before it.
    u32 nleaf_here = 0;
    u32 prev_rank[BUILD_PER_THREAD];   // rank at the previous level, per body
    bool prev_flag[BUILD_PER_THREAD];
#pragma unroll
    for (int s = 0; s < BUILD_PER_THREAD; ++s) { prev_rank[s] = 0; prev_flag[s] = false; }
    for (int L = max(wlo - 1, 0); L <= whi; ++L) {
        const bool counted = L >= Llo;   // level Llo-1: ranks only (parents of the topmost nodes)
        if (!((wmask >> L) & 1u)) {      // no node of this warp at this level: every body has the warp's base rank
            const u32 r = counted ? s_wcnt[warp][L] : s_lvloff[L];
#pragma unroll
            for (int s = 0; s < BUILD_PER_THREAD; ++s) { prev_rank[s] = r; prev_flag[s] = false; }
            continue;
        }
        u32 f[BUILD_PER_THREAD], mine = 0;
#pragma unroll
        for (int s = 0; s < BUILD_PER_THREAD; ++s) { f[s] = (counted && c[s] < L && L <= D[s]) ? 1u : 0u; mine += f[s]; }
        u32 inc = mine;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            u32 t = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += t;
        }
        u32 rank = (counted ? s_wcnt[warp][L] : 0u) + inc - mine;
        if (!counted) {
            // nodes of level Llo-1 all start before this tile or are absent: rank = prefix of the tile
            rank = s_lvloff[L];
        }
#pragma unroll
        for (int s = 0; s < BUILD_PER_THREAD; ++s) {
            if (f[s]) {
                const u32 i = i0 + s;
                if (rank < cell_cap) {
                    cell_start[rank] = i;
                    cell_level[rank] = (u8)L;
                    u32 parent = P3T_NO_PARENT;
                    if (L > 0) {
                        parent = prev_flag[s] ? prev_rank[s] : prev_rank[s] - 1;
                        P3T_DEV_ASSERT(parent < rank);
                        atomicAdd(&cell_nchild[parent], L == D[s] ? 1u : 0x10001u);   // children | internal children << 16
                    }
                    cell_parent[rank] = parent;
                    if (prev_flag[s]) cell_first[prev_rank[s]] = rank;
                    if (L == D[s]) {   // leaf: bodies i .. while c[j] >= L
                        const u32 tl = tid * BUILD_PER_THREAD + s;
                        u32 cnt = 1;
                        while (tl + cnt <= BUILD_TILE + BUILD_HALO && s_c[tl + cnt] >= L) ++cnt;
                        if (tl + cnt > BUILD_TILE + BUILD_HALO)
                            while (i + cnt < n && clev[i + cnt] >= L) ++cnt;   // a deep leaf longer than the window
                        P3T_DEV_ASSERT(i + cnt <= n);
                        cell_meta[rank] = make_uint2(i, cnt | P3T_LEAF_FLAG);
                        ++nleaf_here;
                    } else {
                        cell_meta[rank] = make_uint2(0u, 0u);   // internal: completed by moments_kernel
                    }
                } else {
                    atomicOr(&counters[CNT_ERR_BUILD], (u64)ERR_CELL_CAPACITY);
                }
            }
            prev_rank[s] = rank;
            prev_flag[s] = f[s] != 0;
            rank += f[s];
        }
    }
    u32 nl = __reduce_add_sync(0xffffffffu, nleaf_here);
    if (lane == 0 && nl) atomicAdd(&counters[CNT_NLEAVES], (u64)nl);
    // ---- heads of the tiles before this one: look-back (most predecessors are done by now), then the compaction
    {
        if (tid == 0) {
            const u32 excl = tile_resolve(&tiles[tile].status[24], tile, head_total);
            s_headbase = excl;
            if (tile == ntiles - 1) {
                counters[CNT_NGROUPS] = (u64)(excl + head_total);
                group_start[excl + head_total] = n;
            }
        }
        __syncthreads();
        u32 pos = s_headbase + head_inc - head_mine;
        for (int w = 0; w < warp; ++w) pos += s_whead[w];
#pragma unroll
        for (int s = 0; s < BUILD_PER_THREAD; ++s)
            if ((head_mask >> s) & 1u) { P3T_DEV_ASSERT(pos < n); group_start[pos++] = i0 + s; }
    }
}

__global__ void tile_sentinel_kernel(TileRec *recs)
{
    recs[blockIdx.x].status[threadIdx.x] = TL_FLAG_INC;
}

p3t_status p3t_stage_build(p3t_ctx *ctx)
{
    Workspace &w = ctx->ws;
    u32 n = (u32)ctx->n;
    cudaStream_t s = ctx->stream;
    u32 ntiles = div_up(n, BUILD_TILE);
    TileRec *recs = (TileRec *)w.build_tiles;       // BUILD_LOOKBACK sentinel records, then one per tile
    if (!ctx->tiles_ready) {
        tile_sentinel_kernel<<<BUILD_LOOKBACK, 32, 0, s>>>(recs);
        ctx->tiles_ready = true;
    }
    TileRec *tiles = recs + BUILD_LOOKBACK;
    // (the tile records were zeroed by p3t_stage_sort, at the head of the chain)
    static_assert(sizeof(TileRec) == 256 && BUILD_LOOKBACK == 8, "p3t_stage_sort zeroes the records behind 8 sentinels of 256 bytes");
    P3T_CUDA(ctx, p3t_launch_pdl(levels_kernel, dim3(ntiles), dim3(BUILD_THREADS), 0, s, (const signed char *)w.clev, w.dlev, w.cutflag, tiles,
                                 w.level_total, w.prev_ncells, n, ntiles, ctx->max_level, ctx->nleaf, ctx->ngroup, ctx->merge_levels, w.counters));
    P3T_CUDA(ctx, p3t_launch_pdl(emit_kernel, dim3(ntiles), dim3(BUILD_THREADS), 0, s, (const signed char *)w.clev, (const u8 *)w.dlev,
                                 (const u8 *)w.cutflag, tiles, (const u32 *)w.level_total, n, ntiles, ctx->max_level, ctx->ngroup, (u32)w.cell_cap,
                                 w.cell_start, w.cell_level, w.cell_parent, w.cell_first, w.cell_nchild, w.cell_meta, w.group_start, w.counters));
    P3T_CUDA(ctx, cudaGetLastError());
    return P3T_OK;
}
