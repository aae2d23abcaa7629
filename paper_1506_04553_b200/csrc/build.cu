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

#define BUILD_HALO 64                                  // >= max(NLEAF, NGROUP)
#define BUILD_WIN (BUILD_TILE + 2 * BUILD_HALO + 16)   // window of c values held per tile (16-bit lanes)
#define BUILD_WORDS (BUILD_WIN / 2)
#define BUILD_PER_THREAD (BUILD_TILE / BUILD_THREADS)  // consecutive bodies per thread

// per-tile record written by levels_kernel, completed by the scan of the last tile
struct TileRec {
    u32 cnt[24];        // nodes per level starting in the tile  -> exclusive prefix over tiles
    int lastcut;        // last cut position inside the tile (-1: none) -> last cut BEFORE the tile
    int firstcut;       // first cut position inside the tile (tile end if none)
    u32 heads_after;    // group heads at or after firstcut         -> exclusive prefix of all heads
    u32 pad[5];
};
static_assert(sizeof(TileRec) == 128, "TileRec is one 128-byte line");

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
                                                               u32 *group_start, u32 n, u32 ntiles, int max_level, int nleaf,
                                                               int ngroup, int merge_levels, u64 *counters)
{
    // windows: c, leaf level, group level, minimum over NLEAF entries, two scratch
    __shared__ Window s_c, s_d, s_g, s_m, s_a, s_b;
    __shared__ int s_cnt[32];
    __shared__ int s_wmax[BUILD_THREADS / 32], s_wfirst[BUILD_THREADS / 32];
    __shared__ u32 s_wheads[BUILD_THREADS / 32];
    __shared__ bool s_last;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const long long base = (long long)blockIdx.x * BUILD_TILE;
    // ---- window of biased c values (c + 1 in 0..22; 0 outside the array), two per word
    for (int w = tid; w < BUILD_WORDS; w += BUILD_THREADS) {
        u32 v = 0;
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            long long g = base - BUILD_HALO + 2 * w + h;
            u32 cb = (g >= 0 && g <= (long long)n) ? (u32)((int)clev[g] + 1) : 0u;
            v |= cb << (16 * h);
        }
        s_c.w[w] = v;
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
    int mycut_last = -1, mycut_first = 0x7fffffff;
    int cuts[BUILD_PER_THREAD];
#pragma unroll
    for (int s = 0; s < BUILD_PER_THREAD; ++s) {
        const int t = BUILD_HALO + tid * BUILD_PER_THREAD + s;
        const long long i = base + tid * BUILD_PER_THREAD + s;
        cuts[s] = -1;
        if (i < (long long)n) {
            const int c = win_get(s_c, t) - 1;
            const int D = min(max_level, win_get(s_d, t));
            const int g = min(max_level, win_get(s_g, t)), gp = i > 0 ? min(max_level, win_get(s_g, t - 1)) : 0;
            dlev[i] = (u8)D;
            const bool cut = (i == 0) || c < max(g, gp) - merge_levels;
            cutflag[i] = cut ? 1 : 0;
            if (cut) { cuts[s] = (int)i; mycut_last = (int)i; mycut_first = min(mycut_first, (int)i); }
            if (D > c) { atomicAdd(&s_cnt[c + 1], 1); atomicAdd(&s_cnt[D + 1], -1); }
        }
    }
    // ---- segment start of every body from the cuts inside the tile (inclusive max-scan)
    int run = mycut_last;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        int t = __shfl_up_sync(0xffffffffu, run, o);
        if (lane >= o) run = max(run, t);
    }
    int wfirst = mycut_first;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) wfirst = min(wfirst, __shfl_xor_sync(0xffffffffu, wfirst, o));
    if (lane == 31) s_wmax[warp] = run;
    if (lane == 0) s_wfirst[warp] = wfirst;
    __syncthreads();
    int seg = __shfl_up_sync(0xffffffffu, run, 1);   // last cut strictly before my first body (inside the tile)
    if (lane == 0) seg = -1;
    for (int w = 0; w < warp; ++w) seg = max(seg, s_wmax[w]);
    u32 heads = 0;   // heads at or after the first cut of the tile
#pragma unroll
    for (int s = 0; s < BUILD_PER_THREAD; ++s) {
        const long long i = base + tid * BUILD_PER_THREAD + s;
        if (cuts[s] >= 0) seg = cuts[s];
        if (i < (long long)n && seg >= 0 && ((u32)(i - seg) % (u32)ngroup) == 0) ++heads;
    }
    heads = __reduce_add_sync(0xffffffffu, heads);
    if (lane == 0) s_wheads[warp] = heads;
    __syncthreads();
    if (tid == 0) {
        TileRec &r = tiles[blockIdx.x];
        int acc = 0;
        for (int L = 0; L < 24; ++L) { acc += s_cnt[L]; r.cnt[L] = (u32)acc; }
        int lastcut = -1, firstcut = 0x7fffffff;
        u32 h = 0;
        for (int w = 0; w < BUILD_THREADS / 32; ++w) { lastcut = max(lastcut, s_wmax[w]); firstcut = min(firstcut, s_wfirst[w]); h += s_wheads[w]; }
        const long long tile_end = min((long long)n, base + BUILD_TILE);
        r.lastcut = lastcut;
        r.firstcut = firstcut == 0x7fffffff ? (int)tile_end : firstcut;
        r.heads_after = h;
        __threadfence();
        s_last = atomicAdd(&counters[CNT_HEAD_TICKET], 1ull) + 1ull == (u64)ntiles;
    }
    __syncthreads();
    if (!s_last) return;
    // ---- last tile to finish: prefixes over all tiles.  Thread k owns a contiguous chunk of tiles.
    __threadfence();
    __shared__ u32 s_scan[BUILD_THREADS / 32][26];
    __shared__ u32 s_tot[26];
    const u32 per = (ntiles + BUILD_THREADS - 1) / BUILD_THREADS;
    const u32 t0 = min(ntiles, (u32)tid * per), t1 = min(ntiles, t0 + per);
    // (1) carried cut position: max-scan of lastcut
    int mc = -1;
    for (u32 t = t0; t < t1; ++t) mc = max(mc, __ldcg(&tiles[t].lastcut));
    int mrun = mc;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        int t = __shfl_up_sync(0xffffffffu, mrun, o);
        if (lane >= o) mrun = max(mrun, t);
    }
    if (lane == 31) s_wmax[warp] = mrun;
    __syncthreads();
    int carry = __shfl_up_sync(0xffffffffu, mrun, 1);
    if (lane == 0) carry = -1;
    for (int w = 0; w < warp; ++w) carry = max(carry, s_wmax[w]);
    // (2) sums: 24 level counts + heads (heads of the leading partial segment depend on the carry)
    u32 sums[25];
#pragma unroll
    for (int k = 0; k < 25; ++k) sums[k] = 0;
    {
        int cpos = carry;
        for (u32 t = t0; t < t1; ++t) {
            const uint4 *src = reinterpret_cast<const uint4 *>(tiles[t].cnt);
#pragma unroll
            for (int q = 0; q < 6; ++q) {
                uint4 v = __ldcg(src + q);
                sums[4 * q] += v.x; sums[4 * q + 1] += v.y; sums[4 * q + 2] += v.z; sums[4 * q + 3] += v.w;
            }
            const long long tb = (long long)t * BUILD_TILE;
            const int fc = __ldcg(&tiles[t].firstcut), lc = __ldcg(&tiles[t].lastcut);
            u32 lead = 0;   // heads in [tb, fc) of the segment that started at cpos
            if (cpos >= 0 && fc > tb) {
                const long long first = cpos + (((tb - cpos) + ngroup - 1) / ngroup) * (long long)ngroup;
                if (first < fc) lead = (u32)((fc - 1 - first) / ngroup + 1);
            }
            sums[24] += lead + __ldcg(&tiles[t].heads_after);
            if (lc >= 0) cpos = lc;
        }
    }
    u32 incl[25];
#pragma unroll
    for (int k = 0; k < 25; ++k) {
        u32 v = sums[k];
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            u32 t = __shfl_up_sync(0xffffffffu, v, o);
            if (lane >= o) v += t;
        }
        incl[k] = v;
        if (lane == 31) s_scan[warp][k] = v;
    }
    __syncthreads();
    if (tid < 25) {
        u32 acc = 0;
        for (int w = 0; w < BUILD_THREADS / 32; ++w) { u32 t = s_scan[w][tid]; s_scan[w][tid] = acc; acc += t; }
        s_tot[tid] = acc;
    }
    __syncthreads();
    {   // (3) write the exclusive prefixes back into the tile records
        u32 run25[25];
#pragma unroll
        for (int k = 0; k < 25; ++k) run25[k] = s_scan[warp][k] + incl[k] - sums[k];
        int cpos = carry;
        for (u32 t = t0; t < t1; ++t) {
            TileRec &r = tiles[t];
            uint4 *dst = reinterpret_cast<uint4 *>(r.cnt);
            u32 own[24];
#pragma unroll
            for (int q = 0; q < 6; ++q) {
                uint4 v = __ldcg(reinterpret_cast<const uint4 *>(r.cnt) + q);
                own[4 * q] = v.x; own[4 * q + 1] = v.y; own[4 * q + 2] = v.z; own[4 * q + 3] = v.w;
                dst[q] = make_uint4(run25[4 * q], run25[4 * q + 1], run25[4 * q + 2], run25[4 * q + 3]);
            }
#pragma unroll
            for (int k = 0; k < 24; ++k) run25[k] += own[k];
            const long long tb = (long long)t * BUILD_TILE;
            const int fc = __ldcg(&r.firstcut), lc = __ldcg(&r.lastcut);
            u32 lead = 0;
            if (cpos >= 0 && fc > tb) {
                const long long first = cpos + (((tb - cpos) + ngroup - 1) / ngroup) * (long long)ngroup;
                if (first < fc) lead = (u32)((fc - 1 - first) / ngroup + 1);
            }
            const u32 h = lead + __ldcg(&r.heads_after);
            r.heads_after = run25[24];
            run25[24] += h;
            r.lastcut = cpos;
            if (lc >= 0) cpos = lc;
        }
    }
    if (tid < 24) level_total[tid] = s_tot[tid];
    if (tid == 0) {
        u64 cells = 0, depth = 0;
        for (int L = 0; L <= max_level; ++L) { cells += s_tot[L]; if (s_tot[L]) depth = (u64)L; }
        counters[CNT_NCELLS] = cells;
        counters[CNT_DEPTH] = depth;
        counters[CNT_NGROUPS] = (u64)s_tot[24];
        group_start[s_tot[24]] = n;
    }
}

// ------------------------------------------------------------------------------------------------
// B2: emit the nodes (start, level, parent, first child, leaf range) and the group heads
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(BUILD_THREADS) emit_kernel(
    const signed char *__restrict__ clev, const u8 *__restrict__ dlev, const u8 *__restrict__ cutflag,
    const TileRec *__restrict__ tiles, const u32 *__restrict__ level_total, u32 n, int max_level, int ngroup, u32 cell_cap,
    u32 *__restrict__ cell_start, u8 *__restrict__ cell_level, u32 *__restrict__ cell_parent, u32 *__restrict__ cell_first,
    u32 *cell_nchild, uint2 *__restrict__ cell_meta, u32 *__restrict__ group_start, u64 *counters)
{
    __shared__ signed char s_c[BUILD_TILE + BUILD_HALO + 4];   // c[base .. base + TILE + HALO]
    __shared__ u32 s_wcnt[BUILD_THREADS / 32][24];
    __shared__ u32 s_lvloff[24];
    __shared__ int s_lo, s_hi;
    __shared__ int s_wmax[BUILD_THREADS / 32];
    __shared__ u32 s_whead[BUILD_THREADS / 32];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const u32 base = blockIdx.x * BUILD_TILE;
    for (int t = tid; t < BUILD_TILE + BUILD_HALO + 1; t += BUILD_THREADS) {
        u32 g = base + t;
        s_c[t] = g <= n ? clev[g] : (signed char)-1;
    }
    if (tid == 0) { s_lo = 99; s_hi = -1; }
    if (tid < 24) {
        u32 off = 0;
        for (int L = 0; L < tid; ++L) off += level_total[L];
        s_lvloff[tid] = off + tiles[blockIdx.x].cnt[tid];
    }
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
    lo = __reduce_min_sync(0xffffffffu, lo);
    hi = __reduce_max_sync(0xffffffffu, hi);
    if (lane == 0 && hi >= 0) { atomicMin(&s_lo, lo); atomicMax(&s_hi, hi); }
    __syncthreads();
    const int Llo = s_lo, Lhi = s_hi;   // levels with nodes starting in this tile
    // per-warp node counts per level
    for (int L = Llo; L <= Lhi; ++L) {
        u32 cnt = 0;
#pragma unroll
        for (int s = 0; s < BUILD_PER_THREAD; ++s) cnt += (c[s] < L && L <= D[s]) ? 1u : 0u;
        cnt = __reduce_add_sync(0xffffffffu, cnt);
        if (lane == 0) s_wcnt[warp][L] = cnt;
    }
    __syncthreads();
    if (tid >= Llo && tid <= Lhi) {
        u32 sum = s_lvloff[tid];
        for (int w = 0; w < BUILD_THREADS / 32; ++w) { u32 t = s_wcnt[w][tid]; s_wcnt[w][tid] = sum; sum += t; }
    }
    __syncthreads();
    // ---- nodes.  rank_L(i) = number of level-L nodes starting before body i; a node's parent is the
    //      level-(L-1) node starting at the same body if there is one, else the last one before it.
    u32 nleaf_here = 0;
    u32 prev_rank[BUILD_PER_THREAD];   // rank at the previous level, per body
    bool prev_flag[BUILD_PER_THREAD];
#pragma unroll
    for (int s = 0; s < BUILD_PER_THREAD; ++s) { prev_rank[s] = 0; prev_flag[s] = false; }
    for (int L = max(Llo - 1, 0); L <= Lhi; ++L) {
        const bool counted = L >= Llo;   // level Llo-1: ranks only (parents of the topmost nodes)
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
                        atomicAdd(&cell_nchild[parent], 1u);
                    }
                    cell_parent[rank] = parent;
                    if (prev_flag[s]) cell_first[prev_rank[s]] = rank;
                    if (L == D[s]) {   // leaf: bodies i .. while c[j] >= L
                        const u32 tl = tid * BUILD_PER_THREAD + s;
                        u32 cnt = 1;
                        while (tl + cnt <= BUILD_TILE + BUILD_HALO && s_c[tl + cnt] >= L) ++cnt;
                        if (tl + cnt > BUILD_TILE + BUILD_HALO)
                            while (i + cnt < n && clev[i + cnt] >= L) ++cnt;   // a deep leaf longer than the window
                        cell_meta[rank] = make_uint2(i, cnt | P3T_LEAF_FLAG);
                        ++nleaf_here;
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
    // ---- group heads: every ngroup-th body of a segment (segments start at cut flags)
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
        seg = max(seg, tiles[blockIdx.x].lastcut);   // cut carried in from the tiles before
        for (int w = 0; w < warp; ++w) seg = max(seg, s_wmax[w]);
        bool head[BUILD_PER_THREAD];
        u32 mine = 0;
#pragma unroll
        for (int s = 0; s < BUILD_PER_THREAD; ++s) {
            const u32 i = i0 + s;
            if ((cf >> (8 * s)) & 1u) seg = (int)i;
            head[s] = i < n && ((i - (u32)seg) % (u32)ngroup) == 0;
            mine += head[s] ? 1u : 0u;
        }
        u32 inc = mine;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            u32 t = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += t;
        }
        if (lane == 31) s_whead[warp] = inc;
        __syncthreads();
        u32 pos = tiles[blockIdx.x].heads_after + inc - mine;
        for (int w = 0; w < warp; ++w) pos += s_whead[w];
#pragma unroll
        for (int s = 0; s < BUILD_PER_THREAD; ++s)
            if (head[s]) group_start[pos++] = i0 + s;
    }
}

p3t_status p3t_stage_build(p3t_ctx *ctx)
{
    Workspace &w = ctx->ws;
    u32 n = (u32)ctx->n;
    cudaStream_t s = ctx->stream;
    u32 ntiles = div_up(n, BUILD_TILE);
    // cell_nchild and cell_ready are adjacent in the workspace: one memset zeroes both
    P3T_CUDA(ctx, cudaMemsetAsync(w.cell_nchild, 0, (size_t)((char *)(w.cell_ready + w.cell_cap) - (char *)w.cell_nchild), s));
    levels_kernel<<<ntiles, BUILD_THREADS, 0, s>>>(w.clev, w.dlev, w.cutflag, (TileRec *)w.build_tiles, w.level_total, w.group_start,
                                                  n, ntiles, ctx->max_level, ctx->nleaf, ctx->ngroup, ctx->merge_levels, w.counters);
    emit_kernel<<<ntiles, BUILD_THREADS, 0, s>>>(w.clev, w.dlev, w.cutflag, (const TileRec *)w.build_tiles, w.level_total, n,
                                                ctx->max_level, ctx->ngroup, (u32)w.cell_cap, w.cell_start, w.cell_level,
                                                w.cell_parent, w.cell_first, w.cell_nchild, w.cell_meta, w.group_start, w.counters);
    P3T_CUDA(ctx, cudaGetLastError());
    return P3T_OK;
}
