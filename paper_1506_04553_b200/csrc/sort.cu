// sort.cu -- rows a1-a4 of the hot path:
//   a1 bounding cube, a2 Morton keys, a3 onesweep LSD radix sort of (key, index), a4 body gather.
// The paper only says "Barnes-Hut tree algorithm"; the key/sort formulation is
// this library's own (north_star).  All kernels are HBM/L2-bandwidth bound.
#include "p3t_internal.cuh"

#include <vector>

// ------------------------------------------------------------------------------------------------
// a1: pack (mass, pos) -> float4 bodies in user order, min/max of positions, finiteness check
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) pack_bbox_kernel(const float *__restrict__ mass, const float *__restrict__ pos,
                                                        float4 *__restrict__ body, u32 *bbox_bits, u64 *counters, u32 n)
{
    float lo[3] = {INFINITY, INFINITY, INFINITY}, hi[3] = {-INFINITY, -INFINITY, -INFINITY};
    int bad = 0;
    for (u32 i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        float x = pos[3 * (size_t)i], y = pos[3 * (size_t)i + 1], z = pos[3 * (size_t)i + 2], m = mass[i];
        body[i] = make_float4(x, y, z, m);
        bad |= !(isfinite(x) && isfinite(y) && isfinite(z) && isfinite(m));
        lo[0] = fminf(lo[0], x); hi[0] = fmaxf(hi[0], x);
        lo[1] = fminf(lo[1], y); hi[1] = fmaxf(hi[1], y);
        lo[2] = fminf(lo[2], z); hi[2] = fmaxf(hi[2], z);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            lo[d] = fminf(lo[d], __shfl_xor_sync(0xffffffffu, lo[d], o));
            hi[d] = fmaxf(hi[d], __shfl_xor_sync(0xffffffffu, hi[d], o));
        }
    }
    __shared__ float s_lo[8][3], s_hi[8][3];
    __shared__ int s_bad;
    if (threadIdx.x == 0) s_bad = 0;
    __syncthreads();
    int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (lane == 0) {
        for (int d = 0; d < 3; ++d) { s_lo[warp][d] = lo[d]; s_hi[warp][d] = hi[d]; }
    }
    if (bad) s_bad = 1;
    __syncthreads();
    if (threadIdx.x < 3) {
        int d = threadIdx.x;
        float l = s_lo[0][d], h = s_hi[0][d];
        for (int w = 1; w < 8; ++w) { l = fminf(l, s_lo[w][d]); h = fmaxf(h, s_hi[w][d]); }
        atomicMax(&bbox_bits[d], ~float_to_ordered(l));   // minimum kept inverted: zero is the neutral start of both halves
        atomicMax(&bbox_bits[3 + d], float_to_ordered(h));
    }
    if (threadIdx.x == 0 && s_bad) atomicAdd(&counters[CNT_NONFINITE], 1ull);
}

p3t_status p3t_stage_pack(p3t_ctx *ctx, const float *d_mass, const float *d_pos)
{
    Workspace &w = ctx->ws;
    u32 n = (u32)ctx->n;
    // load words (non-finite flag, bounding-cube accumulators), the build's error word and tickets, the eval words; the
    // tree counts in front (cells, leaves, groups, depth) survive a load: p3t_refit_tree works on the old tree
    P3T_CUDA(ctx, cudaMemsetAsync(w.counters + CNT_ERR_BUILD, 0, (CNT_WORDS - CNT_ERR_BUILD) * sizeof(u64), ctx->stream));
    u32 grid = min(div_up(n, 256 * 4), (u32)ctx->sm_count * 8);
    pack_bbox_kernel<<<grid, 256, 0, ctx->stream>>>(d_mass, d_pos, w.body_user, w.bbox_bits, w.counters, n);
    P3T_CUDA(ctx, cudaGetLastError());
    return P3T_OK;
}

// ------------------------------------------------------------------------------------------------
// unpack: float4 (ax, ay, az, phi) user order -> acc[3n], pot[n]
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) unpack_kernel(const float4 *__restrict__ ap, float *acc, float *pot, u32 n)
{
    P3T_GRID_TRIGGER();
    P3T_GRID_WAIT();
    u32 i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    float4 v = ap[i];
    if (acc) { acc[3 * (size_t)i] = v.x; acc[3 * (size_t)i + 1] = v.y; acc[3 * (size_t)i + 2] = v.z; }
    if (pot) pot[i] = v.w;
}

p3t_status p3t_stage_unpack(p3t_ctx *ctx, float *d_acc, float *d_pot, cudaStream_t stream)
{
    u32 n = (u32)ctx->n;
    if (!d_acc && !d_pot) return P3T_OK;
    P3T_CUDA(ctx, p3t_launch_pdl(unpack_kernel, dim3(div_up(n, 256)), dim3(256), 0, stream ? stream : ctx->stream, (const float4 *)ctx->ws.accpot, d_acc, d_pot, n));
    return P3T_OK;
}

// ------------------------------------------------------------------------------------------------
// a2: root cube + Morton keys + digit histograms of all passes
// ------------------------------------------------------------------------------------------------

// ---- Peano-Hilbert keys by table (A25) ------------------------------------------------------------------
// Skilling's transform (p3t_encode_key) walks all bits of all three coordinates for every level: ~600 instructions per
// body.  The curve it defines is self-similar: inside a cell the order of the eight octants is one of 24 "states"
// (orientations), and the state of a child follows from the parent's state and the child's octant.  The tables are not
// typed in: p3t_hilbert_tables derives them on the host from the plain transform on a 32^3 lattice and checks that
// they are consistent (same state, same octant -> same child state) before any context uses them.
//   tab[state * 64 + two octants (6 bits)] = next state << 6 | two key digits (6 bits)      two levels per step
//   tab[24 * 64 + state * 8 + octant]      = next state << 3 | key digit                     the odd last level
static void host_hilbert_transpose(u32 &x, u32 &y, u32 &z, int bits)   // Skilling's AxestoTranspose, plain
{
    u32 X[3] = {x, y, z};
    for (u32 Q = 1u << (bits - 1); Q > 1u; Q >>= 1) {
        const u32 P = Q - 1u;
        for (int i = 0; i < 3; ++i) {
            if (X[i] & Q) X[0] ^= P;
            else { const u32 t = (X[0] ^ X[i]) & P; X[0] ^= t; X[i] ^= t; }
        }
    }
    for (int i = 1; i < 3; ++i) X[i] ^= X[i - 1];
    u32 t = 0;
    for (u32 Q = 1u << (bits - 1); Q > 1u; Q >>= 1)
        if (X[2] & Q) t ^= Q - 1u;
    x = X[0] ^ t; y = X[1] ^ t; z = X[2] ^ t;
}

bool p3t_hilbert_tables(u32 *tab)
{
    const int B = 5, N = 1 << B;
    // digit[l] of every lattice point, and the octant -> digit map of every cell (level, prefix path of octants)
    std::vector<std::vector<u32>> maps(B);                 // per level: 8 digits per prefix, packed 3 bits each; ~0u = unset
    for (int l = 0; l < B; ++l) maps[l].assign((size_t)1 << (3 * l), 0u);
    std::vector<std::vector<u32>> seen(B);
    for (int l = 0; l < B; ++l) seen[l].assign((size_t)1 << (3 * l), 0u);
    for (u32 x = 0; x < (u32)N; ++x) for (u32 y = 0; y < (u32)N; ++y) for (u32 z = 0; z < (u32)N; ++z) {
        u32 tx = x, ty = y, tz = z;
        host_hilbert_transpose(tx, ty, tz, B);
        u32 pre = 0;
        for (int l = 0; l < B; ++l) {
            const int b = B - 1 - l;
            const u32 oct = ((x >> b) & 1u) << 2 | ((y >> b) & 1u) << 1 | ((z >> b) & 1u);
            const u32 dig = ((tx >> b) & 1u) << 2 | ((ty >> b) & 1u) << 1 | ((tz >> b) & 1u);
            if ((seen[l][pre] >> oct) & 1u) { if (((maps[l][pre] >> (3 * oct)) & 7u) != dig) return false; }
            else { maps[l][pre] |= dig << (3 * oct); seen[l][pre] |= 1u << oct; }
            pre = pre * 8 + oct;
        }
    }
    // states = distinct maps, numbered in order of discovery from the root; transitions must be functions of (state, octant)
    std::vector<u32> state_map;                            // state -> packed map
    auto state_of = [&](u32 m) { for (size_t s = 0; s < state_map.size(); ++s) if (state_map[s] == m) return (int)s; state_map.push_back(m); return (int)state_map.size() - 1; };
    int next[64][8];
    for (auto &r : next) for (int &v : r) v = -1;
    for (int l = 0; l + 1 < B; ++l)
        for (size_t pre = 0; pre < maps[l].size(); ++pre) {
            const int s = state_of(maps[l][pre]);
            if (s >= 64) return false;
            for (u32 oct = 0; oct < 8; ++oct) {
                const int c = state_of(maps[l + 1][pre * 8 + oct]);
                if (c >= 64) return false;
                if (next[s][oct] >= 0 && next[s][oct] != c) return false;
                next[s][oct] = c;
            }
        }
    if (state_map.size() != P3T_HILBERT_STATES || state_of(maps[0][0]) != 0) return false;
    for (int s = 0; s < P3T_HILBERT_STATES; ++s)
        for (u32 oct = 0; oct < 8; ++oct) {
            if (next[s][oct] < 0) return false;
            tab[P3T_HILBERT_STATES * 64 + s * 8 + oct] = (u32)next[s][oct] << 3 | ((state_map[s] >> (3 * oct)) & 7u);
        }
    for (int s = 0; s < P3T_HILBERT_STATES; ++s)
        for (u32 o2 = 0; o2 < 64; ++o2) {
            const u32 e1 = tab[P3T_HILBERT_STATES * 64 + s * 8 + (o2 >> 3)], e2 = tab[P3T_HILBERT_STATES * 64 + (e1 >> 3) * 8 + (o2 & 7u)];
            tab[s * 64 + o2] = (e2 >> 3) << 6 | (e1 & 7u) << 3 | (e2 & 7u);
        }
    return true;
}

// quantised coordinates -> Peano-Hilbert key with the tables in shared memory
__device__ __forceinline__ u64 hilbert_key_tab(const u32 *s_tab, u32 x, u32 y, u32 z, int bits)
{
    // interleave first: the octants of all levels as 3-bit groups (x most significant), then two levels per lookup
    const u64 m = (p3t_spread3(x) << 2) | (p3t_spread3(y) << 1) | p3t_spread3(z);
    u64 key = 0;
    u32 st = 0;
    int b = bits;
    for (; b >= 2; b -= 2) {
        const u32 e = s_tab[st * 64 + (u32)((m >> (3 * (b - 2))) & 63u)];
        key = key << 6 | (e & 63u);
        st = e >> 6;
    }
    if (b) {
        const u32 e = s_tab[P3T_HILBERT_STATES * 64 + st * 8 + (u32)(m & 7u)];
        key = key << 3 | (e & 7u);
    }
    return key;
}

// Root cube from the reduced min/max: centre = midpoint of the AABB, side = largest extent padded
// so that the maximum maps inside.  Every thread recomputes it (6 loads), block 0 publishes it.
__device__ __forceinline__ void root_cube(const u32 *bbox_bits, float &minx, float &miny, float &minz, float &side)
{
    float lo[3], hi[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) { lo[d] = ordered_to_float(~bbox_bits[d]); hi[d] = ordered_to_float(bbox_bits[3 + d]); }
    float ext = fmaxf(hi[0] - lo[0], fmaxf(hi[1] - lo[1], hi[2] - lo[2]));
    side = ext * (1.f + 4e-6f);
    if (!(side > 0.f) || !isfinite(side)) side = 1.f;
    minx = 0.5f * (lo[0] + hi[0]) - 0.5f * side;
    miny = 0.5f * (lo[1] + hi[1]) - 0.5f * side;
    minz = 0.5f * (lo[2] + hi[2]) - 0.5f * side;
}

__global__ void __launch_bounds__(256) keys_hist_kernel(const float4 *__restrict__ body, const u32 *__restrict__ bbox_bits,
                                                        float *cube, u64 *__restrict__ keys, u32 *hist, u32 n,
                                                        int max_level, const u32 *__restrict__ hilbert_tab, int first_pass, int passes, const u32 *__restrict__ prev_ncells,
                                                        u32 cell_cap, u32 *cell_nchild, u32 *cell_ready)
{
    // child counters of the cells of the previous build -> 0 (emit_kernel accumulates into them)
    for (u32 k = blockIdx.x * blockDim.x + threadIdx.x, nc = min(*prev_ncells, cell_cap); k < nc; k += gridDim.x * blockDim.x) {
        cell_nchild[k] = 0;
        cell_ready[k] = 0;
    }
    __shared__ u32 s_hist[8 * 256];
    __shared__ u32 s_tab[P3T_HILBERT_TAB_WORDS];
    for (int t = threadIdx.x; t < 8 * 256; t += blockDim.x) s_hist[t] = 0;
    if (hilbert_tab)
        for (int t = threadIdx.x; t < P3T_HILBERT_TAB_WORDS; t += blockDim.x) s_tab[t] = hilbert_tab[t];
    float minx, miny, minz, side;
    root_cube(bbox_bits, minx, miny, minz, side);
    if (blockIdx.x == 0 && threadIdx.x == 0) { cube[0] = minx; cube[1] = miny; cube[2] = minz; cube[3] = side; }
    const float scale = (float)(1u << max_level) / side;
    const u32 qmax = (1u << max_level) - 1u;
    __syncthreads();
    for (u32 i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        float4 b = body[i];
        u32 qx = min((u32)fmaxf((b.x - minx) * scale, 0.f), qmax);
        u32 qy = min((u32)fmaxf((b.y - miny) * scale, 0.f), qmax);
        u32 qz = min((u32)fmaxf((b.z - minz) * scale, 0.f), qmax);
        u64 key = hilbert_tab ? hilbert_key_tab(s_tab, qx, qy, qz, max_level) : p3t_encode_key(qx, qy, qz, max_level, 0);
        keys[i] = key;
        for (int p = first_pass; p < passes; ++p) atomicAdd(&s_hist[p * 256 + (u32)((key >> (8 * p)) & 255u)], 1u);
    }
    __syncthreads();
    for (int t = first_pass * 256 + threadIdx.x; t < passes * 256; t += blockDim.x) {
        u32 v = s_hist[t];
        if (v) atomicAdd(&hist[t], v);
    }
}

// ------------------------------------------------------------------------------------------------
// a3: one onesweep pass: stable 8-bit digit partition, chained over tiles by decoupled look-back
// ------------------------------------------------------------------------------------------------
// A tile is SORT_TILE consecutive keys, taken in ticket order (so every predecessor of a running tile
// is running or done).  Per tile and bin one status word (flag | count) is published twice: the tile's
// own count (AGG) as soon as it is known, the inclusive prefix (INC) once the look-back has reached
// an INC word.  All tiles of a 1M-body pass are resident at once and publish their AGG words at about
// the same time, so a look-back that reads one predecessor per L2 round trip needs ~sqrt(2 tiles)
// dependent round trips (measured 35 us per pass); here every thread keeps SORT_LOOKBACK loads in
// flight and consumes them in order, which divides the number of round trips by sqrt(SORT_LOOKBACK).
// The status words of pass p live in buffer p & 1; every tile also zeroes its row of the other
// buffer, which the next pass uses, so no memset runs between passes or between builds.
#define OS_FLAG_AGG 0x40000000u
#define OS_FLAG_INC 0x80000000u
#define OS_VAL_MASK 0x3fffffffu
#define SORT_LOOKBACK 16   // sentinel rows in front of row 0 (the widest look-back window)

__device__ __forceinline__ u32 ld_status(const u32 *p)
{
    u32 v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_status(u32 *p, u32 v)
{
    asm volatile("st.relaxed.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

__global__ void fill_u32_kernel(u32 *p, u32 v) { p[blockIdx.x * blockDim.x + threadIdx.x] = v; }

// Lanes of the warp that hold the same 8-bit digit ("peers") come from a per-warp table of lane masks in shared memory:
// every lane ORs its bit into the word of its digit and reads the word back.  (MATCH.ANY gives the same mask in one
// instruction but sustains only about one warp instruction per 35 cycles per SM on B200 -- it was a third of the pass;
// eight ballots per item were 35 % of the pass's instructions; the table costs two shared-memory operations per item:
// a1-a4 at N = 1M 0.131 -> 0.124 ms, at 16M 1.41 -> 1.38 ms.)
struct OnesweepSmem {
    union {
        u32 whist[SORT_THREADS / 32][256];                      // ranking: per-warp digit counts
        struct { u64 key[SORT_TILE]; u32 val[SORT_TILE]; } x;   // exchange: the tile in digit order
    };
    u32 wmask[SORT_THREADS / 32][256];   // ranking: lanes of the warp that hold each digit in the current round
    u32 binstart[256];   // first local position of each bin
    u32 goff[256];       // global position of local position 0 of each bin, minus binstart
    u32 wsum[8];
    u32 tile;
};

// status rows -SORT_LOOKBACK..-1 (in front of row 0) permanently hold INC | 0, so the look-back
// window never needs a bounds check
template <int LB>   // look-back window: 16 when the whole grid is resident (all tiles publish at once), 8 otherwise
__global__ void __launch_bounds__(SORT_THREADS, 1024 / SORT_THREADS) onesweep_kernel(const u64 *__restrict__ kin, const u32 *__restrict__ vin,
                                                                   u64 *__restrict__ kout, u32 *__restrict__ vout, u32 n,
                                                                   int shift, const u32 *__restrict__ ghist, u32 *status,
                                                                   u32 *status_next, u64 *ticket)
{
    extern __shared__ __align__(16) unsigned char os_raw[];
    OnesweepSmem &sm = *reinterpret_cast<OnesweepSmem *>(os_raw);
    const u32 tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    // tiles must start in index order for the look-back to make progress: guaranteed by a ticket, or by the
    // grid being resident as a whole (ticket == nullptr)
    P3T_GRID_TRIGGER();
    if (tid == 0) sm.tile = ticket ? (u32)atomicAdd(ticket, 1ull) : blockIdx.x;
#pragma unroll
    for (u32 t = 0; t < 8; ++t) { sm.whist[warp][t * 32 + lane] = 0; sm.wmask[warp][t * 32 + lane] = 0; }
    __syncthreads();
    P3T_GRID_WAIT();      // the pass before: its keys and values, and its last reads of the status rows zeroed below
    const u32 tile = sm.tile;
    P3T_DEV_ASSERT(tile < (n + SORT_TILE - 1) / SORT_TILE);
    const u32 tile_base = tile * SORT_TILE;
    const u32 tile_valid = min((u32)SORT_TILE, n - tile_base);
    if (tid < 256) status_next[(size_t)tile * 256 + tid] = 0;   // row of the buffer the next pass uses

    u64 key[SORT_ITEMS];
    u32 val[SORT_ITEMS], pos[SORT_ITEMS];
    const u32 wbase = tile_base + warp * (SORT_ITEMS * 32);
#pragma unroll
    for (int k = 0; k < SORT_ITEMS; ++k) {
        u32 i = wbase + k * 32 + lane;
        bool ok = i < n;
        key[k] = ok ? kin[i] : ~0ull;       // padding keys have digit 255 and rank behind every real key
        val[k] = ok ? (vin ? vin[i] : i) : 0u;
    }
    // global base of every bin: exclusive scan of this pass's histogram (256 counts)
    u32 gcount = 0, ginc = 0;
    if (tid < 256) {
        gcount = ghist[tid];
        ginc = gcount;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            u32 t = __shfl_up_sync(0xffffffffu, ginc, o);
            if (lane >= o) ginc += t;
        }
        if (lane == 31) sm.wsum[warp] = ginc;
    }
    // stable rank inside the warp, items in (k, lane) order.  Per item: the peer mask through the warp's table; the
    // lowest peer (the leader) advances the warp's counter of that digit by the number of peers and clears the word for the
    // next round.  Round k's updates are ordered before round k+1's by the __syncwarp()s (different lanes may lead the same
    // digit in different rounds).
    u32 peers[SORT_ITEMS];
#pragma unroll
    for (int k = 0; k < SORT_ITEMS; ++k) {
        const u32 d = (u32)(key[k] >> shift) & 255u;
        atomicOr(&sm.wmask[warp][d], 1u << lane);
        __syncwarp();
        peers[k] = sm.wmask[warp][d];
        __syncwarp();
        pos[k] = 0;
        if ((peers[k] & lanemask_lt()) == 0) {
            sm.wmask[warp][d] = 0;
            pos[k] = atomicAdd(&sm.whist[warp][d], (u32)__popc(peers[k]));
        }
        __syncwarp();
    }
#pragma unroll
    for (int k = 0; k < SORT_ITEMS; ++k)
        pos[k] = __shfl_sync(0xffffffffu, pos[k], __ffs(peers[k]) - 1) + __popc(peers[k] & lanemask_lt());
    __syncthreads();
    // threads 0..255 own one bin each: exclusive over warps, tile total, publish, look back
    u32 sum = 0, gbase = 0;
    if (tid < 256) {
        for (u32 w = 0; w < warp; ++w) gbase += sm.wsum[w];
        gbase += ginc - gcount;
#pragma unroll
        for (int w = 0; w < SORT_THREADS / 32; ++w) {
            u32 t = sm.whist[w][tid];
            sm.whist[w][tid] = sum;
            sum += t;
        }
        if (tid == 255) sum -= SORT_TILE - tile_valid;   // padding keys are not part of the data
        st_status(status + (size_t)tile * 256 + tid, sum | (tile == 0 ? OS_FLAG_INC : OS_FLAG_AGG));
    }
    __syncthreads();          // wsum is read above, rewritten below
    u32 inc = sum;
    if (tid < 256) {
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            u32 t = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += t;
        }
        if (lane == 31) sm.wsum[warp] = inc;
    }
    __syncthreads();
    if (tid < 256) {
        u32 wb = 0;
        for (u32 w = 0; w < warp; ++w) wb += sm.wsum[w];
        const u32 binstart = wb + inc - sum;
        sm.binstart[tid] = binstart;
        u32 excl = 0;
        if (tile > 0) {
            const u32 *p = status + (size_t)(tile - 1) * 256 + tid;
            bool done = false;
            while (!done) {
                u32 v[LB];
#pragma unroll
                for (int k = 0; k < LB; ++k) v[k] = ld_status(p - k * 256);
                bool go = true;
                u32 used = 0;
#pragma unroll
                for (int k = 0; k < LB; ++k) {
                    const bool ready = v[k] >= OS_FLAG_AGG, isinc = v[k] >= OS_FLAG_INC;
                    if (go && ready) { excl += v[k] & OS_VAL_MASK; ++used; }
                    done = done || (go && isinc);
                    go = go && ready && !isinc;
                }
                p -= used * 256;
            }
            st_status(status + (size_t)tile * 256 + tid, (excl + sum) | OS_FLAG_INC);
        }
        sm.goff[tid] = gbase + excl - binstart;
    }
    __syncthreads();
    // final local position of every item (the per-warp counts are dead after this)
#pragma unroll
    for (int k = 0; k < SORT_ITEMS; ++k) {
        u32 d = (u32)(key[k] >> shift) & 255u;
        pos[k] += sm.binstart[d] + sm.whist[warp][d];
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < SORT_ITEMS; ++k) {
        if (pos[k] < tile_valid) {       // padding keys sit behind the valid ones
            sm.x.key[pos[k]] = key[k];
            sm.x.val[pos[k]] = val[k];
        }
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < SORT_ITEMS; ++k) {
        u32 p = k * SORT_THREADS + tid;
        if (p < tile_valid) {
            u64 kk = sm.x.key[p];
            u32 d = (u32)(kk >> shift) & 255u;
            u32 dst = sm.goff[d] + p;
            P3T_DEV_ASSERT(dst < n);
            kout[dst] = kk;
            vout[dst] = sm.x.val[p];
        }
    }
}

// ------------------------------------------------------------------------------------------------
// a3, last step when the radix passes covered only the UPPER key bits (p3t_stage_sort): the keys are then sorted up to
// runs of keys that agree on those bits, each run still in index order (the passes are stable).  Sorting every run by
// the full key, stably, gives exactly the order of the full radix sort.  Runs are short when the upper bits reach below
// the leaf level of the tree (a few keys): the thread at the head of a run sorts it by insertion, in place.  Longer runs
// (a plan that was too optimistic for this distribution: the next build takes more passes, sync_and_check) go to a list
// and are sorted by one CTA each, bitonic on (key, idx) pairs -- idx breaks ties, which is the stable order.
// Every run is touched by one thread or one CTA only; neighbours read no more than the upper bits of a foreign key,
// which do not change while its run is permuted (8-byte loads and stores are single transactions).
// ------------------------------------------------------------------------------------------------
#define SORT_RUN_INLINE 32        // longest run the head thread sorts itself
#define SORT_RUN_SMEM 2048        // longest run sort_long_runs_kernel sorts in shared memory

__global__ void __launch_bounds__(256) sort_fix_kernel(u64 *keys, u32 *idx, u32 n, int tail_bits, u32 *__restrict__ runs, u64 *counters)
{
    P3T_GRID_TRIGGER();
    P3T_GRID_WAIT();
    const u32 i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const volatile u64 *vk = keys;
    const u64 ti = vk[i] >> tail_bits;
    if (i > 0 && (vk[i - 1] >> tail_bits) == ti) return;     // inside a run: its head takes care
    u32 len = 1;
    while (i + len < n && len <= SORT_RUN_INLINE && (vk[i + len] >> tail_bits) == ti) ++len;
    if (len == 1) return;
    if (len > 16) atomicMax(reinterpret_cast<unsigned long long *>(&counters[CNT_SORT_MAXRUN]), (unsigned long long)len);
    if (len > SORT_RUN_INLINE) {
        runs[atomicAdd(reinterpret_cast<unsigned long long *>(&counters[CNT_SORT_NRUNS]), 1ull)] = i;
        return;
    }
    for (u32 a = 1; a < len; ++a) {                           // stable insertion sort of (key, idx)[i, i + len)
        const u64 ka = keys[i + a];
        const u32 va = idx[i + a];
        u32 b = a;
        while (b > 0 && keys[i + b - 1] > ka) {
            keys[i + b] = keys[i + b - 1];
            idx[i + b] = idx[i + b - 1];
            --b;
        }
        if (b != a) { keys[i + b] = ka; idx[i + b] = va; }
    }
}

// bitonic network with all comparisons ascending (first step of every merge is the flip i ^ (k - 1)): positions
// behind the end of the run act as +infinity and never take part, so any length works
template <class KP, class VP>
__device__ __forceinline__ void run_bitonic(KP key, VP val, u32 len)
{
    u32 m = 1;
    while (m < len) m <<= 1;
    for (u32 k = 2; k <= m; k <<= 1) {
        for (u32 j = k >> 1; j > 0; j >>= 1) {
            for (u32 t = threadIdx.x; t < m; t += blockDim.x) {
                const u32 l = (j == (k >> 1)) ? (t ^ (k - 1)) : (t ^ j);
                if (l > t && l < len) {
                    const u64 a = key[t], b = key[l];
                    const u32 va = val[t], vb = val[l];
                    if (a > b || (a == b && va > vb)) { key[t] = b; key[l] = a; val[t] = vb; val[l] = va; }
                }
            }
            __syncthreads();
        }
    }
}

__global__ void __launch_bounds__(256) sort_long_runs_kernel(u64 *keys, u32 *idx, u32 n, int tail_bits, const u32 *__restrict__ runs,
                                                             u64 *counters)
{
    P3T_GRID_TRIGGER();
    P3T_GRID_WAIT();
    __shared__ u64 s_key[SORT_RUN_SMEM];
    __shared__ u32 s_val[SORT_RUN_SMEM];
    __shared__ u32 s_len;
    const u32 nruns = (u32)counters[CNT_SORT_NRUNS];
    for (u32 r = blockIdx.x; r < nruns; r += gridDim.x) {
        const u32 start = runs[r];
        const u64 t0 = keys[start] >> tail_bits;
        if (threadIdx.x == 0) s_len = n - start;
        __syncthreads();
        for (u32 base = 0; start + base < n; base += blockDim.x) {     // first position whose upper bits differ
            const u32 pos = start + base + threadIdx.x;
            if (pos < n && (keys[pos] >> tail_bits) != t0) atomicMin(&s_len, base + threadIdx.x);
            __syncthreads();
            const u32 found = s_len;
            __syncthreads();
            if (found <= base + blockDim.x) break;
        }
        const u32 len = s_len;
        if (threadIdx.x == 0) atomicMax(reinterpret_cast<unsigned long long *>(&counters[CNT_SORT_MAXRUN]), (unsigned long long)len);
        if (len <= SORT_RUN_SMEM) {
            for (u32 t = threadIdx.x; t < len; t += blockDim.x) { s_key[t] = keys[start + t]; s_val[t] = idx[start + t]; }
            __syncthreads();
            run_bitonic(s_key, s_val, len);
            for (u32 t = threadIdx.x; t < len; t += blockDim.x) { keys[start + t] = s_key[t]; idx[start + t] = s_val[t]; }
        } else {
            // Very long runs are what coincident bodies make (equal FULL keys, at any number of passes), and those are in
            // order already: the passes are stable, so equal keys stand in index order.  One look before sorting.
            __shared__ u32 s_inv;
            if (threadIdx.x == 0) s_inv = 0;
            __syncthreads();
            u32 inv = 0;
            for (u32 t = threadIdx.x; t + 1 < len; t += blockDim.x) inv |= keys[start + t] > keys[start + t + 1] ? 1u : 0u;
            if (inv) s_inv = 1;
            __syncthreads();
            if (s_inv) run_bitonic(keys + start, idx + start, len);     // in global memory: slow, and correct
        }
        __syncthreads();
    }
}

// ------------------------------------------------------------------------------------------------
// a4: gather bodies into sorted order; common-prefix level between sorted neighbours
// ------------------------------------------------------------------------------------------------
// clev[i] = number of leading octree levels on which key[i-1] and key[i] agree (0..max_level);
// clev[0] = clev[n] = -1.
__global__ void __launch_bounds__(256) gather_kernel(const float4 *__restrict__ body_user, const u32 *__restrict__ idx,
                                                     const u64 *__restrict__ keys, float4 *__restrict__ body,
                                                     signed char *__restrict__ clev, u32 n, int max_level,
                                                     const u8 *__restrict__ cls_user, u8 *__restrict__ cls_sorted,
                                                     u32 *__restrict__ status_last, u32 status_words)
{
    P3T_GRID_TRIGGER();
    P3T_GRID_WAIT();
    u32 i = blockIdx.x * blockDim.x + threadIdx.x;
    // the look-back rows of the last radix pass -> 0: the first pass of the next build may be any digit, and both status
    // buffers must be clean for it (every pass zeroes the rows of the pass behind it, nobody those of the last one)
    if (i < status_words) status_last[i] = 0;
    if (i > n) return;
    if (i == n) { clev[n] = -1; return; }
    const u32 src = idx[i];
    P3T_DEV_ASSERT(src < n);
    body[i] = body_user[src];
    if (cls_user) cls_sorted[i] = cls_user[src] & 1u;   // pair classes (p3t_set_pair_classes): 0 field star, 1 black hole
    int c = -1;
    if (i > 0) {
        u64 x = keys[i] ^ keys[i - 1];
        if (x == 0) c = max_level;
        else {
            int hb = 63 - __clzll((long long)x);
            c = max_level - hb / 3 - 1;
        }
    }
    clev[i] = (signed char)c;
}

// grid of keys_hist_kernel (instruction-bound at 1M and beyond, where 8 / 4 / 2 / 1 bodies per thread measure alike; at 64K the
// smaller share per thread is worth 6 us)
#ifndef KEYS_BODIES_PER_THREAD
#define KEYS_BODIES_PER_THREAD 2
#define KEYS_CTAS_PER_SM 8
#endif

p3t_status p3t_stage_sort(p3t_ctx *ctx)
{
    Workspace &w = ctx->ws;
    u32 n = (u32)ctx->n;
    cudaStream_t s = ctx->stream;
    const int passes = (3 * ctx->max_level + 7) / 8;   // 8 for 63-bit keys, 4 for 30-bit keys
    // Plan: radix passes over the UPPER digits only, the rest by sort_fix_kernel.  The upper bits must reach below the leaf
    // level of the tree for the runs to be short: log2 n + 14 bits to begin with (n / 16 leaves spread over a cube with a
    // core a few levels deeper than the mean), 8 more after every build that met a run above 24 keys.
    int first_pass = 0;
    if (ctx->sort_passes_user > 0) first_pass = passes - min(ctx->sort_passes_user, passes);
    else if (ctx->max_level == 21) {
        int lg = 0;
        while ((1ull << lg) < (u64)n) ++lg;
        const int need = lg + 14 + ctx->sort_extra_bits;
        first_pass = max(0, min(passes - 1, (3 * ctx->max_level - need) / 8));
    }
    ctx->sort_passes_used = passes - first_pass;
    ++ctx->build_count;
    u32 ntiles = div_up(n, SORT_TILE);
    if (!ctx->sort_attr_set) {   // function attributes are per device: kept per context
        P3T_CUDA(ctx, cudaFuncSetAttribute(onesweep_kernel<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(OnesweepSmem)));
        P3T_CUDA(ctx, cudaFuncSetAttribute(onesweep_kernel<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(OnesweepSmem)));
        P3T_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&ctx->sort_ctas_per_sm, onesweep_kernel<16>, SORT_THREADS, sizeof(OnesweepSmem)));
        ctx->sort_attr_set = true;
    }
    const size_t status_rows = w.n_tiles_max + SORT_LOOKBACK;   // SORT_LOOKBACK sentinel rows in front of row 0
    const int resident = ctx->sort_ctas_per_sm * ctx->sm_count;   // a grid up to this size is co-resident: no ticket needed
    if (!ctx->status_clean) {   // first build of this context: buffers zeroed, sentinel rows = INC | 0 
        P3T_CUDA(ctx, cudaMemsetAsync(w.tile_status, 0, 2 * status_rows * 256 * sizeof(u32), s));
        for (int b = 0; b < 2; ++b)
            fill_u32_kernel<<<SORT_LOOKBACK, 256, 0, s>>>(w.tile_status + b * status_rows * 256, OS_FLAG_INC);
        ctx->status_clean = true;
    }
    // digit histograms + build counters + sort tickets: contiguous, one memset
    P3T_CUDA(ctx, cudaMemsetAsync(w.hist, 0, (size_t)((char *)(w.counters + CNT_NONFINITE) - (char *)w.hist), s));
    u32 grid = min(div_up(n, 256 * KEYS_BODIES_PER_THREAD), (u32)ctx->sm_count * KEYS_CTAS_PER_SM);   // every CTA flushes its non-empty histogram bins with global atomics
    if (ctx->cells_dirty) {   // first build, or the last one ended in an error: all child counters and prev_ncells -> 0
        P3T_CUDA(ctx, cudaMemsetAsync(w.cell_nchild, 0, (size_t)((char *)(w.cell_ready + w.cell_cap) - (char *)w.cell_nchild), s));
        P3T_CUDA(ctx, cudaMemsetAsync(w.prev_ncells, 0, sizeof(u32), s));
        ctx->cells_dirty = false;
    }
    // (the build's tile records are zeroed here, not in front of levels_kernel: a memset between two kernels would break
    //  the chain of programmatic launches)
    P3T_CUDA(ctx, cudaMemsetAsync(reinterpret_cast<char *>(w.build_tiles) + 8 * 256, 0, (size_t)div_up(n, BUILD_TILE) * 256, s));
    keys_hist_kernel<<<grid, 256, 0, s>>>(w.body_user, w.bbox_bits, w.cube, w.keys[0], w.hist, n, ctx->max_level, ctx->key_curve ? w.hilbert_tab : nullptr, first_pass, passes,
                                          w.prev_ncells, (u32)w.cell_cap, w.cell_nchild, w.cell_ready);
    int cur = 0;
    for (int p = first_pass; p < passes; ++p) {
        u32 *st_cur = w.tile_status + ((size_t)(p & 1) * status_rows + SORT_LOOKBACK) * 256;
        u32 *st_next = w.tile_status + ((size_t)((p + 1) & 1) * status_rows + SORT_LOOKBACK) * 256;
        const u32 *vin = p == first_pass ? nullptr : w.idx[cur];   // the first pass makes idx = iota itself
        // (tiles always take their index from the ticket: the order in which resident CTAs of a look-back chain start is
        //  not something CUDA promises, least of all next to other work on the device)
        u64 *ticket = w.counters + CNT_SORT_TICKET + p;
        if (ntiles <= (u32)resident)
            P3T_CUDA(ctx, p3t_launch_pdl(onesweep_kernel<16>, dim3(ntiles), dim3(SORT_THREADS), sizeof(OnesweepSmem), s, (const u64 *)w.keys[cur], vin,
                                         w.keys[cur ^ 1], w.idx[cur ^ 1], n, 8 * p, (const u32 *)(w.hist + p * 256), st_cur, st_next, ticket));
        else
            P3T_CUDA(ctx, p3t_launch_pdl(onesweep_kernel<8>, dim3(ntiles), dim3(SORT_THREADS), sizeof(OnesweepSmem), s, (const u64 *)w.keys[cur], vin,
                                         w.keys[cur ^ 1], w.idx[cur ^ 1], n, 8 * p, (const u32 *)(w.hist + p * 256), st_cur, st_next, ticket));
        cur ^= 1;
    }
    ctx->cur = cur;
    if (first_pass > 0) {   // runs of keys equal on the sorted bits -> full order (group_class: free until the walk stage)
        P3T_CUDA(ctx, p3t_launch_pdl(sort_fix_kernel, dim3(div_up(n, 256)), dim3(256), 0, s, w.keys[cur], w.idx[cur], n, 8 * first_pass, w.group_class,
                                     w.counters));
        P3T_CUDA(ctx, p3t_launch_pdl(sort_long_runs_kernel, dim3((u32)ctx->sm_count), dim3(256), 0, s, w.keys[cur], w.idx[cur], n, 8 * first_pass,
                                     (const u32 *)w.group_class, w.counters));
    }
    // (the last pass is the top digit, an odd one: its look-back rows are in buffer 1)
    P3T_CUDA(ctx, p3t_launch_pdl(gather_kernel, dim3(div_up(n + 1, 256)), dim3(256), 0, s, (const float4 *)w.body_user, (const u32 *)w.idx[cur],
                                 (const u64 *)w.keys[cur], w.body, w.clev, n, ctx->max_level,
                                 (const u8 *)(ctx->cls_n ? w.cls_user : nullptr), w.cls_sorted,
                                 w.tile_status + (status_rows + SORT_LOOKBACK) * 256, ntiles * 256u));
    P3T_CUDA(ctx, cudaGetLastError());
    return P3T_OK;
}
