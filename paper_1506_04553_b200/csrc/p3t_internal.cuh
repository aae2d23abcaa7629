// p3t_internal.cuh -- context, workspace layout and device helpers shared by the
// kernels of the soft-force library (include/p3t.h is the public boundary).
// Nothing here is shared with oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>

#include "p3t.h"

typedef unsigned long long u64;
typedef unsigned int u32;
typedef unsigned char u8;

#define P3T_MAX_LEVELS 22          // levels 0..21 (63-bit keys); 0..10 with 30-bit keys
#define P3T_LEAF_FLAG 0x80000000u
#define P3T_NO_PARENT 0xffffffffu

// ---- tuning constants -------------------------------------------------
#ifndef SORT_THREADS
#define SORT_THREADS 512
#endif
#define SORT_ITEMS 8
#define SORT_TILE (SORT_THREADS * SORT_ITEMS)
#define BUILD_THREADS 256
#define BUILD_TILE 1024               // bodies per CTA of the build kernels (4 per thread)
#define WALK_WARPS 4                 // warps per CTA in the walk kernel
#ifndef WALK_CTAS
#define WALK_CTAS 4                  // resident CTAs per SM the walk kernel is compiled for (register budget)
#endif
#ifndef WALK_STACK_SMEM
#define WALK_STACK_SMEM 512          // stack entries per warp held in shared memory
#endif
#define WALK_STACK_GMEM 7168         // overflow entries per warp in global memory
#ifndef WALK_SPLIT_BELOW_X20
#define WALK_SPLIT_BELOW_X20 26        // auto mode: split walk below 26 / 20 = 1.3 groups (n / ngroup) per resident warp: 2 parts, 4 below 0.65
#endif
#ifndef WALK_SPLIT_CELLS
#define WALK_SPLIT_CELLS 512           // split level: the first tree level with at least this many cells per part
#endif
#ifndef WALK_COOP_BELOW_X20
#define WALK_COOP_BELOW_X20 6          // auto mode: one CTA per group below 6 / 20 = 0.3 groups (n / ngroup) per resident warp; between
                                      // that and 1.3 a split walk (measured, 2368 resident warps, groups of 64: 32K coop 0.36 ms against
                                      // 0.56 split; 64K split x 4 0.56 against coop 0.62; 96K split x 2 0.79 against coop 0.89)
#endif

// Parameters handed to kernels by value.  The coefficients of W are prepared on the host in
// double precision (set_params): for gamma <= y < 1
//   W(y) = sum_{k=0..7} wc[k] y^k + wl * y ln y          (Eq. 16-17 with reading A1)
// and W(y) = cin * y below gamma.  K(x) = x^4 (35 - 84 x + 70 x^2 - 20 x^3)  (Eq. 12).
struct CutoffSet {
    double inv_rout;   // 1 / r_out
    double gamma;      // r_in / r_out
    double inv_1mg;    // 1 / (1 - gamma)
    double cin;        // slope of W below gamma
    double wc[8];
    double wl;
};
// Kinds of pairs when the bodies carry classes (section 3.2.2.1; 0 = field star, 1 = black hole):
// kind = class_i + class_j: 0 FS-FS, 1 BH-FS (its own cutoff radii and neighbour radius, the same softening), 2 BH-BH
// (not split: K = W = 0 in the soft sums, always neighbours, softening eps_bb in the hard part).  Without classes every
// pair is of kind 0.
struct P3TParams {
    float eps2;        // eps^2
    float theta;
    float r_in, r_out, h;
    float rout2;       // r_out^2
    float h2;          // h^2                 (neighbour test  s^2 < h^2, reading A4)
    float hnear2;      // (h (1+1e-5))^2 + slack: bodies whose box distance is below this take the slow path
    int classes;       // bodies carry classes
    float h_bf;        // max(h, h of BH-FS pairs): what a cell with a black hole, or a group with one, keeps clear
    float hnear2_bf;   // hnear2 with h_bf
    float rout2_k[2], h2_k[2];   // per kind of split pair
    double eps2_d;     // eps^2 in double (hard.cu evaluates pairs in fp64)
    double eps2_bb_d;  // softening^2 of the unsplit BH-BH pairs (hard part only)
    CutoffSet cs[2];   // K, W coefficients of kind 0 and kind 1
};

// Device-side counters (one block of 64-bit words in the workspace).  Layout in memory:
//   hist [8][256] u32 | counters: build words, load words, eval words | order_hist [2][1024] u32
// so that each stage zeroes what it needs with ONE memset: the build hist + build words, load the whole
// counter block, an evaluation the eval words + order_hist.
enum {
    // zeroed at every build (together with the digit histograms in front of the block)
    CNT_NCELLS = 0, CNT_NLEAVES, CNT_NGROUPS, CNT_DEPTH, CNT_ERR_BUILD, CNT_HEAD_TICKET, CNT_HEAD_SPARE0,
    CNT_SORT_NRUNS /* runs of keys equal on the sorted upper bits that sort_long_runs_kernel takes */,
    CNT_SORT_TICKET = 8 /* one per pass, 8 */,
    CNT_SORT_MAXRUN = 8 /* longest such run, if above 16: the ticket word of pass 0, which does not run when runs can exist */,
    // words from CNT_ERR_BUILD on are zeroed at load (the tree counts in front survive: a refit needs them)
    CNT_NONFINITE = 16,
    CNT_STRAY = 17 /* refit: bodies that left the cube of their leaf by more than stray_dist leaf sides */,
    CNT_BBOX = 18 /* three words: six 32-bit min/max accumulators of the bounding cube */,
    // zeroed at every eval (together with order_hist behind the block)
    CNT_NPP = 24, CNT_NPC, CNT_NNEAR, CNT_PAIRS, CNT_GROUP_TICKET, CNT_MAXLIST, CNT_ERR_EVAL, CNT_EVAL_SPARE,
    CNT_WORDS = 32
};
enum { ERR_STACK_OVERFLOW = 1, ERR_CELL_CAPACITY = 2 };

struct Workspace {
    // inputs
    float *in_mass, *in_pos;       // staging for host inputs
    float4 *body_user;             // (x,y,z,m) user order
    // a1-a4
    float *cube;                   // [8]: min xyz, side, max xyz, pad   (cube[0..3] = P3T_ARR_ROOT_CUBE)
    u32 *bbox_bits;                // [6] ordered-int accumulators (inverted min, max), inside the counter block
    u64 *keys[2];
    u32 *idx[2];
    u32 *hist;                     // [8][256] digit histograms -> exclusive offsets
    u32 *tile_status;              // [2][ntiles][256] look-back words, ping-pong between passes
    float4 *body;                  // sorted
    // a5
    signed char *clev;             // [n+1]  common-prefix levels between sorted neighbours (c[0] = -1)
    u8 *dlev;                      // [n] leaf level of each body
    u8 *cutflag;                   // [n] segment cut (group construction)
    void *build_tiles;             // [8 + nblk] 256-byte tile records of build.cu (look-back words, exclusive prefixes)
    u32 *level_total;              // [32]
    u32 *prev_ncells;              // [1] cells of the previous build: their child counters are zeroed by the next one
    u32 *group_start;              // [n+1]
    uint4 *group_stats;            // [n] per-group diagnostics of the last walk (P3T_ARR_GROUP_STATS)
    u32 *group_order;              // [n] groups by decreasing cost of the previous walk (ticket -> group)
    u32 *order_meta;               // [4] [0]: number of groups group_order is a permutation of (0: none)
    u32 *group_class;              // [n] predicted cost class of every group of this walk
    u32 *body_class;               // [n] user order: cost class of the group each body was in at the last walk
    u32 *order_hist;               // [2][1024] groups per cost class, scatter cursors
    // cells
    float4 *cell_mac, *cell_mom0, *cell_mom1, *cell_bmin, *cell_bmax;
    uint2 *cell_meta;
    u8 *cell_level;
    u32 *cell_start, *cell_parent, *cell_first, *cell_nchild, *cell_ready;
    // outputs
    float4 *accpot;                // user order (ax, ay, az, phi)
    u32 *nbr_count;                // user order
    u64 *nbr_offset;               // [n+1]
    uint2 *pairs;                  // [cap] (i_user, j_user)
    u32 *nbr;                      // [cap]
    u32 *nbr_cursor;               // [n]
    u32 *subset;                   // [n] staging for eval_direct
    u32 *hilbert_tab;              // [24 * 64 + 24 * 8] state tables of the Peano-Hilbert keys (sort.cu: p3t_hilbert_tables)
    u8 *cls_user, *cls_sorted;     // [n] class of every body (0 field star, 1 black hole), user order and Morton order
    double *hard_out;              // [7n] staging of p3t_eval_hard's host outputs (acc 3n, jerk 3n, pot n); of p3t_hermite_step's pos, vel
    u32 *herm_ids;                 // [n] non-isolated particles by connected component of the neighbour graph (hermite.cu)
    u32 *herm_parent, *herm_root, *herm_csize, *herm_cstart;   // [n] union-find parent, root, component size / fill cursor, first member slot
    uint2 *herm_comps;             // [n/2] (start, size) of the components one warp integrates
    u64 *herm_tdt;                 // [n] t << 8 | log2 dt, in ticks
    double *herm_state;            // [4][3 max_n] a, a1 and the block's new a, a1
    u64 *herm_ctl;                 // [16] counts, cursors, rotating block times, statistics
    u64 *herm_bigctl;              // [8 per cluster-tier component] rotating block times, active count
    u64 *counters;                 // [CNT_WORDS]
    u32 *walk_stack;               // [nwarps][WALK_STACK_GMEM]
    u64 *scan_tmp;                 // [nblk_scan + 1]
    size_t total_bytes;
    size_t cell_cap, n_tiles_max, n_blk_max, walk_warps_max;
};

struct p3t_ctx {
    int device;
    cudaStream_t stream;
    cudaStream_t side_stream;      // Hermite part: warp and cluster tiers beside the grid tier
    cudaEvent_t ev_fork, ev_join;
    size_t max_n, n, nbr_capacity;
    int key_bits, max_level, nleaf, ngroup, merge_levels;
    int key_curve;                 // 0 Morton, 1 Peano-Hilbert (default)
    int walk_parts_used;           // of the last walk: 1, 2, 4 (split) or 0 (cooperative)
    bool merge_user_set;           // p3t_set_group_merge_levels was called: p3t_set_key_curve keeps its value
    int herm_cluster_max;          // largest component a thread-block cluster integrates (larger ones: grid kernel)
    int walk_mode;                 // 0 auto, 1 one warp per group, 2 one CTA per group (cooperative)
    size_t cls_n;                  // 0: no classes; else the particle count the classes were given for
    float r_in_bf, r_out_bf, r_search_bf, eps_bb;
    double herm_eta_bh, herm_eta_s_bh, herm_a0_bh;   // Hermite part: accuracy parameters of class 1 (<= 0 / < 0: those of the call)
    bool shard_classes_fresh;      // p3t_put_shard_classes since the last sharded walk: all ranks hold the same cost classes
    int shard_rank, shard_world;   // this context walks the groups at positions rank, rank + world, ... of the hand-out order
    int sm_count;
    bool have_params, loaded, built, evaluated;
    bool lists_complete;           // the last evaluation made the lists of ALL particles (not a shard, not a subset): they are symmetric
    bool hard_unchecked;           // a device-form p3t_eval_hard whose capacity check is still due (sync_and_check)
    bool sort_attr_set, walk_attr_set;   // cudaFuncSetAttribute done on this context's device
    int sort_ctas_per_sm;
    bool topo_valid;               // sorted order, cells and groups of the last p3t_build_tree are intact (n, tree parameters unchanged)
    size_t topo_n;                 // particles of that build
    int refits, max_refits;        // refits since that build; p3t_refit_tree rebuilds after max_refits of them
    float stray_dist, max_stray_fraction;
    u64 last_stray;                // stray count of the last refit
    bool last_rebuilt;             // the last p3t_refit_tree ended in a rebuild
    bool cells_dirty;              // child counters need a memset before the next build
    bool tiles_ready;              // sentinel records of the build look-back written
    bool status_clean;             // the look-back buffers have been zeroed once (they clean themselves afterwards)
    int cur;                       // which of keys[2]/idx[2] holds the sorted result
    int sort_passes_user;          // p3t_set_sort_passes: 0 = chosen by the library
    int sort_extra_bits;           // upper key bits added to the plan after a build met long runs (sync_and_check)
    int sort_passes_used;          // radix passes of the last build
    u64 build_count, sort_adapted_build;   // builds started; the build whose run statistics were last looked at
    P3TParams prm;
    float eps, theta, r_in, r_out, r_search;
    Workspace ws;
    char *base;
    cudaEvent_t ev[14];            // phase boundaries: 0 build start,1 sort end,2 build end,3 moments end,4 eval start,5 walk end,6 nbr end,7/8 hard,9/10 pack,11/12 hermite
    bool ev_build, ev_eval, ev_hard, ev_pack;
    char err[512];
    // host mirrors (valid after sync)
    u64 h_counters[CNT_WORDS];
};

// coefficients of K and W for one pair of cutoff radii (api.cu)
void p3t_fill_cutoff(CutoffSet &c, float r_in, float r_out);

// Lays the arrays out over `base` (may be NULL to only measure).  Returns total bytes.
size_t p3t_layout(Workspace &ws, char *base, size_t max_n, int key_bits, size_t nbr_capacity, int sm_count);

#define P3T_CUDA(ctx, call)                                                                        \
    do {                                                                                           \
        cudaError_t e_ = (call);                                                                   \
        if (e_ != cudaSuccess) {                                                                   \
            snprintf((ctx)->err, sizeof((ctx)->err), "%s failed: %s (%s:%d)", #call,               \
                     cudaGetErrorString(e_), __FILE__, __LINE__);                                  \
            return P3T_ECUDA;                                                                      \
        }                                                                                          \
    } while (0)

static inline p3t_status p3t_fail(p3t_ctx *ctx, p3t_status st, const char *msg)
{
    if (ctx) snprintf(ctx->err, sizeof(ctx->err), "%s", msg);
    return st;
}

static inline u32 div_up(size_t a, size_t b) { return (u32)((a + b - 1) / b); }

#ifdef __CUDACC__
// Programmatic dependent launch: the kernels of the a1-a6 chain are launched with the stream-serialisation attribute,
// so a kernel's CTAs may become resident and run their prologue (ticket, shared-memory clears, parameter loads) while
// the kernel before it drains; P3T_GRID_WAIT() (griddepcontrol.wait) stands in front of the first access to anything
// a predecessor wrote or still reads, P3T_GRID_TRIGGER() (griddepcontrol.launch_dependents) at the top of each kernel.
// Every kernel launched this way must execute P3T_GRID_WAIT() on all paths: completion is only transitive through it.
#define P3T_GRID_WAIT() cudaGridDependencySynchronize()
#define P3T_GRID_TRIGGER() cudaTriggerProgrammaticLaunchCompletion()
template <class K, class... A>
static inline cudaError_t p3t_launch_pdl(K kernel, dim3 grid, dim3 block, size_t smem, cudaStream_t s, A... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = s;
    cudaLaunchAttribute attr;
    attr.id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr.val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = &attr; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, args...);
}
#endif

// stage entry points (each enqueues kernels on ctx->stream)
p3t_status p3t_stage_pack(p3t_ctx *ctx, const float *d_mass, const float *d_pos);
#define P3T_HILBERT_STATES 24
#define P3T_HILBERT_TAB_WORDS (P3T_HILBERT_STATES * 64 + P3T_HILBERT_STATES * 8)
bool p3t_hilbert_tables(u32 *tab /* [P3T_HILBERT_TAB_WORDS], host */);
p3t_status p3t_stage_sort(p3t_ctx *ctx);
p3t_status p3t_stage_build(p3t_ctx *ctx);
p3t_status p3t_stage_moments(p3t_ctx *ctx);
p3t_status p3t_stage_refit_begin(p3t_ctx *ctx);
p3t_status p3t_stage_refit_finish(p3t_ctx *ctx);
p3t_status p3t_stage_walk(p3t_ctx *ctx);
p3t_status p3t_stage_shard_record(p3t_ctx *ctx, float *d_rec);
p3t_status p3t_stage_shard_classes(p3t_ctx *ctx, const float *d_rec);
p3t_status p3t_stage_direct(p3t_ctx *ctx, const u32 *d_subset, size_t n_subset);
p3t_status p3t_stage_neighbours(p3t_ctx *ctx);
p3t_status p3t_stage_unpack(p3t_ctx *ctx, float *d_acc, float *d_pot, cudaStream_t stream = nullptr);   // nullptr: the context's stream
p3t_status p3t_stage_hard(p3t_ctx *ctx, const float *d_vel, double *d_acc, double *d_jerk, double *d_pot);
p3t_status p3t_stage_hermite(p3t_ctx *ctx, double *d_pos, double *d_vel, double T, int log2_div, double eta, double eta_s,
                             double a0, long long max_blocks, u64 *h_ctl);
p3t_status p3t_stage_kick(p3t_ctx *ctx, double *d_vel, double dt);
p3t_status p3t_stage_narrow(p3t_ctx *ctx, const double *d_pos, float *d_pos32);

#ifdef __CUDACC__
// Checked build (P3T_CHECKED=1 python -m paper_1506_04553_b200.build --force; profiles/sanitizer_r2.md): every index a
// kernel takes from the tree, a list or a look-back result is tested against the size of the array it goes into; a
// violation prints the place and traps (the launch fails, the next API call returns P3T_ECUDA).  Nothing in a normal build.
#ifdef P3T_CHECKED
#define P3T_DEV_ASSERT(cond)                                                                                         \
    do {                                                                                                             \
        if (!(cond)) {                                                                                               \
            printf("P3T_DEV_ASSERT failed: %s (%s:%d) block %u thread %u\n", #cond, __FILE__, __LINE__, blockIdx.x, threadIdx.x); \
            __trap();                                                                                                \
        }                                                                                                            \
    } while (0)
#else
#define P3T_DEV_ASSERT(cond) do { } while (0)
#endif

// ---- device helpers ----------------------------------------------------------------------------

// Cutoff weights on the slow path (pairs with s < r_out), double precision because the closed
// form of W cancels from terms of size ~57 at gamma = 0.1 (hard part 8).
__device__ __forceinline__ void p3t_pair_weights(const CutoffSet &p, float s2, float &K, float &W)
{
    double s = sqrt((double)s2);
    double y = s * p.inv_rout;
    if (y >= 1.0) { K = 1.f; W = 1.f; return; }
    if (y < p.gamma) { K = 0.f; W = (float)(p.cin * y); return; }
    double x = (y - p.gamma) * p.inv_1mg;
    double x2 = x * x;
    double k = x2 * x2 * (35.0 + x * (-84.0 + x * (70.0 - 20.0 * x)));
    double w = p.wc[7];
#pragma unroll
    for (int i = 6; i >= 0; --i) w = w * y + p.wc[i];
    w += p.wl * y * log(y);
    K = (float)k;
    W = (float)w;
}

__device__ __forceinline__ u32 lanemask_lt()
{
    u32 m;
    asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
    return m;
}

// ---- space-filling curve of the keys (A25) -------------------------------------------------------------
// Both curves interleave three `bits`-bit integers (first most significant): for Morton keys these are the quantised
// coordinates themselves, for Peano-Hilbert keys their image under Skilling's transform ("Programming the Hilbert
// curve", AIP Conf. Proc. 707, 2004).  Either way a level-l cell is the run of keys that share their top 3 l bits.
__device__ __forceinline__ u64 p3t_spread3(u32 v)   // bit k -> bit 3k (21 bits)
{
    u64 x = v & 0x1fffffu;
    x = (x | x << 32) & 0x1f00000000ffffull;
    x = (x | x << 16) & 0x1f0000ff0000ffull;
    x = (x | x << 8) & 0x100f00f00f00f00full;
    x = (x | x << 4) & 0x10c30c30c30c30c3ull;
    x = (x | x << 2) & 0x1249249249249249ull;
    return x;
}
__device__ __forceinline__ u32 p3t_compact3(u64 x)   // bit 3k -> bit k
{
    x &= 0x1249249249249249ull;
    x = (x ^ (x >> 2)) & 0x10c30c30c30c30c3ull;
    x = (x ^ (x >> 4)) & 0x100f00f00f00f00full;
    x = (x ^ (x >> 8)) & 0x1f0000ff0000ffull;
    x = (x ^ (x >> 16)) & 0x1f00000000ffffull;
    x = (x ^ (x >> 32)) & 0x1fffffull;
    return (u32)x;
}
// quantised coordinates -> key
__device__ __forceinline__ u64 p3t_encode_key(u32 x, u32 y, u32 z, int bits, int hilbert)
{
    if (hilbert) {
        // Skilling: AxestoTranspose, written without branches (a warp's lanes take all paths anyway):
        //   if (X[i] & Q) X[0] ^= P; else { t = (X[0] ^ X[i]) & P; X[0] ^= t; X[i] ^= t; }    for i = 0, 1, 2
        for (int b = bits - 1; b > 0; --b) {
            const u32 P = (1u << b) - 1u;
            x ^= P & (0u - ((x >> b) & 1u));                    // i = 0: invert (the exchange with itself is void)
            u32 hit = 0u - ((y >> b) & 1u), t = (x ^ y) & P & ~hit;
            x ^= (P & hit) | t; y ^= t;
            hit = 0u - ((z >> b) & 1u); t = (x ^ z) & P & ~hit;
            x ^= (P & hit) | t; z ^= t;
        }
        y ^= x; z ^= y;                                         // Gray encode
        u32 t = 0;
        for (int b = bits - 1; b > 0; --b) t ^= ((1u << b) - 1u) & (0u - ((z >> b) & 1u));
        x ^= t; y ^= t; z ^= t;
    }
    return (p3t_spread3(x) << 2) | (p3t_spread3(y) << 1) | p3t_spread3(z);
}
// key -> quantised coordinates (all `bits` bits; a level-l cell index is the result >> (bits - l))
__device__ __forceinline__ void p3t_decode_key(u64 key, int bits, int hilbert, u32 &x, u32 &y, u32 &z)
{
    x = p3t_compact3(key >> 2); y = p3t_compact3(key >> 1); z = p3t_compact3(key);
    if (hilbert) {
        u32 t = z >> 1;                                         // Skilling: TransposetoAxes
        z ^= y; y ^= x; x ^= t;
        for (u32 Q = 2u; Q != (2u << (bits - 1)); Q <<= 1) {
            const u32 P = Q - 1u;
            if (z & Q) x ^= P; else { t = (x ^ z) & P; x ^= t; z ^= t; }
            if (y & Q) x ^= P; else { t = (x ^ y) & P; x ^= t; y ^= t; }
            if (x & Q) x ^= P;
        }
    }
}

// order-preserving float <-> uint mapping for atomicMin/Max on floats
__device__ __forceinline__ u32 float_to_ordered(float f)
{
    u32 u = __float_as_uint(f);
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float ordered_to_float(u32 u)
{
    return __uint_as_float((u & 0x80000000u) ? (u & 0x7fffffffu) : ~u);
}
#endif
