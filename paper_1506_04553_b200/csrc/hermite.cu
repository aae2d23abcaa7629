// hermite.cu -- NEXT row of SURVEY.md 8(f), rank 2: one soft step under H_hard on the device.
//
// Procedure step 3 (GPU procedure steps 5-6 of section 2.2, which the paper runs on the host):
// particles with an empty neighbour list drift, x += T v; the others are integrated over T with the fourth-order
// Hermite scheme with block timesteps (Eq. 18-20), the force being Eq. 7 (L63) over the particle's list of
// the last evaluation.  Readings A21-A24 of DESIGN.md: time in ticks of T / 2^40, steps are powers of two of ticks,
// at most T / 2^log2_div, dividing the particle's time; Eq. 20 for the first step; Eq. 18 read as Aarseth's criterion
// with |a| -> sqrt(|a|^2 + a0^2); all active particles of a block are evaluated from the state before the block and
// corrected together.
//
// Design.  During a soft step the lists are fixed, so a particle's arithmetic only involves its connected component of
// the neighbour graph ("neighbour cluster"): block times need to be agreed on inside a component only, and the result
// is the same as with global blocks (the oracle's locality pin S6).  The components are found on the device (lock-free
// union-find: hook by compare-and-swap, flatten, count, lay the members out contiguously).  Three tiers:
//  1. a component of up to 64 particles -- nearly all of them: pairs and triples -- is integrated by ONE WARP, its state
//     in shared memory, its block loop synchronised by __syncwarp and a shuffle minimum;
//  2. a component of up to cluster_max (4096) particles by ONE THREAD-BLOCK CLUSTER of 8 CTAs: cluster barriers, active
//     particles compacted per block, several lanes per list;
//  3. the members of all larger components (percolating cores) together in one cooperative kernel on all SMs: two grid
//     barriers per block, a 64-bit atomicMin per CTA over (t + dt) into rotating words.
// Tiers 1 and 2 run on a side stream beside tier 3.  No launch and no host round trip per block.  Everything fp64; the
// state of tiers 2 and 3 lives in global arrays indexed by particle ((t << 8 | log2 dt), a, a1, the block's new a, a1).
#include "p3t_internal.cuh"
#include <cooperative_groups.h>
#include <math_constants.h>
namespace cg = cooperative_groups;

#define HERM_THREADS 256
#define HERM_TICK_BITS 40
#define HERM_WARP_MAX 64        // largest component one warp integrates
#define HERM_CLUSTER 8           // CTAs of the thread-block cluster that integrates one mid-size component
#define HERM_CLUSTER_THREADS 512
enum { HC_COUNT = 0, HC_TMIN0, HC_TMIN1, HC_TMIN2, HC_BLOCKS, HC_STEPS, HC_FLOOR, HC_ERR,
       HC_NSMALL, HC_SMALL_CURSOR, HC_BIG_CURSOR, HC_NCOMP, HC_MAXCOMP, HC_NBIGC, HC_GRID_CURSOR, HC_WORDS = 16 };
#define HERM_GRID_FLAG 0x80000000u   // cstart: the component's members go to the grid tier's own array
#define HERM_NONFINITE 0x80000000u   // high bit of a thread's floor_hits counter: it met a non-finite force (herm_quantise)

__device__ __forceinline__ void herm_weights(const CutoffSet &p, double s, double &omK, double &dKds)
{
    const double y = s * p.inv_rout;
    if (y >= 1.0) { omK = 0.0; dKds = 0.0; return; }
    if (y < p.gamma) { omK = 1.0; dKds = 0.0; return; }
    const double x = (y - p.gamma) * p.inv_1mg;
    const double x2 = x * x;
    omK = 1.0 - x2 * x2 * (35.0 + x * (-84.0 + x * (70.0 - 20.0 * x)));
    const double u = x * (1.0 - x);
    dKds = 140.0 * u * u * u * p.inv_1mg * p.inv_rout;
}

// ---- connected components of the neighbour graph ---------------------------------------------------------------

__device__ __forceinline__ void herm_set_err(u64 *ctl, u32 code)
{
    atomicMax((unsigned long long *)&ctl[7 /* HC_ERR */], (unsigned long long)code);
}

__device__ __forceinline__ u32 cc_find(volatile u32 *parent, u32 i)
{
    u32 p = parent[i];
    while (p != i) {                       // path halving; pointers only ever move towards the root
        const u32 gp = parent[p];
        if (gp != p) parent[i] = gp;
        i = p;
        p = gp;
    }
    return i;
}

__global__ void cc_init_kernel(const u64 *__restrict__ offset, u32 n, u32 *__restrict__ parent, u32 *__restrict__ csize)
{
    // every particle is its own root, isolated ones too: a list entry may then name ANY particle without the finds
    // below leaving initialised memory (lists that are not symmetric are reported by cc_hook_kernel, not trusted)
    const u32 i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    parent[i] = i;
    csize[i] = 0;
}

// HC_ERR values, the largest wins (atomicMax): 1 = more than max_blocks block steps, 2 = the lists are not symmetric,
// 3 = a non-finite force (coincident particles with eps = 0)
__global__ void cc_hook_kernel(const u64 *__restrict__ offset, const u32 *__restrict__ nbr, u32 n, u32 *parent, u64 *ctl)
{
    const u32 i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    // symmetry of the lists (j in L_i <=> i in L_j), which every tier relies on: binary search of i in the ascending L_j
    for (u64 k = offset[i], e = offset[i + 1]; k < e; ++k) {
        const u32 j = nbr[k];
        bool found = false;
        if (j < n) {
            u64 lo = offset[j], hi = offset[j + 1];
            while (lo < hi) {
                const u64 mid = (lo + hi) >> 1;
                const u32 v = nbr[mid];
                if (v == i) { found = true; break; }
                if (v < i) lo = mid + 1; else hi = mid;
            }
        }
        if (!found) { herm_set_err(ctl, 2u); return; }
    }
    for (u64 k = offset[i], e = offset[i + 1]; k < e; ++k) {
        const u32 j = nbr[k];
        if (j >= i) break;                 // lists ascend; every edge is hooked once, from its larger end
        u32 ri = i, rj = j;
        for (;;) {
            ri = cc_find(parent, ri);
            rj = cc_find(parent, rj);
            if (ri == rj) break;
            if (ri < rj) { const u32 t = ri; ri = rj; rj = t; }
            if (atomicCAS(&parent[ri], ri, rj) == ri) break;       // the larger root goes under the smaller
        }
    }
}

// (the roots go to their own array: writing them into parent[] here would race with the path halving of the finds that
// other threads still run through this particle, which may put a non-root ancestor back)
__global__ void cc_count_kernel(const u64 *__restrict__ offset, u32 n, u32 *parent, u32 *__restrict__ root, u32 *csize, u64 *ctl)
{
    const u32 i = blockIdx.x * blockDim.x + threadIdx.x;
    const bool has = i < n && offset[i + 1] > offset[i];
    if (has) {
        const u32 r = cc_find(parent, i);
        root[i] = r;
        atomicAdd(&csize[r], 1u);
    }
    // one atomic per CTA on the shared counter (non-isolated particles are sparse: one per warp would be one per particle)
    __shared__ u32 s_cnt;
    if (threadIdx.x == 0) s_cnt = 0;
    __syncthreads();
    const u32 m = __ballot_sync(0xffffffffu, has);
    if (m && (threadIdx.x & 31) == 0) atomicAdd(&s_cnt, (u32)__popc(m));
    __syncthreads();
    if (threadIdx.x == 0 && s_cnt) atomicAdd((unsigned long long *)&ctl[HC_COUNT], (unsigned long long)s_cnt);
}

// member ranges: small components (one warp each) from the front of members[], mid-size ones (one thread-block cluster
// each, up to cluster_max members) from the back, the members of still larger ones (all together in the cooperative grid
// kernel) in an array of their own.  HC_COUNT is final here.  One atomic per warp and counter for the many small
// components: the roots of a warp take consecutive ranges (warp scan of the sizes); the few large ones take theirs singly.
__global__ void cc_assign_kernel(const u64 *__restrict__ offset, u32 n, const u32 *__restrict__ root, u32 *csize,
                                 u32 *__restrict__ cstart, uint2 *__restrict__ comps, u32 comps_last, u64 *__restrict__ bigctl,
                                 u32 cluster_max, u64 *ctl)
{
    const u32 i = blockIdx.x * blockDim.x + threadIdx.x, lane = threadIdx.x & 31;
    const bool is_root = i < n && offset[i + 1] > offset[i] && root[i] == i;
    const u32 sz = is_root ? csize[i] : 0u;
    const bool small = is_root && sz <= HERM_WARP_MAX;
    const u32 m_root = __ballot_sync(0xffffffffu, is_root);
    const u32 m_small = __ballot_sync(0xffffffffu, small);
    u32 ss = small ? sz : 0u;                              // inclusive warp scan of the small sizes
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const u32 a = __shfl_up_sync(0xffffffffu, ss, o);
        if (lane >= (u32)o) ss += a;
    }
    const u32 tot_s = __shfl_sync(0xffffffffu, ss, 31);
    const u32 mx = __reduce_max_sync(0xffffffffu, sz);
    // CTA level: the warps take ranges of the CTA's totals (shared-memory atomics), one thread takes the CTA's ranges
    // of the global cursors (roots are sparse: per-warp global atomics would be one per root on the same words)
    __shared__ u32 s_tot[4], s_base[2];                    // [0] member slots, [1] small components, [2] roots, [3] max size
    if (threadIdx.x < 4) s_tot[threadIdx.x] = 0;
    __syncthreads();
    u32 off_s = 0, off_c = 0;
    if (lane == 0 && m_root) {
        if (tot_s) off_s = atomicAdd(&s_tot[0], tot_s);
        if (m_small) off_c = atomicAdd(&s_tot[1], (u32)__popc(m_small));
        atomicAdd(&s_tot[2], (u32)__popc(m_root));
        atomicMax(&s_tot[3], mx);
    }
    __syncthreads();
    if (threadIdx.x == 0 && s_tot[2]) {
        s_base[0] = s_tot[0] ? (u32)atomicAdd((unsigned long long *)&ctl[HC_SMALL_CURSOR], (unsigned long long)s_tot[0]) : 0u;
        s_base[1] = s_tot[1] ? (u32)atomicAdd((unsigned long long *)&ctl[HC_NSMALL], (unsigned long long)s_tot[1]) : 0u;
        atomicAdd((unsigned long long *)&ctl[HC_NCOMP], (unsigned long long)s_tot[2]);
        atomicMax((unsigned long long *)&ctl[HC_MAXCOMP], (unsigned long long)s_tot[3]);
    }
    __syncthreads();
    const u32 base_s = s_base[0] + __shfl_sync(0xffffffffu, off_s, 0);
    const u32 base_c = s_base[1] + __shfl_sync(0xffffffffu, off_c, 0);
    if (!is_root) return;
    u32 st;
    if (small) {
        st = base_s + ss - sz;
        comps[base_c + __popc(m_small & ((1u << lane) - 1))] = make_uint2(st, sz);
    } else if (sz <= cluster_max) {
        st = (u32)ctl[HC_COUNT] - ((u32)atomicAdd((unsigned long long *)&ctl[HC_BIG_CURSOR], (unsigned long long)sz) + sz);
        const u32 c = (u32)atomicAdd((unsigned long long *)&ctl[HC_NBIGC], 1ull);
        comps[comps_last - c] = make_uint2(st, sz);
        bigctl[8 * c + 0] = ~0ull; bigctl[8 * c + 1] = ~0ull; bigctl[8 * c + 2] = ~0ull; bigctl[8 * c + 3] = 0ull;
    } else {
        st = (u32)atomicAdd((unsigned long long *)&ctl[HC_GRID_CURSOR], (unsigned long long)sz) | HERM_GRID_FLAG;
    }
    cstart[i] = st;
    csize[i] = 0;                          // becomes the fill cursor of the scatter
}

__global__ void cc_scatter_kernel(const u64 *__restrict__ offset, u32 n, const u32 *__restrict__ root, u32 *csize,
                                  const u32 *__restrict__ cstart, u32 *__restrict__ members, u32 *__restrict__ grid_members)
{
    const u32 i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n || offset[i + 1] == offset[i]) return;
    const u32 r = root[i];
    const u32 st = cstart[r], p = atomicAdd(&csize[r], 1u);            // order inside a component is irrelevant
    P3T_DEV_ASSERT(r < n && (st & ~HERM_GRID_FLAG) + p < n);
    if (st & HERM_GRID_FLAG) grid_members[(st & ~HERM_GRID_FLAG) + p] = i;
    else members[st + p] = i;
}

__global__ void herm_drift_kernel(const u64 *__restrict__ offset, u32 n, double T, double *__restrict__ pos,
                                  const double *__restrict__ vel)
{
    const u32 i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n || offset[i + 1] > offset[i]) return;
#pragma unroll
    for (int c = 0; c < 3; ++c)       // product and sum rounded separately: the same bits as the plain host expression
        pos[3 * (size_t)i + c] = __dadd_rn(pos[3 * (size_t)i + c], __dmul_rn(T, vel[3 * (size_t)i + c]));
}

// ---- the Hermite scheme -----------------------------------------------------------------------------------------

// (constant divisors are multiplied by their rounded reciprocals: the block loop of a cluster is one dependent chain of
// fp64 operations, a division costs ~30 of them; the oracle divides, the difference is an ulp per operation)
constexpr double kSixth = 1.0 / 6.0;

struct HermConst {
    P3TParams prm;
    double tick, rtick, eta, eta_s, a0;
    double c2, c2_s;               // (eta / tick)^2, (eta_s / tick)^2
    double c2k[2], c2_sk[2], a0k[2];   // pair classes: the same per class of the integrated particle (eta_FS, eta_BH)
    u64 max_ticks, max_blocks;
};

// Where a set of particles keeps its state.  Global view: arrays indexed by particle id, lists hold particle ids, masses
// come from body_user.  Local view (one warp's component): arrays in shared memory indexed by the member's slot, lists
// hold slots, masses in `mass`.
struct HermView {
    double *pos, *vel;             // [.][3]
    double *a, *a1, *an, *a1n;     // [.][3]
    u64 *tdt;                      // t << 8 | log2(dt)
    const u32 *nbr;                // list entries
    const float4 *body_user;       // global view: mass in .w (the masses of the evaluation that made the lists)
    const double *mass;            // local view
    const u8 *cls;                 // pair classes only: class of every particle (global view) / member slot (local view)
};

struct HermArgs {
    HermConst C;
    HermView G;                    // the global view
    const u64 *offset;
    const u32 *members;            // particles by component
    const uint2 *comps;            // (start, size): warp-tier components from the front, cluster-tier ones from comps_last down
    u32 comps_last;
    u32 *active;                   // [n] cluster tier: active particles of the block, same ranges as members
    u64 *bigctl;                   // [8 per cluster-tier component] rotating block times, active count
    u32 *lnbr;                     // [capacity] list entries as slots of the particle's component (warp kernel)
    u64 *ctl;
    const u32 *grid_members;       // grid tier: the members of all components above cluster_max
    u32 grid_count;
};

// Eq. 7 and its time derivative over the list [k0, k1) of i at time tn (ticks); the particle and its neighbours are
// predicted from their own last times.  first: t = 0, nothing to predict.
// SPLIT > 1: SPLIT consecutive lanes share the list of one particle (entry k0 + sub, k0 + sub + SPLIT, ...) and add their
// partial sums with shuffles; every lane of the warp must make the call (lanes without a particle pass k0 = k1).
// CLS (pair classes, L287): the kind of a pair, class_i + class_j, selects the softening and the cutoff coefficients; a
// pair of kind 2 (two black holes) is not split: the whole Newtonian term with eps_bb, at every separation.
template <bool LOCAL, int SPLIT = 1, bool CLS = false>
__device__ __forceinline__ void herm_force(const HermConst &C, const HermView &V, u32 i, u64 k0, u64 k1, u64 tn, bool first,
                                           double *a, double *a1)
{
    double xi[3], vi[3];
    {
        const double h = first ? 0.0 : (double)(tn - (V.tdt[i] >> 8)) * C.tick;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const double X = V.pos[3 * (size_t)i + c], Vc = V.vel[3 * (size_t)i + c];
            const double Ac = first ? 0.0 : V.a[3 * (size_t)i + c], Jc = first ? 0.0 : V.a1[3 * (size_t)i + c];
            xi[c] = X + h * (Vc + h * (Ac * 0.5 + h * (Jc * kSixth)));
            vi[c] = Vc + h * (Ac + h * (Jc * 0.5));
        }
    }
    const u32 ci = CLS ? (u32)V.cls[i] : 0u;
    double ax = 0, ay = 0, az = 0, jx = 0, jy = 0, jz = 0;
    for (u64 k = k0 + (SPLIT > 1 ? (threadIdx.x & (SPLIT - 1)) : 0); k < k1; k += SPLIT) {
        const u32 j = V.nbr[k];
        const double h = first ? 0.0 : (double)(tn - (V.tdt[j] >> 8)) * C.tick;
        double d[3], w[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const double X = V.pos[3 * (size_t)j + c], Vc = V.vel[3 * (size_t)j + c];
            const double Ac = first ? 0.0 : V.a[3 * (size_t)j + c], Jc = first ? 0.0 : V.a1[3 * (size_t)j + c];
            d[c] = xi[c] - (X + h * (Vc + h * (Ac * 0.5 + h * (Jc * kSixth))));
            w[c] = vi[c] - (Vc + h * (Ac + h * (Jc * 0.5)));
        }
        const u32 kind = CLS ? ci + (u32)V.cls[j] : 0u;
        const double s2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2] + ((CLS && kind == 2u) ? C.prm.eps2_bb_d : C.prm.eps2_d);
        const double s = sqrt(s2);
        double omK = 1.0, dKds = 0.0;
        if (!(CLS && kind == 2u)) herm_weights(C.prm.cs[CLS ? kind : 0u], s, omK, dKds);
        if (omK == 0.0 && dKds == 0.0) continue;
        const double qv = d[0] * w[0] + d[1] * w[1] + d[2] * w[2];
        const double mj = LOCAL ? V.mass[j] : (double)V.body_user[j].w;
        const double rs2 = 1.0 / s2, rs = s * rs2;          // one division per pair; the block loop is a latency chain
        const double mr3 = mj * rs2 * rs;
        const double c1 = mr3 * omK, c2 = mr3 * qv * (3.0 * omK * rs2 + dKds * rs);
        ax -= c1 * d[0]; ay -= c1 * d[1]; az -= c1 * d[2];
        jx -= c1 * w[0] - c2 * d[0]; jy -= c1 * w[1] - c2 * d[1]; jz -= c1 * w[2] - c2 * d[2];
    }
    if (SPLIT > 1) {
        __syncwarp();
#pragma unroll
        for (int o = SPLIT / 2; o; o >>= 1) {
            ax += __shfl_xor_sync(0xffffffffu, ax, o); ay += __shfl_xor_sync(0xffffffffu, ay, o); az += __shfl_xor_sync(0xffffffffu, az, o);
            jx += __shfl_xor_sync(0xffffffffu, jx, o); jy += __shfl_xor_sync(0xffffffffu, jy, o); jz += __shfl_xor_sync(0xffffffffu, jz, o);
        }
    }
    a[0] = ax; a[1] = ay; a[2] = az;
    a1[0] = jx; a1[1] = jy; a1[2] = jz;
}

__device__ __forceinline__ double norm3(const double *u) { return sqrt(u[0] * u[0] + u[1] * u[1] + u[2] * u[2]); }

// log2 of the largest power of two of ticks <= crit (a time), <= max_ticks, dividing t; at least one tick.  The
// criterion comes as ct^2 = P / Q (ct = crit / tick, P >= 0, Q > 0): floor(log2 ct) = floor(floor(log2(P / Q)) / 2) is
// read off the exponents and mantissas of P and Q, which saves the division and the square root at the end of the
// dependent chain of every step (the oracle takes the root and divides; the two differ only when ct is within
// rounding of a power of two).
__device__ __forceinline__ u32 herm_quantise(const HermConst &C, double P, double Q, u64 t, u32 &floor_hits)
{
    const u32 kmax = 63 - __clzll((long long)C.max_ticks);
    u32 k;
    // (exponent fields first: the test for a non-finite force or jerk is then two integer compares beside the chain,
    //  not two more fp64 operations in it -- as P - P == 0 it cost a quarter of a block step)
    const long long bp = __double_as_longlong(P), bq = __double_as_longlong(Q);
    const int ep = (int)((bp >> 52) & 0x7ff), eq = (int)((bq >> 52) & 0x7ff);
    if (ep == 0x7ff || eq == 0x7ff) {                       // inf or NaN: reported (HERM_NONFINITE), the step is void
        floor_hits |= HERM_NONFINITE;
        k = kmax;
    } else if (!(Q > 0.0)) k = kmax;                       // vanishing denominator: the maximum step
    else {
        const unsigned long long mp = (unsigned long long)bp & 0xfffffffffffffull, mq = (unsigned long long)bq & 0xfffffffffffffull;
        const int L = ep - eq - (mp < mq ? 1 : 0);         // floor(log2(P / Q)) for normal numbers; P = 0 gives a large negative
        if (L >= 2 * (int)kmax) k = kmax;
        else if (L < 0) { k = 0; ++floor_hits; }
        else k = (u32)L >> 1;
    }
    if (t) {
        const u32 tz = __ffsll((long long)t) - 1;          // t % 2^k == 0  <=>  k <= trailing zeros of t
        if (k > tz) k = tz;
    }
    return k;
}

// t = 0: force from the current state, first step from Eq. 20.  Returns the particle's first block time.
template <bool LOCAL, bool CLS = false>
__device__ __forceinline__ u64 herm_start(const HermConst &C, const HermView &V, u32 i, u64 k0, u64 k1, u32 &floor_hits)
{
    double a[3], a1[3];
    herm_force<LOCAL, 1, CLS>(C, V, i, k0, k1, 0, true, a, a1);
    const double d0 = a[0] * a[0] + a[1] * a[1] + a[2] * a[2], d1 = a1[0] * a1[0] + a1[1] * a1[1] + a1[2] * a1[2];
    const double c2s = CLS ? C.c2_sk[V.cls[i]] : C.c2_s, a0 = CLS ? C.a0k[V.cls[i]] : C.a0;
    const u32 k = herm_quantise(C, c2s * (d0 + a0 * a0), d1, 0, floor_hits);          // Eq. 20, squared
#pragma unroll
    for (int c = 0; c < 3; ++c) { V.a[3 * (size_t)i + c] = a[c]; V.a1[3 * (size_t)i + c] = a1[c]; }   // nobody reads a, a1, tdt at t = 0
    V.tdt[i] = k;
    return 1ull << k;
}

// first half of a block: the new force of an active particle from the state before the block.  Returns true if active;
// otherwise te is the particle's own next time (~0 when it has arrived at the end of the soft step).
template <bool LOCAL, bool CLS = false>
__device__ __forceinline__ bool herm_evaluate(const HermConst &C, const HermView &V, u32 i, u64 k0, u64 k1, u64 tn, u64 &te)
{
    const u64 total = 1ull << HERM_TICK_BITS;
    const u64 w = V.tdt[i];
    const u64 t = w >> 8;
    te = t >= total ? ~0ull : t + (1ull << (w & 63));
    if (te != tn) return false;
    double a[3], a1[3];
    herm_force<LOCAL, 1, CLS>(C, V, i, k0, k1, tn, false, a, a1);
#pragma unroll
    for (int c = 0; c < 3; ++c) { V.an[3 * (size_t)i + c] = a[c]; V.a1n[3 * (size_t)i + c] = a1[c]; }
    return true;
}

// second half: corrector and the next step (Eq. 18) of a particle that herm_evaluate found active.  Returns its next time.
template <bool CLS = false>
__device__ __forceinline__ u64 herm_correct(const HermConst &C, const HermView &V, u32 i, u64 tn, u32 &floor_hits)
{
    const u64 total = 1ull << HERM_TICK_BITS;
    const u64 w = V.tdt[i];
    const double h = (double)(1ull << (w & 63)) * C.tick;
    const double rh = __longlong_as_double((long long)(1023 - (int)(w & 63)) << 52) * C.rtick;   // 2^-k / tick, no division
    const double rh2 = rh * rh, rh3 = rh2 * rh;
    double an[3], jn[3], a2e[3], a3[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const size_t o = 3 * (size_t)i + c;
        const double Ac = V.a[o], Jc = V.a1[o], An = V.an[o], Jn = V.a1n[o];
        const double a2 = (-6.0 * (Ac - An) - h * (4.0 * Jc + 2.0 * Jn)) * rh2;
        a3[c] = (12.0 * (Ac - An) + 6.0 * h * (Jc + Jn)) * rh3;
        const double X = V.pos[o], Vc = V.vel[o];
        const double xp = X + h * (Vc + h * (Ac * 0.5 + h * (Jc * kSixth)));
        const double vp = Vc + h * (Ac + h * (Jc * 0.5));
        V.pos[o] = xp + h * h * h * h * (a2 * (1.0 / 24.0) + h * a3[c] * (1.0 / 120.0));
        V.vel[o] = vp + h * h * h * (a2 * kSixth + h * a3[c] * (1.0 / 24.0));
        a2e[c] = a2 + h * a3[c];
        V.a[o] = An; V.a1[o] = Jn;
        an[c] = An; jn[c] = Jn;
    }
    // Eq. 18 squared: ct^2 = (eta / tick)^2 (sqrt(|a|^2 + a0^2) |a2| + |a1|^2) / (|a1| |a3| + |a2|^2), |a1| |a3| as one root
    const double d0 = an[0] * an[0] + an[1] * an[1] + an[2] * an[2], d1 = jn[0] * jn[0] + jn[1] * jn[1] + jn[2] * jn[2];
    const double d2 = a2e[0] * a2e[0] + a2e[1] * a2e[1] + a2e[2] * a2e[2], d3 = a3[0] * a3[0] + a3[1] * a3[1] + a3[2] * a3[2];
    const double den = sqrt(d1 * d3) + d2;
    const double c2 = CLS ? C.c2k[V.cls[i]] : C.c2, a0 = CLS ? C.a0k[V.cls[i]] : C.a0;
    const u32 k = herm_quantise(C, c2 * (sqrt((d0 + a0 * a0) * d2) + d1), den, tn, floor_hits);
    V.tdt[i] = tn << 8 | k;
    return tn < total ? tn + (1ull << k) : ~0ull;
}

__device__ __forceinline__ u64 warp_min_u64(u64 v)
{
#pragma unroll
    for (int o = 16; o; o >>= 1) {
        const u64 x = __shfl_xor_sync(0xffffffffu, v, o);
        v = x < v ? x : v;
    }
    return v;
}

// One warp per component of up to HERM_WARP_MAX particles (two per lane).  The component's whole state lives in shared
// memory for the duration of the soft step (a block then costs shared-memory latencies, not L2 round trips); the lists
// are rewritten once as slots of the component.
#define HERM_WARPS 4
struct WarpState {
    double pos[3 * HERM_WARP_MAX], vel[3 * HERM_WARP_MAX];
    double a[3 * HERM_WARP_MAX], a1[3 * HERM_WARP_MAX], an[3 * HERM_WARP_MAX], a1n[3 * HERM_WARP_MAX];
    u64 tdt[HERM_WARP_MAX];
    double mass[HERM_WARP_MAX];
    u32 gid[HERM_WARP_MAX];
    u8 cls[HERM_WARP_MAX];
};

template <bool CLS>
__global__ void __launch_bounds__(32 * HERM_WARPS) hermite_warp_kernel(HermArgs A)
{
    u32 err = 0;                   // HC_ERR code of this thread, filed at the end of the kernel
    __shared__ WarpState sm_all[HERM_WARPS];
    const u32 wid = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (wid >= (u32)A.ctl[HC_NSMALL]) return;
    WarpState &S = sm_all[threadIdx.x >> 5];
    const uint2 comp = A.comps[wid];
    constexpr int PER = HERM_WARP_MAX / 32;
    u32 slot[PER];
    u64 k0[PER], k1[PER];
    bool have[PER];
#pragma unroll
    for (int q = 0; q < PER; ++q) {
        slot[q] = lane + 32 * q;
        have[q] = slot[q] < comp.y;
        k0[q] = k1[q] = 0;
        if (have[q]) {
            const u32 g = A.members[comp.x + slot[q]];
            S.gid[slot[q]] = g;
            k0[q] = A.offset[g]; k1[q] = A.offset[g + 1];
            S.mass[slot[q]] = (double)A.G.body_user[g].w;
            if (CLS) S.cls[slot[q]] = A.G.cls[g] & 1u;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                S.pos[3 * slot[q] + c] = A.G.pos[3 * (size_t)g + c];
                S.vel[3 * slot[q] + c] = A.G.vel[3 * (size_t)g + c];
            }
        }
    }
    __syncwarp();
#pragma unroll
    for (int q = 0; q < PER; ++q)
        for (u64 k = k0[q]; k < k1[q]; ++k) {             // list entries -> slots (every neighbour is a member)
            const u32 g = A.G.nbr[k];
            u32 sidx = 0;
            while (sidx < comp.y && S.gid[sidx] != g) ++sidx;
            if (sidx == comp.y) { err = max(err, 2u); sidx = slot[q]; }   // a list that is not symmetric: reported, result unusable
            A.lnbr[k] = sidx;
        }
    HermView V;
    V.pos = S.pos; V.vel = S.vel; V.a = S.a; V.a1 = S.a1; V.an = S.an; V.a1n = S.a1n; V.tdt = S.tdt;
    V.nbr = A.lnbr; V.body_user = nullptr; V.mass = S.mass; V.cls = S.cls;
    const HermConst &C = A.C;

    u32 floor_hits = 0, steps = 0;
    u64 next = ~0ull;
#pragma unroll
    for (int q = 0; q < PER; ++q)
        if (have[q]) next = min(next, herm_start<true, CLS>(C, V, slot[q], k0[q], k1[q], floor_hits));
    __syncwarp();
    u64 tn = warp_min_u64(next);
    u64 b = 0;
    while (tn != ~0ull) {
        if (b >= C.max_blocks) { err = max(err, 1u); break; }
        ++b;
        bool act[PER];
        u64 te[PER];
#pragma unroll
        for (int q = 0; q < PER; ++q) act[q] = have[q] && herm_evaluate<true, CLS>(C, V, slot[q], k0[q], k1[q], tn, te[q]);
        __syncwarp();
        next = ~0ull;
#pragma unroll
        for (int q = 0; q < PER; ++q) {
            if (!have[q]) continue;
            if (act[q]) { next = min(next, herm_correct<CLS>(C, V, slot[q], tn, floor_hits)); ++steps; }
            else next = min(next, te[q]);
        }
        __syncwarp();
        tn = warp_min_u64(next);
    }
#pragma unroll
    for (int q = 0; q < PER; ++q)
        if (have[q]) {
            const u32 g = S.gid[slot[q]];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                A.G.pos[3 * (size_t)g + c] = S.pos[3 * slot[q] + c];
                A.G.vel[3 * (size_t)g + c] = S.vel[3 * slot[q] + c];
            }
        }
    if (steps) atomicAdd((unsigned long long *)&A.ctl[HC_STEPS], (unsigned long long)steps);
    // (error codes are kept in a register and filed once, here: an atomic on the error word inside the block loop --
    //  executed or not -- made the warp tier's loop 1.6 times slower, 0.33 -> 0.55 ms for config 2)
    if (floor_hits & HERM_NONFINITE) err = max(err, 3u);
    if (err) herm_set_err(A.ctl, err);
    if (floor_hits & ~HERM_NONFINITE) atomicAdd((unsigned long long *)&A.ctl[HC_FLOOR], (unsigned long long)(floor_hits & ~HERM_NONFINITE));
    if (lane == 0) atomicMax((unsigned long long *)&A.ctl[HC_BLOCKS], (unsigned long long)b);
}

#ifdef P3T_HERM_PROFILE
__device__ unsigned long long g_hprof[8];
#define HPROF(k) do { if (tid == 0 && M > 10000) { unsigned long long t_; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_)); if (k) atomicAdd(&g_hprof[k], t_ - hp_last); hp_last = t_; } } while (0)
extern "C" void p3t_debug_hprof(unsigned long long *out) { cudaDeviceSynchronize(); cudaMemcpyFromSymbol(out, g_hprof, sizeof(g_hprof)); unsigned long long z[8] = {0}; cudaMemcpyToSymbol(g_hprof, z, sizeof(z)); }
#else
#define HPROF(k)
#endif
template <int SPLIT, bool CLS>
__device__ __forceinline__ void cluster_evaluate(const HermArgs &A, const u32 *active, const u32 *ids, u32 na, u32 tid, u32 stride, u64 tn)
{
    const HermView &V = A.G;
    const u32 lane = threadIdx.x & 31;
    constexpr u32 PER_WARP = 32 / SPLIT;
    for (u32 e0 = (tid >> 5) * PER_WARP; e0 < na; e0 += (stride >> 5) * PER_WARP) {
        const u32 e = e0 + lane / SPLIT;
        const bool ok = e < na;
        const u32 i = ok ? active[e] : 0u;
        const u64 k0 = ok ? A.offset[i] : 0ull, k1 = ok ? A.offset[i + 1] : 0ull;
        double a[3], a1[3];
        herm_force<false, SPLIT, CLS>(A.C, V, ok ? i : ids[0], k0, k1, tn, false, a, a1);
        if (ok && (lane & (SPLIT - 1)) == 0) {
#pragma unroll
            for (int k = 0; k < 3; ++k) { V.an[3 * (size_t)i + k] = a[k]; V.a1n[3 * (size_t)i + k] = a1[k]; }
        }
    }
}

// One thread-block cluster (8 CTAs x 512 threads) per mid-size component: the block loop is synchronised by the
// hardware cluster barrier (a fraction of a microsecond, against several for a grid barrier), components run side by
// side.  Per block: scan the members (next block time of the inactive ones, active ones appended to a list), barrier,
// evaluate the active list one particle per thread, barrier, correct, barrier.  State in global memory (L2).
template <bool CLS>
__global__ void __cluster_dims__(HERM_CLUSTER, 1, 1) __launch_bounds__(HERM_CLUSTER_THREADS) hermite_cluster_kernel(HermArgs A)
{
    u32 err = 0;                   // HC_ERR code of this thread, filed at the end of the kernel
    cg::cluster_group cl = cg::this_cluster();
    const u32 c = blockIdx.x / HERM_CLUSTER;
    const uint2 comp = A.comps[A.comps_last - c];
    const u32 M = comp.y;
    const u32 *ids = A.members + comp.x;
    u32 *active = A.active + comp.x;
    u64 *ctl = A.bigctl + 8 * (size_t)c;
    const HermConst &C = A.C;
    const HermView &V = A.G;
    const u32 tid = cl.block_rank() * blockDim.x + threadIdx.x, stride = HERM_CLUSTER * blockDim.x, lane = threadIdx.x & 31;
    u32 floor_hits = 0, steps = 0;
    unsigned long long hp_last = 0; (void)hp_last;
    {
        u64 local_min = ~0ull;
        for (u32 s = tid; s < M; s += stride) {
            const u32 i = ids[s];
            local_min = min(local_min, herm_start<false, CLS>(C, V, i, A.offset[i], A.offset[i + 1], floor_hits));
        }
        local_min = warp_min_u64(local_min);
        if (lane == 0 && local_min != ~0ull) atomicMin((unsigned long long *)&ctl[0], (unsigned long long)local_min);
    }
    cl.sync();
    u64 b = 0;
    for (;; ++b) {
        const u64 tn = *(volatile u64 *)&ctl[b % 3];
        if (tn == ~0ull) break;
        if (b >= C.max_blocks) { err = max(err, 1u); break; }
        u64 local_min = ~0ull;
        HPROF(0);
        // scan: four members per thread and round, their time words requested together
        for (u32 s0 = tid; s0 - lane < M; s0 += 4 * stride) {   // (warp-uniform trip count: the ballots below need every lane)
            u32 id[4];
            u64 w[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) id[q] = s0 + q * stride < M ? ids[s0 + q * stride] : 0xffffffffu;
#pragma unroll
            for (int q = 0; q < 4; ++q) w[q] = id[q] != 0xffffffffu ? V.tdt[id[q]] : ~0ull;
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const u64 t = w[q] >> 8;
                const bool live = id[q] != 0xffffffffu && t < (1ull << HERM_TICK_BITS);
                const u64 te = live ? t + (1ull << (w[q] & 63)) : ~0ull;
                const bool act = live && te == tn;
                if (!act) local_min = min(local_min, te);
                const u32 m = __ballot_sync(0xffffffffu, act);
                if (m) {
                    u32 base = 0;
                    if (lane == 0) base = (u32)atomicAdd((unsigned long long *)&ctl[3], (unsigned long long)__popc(m));
                    base = __shfl_sync(0xffffffffu, base, 0);
                    if (act) active[base + __popc(m & ((1u << lane) - 1))] = id[q];
                }
            }
        }
        HPROF(1);
        cl.sync();
        HPROF(2);
        const u32 na = (u32)*(volatile u64 *)&ctl[3];
        // evaluate the active particles from the state before the block; as many lanes share a particle's list as the
        // cluster has to spare (the longest list of the block is the critical path: every entry is an L2 round trip plus
        // an fp64 chain)
        if (na * 8 <= stride) cluster_evaluate<8, CLS>(A, active, ids, na, tid, stride, tn);
        else if (na * 4 <= stride) cluster_evaluate<4, CLS>(A, active, ids, na, tid, stride, tn);
        else if (na * 2 <= stride) cluster_evaluate<2, CLS>(A, active, ids, na, tid, stride, tn);
        else cluster_evaluate<1, CLS>(A, active, ids, na, tid, stride, tn);
        HPROF(3);
        cl.sync();
        HPROF(4);
        for (u32 e = tid; e < na; e += stride) {           // correct them together
            local_min = min(local_min, herm_correct<CLS>(C, V, active[e], tn, floor_hits));
            ++steps;
        }
        local_min = warp_min_u64(local_min);
        if (lane == 0 && local_min != ~0ull) atomicMin((unsigned long long *)&ctl[(b + 1) % 3], (unsigned long long)local_min);
        if (tid == 0) { ctl[(b + 2) % 3] = ~0ull; ctl[3] = 0ull; }
        HPROF(5);
        cl.sync();
        HPROF(6);
    }
    if (steps) atomicAdd((unsigned long long *)&A.ctl[HC_STEPS], (unsigned long long)steps);
    // (error codes are kept in a register and filed once, here: an atomic on the error word inside the block loop --
    //  executed or not -- made the warp tier's loop 1.6 times slower, 0.33 -> 0.55 ms for config 2)
    if (floor_hits & HERM_NONFINITE) err = max(err, 3u);
    if (err) herm_set_err(A.ctl, err);
    if (floor_hits & ~HERM_NONFINITE) atomicAdd((unsigned long long *)&A.ctl[HC_FLOOR], (unsigned long long)(floor_hits & ~HERM_NONFINITE));
    if (tid == 0) atomicMax((unsigned long long *)&A.ctl[HC_BLOCKS], (unsigned long long)b);
}

// the components above cluster_max, all together: global blocks, two grid barriers per block
// minimum over the CTA, then one atomicMin
__device__ __forceinline__ void cta_min_to(u64 *dst, u64 v, u64 *s_min)
{
    v = warp_min_u64(v);
    if ((threadIdx.x & 31) == 0) s_min[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (u32 w = 1; w < blockDim.x / 32; ++w) v = min(v, s_min[w]);
        if (v != ~0ull) atomicMin((unsigned long long *)dst, (unsigned long long)v);
    }
    __syncthreads();
}

template <bool CLS>
__global__ void __launch_bounds__(HERM_THREADS) hermite_grid_kernel(HermArgs A)
{
    u32 err = 0;                   // HC_ERR code of this thread, filed at the end of the kernel
    __shared__ u64 s_min[HERM_THREADS / 32];
    cg::grid_group grid = cg::this_grid();
    const u32 M = A.grid_count;
    const u32 *ids = A.grid_members;
    const HermConst &C = A.C;
    const HermView &V = A.G;
    const u32 tid = blockIdx.x * blockDim.x + threadIdx.x, stride = gridDim.x * blockDim.x, lane = threadIdx.x & 31;
    u32 floor_hits = 0, steps = 0;
    unsigned long long hp_last = 0; (void)hp_last;
    {
        u64 local_min = ~0ull;
        for (u32 s = tid; s < M; s += stride) {
            const u32 i = ids[s];
            local_min = min(local_min, herm_start<false, CLS>(C, V, i, A.offset[i], A.offset[i + 1], floor_hits));
        }
        cta_min_to(&A.ctl[HC_TMIN0], local_min, s_min);
    }
    grid.sync();
    u64 b = 0;
    for (;; ++b) {
        const u64 tn = *(volatile u64 *)&A.ctl[HC_TMIN0 + b % 3];
        if (tn == ~0ull) break;
        if (b >= C.max_blocks) { err = max(err, 1u); break; }
        u64 local_min = ~0ull;
        HPROF(0);
        // evaluate the active particles from the state before the block: a warp looks at 32 members, then takes its
        // active ones four at a time, eight lanes sharing a particle's list
        for (u32 s0 = tid; s0 - lane < M; s0 += stride) {
            const bool in = s0 < M;
            const u32 i = in ? ids[s0] : 0u;
            const u64 w = in ? V.tdt[i] : ~0ull;
            const u64 t = w >> 8;
            const bool live = in && t < (1ull << HERM_TICK_BITS);
            const u64 te = live ? t + (1ull << (w & 63)) : ~0ull;
            const bool act = live && te == tn;
            if (!act) local_min = min(local_min, te);
            u32 mask = __ballot_sync(0xffffffffu, act);
            while (mask) {
                const u32 src = __fns(mask, 0, (lane >> 3) + 1);       // the (lane / 8 + 1)-th active lane, or none
                const bool ok = src != 0xffffffffu;
                const u32 ii = __shfl_sync(0xffffffffu, i, ok ? src : 0);
                const u64 k0 = ok ? A.offset[ii] : 0ull, k1 = ok ? A.offset[ii + 1] : 0ull;
                double a[3], a1[3];
                herm_force<false, 8, CLS>(C, V, ok ? ii : ids[0], k0, k1, tn, false, a, a1);
                if (ok && (lane & 7) == 0) {
#pragma unroll
                    for (int k = 0; k < 3; ++k) { V.an[3 * (size_t)ii + k] = a[k]; V.a1n[3 * (size_t)ii + k] = a1[k]; }
                }
#pragma unroll
                for (int q = 0; q < 4; ++q) mask &= mask - 1;           // the four lowest set bits are done
            }
        }
        HPROF(3);
        grid.sync();
        HPROF(4);
        for (u32 s = tid; s < M; s += stride) {            // correct them together
            const u32 i = ids[s];
            const u64 w = V.tdt[i];
            if ((w >> 8) + (1ull << (w & 63)) != tn || (w >> 8) >= (1ull << HERM_TICK_BITS)) continue;
            local_min = min(local_min, herm_correct<CLS>(C, V, i, tn, floor_hits));
            ++steps;
        }
        cta_min_to(&A.ctl[HC_TMIN0 + (b + 1) % 3], local_min, s_min);     // (one atomic per CTA: one per thread on the same
                                                                          //  word cost 20 us per block)
        if (tid == 0) A.ctl[HC_TMIN0 + (b + 2) % 3] = ~0ull;
        HPROF(5);
        grid.sync();
        HPROF(6);
    }
    if (steps) atomicAdd((unsigned long long *)&A.ctl[HC_STEPS], (unsigned long long)steps);
    // (error codes are kept in a register and filed once, here: an atomic on the error word inside the block loop --
    //  executed or not -- made the warp tier's loop 1.6 times slower, 0.33 -> 0.55 ms for config 2)
    if (floor_hits & HERM_NONFINITE) err = max(err, 3u);
    if (err) herm_set_err(A.ctl, err);
    if (floor_hits & ~HERM_NONFINITE) atomicAdd((unsigned long long *)&A.ctl[HC_FLOOR], (unsigned long long)(floor_hits & ~HERM_NONFINITE));
    if (tid == 0) atomicMax((unsigned long long *)&A.ctl[HC_BLOCKS], (unsigned long long)b);
}

// Enqueues the component search, reads the counts back (one synchronisation: the grids are sized by them), then the two
// integration kernels and the drift.  d_pos, d_vel: device [n][3] doubles, updated in place.  h_ctl[HC_WORDS].
p3t_status p3t_stage_hermite(p3t_ctx *ctx, double *d_pos, double *d_vel, double T, int log2_div, double eta, double eta_s,
                             double a0, long long max_blocks, u64 *h_ctl)
{
    Workspace &w = ctx->ws;
    const u32 n = (u32)ctx->n;
    const u32 g = div_up(n, 256);
    P3T_CUDA(ctx, cudaMemsetAsync(w.herm_ctl, 0, HC_WORDS * sizeof(u64), ctx->stream));
    P3T_CUDA(ctx, cudaMemsetAsync(w.herm_ctl + HC_TMIN0, 0xff, 3 * sizeof(u64), ctx->stream));
    cc_init_kernel<<<g, 256, 0, ctx->stream>>>(w.nbr_offset, n, w.herm_parent, w.herm_csize);
    cc_hook_kernel<<<g, 256, 0, ctx->stream>>>(w.nbr_offset, w.nbr, n, w.herm_parent, w.herm_ctl);
    cc_count_kernel<<<div_up(n, 1024), 1024, 0, ctx->stream>>>(w.nbr_offset, n, w.herm_parent, w.herm_root, w.herm_csize, w.herm_ctl);
    const u32 comps_last = (u32)(ctx->max_n / 2);
    cc_assign_kernel<<<div_up(n, 1024), 1024, 0, ctx->stream>>>(w.nbr_offset, n, w.herm_root, w.herm_csize, w.herm_cstart, w.herm_comps, comps_last,
                                                 w.herm_bigctl, (u32)ctx->herm_cluster_max, w.herm_ctl);
    cc_scatter_kernel<<<g, 256, 0, ctx->stream>>>(w.nbr_offset, n, w.herm_root, w.herm_csize, w.herm_cstart, w.herm_ids, w.herm_parent);
    P3T_CUDA(ctx, cudaGetLastError());
    P3T_CUDA(ctx, cudaMemcpyAsync(h_ctl, w.herm_ctl, HC_WORDS * sizeof(u64), cudaMemcpyDeviceToHost, ctx->stream));
    P3T_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    const u64 M = h_ctl[HC_COUNT], nsmall = h_ctl[HC_NSMALL], nbigc = h_ctl[HC_NBIGC], ngrid = h_ctl[HC_GRID_CURSOR];
    if (M) {
        HermArgs A;
        A.G.body_user = w.body_user; A.G.nbr = w.nbr; A.G.mass = nullptr;
        A.G.pos = d_pos; A.G.vel = d_vel;
        A.G.tdt = w.herm_tdt; A.G.a = w.herm_state; A.G.a1 = w.herm_state + 3 * (size_t)ctx->max_n;
        A.G.an = w.herm_state + 6 * (size_t)ctx->max_n; A.G.a1n = w.herm_state + 9 * (size_t)ctx->max_n;
        A.offset = w.nbr_offset; A.members = w.herm_ids; A.comps = w.herm_comps; A.comps_last = comps_last;
        A.active = w.herm_cstart;                           // free once the members are laid out
        A.bigctl = w.herm_bigctl;
        A.grid_members = w.herm_parent; A.grid_count = (u32)ngrid;   // parent[] is free once the roots are known
        A.lnbr = reinterpret_cast<u32 *>(w.pairs);          // the walk's pair buffer is free once the lists are built
        A.ctl = w.herm_ctl;
        A.C.prm = ctx->prm;
        A.C.tick = T / (double)(1ull << HERM_TICK_BITS);
        A.C.rtick = (double)(1ull << HERM_TICK_BITS) / T;
        A.C.eta = eta; A.C.eta_s = eta_s; A.C.a0 = a0;
        A.C.c2 = (eta * A.C.rtick) * (eta * A.C.rtick); A.C.c2_s = (eta_s * A.C.rtick) * (eta_s * A.C.rtick);
        {   // pair classes: accuracy parameters per class of the integrated particle (class 1: p3t_set_hermite_class_params)
            const double e1 = ctx->herm_eta_bh > 0.0 ? ctx->herm_eta_bh : eta, es1 = ctx->herm_eta_s_bh > 0.0 ? ctx->herm_eta_s_bh : eta_s;
            A.C.c2k[0] = A.C.c2; A.C.c2_sk[0] = A.C.c2_s; A.C.a0k[0] = a0;
            A.C.c2k[1] = (e1 * A.C.rtick) * (e1 * A.C.rtick); A.C.c2_sk[1] = (es1 * A.C.rtick) * (es1 * A.C.rtick);
            A.C.a0k[1] = ctx->herm_a0_bh >= 0.0 ? ctx->herm_a0_bh : a0;
        }
        A.G.cls = w.cls_user;
        const bool cls = ctx->cls_n != 0;
        A.C.max_ticks = (1ull << HERM_TICK_BITS) >> log2_div;
        A.C.max_blocks = (u64)max_blocks;
        // The grid tier (if any) goes first on the caller's stream: one CTA per SM, mostly waiting at its barriers; the
        // warp and cluster tiers run beside it on the side stream (disjoint particles), joined before the drift.
        cudaStream_t rest = ctx->stream;
        if (ngrid) {
            int per_sm = 0;
            P3T_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, hermite_grid_kernel<false>, HERM_THREADS, 0));
            if (per_sm < 1) return p3t_fail(ctx, P3T_ECUDA, "hermite_grid_kernel does not fit an SM");
            u32 grid = (u32)((ngrid + HERM_THREADS - 1) / HERM_THREADS);
            if (grid > (u32)ctx->sm_count) grid = (u32)ctx->sm_count;   // one CTA per SM: the barrier is the cost of a block
            if (nsmall || nbigc) {
                P3T_CUDA(ctx, cudaEventRecord(ctx->ev_fork, ctx->stream));
                P3T_CUDA(ctx, cudaStreamWaitEvent(ctx->side_stream, ctx->ev_fork, 0));
                rest = ctx->side_stream;
            }
            void *args[] = {&A};
            P3T_CUDA(ctx, cudaLaunchCooperativeKernel(cls ? (void *)hermite_grid_kernel<true> : (void *)hermite_grid_kernel<false>, dim3(grid),
                                                      dim3(HERM_THREADS), args, 0, ctx->stream));
        }
        if (nsmall) {
            if (cls) hermite_warp_kernel<true><<<div_up(nsmall, HERM_WARPS), 32 * HERM_WARPS, 0, rest>>>(A);
            else hermite_warp_kernel<false><<<div_up(nsmall, HERM_WARPS), 32 * HERM_WARPS, 0, rest>>>(A);
            P3T_CUDA(ctx, cudaGetLastError());
        }
        if (nbigc) {
            if (cls) hermite_cluster_kernel<true><<<(u32)nbigc * HERM_CLUSTER, HERM_CLUSTER_THREADS, 0, rest>>>(A);
            else hermite_cluster_kernel<false><<<(u32)nbigc * HERM_CLUSTER, HERM_CLUSTER_THREADS, 0, rest>>>(A);
            P3T_CUDA(ctx, cudaGetLastError());
        }
        if (rest != ctx->stream) {
            P3T_CUDA(ctx, cudaEventRecord(ctx->ev_join, rest));
            P3T_CUDA(ctx, cudaStreamWaitEvent(ctx->stream, ctx->ev_join, 0));
        }
    }
    (void)M;
    herm_drift_kernel<<<g, 256, 0, ctx->stream>>>(w.nbr_offset, n, T, d_pos, d_vel);
    P3T_CUDA(ctx, cudaGetLastError());
    return P3T_OK;
}

// ---- the rest of the scheme's step (L142-153): soft kick, fp64 state -> fp32 input of the tree --------------------

// v += dt a_soft (procedure steps 2 and 4): a_soft of the last evaluation (fp32, user order), velocities fp64
__global__ void kick_kernel(const float4 *__restrict__ accpot, u32 n, double dt, double *__restrict__ vel)
{
    const u32 i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float4 a = accpot[i];
    vel[3 * (size_t)i] += dt * (double)a.x;
    vel[3 * (size_t)i + 1] += dt * (double)a.y;
    vel[3 * (size_t)i + 2] += dt * (double)a.z;
}

__global__ void narrow_kernel(const double *__restrict__ src, size_t count, float *__restrict__ dst)
{
    const size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k < count) dst[k] = (float)src[k];
}

p3t_status p3t_stage_kick(p3t_ctx *ctx, double *d_vel, double dt)
{
    const u32 n = (u32)ctx->n;
    kick_kernel<<<div_up(n, 256), 256, 0, ctx->stream>>>(ctx->ws.accpot, n, dt, d_vel);
    P3T_CUDA(ctx, cudaGetLastError());
    return P3T_OK;
}

p3t_status p3t_stage_narrow(p3t_ctx *ctx, const double *d_pos, float *d_pos32)
{
    const size_t count = 3 * ctx->n;
    narrow_kernel<<<div_up(count, 256), 256, 0, ctx->stream>>>(d_pos, count, d_pos32);
    P3T_CUDA(ctx, cudaGetLastError());
    return P3T_OK;
}
