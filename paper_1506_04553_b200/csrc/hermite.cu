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
// is the same as with global blocks (the oracle's locality pin P6).  The components are found on the device (lock-free
// union-find: hook by compare-and-swap, flatten, count, lay the members out contiguously).  A component of up to 64
// particles -- nearly all of them: pairs and triples -- is integrated by ONE WARP, its block loop synchronised by
// __syncwarp and a shuffle minimum: no grid barrier, no launch per block, thousands of components in flight.  The
// members of all larger components (dense cores, where the spheres percolate) go through one cooperative kernel whose
// block loop uses two grid barriers per block and a 64-bit atomicMin over (t + dt) into rotating words.  A warp keeps
// its component's state ((t << 8 | log2 dt), x, v, a, a1 and the block's new a, a1) in shared memory, the grid kernel in
// global arrays indexed by particle; everything fp64.
#include "p3t_internal.cuh"
#include <cooperative_groups.h>
#include <math_constants.h>
namespace cg = cooperative_groups;

#define HERM_THREADS 256
#define HERM_TICK_BITS 40
#define HERM_WARP_MAX 64        // largest component one warp integrates
enum { HC_COUNT = 0, HC_TMIN0, HC_TMIN1, HC_TMIN2, HC_BLOCKS, HC_STEPS, HC_FLOOR, HC_ERR,
       HC_NSMALL, HC_SMALL_CURSOR, HC_BIG_CURSOR, HC_NCOMP, HC_MAXCOMP, HC_WORDS = 16 };

__device__ __forceinline__ void herm_weights(const P3TParams &p, double s, double &omK, double &dKds)
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
    const u32 i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n || offset[i + 1] == offset[i]) return;
    parent[i] = i;
    csize[i] = 0;
}

__global__ void cc_hook_kernel(const u64 *__restrict__ offset, const u32 *__restrict__ nbr, u32 n, u32 *parent)
{
    const u32 i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
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
    const u32 m = __ballot_sync(0xffffffffu, has);
    if (m && (threadIdx.x & 31) == 0) atomicAdd((unsigned long long *)&ctl[HC_COUNT], (unsigned long long)__popc(m));
}

// member ranges: small components from the front of members[], the others from the back (HC_COUNT is final here).
// One atomic per warp and counter: the roots of a warp take consecutive ranges (warp scans of the sizes).
__global__ void cc_assign_kernel(const u64 *__restrict__ offset, u32 n, const u32 *__restrict__ root, u32 *csize,
                                 u32 *__restrict__ cstart, uint2 *__restrict__ comps, u64 *ctl)
{
    const u32 i = blockIdx.x * blockDim.x + threadIdx.x, lane = threadIdx.x & 31;
    const bool is_root = i < n && offset[i + 1] > offset[i] && root[i] == i;
    const u32 sz = is_root ? csize[i] : 0u;
    const bool small = is_root && sz <= HERM_WARP_MAX, big = is_root && !small;
    const u32 m_root = __ballot_sync(0xffffffffu, is_root);
    if (!m_root) return;
    const u32 m_small = __ballot_sync(0xffffffffu, small);
    u32 ss = small ? sz : 0u, sb = big ? sz : 0u;          // inclusive warp scans of the sizes
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const u32 a = __shfl_up_sync(0xffffffffu, ss, o), c = __shfl_up_sync(0xffffffffu, sb, o);
        if (lane >= (u32)o) { ss += a; sb += c; }
    }
    const u32 tot_s = __shfl_sync(0xffffffffu, ss, 31), tot_b = __shfl_sync(0xffffffffu, sb, 31);
    const u32 mx = __reduce_max_sync(0xffffffffu, sz);
    u32 base_s = 0, base_b = 0, base_c = 0;
    if (lane == 0) {
        if (tot_s) base_s = (u32)atomicAdd((unsigned long long *)&ctl[HC_SMALL_CURSOR], (unsigned long long)tot_s);
        if (tot_b) base_b = (u32)atomicAdd((unsigned long long *)&ctl[HC_BIG_CURSOR], (unsigned long long)tot_b);
        if (m_small) base_c = (u32)atomicAdd((unsigned long long *)&ctl[HC_NSMALL], (unsigned long long)__popc(m_small));
        atomicAdd((unsigned long long *)&ctl[HC_NCOMP], (unsigned long long)__popc(m_root));
        atomicMax((unsigned long long *)&ctl[HC_MAXCOMP], (unsigned long long)mx);
    }
    base_s = __shfl_sync(0xffffffffu, base_s, 0);
    base_b = __shfl_sync(0xffffffffu, base_b, 0);
    base_c = __shfl_sync(0xffffffffu, base_c, 0);
    if (!is_root) return;
    u32 st;
    if (small) {
        st = base_s + ss - sz;
        comps[base_c + __popc(m_small & ((1u << lane) - 1))] = make_uint2(st, sz);
    } else {
        st = (u32)ctl[HC_COUNT] - (base_b + sb);
    }
    cstart[i] = st;
    csize[i] = 0;                          // becomes the fill cursor of the scatter
}

__global__ void cc_scatter_kernel(const u64 *__restrict__ offset, u32 n, const u32 *__restrict__ root, u32 *csize,
                                  const u32 *__restrict__ cstart, u32 *__restrict__ members)
{
    const u32 i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n || offset[i + 1] == offset[i]) return;
    const u32 r = root[i];
    members[cstart[r] + atomicAdd(&csize[r], 1u)] = i;     // order inside a component is irrelevant
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
};

struct HermArgs {
    HermConst C;
    HermView G;                    // the global view
    const u64 *offset;
    const u32 *members;            // particles by component
    const uint2 *comps;            // (start, size) of the components of up to HERM_WARP_MAX members
    u32 *lnbr;                     // [capacity] list entries as slots of the particle's component (warp kernel)
    u64 *ctl;
    u32 big_begin, big_count;      // members[big_begin .. big_begin + big_count): the larger components
};

// Eq. 7 and its time derivative over the list [k0, k1) of i at time tn (ticks); the particle and its neighbours are
// predicted from their own last times.  first: t = 0, nothing to predict.
template <bool LOCAL>
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
    const double eps2 = C.prm.eps2_d;
    double ax = 0, ay = 0, az = 0, jx = 0, jy = 0, jz = 0;
    for (u64 k = k0; k < k1; ++k) {
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
        const double s2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2] + eps2;
        const double s = sqrt(s2);
        double omK, dKds;
        herm_weights(C.prm, s, omK, dKds);
        if (omK == 0.0 && dKds == 0.0) continue;
        const double qv = d[0] * w[0] + d[1] * w[1] + d[2] * w[2];
        const double mj = LOCAL ? V.mass[j] : (double)V.body_user[j].w;
        const double rs2 = 1.0 / s2, rs = s * rs2;          // one division per pair; the block loop is a latency chain
        const double mr3 = mj * rs2 * rs;
        const double c1 = mr3 * omK, c2 = mr3 * qv * (3.0 * omK * rs2 + dKds * rs);
        ax -= c1 * d[0]; ay -= c1 * d[1]; az -= c1 * d[2];
        jx -= c1 * w[0] - c2 * d[0]; jy -= c1 * w[1] - c2 * d[1]; jz -= c1 * w[2] - c2 * d[2];
    }
    a[0] = ax; a[1] = ay; a[2] = az;
    a1[0] = jx; a1[1] = jy; a1[2] = jz;
}

__device__ __forceinline__ double norm3(const double *u) { return sqrt(u[0] * u[0] + u[1] * u[1] + u[2] * u[2]); }

// log2 of the largest power of two of ticks <= crit (a time), <= max_ticks, dividing t; at least one tick
__device__ __forceinline__ u32 herm_quantise(const HermConst &C, double crit, u64 t, u32 &floor_hits)
{
    const double ct = crit * C.rtick;
    u32 k;
    const u32 kmax = 63 - __clzll((long long)C.max_ticks);
    if (!(ct < (double)C.max_ticks)) k = kmax;
    else if (ct < 1.0) { k = 0; ++floor_hits; }
    else k = (u32)((__double2hiint(ct) >> 20) & 0x7ff) - 1023u;
    if (t) {
        const u32 tz = __ffsll((long long)t) - 1;          // t % 2^k == 0  <=>  k <= trailing zeros of t
        if (k > tz) k = tz;
    }
    return k;
}

// t = 0: force from the current state, first step from Eq. 20.  Returns the particle's first block time.
template <bool LOCAL>
__device__ __forceinline__ u64 herm_start(const HermConst &C, const HermView &V, u32 i, u64 k0, u64 k1, u32 &floor_hits)
{
    double a[3], a1[3];
    herm_force<LOCAL>(C, V, i, k0, k1, 0, true, a, a1);
    const double na = norm3(a), n1 = norm3(a1);
    const double crit = n1 > 0.0 ? C.eta_s * sqrt((na * na + C.a0 * C.a0) / (n1 * n1)) : CUDART_INF;
    const u32 k = herm_quantise(C, crit, 0, floor_hits);
#pragma unroll
    for (int c = 0; c < 3; ++c) { V.a[3 * (size_t)i + c] = a[c]; V.a1[3 * (size_t)i + c] = a1[c]; }   // nobody reads a, a1, tdt at t = 0
    V.tdt[i] = k;
    return 1ull << k;
}

// first half of a block: the new force of an active particle from the state before the block.  Returns true if active;
// otherwise te is the particle's own next time (~0 when it has arrived at the end of the soft step).
template <bool LOCAL>
__device__ __forceinline__ bool herm_evaluate(const HermConst &C, const HermView &V, u32 i, u64 k0, u64 k1, u64 tn, u64 &te)
{
    const u64 total = 1ull << HERM_TICK_BITS;
    const u64 w = V.tdt[i];
    const u64 t = w >> 8;
    te = t >= total ? ~0ull : t + (1ull << (w & 63));
    if (te != tn) return false;
    double a[3], a1[3];
    herm_force<LOCAL>(C, V, i, k0, k1, tn, false, a, a1);
#pragma unroll
    for (int c = 0; c < 3; ++c) { V.an[3 * (size_t)i + c] = a[c]; V.a1n[3 * (size_t)i + c] = a1[c]; }
    return true;
}

// second half: corrector and the next step (Eq. 18) of a particle that herm_evaluate found active.  Returns its next time.
__device__ __forceinline__ u64 herm_correct(const HermConst &C, const HermView &V, u32 i, u64 tn, u32 &floor_hits)
{
    const u64 total = 1ull << HERM_TICK_BITS;
    const u64 w = V.tdt[i];
    const double h = (double)(1ull << (w & 63)) * C.tick;
    const double rh = 1.0 / h, rh2 = rh * rh, rh3 = rh2 * rh;
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
    const double na = norm3(an), n1 = norm3(jn), n2 = norm3(a2e), n3 = norm3(a3);
    const double den = n1 * n3 + n2 * n2;
    const double crit = den > 0.0 ? C.eta * sqrt((sqrt(na * na + C.a0 * C.a0) * n2 + n1 * n1) / den) : CUDART_INF;
    const u32 k = herm_quantise(C, crit, tn, floor_hits);
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
};

__global__ void __launch_bounds__(32 * HERM_WARPS) hermite_warp_kernel(HermArgs A)
{
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
            if (sidx == comp.y) { A.ctl[HC_ERR] = 2; sidx = slot[q]; }   // a list that is not symmetric: reported, result unusable
            A.lnbr[k] = sidx;
        }
    HermView V;
    V.pos = S.pos; V.vel = S.vel; V.a = S.a; V.a1 = S.a1; V.an = S.an; V.a1n = S.a1n; V.tdt = S.tdt;
    V.nbr = A.lnbr; V.body_user = nullptr; V.mass = S.mass;
    const HermConst &C = A.C;

    u32 floor_hits = 0, steps = 0;
    u64 next = ~0ull;
#pragma unroll
    for (int q = 0; q < PER; ++q)
        if (have[q]) next = min(next, herm_start<true>(C, V, slot[q], k0[q], k1[q], floor_hits));
    __syncwarp();
    u64 tn = warp_min_u64(next);
    u64 b = 0;
    while (tn != ~0ull) {
        if (b >= C.max_blocks) { if (lane == 0) A.ctl[HC_ERR] = 1; break; }
        ++b;
        bool act[PER];
        u64 te[PER];
#pragma unroll
        for (int q = 0; q < PER; ++q) act[q] = have[q] && herm_evaluate<true>(C, V, slot[q], k0[q], k1[q], tn, te[q]);
        __syncwarp();
        next = ~0ull;
#pragma unroll
        for (int q = 0; q < PER; ++q) {
            if (!have[q]) continue;
            if (act[q]) { next = min(next, herm_correct(C, V, slot[q], tn, floor_hits)); ++steps; }
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
    if (floor_hits) atomicAdd((unsigned long long *)&A.ctl[HC_FLOOR], (unsigned long long)floor_hits);
    if (lane == 0) atomicMax((unsigned long long *)&A.ctl[HC_BLOCKS], (unsigned long long)b);
}

// all larger components together: global blocks, two grid barriers per block
__global__ void __launch_bounds__(HERM_THREADS) hermite_grid_kernel(HermArgs A)
{
    cg::grid_group grid = cg::this_grid();
    const u32 M = A.big_count;
    const u32 *ids = A.members + A.big_begin;
    const HermConst &C = A.C;
    const HermView &V = A.G;
    const u32 tid = blockIdx.x * blockDim.x + threadIdx.x, stride = gridDim.x * blockDim.x;
    u32 floor_hits = 0, steps = 0;
    {
        u64 local_min = ~0ull;
        for (u32 s = tid; s < M; s += stride) {
            const u32 i = ids[s];
            local_min = min(local_min, herm_start<false>(C, V, i, A.offset[i], A.offset[i + 1], floor_hits));
        }
        if (local_min != ~0ull) atomicMin((unsigned long long *)&A.ctl[HC_TMIN0], (unsigned long long)local_min);
    }
    grid.sync();
    u64 b = 0;
    for (;; ++b) {
        const u64 tn = *(volatile u64 *)&A.ctl[HC_TMIN0 + b % 3];
        if (tn == ~0ull) break;
        if (b >= C.max_blocks) { if (tid == 0) A.ctl[HC_ERR] = 1; break; }
        u64 local_min = ~0ull;
        for (u32 s = tid; s < M; s += stride) {            // evaluate the active particles from the state before the block
            const u32 i = ids[s];
            u64 te;
            if (!herm_evaluate<false>(C, V, i, A.offset[i], A.offset[i + 1], tn, te)) local_min = min(local_min, te);
        }
        grid.sync();
        for (u32 s = tid; s < M; s += stride) {            // correct them together
            const u32 i = ids[s];
            const u64 w = V.tdt[i];
            if ((w >> 8) + (1ull << (w & 63)) != tn || (w >> 8) >= (1ull << HERM_TICK_BITS)) continue;
            local_min = min(local_min, herm_correct(C, V, i, tn, floor_hits));
            ++steps;
        }
        if (local_min != ~0ull) atomicMin((unsigned long long *)&A.ctl[HC_TMIN0 + (b + 1) % 3], (unsigned long long)local_min);
        if (tid == 0) A.ctl[HC_TMIN0 + (b + 2) % 3] = ~0ull;
        grid.sync();
    }
    if (steps) atomicAdd((unsigned long long *)&A.ctl[HC_STEPS], (unsigned long long)steps);
    if (floor_hits) atomicAdd((unsigned long long *)&A.ctl[HC_FLOOR], (unsigned long long)floor_hits);
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
    cc_hook_kernel<<<g, 256, 0, ctx->stream>>>(w.nbr_offset, w.nbr, n, w.herm_parent);
    cc_count_kernel<<<g, 256, 0, ctx->stream>>>(w.nbr_offset, n, w.herm_parent, w.herm_root, w.herm_csize, w.herm_ctl);
    cc_assign_kernel<<<g, 256, 0, ctx->stream>>>(w.nbr_offset, n, w.herm_root, w.herm_csize, w.herm_cstart, w.herm_comps, w.herm_ctl);
    cc_scatter_kernel<<<g, 256, 0, ctx->stream>>>(w.nbr_offset, n, w.herm_root, w.herm_csize, w.herm_cstart, w.herm_ids);
    P3T_CUDA(ctx, cudaGetLastError());
    P3T_CUDA(ctx, cudaMemcpyAsync(h_ctl, w.herm_ctl, HC_WORDS * sizeof(u64), cudaMemcpyDeviceToHost, ctx->stream));
    P3T_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    const u64 M = h_ctl[HC_COUNT], nsmall = h_ctl[HC_NSMALL], nbig = h_ctl[HC_BIG_CURSOR];
    if (M) {
        HermArgs A;
        A.G.body_user = w.body_user; A.G.nbr = w.nbr; A.G.mass = nullptr;
        A.G.pos = d_pos; A.G.vel = d_vel;
        A.G.tdt = w.herm_tdt; A.G.a = w.herm_state; A.G.a1 = w.herm_state + 3 * (size_t)ctx->max_n;
        A.G.an = w.herm_state + 6 * (size_t)ctx->max_n; A.G.a1n = w.herm_state + 9 * (size_t)ctx->max_n;
        A.offset = w.nbr_offset; A.members = w.herm_ids; A.comps = w.herm_comps;
        A.lnbr = reinterpret_cast<u32 *>(w.pairs);          // the walk's pair buffer is free once the lists are built
        A.ctl = w.herm_ctl;
        A.C.prm = ctx->prm;
        A.C.tick = T / (double)(1ull << HERM_TICK_BITS);
        A.C.rtick = (double)(1ull << HERM_TICK_BITS) / T;
        A.C.eta = eta; A.C.eta_s = eta_s; A.C.a0 = a0;
        A.C.max_ticks = (1ull << HERM_TICK_BITS) >> log2_div;
        A.C.max_blocks = (u64)max_blocks;
        A.big_begin = (u32)(M - nbig); A.big_count = (u32)nbig;
        if (nsmall) {
            hermite_warp_kernel<<<div_up(nsmall, HERM_WARPS), 32 * HERM_WARPS, 0, ctx->stream>>>(A);
            P3T_CUDA(ctx, cudaGetLastError());
        }
        if (nbig) {
            int per_sm = 0;
            P3T_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, hermite_grid_kernel, HERM_THREADS, 0));
            if (per_sm < 1) return p3t_fail(ctx, P3T_ECUDA, "hermite_grid_kernel does not fit an SM");
            u32 grid = (u32)((nbig + HERM_THREADS - 1) / HERM_THREADS);
            if (grid > (u32)ctx->sm_count) grid = (u32)ctx->sm_count;   // one CTA per SM: the barrier is the cost of a block
            void *args[] = {&A};
            P3T_CUDA(ctx, cudaLaunchCooperativeKernel((void *)hermite_grid_kernel, dim3(grid), dim3(HERM_THREADS), args, 0, ctx->stream));
        }
    }
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
