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

// unroll factors of the interaction loops (list entries in flight per warp)
#ifndef WALK_PP_UNROLL
#define WALK_PP_UNROLL 8
#endif
#ifndef WALK_PC_UNROLL
#define WALK_PC_UNROLL 2
#endif
// full batches of 32 list entries summed in fp32 before the sums go to the fp64 accumulators
#ifndef WALK_FLUSH_EVERY
#define WALK_FLUSH_EVERY 4
#endif
constexpr int kPpUnroll = WALK_PP_UNROLL, kPcUnroll = WALK_PC_UNROLL;

#ifdef P3T_WALK_PROFILE
// sequential attribution of a warp's cycles to phases (diagnostic builds only)
#define WP_SLOTS 12
__device__ unsigned long long g_wprof[WP_SLOTS];
#define WPROF_DECL u32 wp_acc[WP_SLOTS]; for (int k_ = 0; k_ < WP_SLOTS; ++k_) wp_acc[k_] = 0; u32 wp_last = (u32)clock64()
#define WP(k) do { u32 t_ = (u32)clock64(); wp_acc[k] += t_ - wp_last; wp_last = t_; } while (0)
#define WPC(k) (++wp_acc[k])
#else
#define WPROF_DECL
#define WP(k)
#define WPC(k)
#endif

struct WarpShared {
    // far ring: (x, y, z, m) of each body, stored once.  The loops use a list entry as the scalar
    // (broadcast) operand of the packed instructions (SASS: FFMA2 Rd, Rj.F32, Ra.F32x2, Rb.F32x2), so
    // no duplicated pairs are needed: half the shared-memory traffic of a {x,x,y,y} layout, and a
    // scalar operand costs one register-file read instead of two (profiles/ffma2_operand_bandwidth_r1.md)
    float4 far[64];
    float4 near_buf[64];
    u32 near_idx[64];
    float4 pc[3][64];   // p-c ring: staged cells (see stage_pc)
    // landing area of the asynchronous copies (cp.async) of the 32 cells popped for the NEXT walk
    // step: their latency is hidden behind the interaction batches of the current step
    float4 l_mac[32], l_mom0[32], l_mom1[32];
    uint2 l_meta[32];
    u32 l_cell[32];     // their indices (written and read by a split walk only)
};

__device__ __forceinline__ void cp_async16(void *smem, const void *gmem)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"((u32)__cvta_generic_to_shared(smem)), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async8(void *smem, const void *gmem)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((u32)__cvta_generic_to_shared(smem)), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// ---- arithmetic on V = float (one body per lane) or float2 (two bodies per lane, packed) -----------
// Blackwell's FFMA2/FMUL2/FADD2 do two fp32 operations per issue slot at the full FP32 pipe rate
// (measured 73.7 TFLOP/s against 72.2 for scalar FFMA, profiles/), which leaves issue slots for
// the LDS, MUFU and integer instructions of the loop.
__device__ __forceinline__ float vfma(float a, float b, float c) { return fmaf(a, b, c); }
__device__ __forceinline__ float vmul(float a, float b) { return a * b; }
__device__ __forceinline__ float vadd(float a, float b) { return a + b; }
__device__ __forceinline__ float2 vfma(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ float2 vmul(float2 a, float2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ float2 vadd(float2 a, float2 b) { return __fadd2_rn(a, b); }
// (Issuing the accumulator updates -- three distinct register pairs, three cycles as FFMA2 -- as two scalar FFMAs each
// makes an eval-only probe of the quadrupole loop 9 % faster, 85 -> 78 cycles per entry, but the whole kernel 1.4 % slower:
// the six extra instructions per entry compete with the walk's own instructions for the issue port.)
__device__ __forceinline__ float rsq(float x)
{
    float r;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ float vrsqrt(float a) { return rsq(a); }
__device__ __forceinline__ float2 vrsqrt(float2 a) { return make_float2(rsq(a.x), rsq(a.y)); }
template <class V> __device__ __forceinline__ V vdup(float a);
template <> __device__ __forceinline__ float vdup<float>(float a) { return a; }
template <> __device__ __forceinline__ float2 vdup<float2>(float a) { return make_float2(a, a); }
__device__ __forceinline__ float vget(float a, int) { return a; }
__device__ __forceinline__ float vget(float2 a, int b) { return b ? a.y : a.x; }
__device__ __forceinline__ float &vref(float &a, int) { return a; }
__device__ __forceinline__ float &vref(float2 &a, int b) { return b ? a.y : a.x; }
template <int NI> struct VecOf { typedef float type; };
template <> struct VecOf<2> { typedef float2 type; };

template <int NI> struct Acc {
    typedef typename VecOf<NI>::type V;
    V ax, ay, az, ph;                          // current batch (fp32)
    double dax[NI], day[NI], daz[NI], dph[NI]; // running totals (fp64)
    __device__ __forceinline__ void zero()
    {
        ax = ay = az = ph = vdup<V>(0.f);
#pragma unroll
        for (int b = 0; b < NI; ++b) dax[b] = day[b] = daz[b] = dph[b] = 0.0;
    }
    int pending = 0;                           // batches added to the fp32 sums since the last flush
    __device__ __forceinline__ void flush_lazy()
    {
        if (++pending >= WALK_FLUSH_EVERY) flush();
    }
    __device__ __forceinline__ void flush()
    {
        pending = 0;
#pragma unroll
        for (int b = 0; b < NI; ++b) {
            dax[b] += (double)vget(ax, b); day[b] += (double)vget(ay, b);
            daz[b] += (double)vget(az, b); dph[b] += (double)vget(ph, b);
        }
        ax = ay = az = ph = vdup<V>(0.f);
    }
};

// the group's bodies as the loops consume them: negated coordinates (d = q_j + (-q_i) is one FADD2)
// seal(): passes each component through an identity shuffle, which makes the pairs opaque to ptxas:
// it then keeps them in aligned register pairs for the whole walk instead of rebuilding them from
// the registers of the body load with two MOVs at every use (once per group, 3*NI SHFLs).
__device__ __forceinline__ float vseal1(float a) { return __shfl_sync(0xffffffffu, a, threadIdx.x & 31); }
__device__ __forceinline__ void vseal(float &a) { a = vseal1(a); }
__device__ __forceinline__ void vseal(float2 &a) { a = make_float2(vseal1(a.x), vseal1(a.y)); }
template <int NI> struct Targets {
    typedef typename VecOf<NI>::type V;
    V nx, ny, nz;
    __device__ __forceinline__ void seal() { vseal(nx); vseal(ny); vseal(nz); }
};

// Walk stack: the first `cap` entries live in shared memory, the rest in a global overflow area.
// One warp per group: each warp owns WALK_STACK_SMEM + WALK_STACK_GMEM entries.  Cooperative mode
// (one CTA per group): the four regions form one stack shared by the CTA's warps.
struct StackRef {
    u32 *smem;
    u32 *gmem;
    u32 cap;       // shared-memory entries
    u32 limit;     // total entries
};
__device__ __forceinline__ u32 stack_read(const StackRef &st, u32 pos)
{
    P3T_DEV_ASSERT(pos < st.limit);
    return pos < st.cap ? st.smem[pos] : st.gmem[pos - st.cap];
}
__device__ __forceinline__ void stack_write(const StackRef &st, u32 pos, u32 v)
{
    P3T_DEV_ASSERT(pos < st.limit);
    if (pos < st.cap) st.smem[pos] = v;
    else st.gmem[pos - st.cap] = v;
}

// Control block of the cooperative mode (one per CTA, shared memory).  Invariant: top > 0 implies
// busy > 0 (or nobody has started), so top == 0 && busy == 0 means the walk of the group is over.
struct CtaCtl {
    u32 top;       // entries on the shared stack
    u32 busy;      // warps that hold popped cells whose children are not pushed yet
    u32 lock;
    u32 group;     // ticket of the group in flight
    u32 err;
    u32 stat[2];   // list lengths (p-p, p-c entries) summed over the warps, for P3T_ARR_GROUP_STATS
    u32 cls;       // cost class of the group just finished (read by all threads after the barrier)
};
__device__ __forceinline__ u32 vload(const u32 *p) { return *reinterpret_cast<const volatile u32 *>(p); }
__device__ __forceinline__ void vstore(u32 *p, u32 v) { *reinterpret_cast<volatile u32 *>(p) = v; }
__device__ __forceinline__ void ctl_lock(CtaCtl *c)
{
    while (atomicCAS(&c->lock, 0u, 1u) != 0u) { }
    __threadfence_block();
}
__device__ __forceinline__ void ctl_unlock(CtaCtl *c)
{
    __threadfence_block();
    atomicExch(&c->lock, 0u);
}

// ---- p-p, plain softened Newtonian (K = W = 1): 13 FP32-pipe operations per interaction; counted as
//      23 flop by the convention of DESIGN.md section 8 ---------------------------------------------
template <int NI>
__device__ __forceinline__ void pp_body(const float4 &B, const Targets<NI> &t, typename VecOf<NI>::type eps2, Acc<NI> &acc)
{
    typedef typename VecOf<NI>::type V;
    V dx = vadd(vdup<V>(B.x), t.nx), dy = vadd(vdup<V>(B.y), t.ny), dz = vadd(vdup<V>(B.z), t.nz);
    V r2 = vfma(dx, dx, vfma(dy, dy, vfma(dz, dz, eps2)));
    V rinv = vrsqrt(r2);
    V mrinv = vmul(vdup<V>(B.w), rinv);
    V mr3 = vmul(mrinv, vmul(rinv, rinv));
    acc.ax = vfma(mr3, dx, acc.ax);
    acc.ay = vfma(mr3, dy, acc.ay);
    acc.az = vfma(mr3, dz, acc.az);
    acc.ph = vadd(acc.ph, mrinv);
}

template <int NI>
__device__ __forceinline__ void eval_far(const WarpShared &ws, u32 head, u32 cnt, const Targets<NI> &t, float eps2s,
                                         Acc<NI> &acc)
{
    typedef typename VecOf<NI>::type V;
    const V eps2 = vdup<V>(eps2s);
    if (cnt == 32) {
#pragma unroll kPpUnroll
        for (u32 j = 0; j < 32; ++j) pp_body<NI>(ws.far[head + j], t, eps2, acc);
    } else {
        for (u32 j = 0; j < cnt; ++j) pp_body<NI>(ws.far[head + j], t, eps2, acc);
    }
    acc.flush_lazy();
}

// ---- p-c, softened monopole + quadrupole about the centre of mass (rule R-QUAD), K = W = 1 ----------
//   with d = c - q_i, s^2 = |d|^2 + eps^2 and the traceful Q of moments.cu, R-QUAD reads
//     -phi = M/s + 1.5 dQd/s^5 - 0.5 trQ/s^3,   a = d (M/s^3 + 7.5 dQd/s^7 - 1.5 trQ/s^5) - 3 Qd/s^5.
//   Staged per cell (stage_pc):  Q5 = 7.5 Q - 2.5 trQ I,  te5 = -2.5 trQ eps^2,  so that
//     T = d.Q5 d + te5 = 7.5 dQd - 2.5 trQ s^2,   c1 = M + T/s^4,
//     -phi = (0.8 M + 0.2 c1)/s,                   a = d c1/s^3 - 0.4 (Q5 d)/s^5
//   which is the same expression (the eps^2 of the softened trace term is carried by te5), in
//   33 FP32-pipe operations per interaction; counted as 65 flop by the convention of DESIGN.md.
__device__ __forceinline__ void stage_pc(WarpShared &ws, u32 slot, const float4 &a, const float4 &q0, const float4 &q1, float eps2)
{
    float tr25 = 2.5f * (q0.y + q0.z + q0.w);
    float qxx = fmaf(7.5f, q0.y, -tr25), qyy = fmaf(7.5f, q0.z, -tr25), qzz = fmaf(7.5f, q0.w, -tr25);
    float qxy = 7.5f * q1.x, qxz = 7.5f * q1.y, qyz = 7.5f * q1.z;
    float te5 = -tr25 * eps2, m08 = 0.8f * q0.x;
    ws.pc[0][slot] = make_float4(a.x, a.y, a.z, q0.x);
    ws.pc[1][slot] = make_float4(qxx, qyy, qzz, qxy);
    ws.pc[2][slot] = make_float4(qxz, qyz, te5, m08);
}

template <int NI>
__device__ __forceinline__ void eval_pc(const WarpShared &ws, u32 head, u32 cnt, const Targets<NI> &t, float eps2s, Acc<NI> &acc)
{
    typedef typename VecOf<NI>::type V;
    const V eps2 = vdup<V>(eps2s), c02 = vdup<V>(0.2f), cm04 = vdup<V>(-0.4f);
#pragma unroll kPcUnroll
    for (u32 j = 0; j < cnt; ++j) {
        const u32 e = head + j;
        const float4 P0 = ws.pc[0][e], P1 = ws.pc[1][e], P2 = ws.pc[2][e];
        const V M = vdup<V>(P0.w);
        const V qxx = vdup<V>(P1.x), qyy = vdup<V>(P1.y), qzz = vdup<V>(P1.z);
        const V qxy = vdup<V>(P1.w), qxz = vdup<V>(P2.x), qyz = vdup<V>(P2.y);
        V dx = vadd(vdup<V>(P0.x), t.nx), dy = vadd(vdup<V>(P0.y), t.ny), dz = vadd(vdup<V>(P0.z), t.nz);
        V r2 = vfma(dx, dx, vfma(dy, dy, vfma(dz, dz, eps2)));
        V rinv = vrsqrt(r2);
        V r2i = vmul(rinv, rinv);
        V r3i = vmul(r2i, rinv);
        V r4i = vmul(r2i, r2i);
        V n5 = vmul(r3i, vmul(cm04, r2i));                          // -0.4 / s^5
        // (source order: the three lines of Q5 d by shared operand, then the accumulator updates by shared factor -- ptxas keeps
        // part of it, and consecutive packed instructions that share a source register read it once: SASS .reuse)
        V qdx = vmul(qxz, dz), qdy = vmul(qyz, dz), qdz = vmul(qzz, dz);
        qdx = vfma(qxy, dy, qdx); qdy = vfma(qyy, dy, qdy); qdz = vfma(qyz, dy, qdz);
        qdx = vfma(qxx, dx, qdx); qdy = vfma(qxy, dx, qdy); qdz = vfma(qxz, dx, qdz);
        V T = vfma(dx, qdx, vfma(dy, qdy, vfma(dz, qdz, vdup<V>(P2.z))));
        acc.ax = vfma(n5, qdx, acc.ax); acc.ay = vfma(n5, qdy, acc.ay); acc.az = vfma(n5, qdz, acc.az);
        V c1 = vfma(T, r4i, M);
        V pphi = vfma(c02, c1, vdup<V>(P2.w));
        V coef = vmul(c1, r3i);
        acc.ax = vfma(coef, dx, acc.ax); acc.ay = vfma(coef, dy, acc.ay); acc.az = vfma(coef, dz, acc.az);
        acc.ph = vfma(pphi, rinv, acc.ph);
    }
    acc.flush_lazy();
}

// ---- p-p slow path: K (Eq. 12) on the force, W (Eq. 16-17) on the potential, j != i by index,
//      neighbour emission for s_ij < h (reading A4) -------------------------------------------------
//      With pair classes (CLS): the kind of the pair, class_i + class_j, selects the cutoff radii and the
//      neighbour radius; a pair of kind 2 (two black holes) is not split: nothing in the soft sums, always neighbours.
template <int NI, bool CLS>
__device__ __forceinline__ void eval_near(const WarpShared &ws, u32 head, u32 cnt, const Targets<NI> &t,
                                          const u32 (&isorted)[NI], const u32 (&iuser)[NI], const u32 (&icls)[NI],
                                          const P3TParams &prm, const u32 *__restrict__ sorted_idx, uint2 *pairs, u64 pair_cap,
                                          u64 *counters, u32 (&nnb)[NI], Acc<NI> &acc, u32 lane)
{
    // Nearly all near entries are plain Newtonian partners of all the group's bodies (they are "near" the group's BOX):
    // the packed plain term is evaluated for everybody, with the mass of a pair that is not plain (self, closer than
    // the neighbour radius, two black holes) set to zero -- masked, not subtracted afterwards: a close pair's plain term
    // would be many orders of magnitude above the sum -- and the K/W term and the list entry of such pairs are done by a
    // branch that a warp takes for about one entry in fifty.
    typedef typename VecOf<NI>::type V;
    const V eps2v = vdup<V>(prm.eps2);
    for (u32 j = 0; j < cnt; ++j) {
        float4 bj = ws.near_buf[head + j];
        u32 js = ws.near_idx[head + j];
        u32 cj = 0;
        if (CLS) { cj = js >> 31; js &= 0x7fffffffu; }
        V dx = vadd(vdup<V>(bj.x), t.nx), dy = vadd(vdup<V>(bj.y), t.ny), dz = vadd(vdup<V>(bj.z), t.nz);
        V r2 = vfma(dx, dx, vfma(dy, dy, vfma(dz, dz, eps2v)));
        V r2s = r2, meff;
        bool slow[NI], anyslow = false;
#pragma unroll
        for (int b = 0; b < NI; ++b) {
            const u32 kind = CLS ? icls[b] + cj : 0u;
            const bool live = isorted[b] != 0xffffffffu && isorted[b] != js;
            const float thr = CLS ? (kind == 2u ? INFINITY : prm.h2_k[kind & 1u]) : prm.h2;
            slow[b] = live && vget(r2, b) < thr;
            const bool plain = live && !slow[b];
            vref(meff, b) = plain ? bj.w : 0.f;
            if (!plain) vref(r2s, b) = 1.f;           // keeps 0 * rsqrt(0) out of the sums (self pair with eps = 0)
            anyslow = anyslow || slow[b];
        }
        {
            V rinv = vrsqrt(r2s);
            V mrinv = vmul(meff, rinv);
            V mr3 = vmul(mrinv, vmul(rinv, rinv));
            acc.ax = vfma(mr3, dx, acc.ax);
            acc.ay = vfma(mr3, dy, acc.ay);
            acc.az = vfma(mr3, dz, acc.az);
            acc.ph = vadd(acc.ph, mrinv);
        }
        if (__any_sync(0xffffffffu, anyslow)) {
#pragma unroll
            for (int b = 0; b < NI; ++b) {
                const u32 kind = CLS ? icls[b] + cj : 0u;
                const bool hit = slow[b];                 // within the neighbour radius of its kind (always, for kind 2)
                if (hit && !(CLS && kind == 2u)) {
                    const float s2 = vget(r2, b);
                    float rinv = rsq(s2);
                    float mrinv = bj.w * rinv;
                    float mr3 = mrinv * (rinv * rinv);
                    float K = 1.f, W = 1.f;
                    if (CLS) { if (s2 < prm.rout2_k[kind]) p3t_pair_weights(prm.cs[kind], s2, K, W); }
                    else if (s2 < prm.rout2) p3t_pair_weights(prm.cs[0], s2, K, W);
                    mr3 *= K;
                    vref(acc.ax, b) = fmaf(mr3, vget(dx, b), vget(acc.ax, b));
                    vref(acc.ay, b) = fmaf(mr3, vget(dy, b), vget(acc.ay, b));
                    vref(acc.az, b) = fmaf(mr3, vget(dz, b), vget(acc.az, b));
                    vref(acc.ph, b) = fmaf(W, mrinv, vget(acc.ph, b));
                }
                u32 hb = __ballot_sync(0xffffffffu, hit);
                if (hb) {
                    u64 base = 0;
                    if (lane == 0) base = atomicAdd(&counters[CNT_PAIRS], (u64)__popc(hb));
                    base = __shfl_sync(0xffffffffu, base, 0);
                    if (hit) {
                        u64 pos = base + __popc(hb & lanemask_lt());
                        P3T_DEV_ASSERT(js < 0x40000000u);
                        if (pos < pair_cap) pairs[pos] = make_uint2(iuser[b], sorted_idx[js]);
                        ++nnb[b];
                    }
                }
            }
        }
    }
    acc.flush_lazy();
}

__device__ __forceinline__ u64 globaltimer_ns()
{
    u64 t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}

// cost class of a finished group (see group_order_kernel)
#define ORDER_CLASSES 1024
__device__ __forceinline__ u32 cost_class(u32 pp_len, u32 pc_len, bool packed)
{
    const u32 c = (13u * pp_len + 33u * pc_len) * (packed ? 2u : 1u);
    const u32 bits = __float_as_uint((float)max(c, 1u)) >> 20;        // exponent and three mantissa bits
    const u32 lo = 127u << 3;                                         // cost 1
    return ORDER_CLASSES - 1u - min(bits - lo, (u32)ORDER_CLASSES - 1u);   // class 0 = most expensive
}

// Arguments of the walk that do not change between groups.
struct WalkArgs {
    const float4 *__restrict__ body;
    const u32 *__restrict__ sorted_idx;
    const float4 *__restrict__ cell_mac, *__restrict__ cell_mom0, *__restrict__ cell_mom1;
    const uint2 *__restrict__ cell_meta;
    float4 *__restrict__ accpot;
    u32 *__restrict__ nbr_count;
    uint4 *__restrict__ group_stats;
    const u32 *__restrict__ group_order;   // position -> group of the previous call, a permutation of 0..order_meta[0]-1
    const u32 *__restrict__ order_meta;
    u32 *__restrict__ body_class;    // [n] user order: cost class of the group each body was in (this walk's record for the next call)
    u32 *order_hist;                 // [ORDER_CLASSES] groups per class
    u32 shard_rank, shard_world;     // this launch walks positions rank, rank + world, ... of the hand-out order
    u32 use_order;                   // 0: positions are group numbers (a sharded walk whose ranks have not exchanged cost classes)
    uint2 *pairs;
    u64 pair_cap;
    u64 *counters;
    const u8 *__restrict__ cls_sorted;   // pair classes (walk_kernel<.., .., true> only)
    const float *__restrict__ cube;
    u32 n;                               // bodies (checked builds test indices against it)
    // split walk (mid-size n: about as many groups as warps, so that all of them start at once and the launch ends in a
    // long tail of lone warps): every group is walked by `nparts` warps, each taking every nparts-th cell of one tree
    // level (and everything below those); what is accepted or is a leaf above that level is dealt out likewise.  Parts 1..
    // write their sums to split_acc / split_cnt, a small kernel adds them in fixed order.
    u32 nparts;                          // 1, 2 or 4
    const u32 *__restrict__ level_total; // cells per level (build.cu)
    float4 *__restrict__ split_acc;      // [nparts - 1][n]
    u32 *__restrict__ split_cnt;         // [nparts - 1][n]
};
struct SplitRule { u32 part, nparts, lo, hi; };   // this warp's part; cell indices [lo, hi) of the split level

// starts the asynchronous copy of the records of the popped cells into the landing area
template <bool SPLIT = false>
__device__ __forceinline__ void request_cells(WarpShared &ws, const WalkArgs &A, u32 take, u32 lane, u32 cell)
{
    if (lane < take) {
        P3T_DEV_ASSERT((u64)cell < A.counters[CNT_NCELLS]);
        if (SPLIT) ws.l_cell[lane] = cell;
        cp_async16(&ws.l_mac[lane], &A.cell_mac[cell]);
        cp_async8(&ws.l_meta[lane], &A.cell_meta[cell]);
        cp_async16(&ws.l_mom0[lane], &A.cell_mom0[cell]);
        cp_async16(&ws.l_mom1[lane], &A.cell_mom1[cell]);
    }
    cp_async_commit();
}
// pops up to 32 cells of a warp-private stack
template <bool SPLIT = false>
__device__ __forceinline__ u32 pop_cells(WarpShared &ws, const StackRef &st, const WalkArgs &A, u32 &top, u32 lane)
{
    const u32 take = min(32u, top);
    top -= take;
    const u32 cell = lane < take ? stack_read(st, top + lane) : 0u;
    request_cells<SPLIT>(ws, A, take, lane, cell);
    return take;
}
// cooperative mode: a warp without cells takes up to 32 from the shared stack; waits while other warps may
// still push; returns 0 when the walk of the group is over
__device__ __forceinline__ u32 coop_acquire(WarpShared &ws, const StackRef &st, CtaCtl *c, const WalkArgs &A, u32 lane)
{
    for (;;) {
        u32 state = 0;   // 0: wait, 1: try, 2: maybe over
        if (lane == 0) {
            const u32 t = vload(&c->top), b = vload(&c->busy);
            state = t > 0 ? 1u : (b == 0 ? 2u : 0u);
        }
        state = __shfl_sync(0xffffffffu, state, 0);
        if (state == 0) { __nanosleep(200); continue; }
        u32 t = 0;
        if (lane == 0) { ctl_lock(c); t = vload(&c->top); }
        t = __shfl_sync(0xffffffffu, t, 0);
        const u32 take = min(32u, t);
        if (take == 0) {
            u32 b = 0;
            if (lane == 0) { b = vload(&c->busy); ctl_unlock(c); }
            b = __shfl_sync(0xffffffffu, b, 0);
            if (b == 0) return 0u;
            continue;
        }
        const u32 cell = lane < take ? stack_read(st, t - take + lane) : 0u;
        __syncwarp();
        if (lane == 0) { vstore(&c->top, t - take); vstore(&c->busy, vload(&c->busy) + 1u); ctl_unlock(c); }
        request_cells(ws, A, take, lane, cell);
        return take;
    }
}

// One i-group: walk + interactions.  Walk step k consumes the 32 cell records that were requested
// during step k-1, pushes children, requests the records of step k+1, and only then evaluates the
// leaf bodies and the full interaction batches, so that the requests are in flight behind FP32 work.
// COOP: the four warps of the CTA work on the same group.  Each warp holds all the group's bodies, takes
// cells from the shared stack (under a lock, lane 0), builds and evaluates its own lists; the partial
// sums of warps 1-3 are added to warp 0's at the end.  Which warp meets which cell depends on timing,
// so results are reproducible to fp32 rounding of the batch sums, not bitwise.
// CLS (pair classes): a group that holds a black hole keeps every cell with a body within h_bf of its box
// open (cells were given their radius for field-star groups: h, or h_bf if the cell itself holds a black hole) and never
// accepts a cell that holds a black hole (BH-BH pairs are not split); bodies go to the K/W path when they are within
// the neighbour radius of the kinds of pairs they can form with the group, black holes met by such a group always.
template <int NI, bool COOP, bool CLS, bool SPLIT>
__device__ __forceinline__ void walk_group(WarpShared *wsall, const StackRef &st, CtaCtl *ctl, const WalkArgs &A,
                                           const P3TParams &prm, u32 gs, u32 ge, u32 lane, u32 warp, u64 &tot_pp, u64 &tot_pc,
                                           u64 &tot_near, const SplitRule &sr, u32 &len_pp, u32 &len_pc)
{
    WarpShared &ws = wsall[warp];
    const u32 gcount = ge - gs;
    WPROF_DECL;
    // ---- my bodies; empty slots replicate the group's first body and are flagged dead
    Targets<NI> tg;
    u32 isorted[NI], iuser[NI], nnb[NI], icls[NI];
    float lo[3] = {INFINITY, INFINITY, INFINITY}, hi[3] = {-INFINITY, -INFINITY, -INFINITY};
#pragma unroll
    for (int b = 0; b < NI; ++b) {
        u32 k = gs + b * 32 + lane;
        bool ok = k < ge;
        float4 p = A.body[ok ? k : gs];
        vref(tg.nx, b) = -p.x; vref(tg.ny, b) = -p.y; vref(tg.nz, b) = -p.z;
        isorted[b] = ok ? k : 0xffffffffu;
        iuser[b] = ok ? A.sorted_idx[k] : 0u;
        icls[b] = (CLS && ok) ? (u32)A.cls_sorted[k] : 0u;
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
    tg.seal();
    WP(9);
    bool heavy_group = false;
    float slack = 0.f;
    if (CLS) {
        u32 any = 0;
#pragma unroll
        for (int b = 0; b < NI; ++b) any |= icls[b];
        heavy_group = __any_sync(0xffffffffu, any != 0);
        slack = 8.f * 1.1920929e-7f * (fabsf(A.cube[0]) + fabsf(A.cube[1]) + fabsf(A.cube[2]) + 2.f * A.cube[3]);   // as moments.cu
    }

    u32 top = 1;
    if (!COOP && lane == 0) st.smem[0] = 0;   // root (cooperative mode: placed by the kernel)
    u32 far_head = 0, far_cnt = 0, near_head = 0, near_cnt = 0, pc_head = 0, pc_cnt = 0;
    u32 n_far = 0, n_near = 0, n_pc = 0;
    bool overflow = false;
    __syncwarp();
    u32 take = COOP ? coop_acquire(ws, st, ctl, A, lane) : pop_cells<SPLIT>(ws, st, A, top, lane);
    while (take > 0) {
        const bool have = lane < take;
        WP(8);
        cp_async_wait_all();
        WP(2); WPC(10);
        // ---- consume the landed records: acceptance test (R-MAC, folded radius of moments.cu)
        bool accept = false, skip = false;
        u32 nch = 0, first = 0, lcount = 0, lstart = 0;
        float4 a = make_float4(0.f, 0.f, 0.f, 0.f);
        if (have) {
            a = ws.l_mac[lane];
            float ex = fmaxf(0.f, fmaxf(lo[0] - a.x, a.x - hi[0]));
            float ey = fmaxf(0.f, fmaxf(lo[1] - a.y, a.y - hi[1]));
            float ez = fmaxf(0.f, fmaxf(lo[2] - a.z, a.z - hi[2]));
            float d2 = fmaf(ex, ex, fmaf(ey, ey, ez * ez));
            accept = d2 > a.w;
            if (CLS && heavy_group && accept) {
                const float rm = ws.l_mom1[lane].w;                       // bounding radius; sign bit: the cell holds a black hole
                const float rc = (prm.h_bf + fabsf(rm)) * (1.f + 1e-5f) + slack;
                accept = !(__float_as_uint(rm) >> 31) && d2 > rc * rc;
            }
            // (after the acceptance is final: a part that drops a cell as "accepted, someone else's" must not find out
            //  later that it has to be opened)
            if (SPLIT) {      // is this cell mine?
                const u32 c = ws.l_cell[lane];
                if (c >= sr.lo) {
                    if (c < sr.hi && ((c - sr.lo) & (sr.nparts - 1u)) != sr.part) { skip = true; accept = false; }
                } else if ((c & (sr.nparts - 1u)) != sr.part) {      // above the split level all parts meet the cell: what is
                    skip = accept || (ws.l_meta[lane].y & P3T_LEAF_FLAG) != 0;   // accepted or a leaf there goes to one of them
                    accept = false;
                }
            }
            if (!accept && !(SPLIT && skip)) {
                uint2 meta = ws.l_meta[lane];
                if (meta.y & P3T_LEAF_FLAG) { lstart = meta.x; lcount = meta.y & ~P3T_LEAF_FLAG; P3T_DEV_ASSERT(lcount >= 1 && lstart + lcount <= A.n); }
                else { first = meta.x; nch = meta.y; P3T_DEV_ASSERT(nch >= 1 && nch <= 8 && (u64)first + nch <= A.counters[CNT_NCELLS]); }
            }
        }
        // ---- accepted cells -> p-c ring (at most 31 pending + 32 new entries, capacity 64)
        {
            u32 ab = __ballot_sync(0xffffffffu, accept);
            if (accept)
                stage_pc(ws, (pc_head + pc_cnt + __popc(ab & lanemask_lt())) & 63u, a, ws.l_mom0[lane], ws.l_mom1[lane], prm.eps2);
            pc_cnt += __popc(ab);
        }
        WP(3);
        // ---- children of opened internal cells -> stack
        {
            u32 inc = nch, total = 0;
            if (__any_sync(0xffffffffu, nch != 0)) {      // (a step of accepted cells and leaves only pushes nothing)
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    u32 t = __shfl_up_sync(0xffffffffu, inc, o);
                    if (lane >= o) inc += t;
                }
                total = __shfl_sync(0xffffffffu, inc, 31);
            }
            if (!COOP) {
                if (top + total > st.limit) { overflow = true; break; }
                u32 pos = top + inc - nch;
                if (top + total <= st.cap) {      // (warp-uniform) everything lands in shared memory: no per-entry test
#pragma unroll
                    for (u32 c = 0; c < 8; ++c)
                        if (c < nch) st.smem[pos + c] = first + c;
                } else {
                    for (u32 c = 0; c < nch; ++c) stack_write(st, pos + c, first + c);
                }
                top += total;
                __syncwarp();
                // ---- request the records of the next step before any interaction work
                take = top > 0 ? pop_cells<SPLIT>(ws, st, A, top, lane) : 0u;
            } else {
                // one critical section: push the children, take the next 32 cells (mostly my own children)
                u32 base = 0;
                if (lane == 0) { ctl_lock(ctl); base = vload(&ctl->top); }
                base = __shfl_sync(0xffffffffu, base, 0);
                if (base + total > st.limit) {
                    if (lane == 0) { vstore(&ctl->top, 0u); vstore(&ctl->busy, vload(&ctl->busy) - 1u); vstore(&ctl->err, 1u); ctl_unlock(ctl); }
                    overflow = true;
                    break;
                }
                u32 pos = base + inc - nch;
                for (u32 c = 0; c < nch; ++c) stack_write(st, pos + c, first + c);
                __syncwarp();
                const u32 ntop = base + total;
                take = min(32u, ntop);
                const u32 cell = lane < take ? stack_read(st, ntop - take + lane) : 0u;
                __syncwarp();
                if (lane == 0) {
                    vstore(&ctl->top, ntop - take);
                    if (take == 0) vstore(&ctl->busy, vload(&ctl->busy) - 1u);
                    ctl_unlock(ctl);
                }
                request_cells(ws, A, take, lane, cell);
            }
        }
        WP(4);
        // ---- bodies of opened leaves -> near / far rings; the next chunk of 32 bodies is loaded
        //      while the current one is tested and (when a ring fills) evaluated
        if (__any_sync(0xffffffffu, lcount != 0)) {      // (steps near the top of the tree open no leaf: no scan then)
            u32 inc = lcount;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                u32 t = __shfl_up_sync(0xffffffffu, inc, o);
                if (lane >= o) inc += t;
            }
            const u32 total = __shfl_sync(0xffffffffu, inc, 31);
            const u32 excl = inc - lcount;
            auto fetch = [&](u32 v0, float4 &bj, u32 &bidx, bool &hv, u32 &cj) {
                u32 v = v0 + lane;
                u32 s = 0;   // owner lane: largest s with excl[s] <= v
#pragma unroll
                for (int step = 16; step > 0; step >>= 1) {
                    u32 cand = s + step;
                    u32 t = __shfl_sync(0xffffffffu, inc, cand - 1);   // = excl[cand]
                    if (t <= v) s = cand;
                }
                u32 s_start = __shfl_sync(0xffffffffu, lstart, s);
                u32 s_excl = __shfl_sync(0xffffffffu, excl, s);
                hv = v < total;
                bidx = s_start + (v - s_excl);
                P3T_DEV_ASSERT(!hv || bidx < A.n);
                bj = A.body[hv ? bidx : gs];
                if (CLS) cj = A.cls_sorted[hv ? bidx : gs];
            };
            float4 bj = make_float4(0.f, 0.f, 0.f, 0.f), bn = bj;
            u32 bidx = 0, bidxn = 0, cj = 0, cjn = 0;
            bool hv = false, hvn = false;
            if (total) fetch(0, bj, bidx, hv, cj);
            for (u32 v0 = 0; v0 < total; v0 += 32) {
                WPC(11);
                hvn = false;
                if (v0 + 32 < total) fetch(v0 + 32, bn, bidxn, hvn, cjn);
                float ex = fmaxf(0.f, fmaxf(lo[0] - bj.x, bj.x - hi[0]));
                float ey = fmaxf(0.f, fmaxf(lo[1] - bj.y, bj.y - hi[1]));
                float ez = fmaxf(0.f, fmaxf(lo[2] - bj.z, bj.z - hi[2]));
                float d2 = fmaf(ex, ex, fmaf(ey, ey, ez * ez));
                float thr = prm.hnear2;
                if (CLS) {
                    if (cj != 0 || heavy_group) thr = prm.hnear2_bf;
                    if (cj != 0 && heavy_group) thr = INFINITY;          // two black holes: always the slow path
                }
                bool isnear = hv && d2 < thr;
                bool isfar = hv && !isnear;
                u32 fb = __ballot_sync(0xffffffffu, isfar), nb = __ballot_sync(0xffffffffu, isnear);
                if (isfar) {
                    u32 slot = (far_head + far_cnt + __popc(fb & lanemask_lt())) & 63u;
                    ws.far[slot] = bj;
                }
                if (isnear) {
                    u32 slot = (near_head + near_cnt + __popc(nb & lanemask_lt())) & 63u;
                    ws.near_buf[slot] = bj;
                    ws.near_idx[slot] = CLS ? (bidx | (cj << 31)) : bidx;
                }
                far_cnt += __popc(fb);
                near_cnt += __popc(nb);
                __syncwarp();
                if (far_cnt >= 32) {
                    WP(5);
                    eval_far<NI>(ws, far_head, 32, tg, prm.eps2, acc);
                    WP(0);
                    far_head = (far_head + 32) & 63u; far_cnt -= 32; n_far += 32;
                }
                if (near_cnt >= 32) {
                    WP(5);
                    eval_near<NI, CLS>(ws, near_head, 32, tg, isorted, iuser, icls, prm, A.sorted_idx, A.pairs, A.pair_cap, A.counters, nnb,
                                  acc, lane);
                    WP(6);
                    near_head = (near_head + 32) & 63u; near_cnt -= 32; n_near += 32;
                }
                __syncwarp();
                bj = bn; bidx = bidxn; hv = hvn; cj = cjn;
            }
        }
        // ---- a full batch of accepted cells
        if (pc_cnt >= 32) {
            WP(5);
            eval_pc<NI>(ws, pc_head, 32, tg, prm.eps2, acc);
            WP(1);
            pc_head = (pc_head + 32) & 63u; pc_cnt -= 32; n_pc += 32;
            __syncwarp();
        }
        if (COOP && take == 0) take = coop_acquire(ws, st, ctl, A, lane);
    }
    cp_async_wait_all();
    WP(5);
    if (overflow) {
        if (lane == 0) atomicOr(&A.counters[CNT_ERR_EVAL], (u64)ERR_STACK_OVERFLOW);
    }
    // ---- flush what is left in the rings
    __syncwarp();
    if (pc_cnt) { eval_pc<NI>(ws, pc_head, pc_cnt, tg, prm.eps2, acc); n_pc += pc_cnt; }
    if (far_cnt) { eval_far<NI>(ws, far_head, far_cnt, tg, prm.eps2, acc); n_far += far_cnt; }
    if (near_cnt) {
        eval_near<NI, CLS>(ws, near_head, near_cnt, tg, isorted, iuser, icls, prm, A.sorted_idx, A.pairs, A.pair_cap, A.counters, nnb, acc, lane);
        n_near += near_cnt;
    }
    acc.flush();
    __syncwarp();
    if (COOP) {
        // partial sums of warps 1-3 -> their own (now dead) p-c ring, neighbour counts -> far ring; warp 0 adds
        // them in warp order and writes the results
        double *red = reinterpret_cast<double *>(&ws.pc[0][0]);
        u32 *rnb = reinterpret_cast<u32 *>(&ws.far[0]);
        if (lane == 0) { atomicAdd(&ctl->stat[0], n_far + n_near); atomicAdd(&ctl->stat[1], n_pc); }
        if (warp != 0) {
#pragma unroll
            for (int b = 0; b < NI; ++b) {
                red[(4 * b + 0) * 32 + lane] = acc.dax[b]; red[(4 * b + 1) * 32 + lane] = acc.day[b];
                red[(4 * b + 2) * 32 + lane] = acc.daz[b]; red[(4 * b + 3) * 32 + lane] = acc.dph[b];
                rnb[b * 32 + lane] = nnb[b];
            }
        }
        __syncthreads();
        if (warp == 0) {
            for (u32 w = 1; w < WALK_WARPS; ++w) {
                const double *ro = reinterpret_cast<const double *>(&wsall[w].pc[0][0]);
                const u32 *rn = reinterpret_cast<const u32 *>(&wsall[w].far[0]);
#pragma unroll
                for (int b = 0; b < NI; ++b) {
                    acc.dax[b] += ro[(4 * b + 0) * 32 + lane]; acc.day[b] += ro[(4 * b + 1) * 32 + lane];
                    acc.daz[b] += ro[(4 * b + 2) * 32 + lane]; acc.dph[b] += ro[(4 * b + 3) * 32 + lane];
                    nnb[b] += rn[b * 32 + lane];
                }
            }
        }
    }
    // ---- results, user order (split walk: parts 1.. to their own arrays)
    if (!COOP || warp == 0) {
        float4 *out = A.accpot;
        u32 *cnt = A.nbr_count;
        if (SPLIT && sr.part) { out = A.split_acc + (size_t)(sr.part - 1u) * A.n; cnt = A.split_cnt + (size_t)(sr.part - 1u) * A.n; }
#pragma unroll
    for (int b = 0; b < NI; ++b) {
        if (isorted[b] != 0xffffffffu) {
            out[iuser[b]] = make_float4((float)acc.dax[b], (float)acc.day[b], (float)acc.daz[b], (float)(-acc.dph[b]));
            cnt[iuser[b]] = nnb[b];
        }
    }
    }
    if (COOP) __syncthreads();   // the rings are reused by the next group
#ifdef P3T_WALK_PROFILE
    WP(7);
    if (lane == 0) for (int k_ = 0; k_ < WP_SLOTS; ++k_) atomicAdd(&g_wprof[k_], (unsigned long long)wp_acc[k_]);
#endif
    // each live body met itself once on the near path (distance 0 to its own group's box): removed once per group, by
    // warp 0 / part 0 (the per-warp totals are u64 and wrap harmlessly; their sum is right)
    const u64 self = (COOP ? warp == 0 : (!SPLIT || sr.part == 0)) ? gcount : 0;
    tot_pp += (u64)(n_far + n_near) * gcount - self;
    tot_near += (u64)n_near * gcount - self;
    tot_pc += (u64)n_pc * gcount;
    len_pp = n_far + n_near; len_pc = n_pc;
}

// split walk: accpot += the sums of parts 1.., nbr_count likewise, in fixed order (deterministic)
__global__ void __launch_bounds__(256) split_combine_kernel(float4 *__restrict__ accpot, u32 *__restrict__ nbr_count,
                                                            const float4 *__restrict__ split_acc, const u32 *__restrict__ split_cnt,
                                                            u32 n, u32 nparts)
{
    const u32 i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    float4 a = accpot[i];
    u32 c = nbr_count[i];
    for (u32 p = 0; p + 1 < nparts; ++p) {
        const float4 b = split_acc[(size_t)p * n + i];
        a.x += b.x; a.y += b.y; a.z += b.z; a.w += b.w;
        c += split_cnt[(size_t)p * n + i];
    }
    accpot[i] = a;
    nbr_count[i] = c;
}

// Persistent grid: 148 SMs x 4 CTAs x 4 warps; groups are handed out by an atomic ticket, one per warp
// (COOP = false) or one per CTA (COOP = true).  A group of at most 32 bodies takes the one-body-per-lane
// path (half the FP32 work of the packed path).
// Shared memory: WALK_WARPS x WarpShared | WALK_WARPS x WALK_STACK_SMEM stack words | CtaCtl
template <int NIMAX, bool COOP, bool CLS, bool SPLIT = false>
__global__ void __launch_bounds__(WALK_WARPS * 32, WALK_CTAS)
walk_kernel(WalkArgs A, const u32 *__restrict__ group_start, P3TParams prm, u32 *walk_stack)
{
    extern __shared__ __align__(16) unsigned char s_raw[];
    const u32 lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    WarpShared *wsall = reinterpret_cast<WarpShared *>(s_raw);
    u32 *sstack = reinterpret_cast<u32 *>(s_raw + sizeof(WarpShared) * WALK_WARPS);
    CtaCtl *ctl = reinterpret_cast<CtaCtl *>(sstack + WALK_WARPS * WALK_STACK_SMEM);
    StackRef st;
    if (COOP) {
        st.smem = sstack; st.cap = WALK_WARPS * WALK_STACK_SMEM;
        st.gmem = walk_stack + (size_t)blockIdx.x * WALK_WARPS * WALK_STACK_GMEM;
        st.limit = WALK_WARPS * (WALK_STACK_SMEM + WALK_STACK_GMEM);
    } else {
        st.smem = sstack + warp * WALK_STACK_SMEM; st.cap = WALK_STACK_SMEM;
        st.gmem = walk_stack + (size_t)(blockIdx.x * WALK_WARPS + warp) * WALK_STACK_GMEM;
        st.limit = WALK_STACK_SMEM + WALK_STACK_GMEM;
    }
    const u32 ngroups = (u32)A.counters[CNT_NGROUPS];
    // Hand-out order: this call's groups by decreasing PREDICTED cost (group_order, a permutation of 0..ngroups-1 made
    // by group_predict_kernel + group_order_kernel just before this launch: a group is expected to cost what the group
    // that held its first body cost in the previous call).
    // Every rank of a sharded walk must map positions to groups alike: it uses the order only if the ranks have exchanged
    // their cost classes since the last walk (p3t_put_shard_classes), else positions are group numbers (key order).
    const u32 ng_prev = A.use_order ? A.order_meta[0] : 0u;
    const u32 npos = max(ngroups, ng_prev);
    u64 tot_pp = 0, tot_pc = 0, tot_near = 0;
    // split walk: the level whose cells are dealt to the parts = the first one with at least WALK_SPLIT_CELLS cells per
    // part (fine enough for the near field of a group to spread over all parts), or the deepest level
    SplitRule sr = {0u, SPLIT ? A.nparts : 1u, 0u, 0u};
    if (SPLIT) {
        u32 lo = 0, cnt = 0;
        for (int L = 0; L < 24; ++L) {
            cnt = A.level_total[L];
            if (cnt >= (u32)WALK_SPLIT_CELLS * sr.nparts || (L < 23 && A.level_total[L + 1] == 0)) break;
            lo += cnt;
        }
        sr.lo = lo; sr.hi = lo + cnt;
    }

    while (true) {
        u32 g = 0;
        if (COOP) {
            if (threadIdx.x == 0) {
                ctl->group = (u32)atomicAdd(&A.counters[CNT_GROUP_TICKET], 1ull);
                ctl->top = 1; ctl->busy = 0; ctl->lock = 0; ctl->err = 0; ctl->stat[0] = 0; ctl->stat[1] = 0;
                sstack[0] = 0;   // root
            }
            __syncthreads();
            g = ctl->group;
        } else {
            if (lane == 0) g = (u32)atomicAdd(&A.counters[CNT_GROUP_TICKET], 1ull);
            g = __shfl_sync(0xffffffffu, g, 0);
        }
        g = g * A.shard_world + A.shard_rank;   // (overflow-free: tickets stop at npos / world)
        if (SPLIT) { sr.part = g & (sr.nparts - 1u); g /= sr.nparts; }   // the parts of a group: consecutive tickets
        if (g >= npos) break;
        if (g < ng_prev) g = A.group_order[g];
        if (g >= ngroups) {                      // a group of the previous call that is gone
            if (COOP) __syncthreads();           // ctl is rewritten for the next ticket
            continue;
        }
        const u32 gs = group_start[g], ge = group_start[g + 1];
        P3T_DEV_ASSERT(gs < ge && ge <= A.n && ge - gs <= 32u * NIMAX);
        const u32 t0 = (u32)globaltimer_ns();
        u32 len_pp = 0, len_pc = 0;
        if (NIMAX == 2 && ge - gs > 32) walk_group<2, COOP, CLS, SPLIT>(wsall, st, ctl, A, prm, gs, ge, lane, warp, tot_pp, tot_pc, tot_near, sr, len_pp, len_pc);
        else walk_group<1, COOP, CLS, SPLIT>(wsall, st, ctl, A, prm, gs, ge, lane, warp, tot_pp, tot_pc, tot_near, sr, len_pp, len_pc);
        __syncwarp();
        // diagnostics: list lengths of this group (+1: the self term removed from tot_pp) and its time window
        if (COOP) {
            if (threadIdx.x == 0) {
                A.group_stats[g] = make_uint4(ctl->stat[0], ctl->stat[1], t0, (u32)globaltimer_ns());
                ctl->cls = cost_class(ctl->stat[0], ctl->stat[1], ge - gs > 32);
            }
            __syncthreads();   // ctl is rewritten for the next group (cls only at the end of that group)
            for (u32 bb = gs + threadIdx.x; bb < ge; bb += blockDim.x) A.body_class[A.sorted_idx[bb]] = ctl->cls;
        } else if (!SPLIT || sr.part == 0) {
            // (a split walk files the group under nparts x part 0's list lengths: the parts take alike shares)
            u32 c = 0;
            if (lane == 0) {
                const u32 lpp = len_pp * sr.nparts, lpc = len_pc * sr.nparts;
#ifdef P3T_DIAG_SLOT
                u32 smid_, wid_;
                asm volatile("mov.u32 %0, %%smid;" : "=r"(smid_));
                asm volatile("mov.u32 %0, %%warpid;" : "=r"(wid_));
                A.group_stats[g] = make_uint4((smid_ << 16) | (wid_ << 8) | ((blockIdx.x / 148u) << 4) | warp, 26 * lpp / 66 + lpc, t0, (u32)globaltimer_ns());
#else
                A.group_stats[g] = make_uint4(lpp, lpc, t0, (u32)globaltimer_ns());
#endif
                c = cost_class(lpp, lpc, ge - gs > 32);
            }
            c = __shfl_sync(0xffffffffu, c, 0);
            for (u32 bb = gs + lane; bb < ge; bb += 32) A.body_class[A.sorted_idx[bb]] = c;
        }
    }
    if (lane == 0) {
        atomicAdd(&A.counters[CNT_NPP], tot_pp);
        atomicAdd(&A.counters[CNT_NPC], tot_pc);
        atomicAdd(&A.counters[CNT_NNEAR], tot_near);
    }
}

// Groups by decreasing predicted cost, so that the long ones start first and the tail of the persistent launch is made
// of short ones.  The walk files every body under the cost class of its group (list lengths x 13 / 33 packed
// operations, halved for the one-body-per-lane path; top bits of the cost as a float: 8 classes per octave).  The next
// call, whose tree is a little different (bodies have moved, group boundaries and numbers have shifted), predicts for
// each of ITS groups the class its first body had (group_predict_kernel) and counts the classes; group_order_kernel
// turns the counts into offsets (every CTA scans the 1024 counters itself) and scatters the group ids.  (Keyed by group
// number instead, the order of the previous call was worth 0.32 ms of 9 at N = 1M when the positions did not change and
// almost nothing when they did.)  The order is only a schedule: results do not depend on it.
__global__ void __launch_bounds__(256) group_predict_kernel(const u32 *__restrict__ group_start, const u32 *__restrict__ sorted_idx,
                                                            const u32 *__restrict__ body_class, const u64 *__restrict__ counters,
                                                            u32 *__restrict__ gclass, u32 *hist)
{
    const u32 ng = (u32)counters[CNT_NGROUPS];
    // (the group count lives on the device: a fixed grid strides over it)
    for (u32 g = blockIdx.x * blockDim.x + threadIdx.x; g < ng; g += gridDim.x * blockDim.x) {
        // (class 0 = most expensive: the minimum over the first, middle and last body guards against a group that
        //  inherited its first body from a cheaper neighbour)
        const u32 gs = group_start[g], ge = group_start[g + 1];
        const u32 c = min(min(body_class[sorted_idx[gs]], body_class[sorted_idx[gs + (ge - gs) / 2]]),
                          min(body_class[sorted_idx[ge - 1]], (u32)ORDER_CLASSES - 1u));
        gclass[g] = c;
        atomicAdd(&hist[c], 1u);
    }
}

__global__ void __launch_bounds__(256) group_order_kernel(const u32 *__restrict__ gclass, const u32 *__restrict__ hist, u32 *cursor,
                                                          const u64 *__restrict__ counters, u32 *__restrict__ order, u32 *order_meta)
{
    __shared__ u32 s_base[ORDER_CLASSES];
    __shared__ u32 s_warp[8];
    const u32 ng = (u32)counters[CNT_NGROUPS], tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    // exclusive scan of the class counts: four consecutive classes per thread
    u32 v[4], sum = 0;
#pragma unroll
    for (int k = 0; k < 4; ++k) { v[k] = hist[4 * tid + k]; sum += v[k]; }
    u32 inc = sum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        u32 t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) s_warp[warp] = inc;
    __syncthreads();
    u32 base = inc - sum;
    for (u32 w = 0; w < warp; ++w) base += s_warp[w];
#pragma unroll
    for (int k = 0; k < 4; ++k) { s_base[4 * tid + k] = base; base += v[k]; }
    __syncthreads();
    for (u32 g = blockIdx.x * blockDim.x + tid; g < ng; g += gridDim.x * blockDim.x) {
        const u32 c = gclass[g];
        order[s_base[c] + atomicAdd(&cursor[c], 1u)] = g;
    }
    if (blockIdx.x == 0 && tid == 0) order_meta[0] = ng;
}

// The same order without atomics: one CTA, groups taken 1024 at a time, a group's place inside its class = the places
// taken by earlier chunks + the number of groups of its class before it in the chunk.  Slower (about 50 us per 20 000
// groups) but a function of the classes alone: the ranks of a sharded walk all get the SAME order, which is what lets
// them deal its positions out among themselves (p3t_set_shard).
__global__ void __launch_bounds__(1024) group_order_det_kernel(const u32 *__restrict__ gclass, const u32 *__restrict__ hist,
                                                               const u64 *__restrict__ counters, u32 *__restrict__ order, u32 *order_meta)
{
    __shared__ u32 s_base[ORDER_CLASSES], s_cur[ORDER_CLASSES], s_cls[1024];
    const u32 ng = (u32)counters[CNT_NGROUPS], tid = threadIdx.x;
    if (tid == 0) {
        u32 run = 0;
        for (u32 c = 0; c < ORDER_CLASSES; ++c) { s_base[c] = run; run += hist[c]; }
    }
    s_cur[tid] = 0;
    __syncthreads();
    for (u32 g0 = 0; g0 < ng; g0 += 1024) {
        const u32 g = g0 + tid;
        const u32 c = g < ng ? gclass[g] : 0xffffffffu;
        s_cls[tid] = c;
        __syncthreads();
        if (g < ng) {
            u32 r = 0;
            for (u32 t = 0; t < tid; ++t) r += s_cls[t] == c ? 1u : 0u;
            order[s_base[c] + s_cur[c] + r] = g;
        }
        __syncthreads();
        if (g < ng) atomicAdd(&s_cur[c], 1u);     // counts only: the order of these additions does not matter
        __syncthreads();
    }
    if (tid == 0) order_meta[0] = ng;
}

// records of a sharded evaluation for ONE all-reduce (sum) over the ranks: (ax, ay, az, phi, cost class + 1) per particle
// in user order, all zero for the particles of the groups other ranks walked
__global__ void __launch_bounds__(256) shard_record_kernel(const float4 *__restrict__ accpot, const u32 *__restrict__ body_class,
                                                           float *__restrict__ rec, u32 n)
{
    const u32 i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float4 a = accpot[i];
    const u32 c = body_class[i];
    float *r = rec + 5 * (size_t)i;
    r[0] = a.x; r[1] = a.y; r[2] = a.z; r[3] = a.w;
    r[4] = c == 0xffffffffu ? 0.f : (float)(c + 1u);
}
__global__ void __launch_bounds__(256) shard_classes_kernel(const float *__restrict__ rec, u32 *__restrict__ body_class, u32 n)
{
    const u32 i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float v = rec[5 * (size_t)i + 4];
    body_class[i] = v >= 0.5f ? min((u32)(v - 0.5f), (u32)ORDER_CLASSES - 1u) : (u32)ORDER_CLASSES - 1u;
}
p3t_status p3t_stage_shard_record(p3t_ctx *ctx, float *d_rec)
{
    shard_record_kernel<<<div_up(ctx->n, 256), 256, 0, ctx->stream>>>(ctx->ws.accpot, ctx->ws.body_class, d_rec, (u32)ctx->n);
    P3T_CUDA(ctx, cudaGetLastError());
    return P3T_OK;
}
p3t_status p3t_stage_shard_classes(p3t_ctx *ctx, const float *d_rec)
{
    shard_classes_kernel<<<div_up(ctx->n, 256), 256, 0, ctx->stream>>>(d_rec, ctx->ws.body_class, (u32)ctx->n);
    P3T_CUDA(ctx, cudaGetLastError());
    return P3T_OK;
}

#ifdef P3T_WALK_PROFILE
extern "C" void p3t_debug_wprof(unsigned long long *out)
{
    cudaDeviceSynchronize();
    cudaMemcpyFromSymbol(out, g_wprof, sizeof(g_wprof));
    unsigned long long z[WP_SLOTS] = {0};
    cudaMemcpyToSymbol(g_wprof, z, sizeof(z));
}
#endif

p3t_status p3t_stage_walk(p3t_ctx *ctx)
{
    Workspace &w = ctx->ws;
    cudaStream_t s = ctx->stream;
    // eval counters + cost-class counts and scatter cursors of the group order: contiguous, one memset
    P3T_CUDA(ctx, cudaMemsetAsync(w.counters + CNT_NPP, 0, 8 * sizeof(u64) + 2 * ORDER_CLASSES * sizeof(u32), s));
    P3T_CUDA(ctx, cudaMemsetAsync(w.nbr_cursor, 0, ctx->n * sizeof(u32), s));     // scatter cursors of the neighbour stage (no memset inside its chain)
    u32 grid = (u32)ctx->sm_count * WALK_CTAS;
    if ((size_t)grid * WALK_WARPS > w.walk_warps_max) grid = (u32)(w.walk_warps_max / WALK_WARPS);
    const size_t smem = (sizeof(WarpShared) + WALK_STACK_SMEM * sizeof(u32)) * WALK_WARPS + sizeof(CtaCtl);
    typedef void (*walk_fn)(WalkArgs, const u32 *, P3TParams, u32 *);
    static const walk_fn fns[12] = {walk_kernel<1, false, false>, walk_kernel<2, false, false>, walk_kernel<1, true, false>, walk_kernel<2, true, false>,
                                    walk_kernel<1, false, true>,  walk_kernel<2, false, true>,  walk_kernel<1, true, true>,  walk_kernel<2, true, true>,
                                    walk_kernel<1, false, false, true>, walk_kernel<2, false, false, true>,      // split walk
                                    walk_kernel<1, false, true, true>,  walk_kernel<2, false, true, true>};
    if (!ctx->walk_attr_set) {   // function attributes are per device: kept per context
        for (int k = 0; k < 12; ++k) P3T_CUDA(ctx, cudaFuncSetAttribute(fns[k], cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        ctx->walk_attr_set = true;
    }
    WalkArgs A;
    A.body = w.body; A.sorted_idx = w.idx[ctx->cur];
    A.cell_mac = w.cell_mac; A.cell_mom0 = w.cell_mom0; A.cell_mom1 = w.cell_mom1; A.cell_meta = w.cell_meta;
    A.accpot = w.accpot; A.nbr_count = w.nbr_count; A.group_stats = w.group_stats; A.pairs = w.pairs; A.pair_cap = (u64)ctx->nbr_capacity;
    A.counters = w.counters;
    A.group_order = w.group_order;
    A.order_meta = w.order_meta;
    A.body_class = w.body_class;
    A.order_hist = w.order_hist;
    A.shard_rank = (u32)ctx->shard_rank;
    A.shard_world = (u32)ctx->shard_world;
    A.cls_sorted = w.cls_sorted;
    A.cube = w.cube;
    A.n = (u32)ctx->n;
    if (ctx->shard_world > 1) {   // particles of the groups other ranks walk: zero acceleration, potential, neighbour count
        P3T_CUDA(ctx, cudaMemsetAsync(w.accpot, 0, ctx->n * sizeof(float4), s));
        P3T_CUDA(ctx, cudaMemsetAsync(w.nbr_count, 0, ctx->n * sizeof(u32), s));
    }
    // hand-out order of this call's groups from the classes the previous call left per body (the group count lives on
    // the device).  A sharded walk orders its groups only if the ranks have exchanged their classes since the last walk
    // (then all ranks hold the same classes, and the atomic-free order kernel gives all of them the same order); it then
    // marks every body "not mine" so that the next exchange can tell whose class is whose.
    A.use_order = (ctx->shard_world == 1 || ctx->shard_classes_fresh) ? 1u : 0u;
    if (A.use_order) {
        const u32 ogrid = min(div_up(ctx->n, 256 * 32), (u32)ctx->sm_count * 4);     // about n / 50 groups: a few per thread
        group_predict_kernel<<<ogrid, 256, 0, s>>>(w.group_start, w.idx[ctx->cur], w.body_class, w.counters, w.group_class, w.order_hist);
        if (ctx->shard_world == 1)
            group_order_kernel<<<ogrid, 256, 0, s>>>(w.group_class, w.order_hist, w.order_hist + ORDER_CLASSES, w.counters,
                                                                  w.group_order, w.order_meta);
        else
            group_order_det_kernel<<<1, 1024, 0, s>>>(w.group_class, w.order_hist, w.counters, w.group_order, w.order_meta);
    }
    if (ctx->shard_world > 1) {
        P3T_CUDA(ctx, cudaMemsetAsync(w.body_class, 0xff, ctx->n * sizeof(u32), s));
        ctx->shard_classes_fresh = false;
    }
    // one CTA per group when there are too few groups to keep every warp busy to the end of the launch
    // (the group count lives on the device; n / ngroup is its lower bound up to the fill of the groups)
    bool coop = ctx->walk_mode == 2 || (ctx->walk_mode == 0 && 20 * (ctx->n / (size_t)ctx->ngroup) < (size_t)WALK_COOP_BELOW_X20 * grid * WALK_WARPS);
    // split walk (modes 3, 4: 2 or 4 warps per group; auto: 2 below 1.3 groups per resident warp, 4 below 0.65), so that
    // the hand-out has about two items per warp to balance with
    u32 nparts = ctx->walk_mode == 3 ? 2u : ctx->walk_mode == 4 ? 4u : 1u;
    if (ctx->walk_mode == 0 && !coop) {
        const size_t groups = ctx->n / (size_t)ctx->ngroup, warps = (size_t)grid * WALK_WARPS;
        nparts = 20 * groups >= WALK_SPLIT_BELOW_X20 * warps ? 1u : 40 * groups >= WALK_SPLIT_BELOW_X20 * warps ? 2u : 4u;
    }
    if (ctx->shard_world > 1 || coop) nparts = 1;
    A.nparts = nparts;
    ctx->walk_parts_used = coop ? 0 : (int)nparts;
    A.level_total = w.level_total;
    A.split_acc = reinterpret_cast<float4 *>(w.hard_out);          // 48 n bytes of the 56 n (free until p3t_eval_hard)
    A.split_cnt = reinterpret_cast<u32 *>(w.herm_state);           // 12 n bytes of 96 n (free until p3t_hermite_step)
    const dim3 block(WALK_WARPS * 32);
    const int fi = nparts > 1 ? 8 + (ctx->ngroup == 64 ? 1 : 0) + (ctx->cls_n ? 2 : 0)
                              : (ctx->ngroup == 64 ? 1 : 0) + (coop ? 2 : 0) + (ctx->cls_n ? 4 : 0);
    fns[fi]<<<grid, block, smem, s>>>(A, w.group_start, ctx->prm, w.walk_stack);
    if (nparts > 1)
        split_combine_kernel<<<div_up(ctx->n, 256), 256, 0, s>>>(w.accpot, w.nbr_count, A.split_acc, A.split_cnt, (u32)ctx->n, nparts);
    P3T_CUDA(ctx, cudaGetLastError());
    return P3T_OK;
}
