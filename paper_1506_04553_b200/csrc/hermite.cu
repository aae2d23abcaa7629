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
// Design.  The whole block loop runs inside ONE cooperative kernel: the non-isolated particles are compacted into a slot
// list; every block each thread looks at its slots, evaluates the active ones (predicting the particle and each of
// its neighbours from that neighbour's own time, fp64), grid barrier, corrects them and chooses the next step, grid
// barrier.  The next block time is a 64-bit atomicMin over (t + dt) into one of three rotating words, so no host
// round trip and no launch per block: a block costs two grid barriers.  The grid is only as large as the slot count
// needs (a handful of particles: one CTA, the barrier is then a __syncthreads).  State is indexed by particle:
// (t << 8 | log2 dt), a, a1, and the new a, a1 of the block.
#include "p3t_internal.cuh"
#include <cooperative_groups.h>
#include <math_constants.h>
namespace cg = cooperative_groups;

#define HERM_THREADS 256
#define HERM_TICK_BITS 40
enum { HC_COUNT = 0, HC_TMIN0, HC_TMIN1, HC_TMIN2, HC_BLOCKS, HC_STEPS, HC_FLOOR, HC_ERR, HC_WORDS = 8 };

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

// slot list of the particles whose list is not empty (order is irrelevant: a particle's arithmetic only involves its list)
__global__ void herm_collect_kernel(const u64 *__restrict__ offset, u32 n, u32 *__restrict__ ids, u64 *__restrict__ ctl)
{
    const u32 i = blockIdx.x * blockDim.x + threadIdx.x;
    const bool has = i < n && offset[i + 1] > offset[i];
    const u32 m = __ballot_sync(0xffffffffu, has);
    if (!m) return;
    const u32 lane = threadIdx.x & 31;
    u32 base = 0;
    if (lane == 0) base = (u32)atomicAdd((unsigned long long *)&ctl[HC_COUNT], (unsigned long long)__popc(m));
    base = __shfl_sync(0xffffffffu, base, 0);
    if (has) ids[base + __popc(m & ((1u << lane) - 1))] = i;
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

struct HermArgs {
    const float4 *body_user;       // mass in .w (the masses of the evaluation that made the lists)
    const u64 *offset;
    const u32 *nbr;
    const u32 *ids;
    double *pos, *vel;             // [n][3] in/out
    u64 *tdt;                      // [n] t << 8 | log2(dt)
    double *a, *a1, *an, *a1n;     // [n][3]
    u64 *ctl;
    P3TParams prm;
    double tick, eta, eta_s, a0;
    u64 max_ticks, max_blocks;
};

// Eq. 7 and its time derivative over the list of i at time tn (ticks); the particle and its neighbours are predicted
// from their own last times.  first: t = 0, nothing to predict.
__device__ __forceinline__ void herm_force(const HermArgs &A, u32 i, u64 tn, bool first, double *a, double *a1)
{
    double xi[3], vi[3];
    {
        const double h = first ? 0.0 : (double)(tn - (A.tdt[i] >> 8)) * A.tick;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const double X = A.pos[3 * (size_t)i + c], V = A.vel[3 * (size_t)i + c];
            const double Ac = first ? 0.0 : A.a[3 * (size_t)i + c], Jc = first ? 0.0 : A.a1[3 * (size_t)i + c];
            xi[c] = X + h * (V + h * (Ac / 2.0 + h * (Jc / 6.0)));
            vi[c] = V + h * (Ac + h * (Jc / 2.0));
        }
    }
    const double eps2 = A.prm.eps2_d;
    double ax = 0, ay = 0, az = 0, jx = 0, jy = 0, jz = 0;
    for (u64 k = A.offset[i], e = A.offset[i + 1]; k < e; ++k) {
        const u32 j = A.nbr[k];
        const double h = first ? 0.0 : (double)(tn - (A.tdt[j] >> 8)) * A.tick;
        double d[3], w[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const double X = A.pos[3 * (size_t)j + c], V = A.vel[3 * (size_t)j + c];
            const double Ac = first ? 0.0 : A.a[3 * (size_t)j + c], Jc = first ? 0.0 : A.a1[3 * (size_t)j + c];
            d[c] = xi[c] - (X + h * (V + h * (Ac / 2.0 + h * (Jc / 6.0))));
            w[c] = vi[c] - (V + h * (Ac + h * (Jc / 2.0)));
        }
        const double s2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2] + eps2;
        const double s = sqrt(s2);
        double omK, dKds;
        herm_weights(A.prm, s, omK, dKds);
        if (omK == 0.0 && dKds == 0.0) continue;
        const double qv = d[0] * w[0] + d[1] * w[1] + d[2] * w[2];
        const double mr3 = (double)A.body_user[j].w / (s2 * s);
        const double c1 = mr3 * omK, c2 = mr3 * (3.0 * omK * qv / s2 + dKds * qv / s);
        ax -= c1 * d[0]; ay -= c1 * d[1]; az -= c1 * d[2];
        jx -= c1 * w[0] - c2 * d[0]; jy -= c1 * w[1] - c2 * d[1]; jz -= c1 * w[2] - c2 * d[2];
    }
    a[0] = ax; a[1] = ay; a[2] = az;
    a1[0] = jx; a1[1] = jy; a1[2] = jz;
}

__device__ __forceinline__ double norm3(const double *u) { return sqrt(u[0] * u[0] + u[1] * u[1] + u[2] * u[2]); }

// log2 of the largest power of two of ticks <= crit (a time), <= max_ticks, dividing t; at least one tick
__device__ __forceinline__ u32 herm_quantise(const HermArgs &A, double crit, u64 t, u32 &floor_hits)
{
    const double ct = crit / A.tick;
    u32 k;
    const u32 kmax = 63 - __clzll((long long)A.max_ticks);
    if (!(ct < (double)A.max_ticks)) k = kmax;
    else if (ct < 1.0) { k = 0; ++floor_hits; }
    else k = (u32)((__double2hiint(ct) >> 20) & 0x7ff) - 1023u;
    if (t) {
        const u32 tz = __ffsll((long long)t) - 1;          // t % 2^k == 0  <=>  k <= trailing zeros of t
        if (k > tz) k = tz;
    }
    return k;
}

__global__ void __launch_bounds__(HERM_THREADS) hermite_kernel(HermArgs A)
{
    cg::grid_group grid = cg::this_grid();
    const u32 M = (u32)A.ctl[HC_COUNT];
    const u32 tid = blockIdx.x * blockDim.x + threadIdx.x, stride = gridDim.x * blockDim.x;
    const u64 total = 1ull << HERM_TICK_BITS;
    u32 floor_hits = 0, steps = 0;

    // t = 0: forces from the current state, first steps from Eq. 20
    {
        u64 local_min = ~0ull;
        for (u32 s = tid; s < M; s += stride) {
            const u32 i = A.ids[s];
            double a[3], a1[3];
            herm_force(A, i, 0, true, a, a1);
            const double na = norm3(a), n1 = norm3(a1);
            const double crit = n1 > 0.0 ? A.eta_s * sqrt((na * na + A.a0 * A.a0) / (n1 * n1)) : CUDART_INF;
            const u32 k = herm_quantise(A, crit, 0, floor_hits);
#pragma unroll
            for (int c = 0; c < 3; ++c) { A.a[3 * (size_t)i + c] = a[c]; A.a1[3 * (size_t)i + c] = a1[c]; }   // nobody reads a, a1, tdt at t = 0
            A.tdt[i] = k;                                   // t = 0
            local_min = min(local_min, 1ull << k);
        }
        if (local_min != ~0ull) atomicMin((unsigned long long *)&A.ctl[HC_TMIN0], (unsigned long long)local_min);
    }
    grid.sync();

    u64 b = 0;
    for (;; ++b) {
        const u64 tn = *(volatile u64 *)&A.ctl[HC_TMIN0 + b % 3];
        if (tn == ~0ull) break;
        if (b >= A.max_blocks) { if (tid == 0) A.ctl[HC_ERR] = 1; break; }
        u64 *next = &A.ctl[HC_TMIN0 + (b + 1) % 3];
        u64 local_min = ~0ull;
        // evaluate the active particles from the state before the block
        for (u32 s = tid; s < M; s += stride) {
            const u32 i = A.ids[s];
            const u64 w = A.tdt[i];
            const u64 t = w >> 8, te = t + (1ull << (w & 63));
            if (t >= total) continue;
            if (te != tn) { local_min = min(local_min, te); continue; }
            double a[3], a1[3];
            herm_force(A, i, tn, false, a, a1);
#pragma unroll
            for (int c = 0; c < 3; ++c) { A.an[3 * (size_t)i + c] = a[c]; A.a1n[3 * (size_t)i + c] = a1[c]; }
        }
        grid.sync();
        // correct them together, choose the next steps (Eq. 18)
        for (u32 s = tid; s < M; s += stride) {
            const u32 i = A.ids[s];
            const u64 w = A.tdt[i];
            const u64 t = w >> 8;
            if (t >= total || t + (1ull << (w & 63)) != tn) continue;
            const double h = (double)(1ull << (w & 63)) * A.tick;
            double an[3], jn[3], a2e[3], a3[3];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const size_t o = 3 * (size_t)i + c;
                const double Ac = A.a[o], Jc = A.a1[o], An = A.an[o], Jn = A.a1n[o];
                const double a2 = (-6.0 * (Ac - An) - h * (4.0 * Jc + 2.0 * Jn)) / (h * h);
                a3[c] = (12.0 * (Ac - An) + 6.0 * h * (Jc + Jn)) / (h * h * h);
                const double X = A.pos[o], V = A.vel[o];
                const double xp = X + h * (V + h * (Ac / 2.0 + h * (Jc / 6.0)));
                const double vp = V + h * (Ac + h * (Jc / 2.0));
                A.pos[o] = xp + h * h * h * h * (a2 / 24.0 + h * a3[c] / 120.0);
                A.vel[o] = vp + h * h * h * (a2 / 6.0 + h * a3[c] / 24.0);
                a2e[c] = a2 + h * a3[c];
                A.a[o] = An; A.a1[o] = Jn;
                an[c] = An; jn[c] = Jn;
            }
            ++steps;
            const double na = norm3(an), n1 = norm3(jn), n2 = norm3(a2e), n3 = norm3(a3);
            const double den = n1 * n3 + n2 * n2;
            const double crit = den > 0.0 ? A.eta * sqrt((sqrt(na * na + A.a0 * A.a0) * n2 + n1 * n1) / den) : CUDART_INF;
            const u32 k = herm_quantise(A, crit, tn, floor_hits);
            A.tdt[i] = tn << 8 | k;
            if (tn < total) local_min = min(local_min, tn + (1ull << k));
        }
        if (local_min != ~0ull) atomicMin((unsigned long long *)next, (unsigned long long)local_min);
        if (tid == 0) A.ctl[HC_TMIN0 + (b + 2) % 3] = ~0ull;
        grid.sync();
    }
    if (steps) atomicAdd((unsigned long long *)&A.ctl[HC_STEPS], (unsigned long long)steps);
    if (floor_hits) atomicAdd((unsigned long long *)&A.ctl[HC_FLOOR], (unsigned long long)floor_hits);
    if (tid == 0) A.ctl[HC_BLOCKS] = b;
}

// Enqueues the collection, reads the slot count back (one synchronisation: the grid is sized by it), then the block
// loop and the drift.  d_pos, d_vel: device [n][3] doubles, updated in place.
p3t_status p3t_stage_hermite(p3t_ctx *ctx, double *d_pos, double *d_vel, double T, int log2_div, double eta, double eta_s,
                             double a0, long long max_blocks, u64 *h_ctl)
{
    Workspace &w = ctx->ws;
    const u32 n = (u32)ctx->n;
    P3T_CUDA(ctx, cudaMemsetAsync(w.herm_ctl, 0, HC_WORDS * sizeof(u64), ctx->stream));
    P3T_CUDA(ctx, cudaMemsetAsync(w.herm_ctl + HC_TMIN0, 0xff, 3 * sizeof(u64), ctx->stream));
    herm_collect_kernel<<<div_up(n, 256), 256, 0, ctx->stream>>>(w.nbr_offset, n, w.herm_ids, w.herm_ctl);
    P3T_CUDA(ctx, cudaGetLastError());
    P3T_CUDA(ctx, cudaMemcpyAsync(h_ctl, w.herm_ctl, sizeof(u64), cudaMemcpyDeviceToHost, ctx->stream));
    P3T_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    const u64 M = h_ctl[HC_COUNT];
    if (M) {
        HermArgs A;
        A.body_user = w.body_user; A.offset = w.nbr_offset; A.nbr = w.nbr; A.ids = w.herm_ids;
        A.pos = d_pos; A.vel = d_vel;
        A.tdt = w.herm_tdt; A.a = w.herm_state; A.a1 = w.herm_state + 3 * (size_t)ctx->max_n;
        A.an = w.herm_state + 6 * (size_t)ctx->max_n; A.a1n = w.herm_state + 9 * (size_t)ctx->max_n;
        A.ctl = w.herm_ctl;
        A.prm = ctx->prm;
        A.tick = T / (double)(1ull << HERM_TICK_BITS);
        A.eta = eta; A.eta_s = eta_s; A.a0 = a0;
        A.max_ticks = (1ull << HERM_TICK_BITS) >> log2_div;
        A.max_blocks = (u64)max_blocks;
        int per_sm = 0;
        P3T_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, hermite_kernel, HERM_THREADS, 0));
        if (per_sm < 1) return p3t_fail(ctx, P3T_ECUDA, "hermite_kernel does not fit an SM");
        u32 grid = (u32)((M + HERM_THREADS - 1) / HERM_THREADS);
        if (grid > (u32)ctx->sm_count) grid = (u32)ctx->sm_count;       // one CTA per SM: the barrier is the cost of a block
        void *args[] = {&A};
        P3T_CUDA(ctx, cudaLaunchCooperativeKernel((void *)hermite_kernel, dim3(grid), dim3(HERM_THREADS), args, 0, ctx->stream));
    }
    herm_drift_kernel<<<div_up(n, 256), 256, 0, ctx->stream>>>(w.nbr_offset, n, T, d_pos, d_vel);
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
