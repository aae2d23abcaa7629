// hard.cu -- NEXT row of SURVEY.md 8(f), rank 1: the hard force over the neighbour lists.
//
// For every particle i, from the CSR lists L_i of the last p3t_eval_soft (all j with s_ij < h, h >= r_cut):
//   a_i   = - sum_{j in L_i} m_j (1 - K(s_ij)) q_ij / s_ij^3                       Eq. 7, per unit mass
//   j_i   = d a_i / dt  for  q_ij -> q_ij + v_ij t,   ds/dt = (q_ij . v_ij) / s
//         = - sum_j m_j [ (1 - K) (v_ij / s^3 - 3 (q.v) q_ij / s^5) - K'(s) ((q.v)/s) q_ij / s^3 ]
//   phi_i = - sum_{j in L_i} m_j (1 - W(s_ij)) / s_ij                              Eq. 5 (L53)
// These are what the fourth-order Hermite integrator of the non-isolated particles consumes (procedure
// step 3, L147; the paper evaluates them on the host).  1 - K = 1 - W = 0 for s >= r_cut, so the sum over
// L_i equals the sum over all j.  The lists are short (0.017 entries per particle at the headline workload) and
// the terms span many orders of magnitude: every pair is evaluated in fp64; one thread per particle.
#include "p3t_internal.cuh"

// K, dK/ds and W in double for gamma <= y < 1 (Eq. 12, 16-17 with reading A1); coefficients from set_params
__device__ __forceinline__ void hard_weights(const CutoffSet &p, double s, double &omK, double &dKds, double &omW)
{
    const double y = s * p.inv_rout;
    if (y >= 1.0) { omK = 0.0; dKds = 0.0; omW = 0.0; return; }
    if (y < p.gamma) { omK = 1.0; dKds = 0.0; omW = 1.0 - p.cin * y; return; }
    const double x = (y - p.gamma) * p.inv_1mg;
    const double x2 = x * x;
    omK = 1.0 - x2 * x2 * (35.0 + x * (-84.0 + x * (70.0 - 20.0 * x)));
    const double u = x * (1.0 - x);
    dKds = 140.0 * u * u * u * p.inv_1mg * p.inv_rout;
    double w = p.wc[7];
#pragma unroll
    for (int i = 6; i >= 0; --i) w = w * y + p.wc[i];
    w += p.wl * y * log(y);
    omW = 1.0 - w;
}

#define HARD_THREADS 128
// (Staging the interleaved xyz arrays through shared memory for contiguous global accesses was tried: 44 us
// against 31 us at N = 1M -- the extra block barriers cost more than the partially used sectors.)
__global__ void __launch_bounds__(HARD_THREADS) hard_kernel(const float4 *__restrict__ body_user, const float *__restrict__ vel,
                                                            const u64 *__restrict__ offset, const u32 *__restrict__ nbr,
                                                            const u64 *__restrict__ counters, u64 capacity, P3TParams prm, u32 n,
                                                            double *__restrict__ acc, double *__restrict__ jerk,
                                                            double *__restrict__ pot, const u8 *__restrict__ cls_user)
{
    const u32 i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    if (counters[CNT_PAIRS] > capacity) return;     // the lists did not fit: the caller gets P3T_ECAPACITY
    const float4 bi = body_user[i];
    const double vix = vel[3 * (size_t)i], viy = vel[3 * (size_t)i + 1], viz = vel[3 * (size_t)i + 2];
    const u32 ci = cls_user ? (cls_user[i] & 1u) : 0u;     // pair classes: kind of a pair = ci + cj
    double ax = 0, ay = 0, az = 0, jx = 0, jy = 0, jz = 0, ph = 0;
    for (u64 k = offset[i], e = offset[i + 1]; k < e; ++k) {
        const u32 j = nbr[k];
        P3T_DEV_ASSERT(j < n && j != i);
        const float4 bj = body_user[j];
        const double dx = (double)bi.x - (double)bj.x, dy = (double)bi.y - (double)bj.y, dz = (double)bi.z - (double)bj.z;
        const double wx = vix - (double)vel[3 * (size_t)j], wy = viy - (double)vel[3 * (size_t)j + 1],
                     wz = viz - (double)vel[3 * (size_t)j + 2];
        const u32 kind = ci + (cls_user ? (cls_user[j] & 1u) : 0u);
        const double s2 = dx * dx + dy * dy + dz * dz + (kind == 2u ? prm.eps2_bb_d : prm.eps2_d);
        const double s = sqrt(s2);
        double omK = 1.0, dKds = 0.0, omW = 1.0;         // kind 2 (two black holes): not split, the whole Newtonian term
        if (kind < 2u) hard_weights(prm.cs[kind], s, omK, dKds, omW);
        const double qv = dx * wx + dy * wy + dz * wz;
        const double mr3 = (double)bj.w / (s2 * s);
        const double c1 = mr3 * omK, c2 = mr3 * (3.0 * omK * qv / s2 + dKds * qv / s);
        ax -= c1 * dx; ay -= c1 * dy; az -= c1 * dz;
        jx -= c1 * wx - c2 * dx; jy -= c1 * wy - c2 * dy; jz -= c1 * wz - c2 * dz;
        ph -= (double)bj.w / s * omW;
    }
    if (acc) { acc[3 * (size_t)i] = ax; acc[3 * (size_t)i + 1] = ay; acc[3 * (size_t)i + 2] = az; }
    if (jerk) { jerk[3 * (size_t)i] = jx; jerk[3 * (size_t)i + 1] = jy; jerk[3 * (size_t)i + 2] = jz; }
    if (pot) pot[i] = ph;
}

p3t_status p3t_stage_hard(p3t_ctx *ctx, const float *d_vel, double *d_acc, double *d_jerk, double *d_pot)
{
    Workspace &w = ctx->ws;
    const u32 n = (u32)ctx->n;
    hard_kernel<<<div_up(n, HARD_THREADS), HARD_THREADS, 0, ctx->stream>>>(w.body_user, d_vel, w.nbr_offset, w.nbr, w.counters, (u64)ctx->nbr_capacity,
                                                        ctx->prm, n, d_acc, d_jerk, d_pot, ctx->cls_n ? w.cls_user : nullptr);
    P3T_CUDA(ctx, cudaGetLastError());
    return P3T_OK;
}
