// moments.cu -- row a6: bottom-up monopole + quadrupole moments ("up to the quadrupole moment",
// PAPER.md L138), tight AABBs and the per-cell acceptance radius, in ONE launch.
//
// One thread per cell.  Leaf threads reduce their bodies, then climb: a thread that finishes cell k
// increments its parent's arrival counter; the thread that brings it to the parent's child count
// merges the children (parallel-axis shift of the quadrupoles) and keeps climbing.  Children are
// always merged in index order, so the result is deterministic.
//
// Acceptance radius (rule R-MAC of DESIGN.md, readings A9/A10): a cell C may be used as a multipole
// by a group with box B iff  d(B, c_C)^2 > rcrit_C^2,
//   rcrit_C = max( l_C / theta + |c_C - g_C| ,  (h + rmax_C) (1 + 1e-5) + slack ),
// l_C the cube side, g_C its geometric centre, c_C the centre of mass, rmax_C a bound of the
// distance from c_C to any body of C (farthest corner of the tight AABB).  The second term
// guarantees that no body of C is within h of any body of the group, so accepted cells carry
// K = W = 1 and hold no neighbours.  theta = 0 gives rcrit = inf (nothing is accepted).
#include "p3t_internal.cuh"

__device__ __forceinline__ u32 compact3(u64 x)
{
    x &= 0x1249249249249249ull;
    x = (x ^ (x >> 2)) & 0x10c30c30c30c30c3ull;
    x = (x ^ (x >> 4)) & 0x100f00f00f00f00full;
    x = (x ^ (x >> 8)) & 0x1f0000ff0000ffull;
    x = (x ^ (x >> 16)) & 0x1f00000000ffffull;
    x = (x ^ (x >> 32)) & 0x1fffffull;
    return (u32)x;
}

struct Mom {
    float cx, cy, cz, M;
    float qxx, qyy, qzz, qxy, qxz, qyz;
    float lox, loy, loz, hix, hiy, hiz;
};

__device__ __forceinline__ void store_cell(u32 k, const Mom &m, int level, u64 key, const float *__restrict__ cube,
                                           int max_level, float theta, float h, float4 *cell_mac, float4 *cell_mom0,
                                           float4 *cell_mom1, float4 *cell_bmin, float4 *cell_bmax)
{
    const float side = cube[3];
    const float l = ldexpf(side, -level);
    // geometric centre from the key prefix
    u64 pre = level ? (key >> (3 * (max_level - level))) : 0ull;
    float gx = cube[0] + ((float)compact3(pre >> 2) + 0.5f) * l;
    float gy = cube[1] + ((float)compact3(pre >> 1) + 0.5f) * l;
    float gz = cube[2] + ((float)compact3(pre) + 0.5f) * l;
    float dx = m.cx - gx, dy = m.cy - gy, dz = m.cz - gz;
    float delta = sqrtf(dx * dx + dy * dy + dz * dz);
    float fx = fmaxf(m.cx - m.lox, m.hix - m.cx), fy = fmaxf(m.cy - m.loy, m.hiy - m.cy),
          fz = fmaxf(m.cz - m.loz, m.hiz - m.cz);
    float rmax = sqrtf(fx * fx + fy * fy + fz * fz) * (1.f + 1e-6f);
    float slack = 8.f * 1.1920929e-7f * (fabsf(cube[0]) + fabsf(cube[1]) + fabsf(cube[2]) + 2.f * side);
    float rc3 = (h + rmax) * (1.f + 1e-5f) + slack;
    float rc1 = theta > 0.f ? l / theta + delta : INFINITY;
    float rc = fmaxf(rc1, rc3);
    cell_mac[k] = make_float4(m.cx, m.cy, m.cz, rc * rc);
    cell_mom0[k] = make_float4(m.M, m.qxx, m.qyy, m.qzz);
    cell_mom1[k] = make_float4(m.qxy, m.qxz, m.qyz, rmax);
    cell_bmin[k] = make_float4(m.lox, m.loy, m.loz, l);
    cell_bmax[k] = make_float4(m.hix, m.hiy, m.hiz, delta);
}

__global__ void __launch_bounds__(128) moments_kernel(
    const float4 *__restrict__ body, const u64 *__restrict__ keys, const float *__restrict__ cube,
    const u8 *__restrict__ cell_level, const u32 *__restrict__ cell_start, const u32 *__restrict__ cell_parent,
    const u32 *__restrict__ cell_first, const u32 *__restrict__ cell_nchild, u32 *cell_ready, uint2 *cell_meta,
    const u8 *__restrict__ dlev, float4 *cell_mac, float4 *cell_mom0, float4 *cell_mom1, float4 *cell_bmin,
    float4 *cell_bmax, const u64 *__restrict__ counters, u32 cell_cap, int max_level, float theta, float h)
{
    u32 ncell = (u32)min((u64)cell_cap, counters[CNT_NCELLS]);
    u32 k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= ncell) return;
    int level = cell_level[k];
    u32 start = cell_start[k];
    if (level != (int)dlev[start]) return;   // internal cell: computed by the last arriving child
    // ---- leaf: two passes over its bodies (offsets from the first body keep the sums well conditioned)
    Mom m;
    {
        uint2 meta = cell_meta[k];
        u32 cnt = meta.y & ~P3T_LEAF_FLAG;
        float4 b0 = body[start];
        float sx = 0.f, sy = 0.f, sz = 0.f, M = 0.f;
        m.lox = m.hix = b0.x; m.loy = m.hiy = b0.y; m.loz = m.hiz = b0.z;
        for (u32 j = 0; j < cnt; ++j) {
            float4 b = body[start + j];
            M += b.w;
            sx += b.w * (b.x - b0.x); sy += b.w * (b.y - b0.y); sz += b.w * (b.z - b0.z);
            m.lox = fminf(m.lox, b.x); m.hix = fmaxf(m.hix, b.x);
            m.loy = fminf(m.loy, b.y); m.hiy = fmaxf(m.hiy, b.y);
            m.loz = fminf(m.loz, b.z); m.hiz = fmaxf(m.hiz, b.z);
        }
        float inv = M > 0.f ? 1.f / M : 0.f;
        m.M = M;
        m.cx = b0.x + sx * inv; m.cy = b0.y + sy * inv; m.cz = b0.z + sz * inv;
        if (!(M > 0.f)) {   // massless leaf: centre of its box
            m.cx = 0.5f * (m.lox + m.hix); m.cy = 0.5f * (m.loy + m.hiy); m.cz = 0.5f * (m.loz + m.hiz);
        }
        m.qxx = m.qyy = m.qzz = m.qxy = m.qxz = m.qyz = 0.f;
        for (u32 j = 0; j < cnt; ++j) {
            float4 b = body[start + j];
            float rx = b.x - m.cx, ry = b.y - m.cy, rz = b.z - m.cz;
            m.qxx += b.w * rx * rx; m.qyy += b.w * ry * ry; m.qzz += b.w * rz * rz;
            m.qxy += b.w * rx * ry; m.qxz += b.w * rx * rz; m.qyz += b.w * ry * rz;
        }
    }
    while (true) {
        store_cell(k, m, level, keys[start], cube, max_level, theta, h, cell_mac, cell_mom0, cell_mom1, cell_bmin, cell_bmax);
        u32 p = cell_parent[k];
        if (p == P3T_NO_PARENT) break;
        __threadfence();
        u32 nch = cell_nchild[p];
        u32 old = atomicAdd(&cell_ready[p], 1u);
        if (old + 1 != nch) break;
        __threadfence();
        // ---- last arrival: merge the children of p in index order
        u32 first = cell_first[p];
        float M = 0.f, sx = 0.f, sy = 0.f, sz = 0.f;
        float4 a0 = __ldcg(&cell_mac[first]);
        m.lox = m.loy = m.loz = INFINITY; m.hix = m.hiy = m.hiz = -INFINITY;
        for (u32 c = 0; c < nch; ++c) {
            float4 a = __ldcg(&cell_mac[first + c]);
            float4 q0 = __ldcg(&cell_mom0[first + c]);
            float4 lo = __ldcg(&cell_bmin[first + c]), hi = __ldcg(&cell_bmax[first + c]);
            M += q0.x;
            sx += q0.x * (a.x - a0.x); sy += q0.x * (a.y - a0.y); sz += q0.x * (a.z - a0.z);
            m.lox = fminf(m.lox, lo.x); m.loy = fminf(m.loy, lo.y); m.loz = fminf(m.loz, lo.z);
            m.hix = fmaxf(m.hix, hi.x); m.hiy = fmaxf(m.hiy, hi.y); m.hiz = fmaxf(m.hiz, hi.z);
        }
        float inv = M > 0.f ? 1.f / M : 0.f;
        m.M = M;
        m.cx = a0.x + sx * inv; m.cy = a0.y + sy * inv; m.cz = a0.z + sz * inv;
        if (!(M > 0.f)) {
            m.cx = 0.5f * (m.lox + m.hix); m.cy = 0.5f * (m.loy + m.hiy); m.cz = 0.5f * (m.loz + m.hiz);
        }
        m.qxx = m.qyy = m.qzz = m.qxy = m.qxz = m.qyz = 0.f;
        for (u32 c = 0; c < nch; ++c) {
            float4 a = __ldcg(&cell_mac[first + c]);
            float4 q0 = __ldcg(&cell_mom0[first + c]);
            float4 q1 = __ldcg(&cell_mom1[first + c]);
            float rx = a.x - m.cx, ry = a.y - m.cy, rz = a.z - m.cz;
            m.qxx += q0.y + q0.x * rx * rx; m.qyy += q0.z + q0.x * ry * ry; m.qzz += q0.w + q0.x * rz * rz;
            m.qxy += q1.x + q0.x * rx * ry; m.qxz += q1.y + q0.x * rx * rz; m.qyz += q1.z + q0.x * ry * rz;
        }
        cell_meta[p] = make_uint2(first, nch);
        k = p;
        level = cell_level[k];
        start = cell_start[k];
    }
}

p3t_status p3t_stage_moments(p3t_ctx *ctx)
{
    Workspace &w = ctx->ws;
    cudaStream_t s = ctx->stream;
    // the number of cells lives on the device; launch for the upper bound the host knows and let
    // surplus threads exit (cells <= min(cell_cap, n * (max_level + 1)))
    size_t bound = ctx->n * (size_t)(ctx->max_level + 1);
    if (bound > w.cell_cap) bound = w.cell_cap;
    moments_kernel<<<div_up(bound, 128), 128, 0, s>>>(w.body, w.keys[ctx->cur], w.cube, w.cell_level, w.cell_start,
                                                      w.cell_parent, w.cell_first, w.cell_nchild, w.cell_ready, w.cell_meta,
                                                      w.dlev, w.cell_mac, w.cell_mom0, w.cell_mom1, w.cell_bmin, w.cell_bmax,
                                                      w.counters, (u32)w.cell_cap, ctx->max_level, ctx->prm.theta, ctx->prm.h);
    P3T_CUDA(ctx, cudaGetLastError());
    return P3T_OK;
}
