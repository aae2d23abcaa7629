// moments.cu -- row a6: bottom-up monopole + quadrupole moments ("up to the quadrupole moment",
// PAPER.md L138), tight AABBs and the per-cell acceptance radius.
//
// Two launches (moments_kernel<0>: leaves, moments_kernel<1>: internal cells), one thread per cell.
//
// Acceptance radius (rule R-MAC of DESIGN.md, readings A9/A10): a cell C may be used as a multipole
// by a group with box B iff  d(B, c_C)^2 > rcrit_C^2,
//   rcrit_C = max( l_C / theta + |c_C - g_C| ,  (h + rmax_C) (1 + 1e-5) + slack ),
// l_C the cube side, g_C its geometric centre, c_C the centre of mass, rmax_C a bound of the
// distance from c_C to any body of C (farthest corner of the tight AABB).  The second term
// guarantees that no body of C is within h of any body of the group, so accepted cells carry
// K = W = 1 and hold no neighbours.  theta = 0 gives rcrit = inf (nothing is accepted).
#include "p3t_internal.cuh"


struct Mom {
    float cx, cy, cz, M;
    float qxx, qyy, qzz, qxy, qxz, qyz;
    float lox, loy, loz, hix, hiy, hiz;
    bool heavy;        // pair classes: the cell holds a black hole (kept in the sign bit of the stored rmax)
};

template <bool REFIT>
__device__ __forceinline__ void store_cell(u32 k, const Mom &m, int level, u64 key, const float4 &b0, const float *__restrict__ cube,
                                           int max_level, int hilbert, float theta, float h, float4 *cell_mac, float4 *cell_mom0,
                                           float4 *cell_mom1, float4 *cell_bmin, float4 *cell_bmax)
{
    const float side = cube[3];
    const float l = ldexpf(side, -level);
    // geometric centre from the cell's first body: its quantised coordinates, cut to `level` bits.  A build takes them
    // from the body's position with the arithmetic of keys_hist_kernel (the same integers, no inverse transform in the
    // latency chain of the climb); a refit, whose bodies have moved, from the body's key.
    u32 qx, qy, qz;
    if (REFIT) p3t_decode_key(key, max_level, hilbert, qx, qy, qz);
    else {
        const float scale = (float)(1u << max_level) / side;
        const u32 qmax = (1u << max_level) - 1u;
        qx = min((u32)fmaxf((b0.x - cube[0]) * scale, 0.f), qmax);
        qy = min((u32)fmaxf((b0.y - cube[1]) * scale, 0.f), qmax);
        qz = min((u32)fmaxf((b0.z - cube[2]) * scale, 0.f), qmax);
    }
    const int sh = max_level - level;
    float gx = cube[0] + ((float)(qx >> sh) + 0.5f) * l;
    float gy = cube[1] + ((float)(qy >> sh) + 0.5f) * l;
    float gz = cube[2] + ((float)(qz >> sh) + 0.5f) * l;
    float dx = m.cx - gx, dy = m.cy - gy, dz = m.cz - gz;
    float delta = sqrtf(dx * dx + dy * dy + dz * dz);
    float fx = fmaxf(m.cx - m.lox, m.hix - m.cx), fy = fmaxf(m.cy - m.loy, m.hiy - m.cy),
          fz = fmaxf(m.cz - m.loz, m.hiz - m.cz);
    float rmax = sqrtf(fx * fx + fy * fy + fz * fz) * (1.f + 1e-6f);
    float slack = 8.f * 1.1920929e-7f * (fabsf(cube[0]) + fabsf(cube[1]) + fabsf(cube[2]) + 2.f * side);
    float rc3 = (h + rmax) * (1.f + 1e-5f) + slack;          // h: the caller passes h_bf for a cell that holds a black hole
    // Refit (p3t_refit_tree): the bodies have moved since the keys were made and may sit outside the cell's cube; the
    // opening test then takes the side of the smallest cube about the geometric centre that holds them all, which
    // keeps the geometric meaning of l / theta (for bodies inside the cube nothing changes).
    float lm = l;
    if (REFIT) {
        const float ox = fmaxf(gx - m.lox, m.hix - gx), oy = fmaxf(gy - m.loy, m.hiy - gy), oz = fmaxf(gz - m.loz, m.hiz - gz);
        lm = fmaxf(l, 2.f * fmaxf(ox, fmaxf(oy, oz)) * (1.f + 1e-6f));
    }
    float rc1 = theta > 0.f ? lm / theta + delta : INFINITY;
    float rc = fmaxf(rc1, rc3);
    cell_mac[k] = make_float4(m.cx, m.cy, m.cz, rc * rc);
    cell_mom0[k] = make_float4(m.M, m.qxx, m.qyy, m.qzz);
    cell_mom1[k] = make_float4(m.qxy, m.qxz, m.qyz, m.heavy ? -rmax : rmax);
    cell_bmin[k] = make_float4(m.lox, m.loy, m.loz, l);
    cell_bmax[k] = make_float4(m.hix, m.hiy, m.hiz, delta);
}

// One cell from its children [first, first + nch), merged in index order: sums about the first child's
// centre of mass (well conditioned), then the quadrupole is shifted to the centre of mass of the cell
// (parallel-axis theorem).  All loads go to L2 (the records were written by other SMs in this launch).
__device__ __forceinline__ void merge_children(u32 first, u32 nch, const float4 *cell_mac, const float4 *cell_mom0,
                                               const float4 *cell_mom1, const float4 *cell_bmin, const float4 *cell_bmax, Mom &m)
{
    const float4 a0 = __ldcg(&cell_mac[first]);
    float M = 0.f, sx = 0.f, sy = 0.f, sz = 0.f;
    float qxx = 0.f, qyy = 0.f, qzz = 0.f, qxy = 0.f, qxz = 0.f, qyz = 0.f;
    m.lox = m.loy = m.loz = INFINITY; m.hix = m.hiy = m.hiz = -INFINITY;
    m.heavy = false;
#pragma unroll
    for (int c = 0; c < 8; ++c) {
        if ((u32)c < nch) {
            const u32 ci = first + c;
            const float4 a = __ldcg(&cell_mac[ci]), q0 = __ldcg(&cell_mom0[ci]), q1 = __ldcg(&cell_mom1[ci]);
            const float4 lo = __ldcg(&cell_bmin[ci]), hi = __ldcg(&cell_bmax[ci]);
            const float mc = q0.x, rx = a.x - a0.x, ry = a.y - a0.y, rz = a.z - a0.z;
            m.heavy = m.heavy || (__float_as_uint(q1.w) >> 31);
            M += mc;
            sx += mc * rx; sy += mc * ry; sz += mc * rz;
            qxx += q0.y + mc * rx * rx; qyy += q0.z + mc * ry * ry; qzz += q0.w + mc * rz * rz;
            qxy += q1.x + mc * rx * ry; qxz += q1.y + mc * rx * rz; qyz += q1.z + mc * ry * rz;
            m.lox = fminf(m.lox, lo.x); m.loy = fminf(m.loy, lo.y); m.loz = fminf(m.loz, lo.z);
            m.hix = fmaxf(m.hix, hi.x); m.hiy = fmaxf(m.hiy, hi.y); m.hiz = fmaxf(m.hiz, hi.z);
        }
    }
    const float inv = M > 0.f ? 1.f / M : 0.f;
    const float dx = sx * inv, dy = sy * inv, dz = sz * inv;
    m.M = M;
    m.cx = a0.x + dx; m.cy = a0.y + dy; m.cz = a0.z + dz;
    m.qxx = fmaxf(qxx - M * dx * dx, 0.f); m.qyy = fmaxf(qyy - M * dy * dy, 0.f); m.qzz = fmaxf(qzz - M * dz * dz, 0.f);
    m.qxy = qxy - M * dx * dy; m.qxz = qxz - M * dx * dz; m.qyz = qyz - M * dy * dz;
    if (!(M > 0.f)) {
        m.cx = 0.5f * (m.lox + m.hix); m.cy = 0.5f * (m.loy + m.hiy); m.cz = 0.5f * (m.loz + m.hiz);
        m.qxx = m.qyy = m.qzz = m.qxy = m.qxz = m.qyz = 0.f;
    }
}

// PHASE 0: every leaf from its bodies -- a streaming pass without atomics or fences.
// PHASE 1: the internal cells.  cell_nchild[p] holds (children | internal children << 16), counted by
//   emit_kernel.  A cell whose children are all leaves is computed at once; its thread then climbs:
//   it arrives at the parent's counter and the last internal child to arrive merges the parent.
//   Only internal cells (about one cell in eight) pay for a fence and an atomic, and the loads of a
//   merge go to L2, so no acquire (L1 invalidation) is needed.  Children are merged in index order:
//   the result is deterministic.  The counters are read-only here (a late thread must still see whether
//   its cell waits for children); keys_hist_kernel of the next build zeroes them.
template <int PHASE, bool REFIT>
__global__ void __launch_bounds__(128, 4) moments_kernel(
    const float4 *__restrict__ body, const u64 *__restrict__ keys, const float *__restrict__ cube,
    const u8 *__restrict__ cell_level, const u32 *__restrict__ cell_start, const u32 *__restrict__ cell_parent,
    const u32 *__restrict__ cell_first, u32 *cell_nchild, u32 *cell_ready, uint2 *cell_meta,
    float4 *cell_mac, float4 *cell_mom0, float4 *cell_mom1, float4 *cell_bmin,
    float4 *cell_bmax, const u64 *__restrict__ counters, u32 cell_cap, int max_level, int hilbert, float theta, float h,
    const u8 *__restrict__ cls_sorted, float h_bf)
{
    P3T_GRID_TRIGGER();
    P3T_GRID_WAIT();
    const u32 ncell = (u32)min((u64)cell_cap, counters[CNT_NCELLS]);
    for (u32 k0 = blockIdx.x * blockDim.x + threadIdx.x; k0 < ncell; k0 += gridDim.x * blockDim.x) {
        u32 k = k0;
        // emit_kernel writes cell_meta of internal cells as (0, 0): the leaf flag is valid for every cell
        const uint2 meta = cell_meta[k];
        const bool leaf = (meta.y & P3T_LEAF_FLAG) != 0;
        if (leaf != (PHASE == 0)) continue;
        int level = cell_level[k];
        u32 start = cell_start[k];
        Mom m;
        if (PHASE == 0) {
            // ---- leaf: one pass over its bodies, sums about the first body, then shifted to the centre of mass
            const u32 cnt = meta.y & ~P3T_LEAF_FLAG;
            P3T_DEV_ASSERT(cnt >= 1 && meta.x == start);
            const float4 b0 = body[start];
            float sx = 0.f, sy = 0.f, sz = 0.f, M = 0.f;
            float qxx = 0.f, qyy = 0.f, qzz = 0.f, qxy = 0.f, qxz = 0.f, qyz = 0.f;
            m.lox = m.hix = b0.x; m.loy = m.hiy = b0.y; m.loz = m.hiz = b0.z;
            m.heavy = false;
            if (cls_sorted)
                for (u32 j = 0; j < cnt; ++j) m.heavy = m.heavy || cls_sorted[start + j] != 0;
            for (u32 j0 = 0; j0 < cnt; j0 += 4) {
                float4 bb[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) bb[u] = body[start + min(j0 + u, cnt - 1)];
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    if (j0 + u < cnt) {
                        const float4 b = bb[u];
                        const float rx = b.x - b0.x, ry = b.y - b0.y, rz = b.z - b0.z;
                        M += b.w;
                        sx += b.w * rx; sy += b.w * ry; sz += b.w * rz;
                        qxx += b.w * rx * rx; qyy += b.w * ry * ry; qzz += b.w * rz * rz;
                        qxy += b.w * rx * ry; qxz += b.w * rx * rz; qyz += b.w * ry * rz;
                        m.lox = fminf(m.lox, b.x); m.hix = fmaxf(m.hix, b.x);
                        m.loy = fminf(m.loy, b.y); m.hiy = fmaxf(m.hiy, b.y);
                        m.loz = fminf(m.loz, b.z); m.hiz = fmaxf(m.hiz, b.z);
                    }
                }
            }
            const float inv = M > 0.f ? 1.f / M : 0.f;
            const float dx = sx * inv, dy = sy * inv, dz = sz * inv;   // centre of mass - first body
            m.M = M;
            m.cx = b0.x + dx; m.cy = b0.y + dy; m.cz = b0.z + dz;
            m.qxx = fmaxf(qxx - M * dx * dx, 0.f); m.qyy = fmaxf(qyy - M * dy * dy, 0.f); m.qzz = fmaxf(qzz - M * dz * dz, 0.f);
            m.qxy = qxy - M * dx * dy; m.qxz = qxz - M * dx * dz; m.qyz = qyz - M * dy * dz;
            if (!(M > 0.f)) {   // massless leaf: centre of its box
                m.cx = 0.5f * (m.lox + m.hix); m.cy = 0.5f * (m.loy + m.hiy); m.cz = 0.5f * (m.loz + m.hiz);
                m.qxx = m.qyy = m.qzz = m.qxy = m.qxz = m.qyz = 0.f;
            }
            store_cell<REFIT>(k, m, level, REFIT ? keys[start] : 0ull, b0, cube, max_level, hilbert, theta, m.heavy ? h_bf : h, cell_mac, cell_mom0, cell_mom1, cell_bmin, cell_bmax);
            continue;
        }
        // ---- internal cell
        u32 cw = cell_nchild[k];
        if (cw >> 16) continue;          // has internal children: computed by the last of them to arrive
        u32 first = cell_first[k], parent = cell_parent[k];
        u64 key = REFIT ? keys[start] : 0ull;
        float4 bfirst = REFIT ? make_float4(0.f, 0.f, 0.f, 0.f) : body[start];
        while (true) {
            const u32 nch = cw & 0xffffu;
            P3T_DEV_ASSERT(nch >= 1 && nch <= 8 && first > k && first + nch <= ncell && (parent == P3T_NO_PARENT || parent < k));
            // what the next step needs of the parent does not depend on this merge: requested now, so that
            // one level of the climb costs the merge loads, a fence and an atomic, nothing more
            u32 pcw = 0, pfirst = 0, pparent = P3T_NO_PARENT, pstart = 0;
            int plevel = 0;
            if (parent != P3T_NO_PARENT) {
                pcw = cell_nchild[parent]; pfirst = cell_first[parent]; pparent = cell_parent[parent];
                plevel = cell_level[parent]; pstart = cell_start[parent];
            }
            merge_children(first, nch, cell_mac, cell_mom0, cell_mom1, cell_bmin, cell_bmax, m);
            const u64 pkey = (REFIT && parent != P3T_NO_PARENT) ? keys[pstart] : 0ull;
            const float4 pb = (!REFIT && parent != P3T_NO_PARENT) ? body[pstart] : make_float4(0.f, 0.f, 0.f, 0.f);
            store_cell<REFIT>(k, m, level, key, bfirst, cube, max_level, hilbert, theta, m.heavy ? h_bf : h, cell_mac, cell_mom0, cell_mom1, cell_bmin, cell_bmax);
            cell_meta[k] = make_uint2(first, nch);
            if (parent == P3T_NO_PARENT) break;
            __threadfence();             // my record is visible before my arrival is
            if (atomicAdd(&cell_ready[parent], 1u) + 1 != (pcw >> 16)) break;
            k = parent; cw = pcw; first = pfirst; parent = pparent; level = plevel; start = pstart; key = pkey; bfirst = pb;
        }
    }
}

p3t_status p3t_stage_moments(p3t_ctx *ctx)
{
    Workspace &w = ctx->ws;
    cudaStream_t s = ctx->stream;
    // the number of cells lives on the device: grid-stride loops over it
    size_t bound = ctx->n * (size_t)(ctx->max_level + 1);
    if (bound > w.cell_cap) bound = w.cell_cap;
    const u32 grid = (u32)min((size_t)div_up(bound, 128), (size_t)ctx->sm_count * 16);
    P3T_CUDA(ctx, p3t_launch_pdl(moments_kernel<0, false>, dim3(grid), dim3(128), 0, s, (const float4 *)w.body, (const u64 *)w.keys[ctx->cur],
                                 (const float *)w.cube, (const u8 *)w.cell_level, (const u32 *)w.cell_start, (const u32 *)w.cell_parent,
                                 (const u32 *)w.cell_first, w.cell_nchild, w.cell_ready, w.cell_meta, w.cell_mac, w.cell_mom0, w.cell_mom1,
                                 w.cell_bmin, w.cell_bmax, (const u64 *)w.counters, (u32)w.cell_cap, ctx->max_level, ctx->key_curve,
                                 ctx->prm.theta, ctx->prm.h, (const u8 *)(ctx->cls_n ? w.cls_sorted : nullptr), ctx->prm.h_bf));
    P3T_CUDA(ctx, p3t_launch_pdl(moments_kernel<1, false>, dim3(grid), dim3(128), 0, s, (const float4 *)w.body, (const u64 *)w.keys[ctx->cur],
                                 (const float *)w.cube, (const u8 *)w.cell_level, (const u32 *)w.cell_start, (const u32 *)w.cell_parent,
                                 (const u32 *)w.cell_first, w.cell_nchild, w.cell_ready, w.cell_meta, w.cell_mac, w.cell_mom0, w.cell_mom1,
                                 w.cell_bmin, w.cell_bmax, (const u64 *)w.counters, (u32)w.cell_cap, ctx->max_level, ctx->key_curve,
                                 ctx->prm.theta, ctx->prm.h, (const u8 *)(ctx->cls_n ? w.cls_sorted : nullptr), ctx->prm.h_bf));
    P3T_CUDA(ctx, cudaGetLastError());
    return P3T_OK;
}

// ------------------------------------------------------------------------------------------------
// Tree reuse between soft steps ("the cost of the usual complete
// reconstruction of the tree is O(N log N) and not negligible"): the bodies have moved a little, the sorted order, the
// cells and the groups of the last build are kept, and only what depends on the positions is made again -- the
// gathered bodies, then moments, tight boxes and acceptance radii on the old topology.  Lists and forces stay exact in
// the sense of R-MAC (boxes and radii come from the new positions); what degrades is the tightness of cells and
// groups, so the refit also counts the bodies that left the cube of their leaf by more than stray_dist leaf sides.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) refit_gather_kernel(const float4 *__restrict__ body_user, const u32 *__restrict__ idx,
                                                           const u64 *__restrict__ keys, const u8 *__restrict__ dlev,
                                                           const float *__restrict__ cube, float4 *__restrict__ body, u32 n,
                                                           int max_level, int hilbert, float stray_dist, u32 *cell_ready,
                                                           const u32 *__restrict__ prev_ncells, u32 cell_cap, u64 *counters)
{
    // arrival counters of the climb -> 0 (a build has keys_hist_kernel do this)
    for (u32 k = blockIdx.x * blockDim.x + threadIdx.x, nc = min(*prev_ncells, cell_cap); k < nc; k += gridDim.x * blockDim.x)
        cell_ready[k] = 0;
    const float side = cube[3];
    u32 stray = 0;
    for (u32 i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const float4 b = body_user[idx[i]];
        body[i] = b;
        const int D = dlev[i];
        u32 qx, qy, qz;
        p3t_decode_key(keys[i], max_level, hilbert, qx, qy, qz);
        const int sh = max_level - D;
        const float l = ldexpf(side, -D);
        const float lx = cube[0] + (float)(qx >> sh) * l, ly = cube[1] + (float)(qy >> sh) * l, lz = cube[2] + (float)(qz >> sh) * l;
        const float ex = fmaxf(fmaxf(lx - b.x, b.x - (lx + l)), 0.f), ey = fmaxf(fmaxf(ly - b.y, b.y - (ly + l)), 0.f),
                    ez = fmaxf(fmaxf(lz - b.z, b.z - (lz + l)), 0.f);
        stray += fmaxf(ex, fmaxf(ey, ez)) > stray_dist * l ? 1u : 0u;
    }
    stray = __reduce_add_sync(0xffffffffu, stray);
    if ((threadIdx.x & 31) == 0 && stray) atomicAdd(&counters[CNT_STRAY], (u64)stray);
}

// first half: gather + stray count + leaf moments (the caller reads the stray count, then either finishes the refit
// with p3t_stage_refit_finish or rebuilds)
p3t_status p3t_stage_refit_begin(p3t_ctx *ctx)
{
    Workspace &w = ctx->ws;
    cudaStream_t s = ctx->stream;
    const u32 n = (u32)ctx->n;
    P3T_CUDA(ctx, cudaMemsetAsync(w.counters + CNT_STRAY, 0, sizeof(u64), s));
    refit_gather_kernel<<<min(div_up(n, 256), (u32)ctx->sm_count * 8), 256, 0, s>>>(
        w.body_user, w.idx[ctx->cur], w.keys[ctx->cur], w.dlev, w.cube, w.body, n, ctx->max_level, ctx->key_curve, ctx->stray_dist, w.cell_ready,
        w.prev_ncells, (u32)w.cell_cap, w.counters);
    size_t bound = ctx->n * (size_t)(ctx->max_level + 1);
    if (bound > w.cell_cap) bound = w.cell_cap;
    const u32 grid = (u32)min((size_t)div_up(bound, 128), (size_t)ctx->sm_count * 16);
    moments_kernel<0, true><<<grid, 128, 0, s>>>(w.body, w.keys[ctx->cur], w.cube, w.cell_level, w.cell_start, w.cell_parent, w.cell_first,
                                                 w.cell_nchild, w.cell_ready, w.cell_meta, w.cell_mac, w.cell_mom0, w.cell_mom1,
                                                 w.cell_bmin, w.cell_bmax, w.counters, (u32)w.cell_cap, ctx->max_level, ctx->key_curve, ctx->prm.theta,
                                                 ctx->prm.h, ctx->cls_n ? w.cls_sorted : nullptr, ctx->prm.h_bf);
    P3T_CUDA(ctx, cudaGetLastError());
    return P3T_OK;
}

p3t_status p3t_stage_refit_finish(p3t_ctx *ctx)
{
    Workspace &w = ctx->ws;
    cudaStream_t s = ctx->stream;
    size_t bound = ctx->n * (size_t)(ctx->max_level + 1);
    if (bound > w.cell_cap) bound = w.cell_cap;
    const u32 grid = (u32)min((size_t)div_up(bound, 128), (size_t)ctx->sm_count * 16);
    moments_kernel<1, true><<<grid, 128, 0, s>>>(w.body, w.keys[ctx->cur], w.cube, w.cell_level, w.cell_start, w.cell_parent, w.cell_first,
                                                 w.cell_nchild, w.cell_ready, w.cell_meta, w.cell_mac, w.cell_mom0, w.cell_mom1,
                                                 w.cell_bmin, w.cell_bmax, w.counters, (u32)w.cell_cap, ctx->max_level, ctx->key_curve, ctx->prm.theta,
                                                 ctx->prm.h, ctx->cls_n ? w.cls_sorted : nullptr, ctx->prm.h_bf);
    P3T_CUDA(ctx, cudaGetLastError());
    return P3T_OK;
}
