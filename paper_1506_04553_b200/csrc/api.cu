// api.cu -- the C ABI of include/p3t.h: argument checks, workspace layout, stage sequencing.
// Every numerical step is a CUDA kernel in the other files of this directory; no CPU fallback.
#include <math.h>
#include <cmath>
#include <new>
#include <stdlib.h>
#include <thread>
#include <vector>

#include "p3t_internal.cuh"

// ------------------------------------------------------------------------------------------------
// workspace layout
// ------------------------------------------------------------------------------------------------
namespace {
struct Bump {
    char *base;
    size_t off;
    template <class T> T *take(size_t count)
    {
        off = (off + 255) & ~size_t(255);
        T *p = base ? reinterpret_cast<T *>(base + off) : nullptr;
        off += count * sizeof(T);
        return p;
    }
};
} // namespace

size_t p3t_layout(Workspace &ws, char *base, size_t max_n, int key_bits, size_t nbr_capacity, int sm_count)
{
    (void)key_bits;
    Bump b{base, 0};
    size_t n = max_n;
    ws.cell_cap = 3 * n + 1024;
    ws.n_tiles_max = (n + SORT_TILE - 1) / SORT_TILE;
    ws.n_blk_max = (n + BUILD_TILE - 1) / BUILD_TILE;
    ws.walk_warps_max = (size_t)sm_count * WALK_WARPS * WALK_CTAS;   // upper bound of resident walk warps
    ws.in_mass = b.take<float>(n);
    ws.in_pos = b.take<float>(3 * n);
    ws.body_user = b.take<float4>(n);
    ws.cube = b.take<float>(8);
    ws.keys[0] = b.take<u64>(n);
    ws.keys[1] = b.take<u64>(n);
    ws.idx[0] = b.take<u32>(n);
    ws.idx[1] = b.take<u32>(n);
    ws.tile_status = b.take<u32>(2 * (ws.n_tiles_max + 64) * 256);   // + sentinel rows (sort.cu)
    ws.body = b.take<float4>(n);
    ws.clev = b.take<signed char>(n + 8);
    ws.dlev = b.take<u8>(n + 4);
    ws.cutflag = b.take<u8>(n + 4);
    ws.build_tiles = b.take<uint4>((ws.n_blk_max + 8) * 16);
    ws.level_total = b.take<u32>(64);
    ws.prev_ncells = b.take<u32>(4);
    ws.group_start = b.take<u32>(n + 1);
    ws.group_stats = b.take<uint4>(n);
    ws.group_order = b.take<u32>(n);
    ws.order_meta = b.take<u32>(4);
    ws.group_class = b.take<u32>(n);
    ws.body_class = b.take<u32>(n);
    ws.cell_mac = b.take<float4>(ws.cell_cap);
    ws.cell_mom0 = b.take<float4>(ws.cell_cap);
    ws.cell_mom1 = b.take<float4>(ws.cell_cap);
    ws.cell_bmin = b.take<float4>(ws.cell_cap);
    ws.cell_bmax = b.take<float4>(ws.cell_cap);
    ws.cell_meta = b.take<uint2>(ws.cell_cap);
    ws.cell_level = b.take<u8>(ws.cell_cap);
    ws.cell_start = b.take<u32>(ws.cell_cap);
    ws.cell_parent = b.take<u32>(ws.cell_cap);
    ws.cell_first = b.take<u32>(ws.cell_cap);
    ws.cell_nchild = b.take<u32>(ws.cell_cap);
    ws.cell_ready = b.take<u32>(ws.cell_cap);
    ws.accpot = b.take<float4>(n);
    ws.nbr_count = b.take<u32>(n);
    ws.nbr_offset = b.take<u64>(n + 1);
    ws.pairs = b.take<uint2>(nbr_capacity ? nbr_capacity : 1);
    ws.nbr = b.take<u32>(nbr_capacity ? nbr_capacity : 1);
    ws.nbr_cursor = b.take<u32>(n);
    ws.subset = b.take<u32>(n);
    ws.hilbert_tab = b.take<u32>(P3T_HILBERT_TAB_WORDS);
    ws.cls_user = b.take<u8>(n + 4);
    ws.cls_sorted = b.take<u8>(n + 4);
    ws.hard_out = b.take<double>(7 * n);
    ws.herm_ids = b.take<u32>(n);
    ws.herm_tdt = b.take<u64>(n);
    ws.herm_state = b.take<double>(12 * n);
    ws.herm_parent = b.take<u32>(n);
    ws.herm_root = b.take<u32>(n);
    ws.herm_csize = b.take<u32>(n);
    ws.herm_cstart = b.take<u32>(n);
    ws.herm_comps = b.take<uint2>(n / 2 + 1);
    ws.herm_ctl = b.take<u64>(16);
    ws.herm_bigctl = b.take<u64>(8 * (n / 65 + 1));
    ws.hist = b.take<u32>(8 * 256);            // hist | counters | order_hist are contiguous (p3t_internal.cuh)
    ws.counters = b.take<u64>(CNT_WORDS);
    ws.order_hist = b.take<u32>(2048);
    ws.bbox_bits = reinterpret_cast<u32 *>(ws.counters + CNT_BBOX);   // zeroed with the counters at load
    ws.walk_stack = b.take<u32>(ws.walk_warps_max * WALK_STACK_GMEM);
    ws.scan_tmp = b.take<u64>((n + 1023) / 1024 + 2);
    b.off = (b.off + 255) & ~size_t(255);
    ws.total_bytes = b.off;
    return b.off;
}

static bool valid_sizes(size_t max_n, int key_bits)
{
    return max_n >= 1 && max_n < (size_t(1) << 30) && (key_bits == 30 || key_bits == 63);
}

extern "C" size_t p3t_workspace_bytes(size_t max_n, int key_bits, size_t nbr_capacity)
{
    if (!valid_sizes(max_n, key_bits)) return 0;
    Workspace ws;
    return p3t_layout(ws, nullptr, max_n, key_bits, nbr_capacity, 160 /* >= SMs of any B200 */);
}

// ------------------------------------------------------------------------------------------------
// lifetime
// ------------------------------------------------------------------------------------------------
extern "C" p3t_status p3t_create(p3t_ctx **out, int device, size_t max_n, int key_bits, void *workspace,
                                 size_t workspace_bytes, size_t nbr_capacity, void *cuda_stream)
{
    if (!out) return P3T_EINVAL;
    *out = nullptr;
    if (!valid_sizes(max_n, key_bits) || !workspace) return P3T_EINVAL;
    if ((reinterpret_cast<uintptr_t>(workspace) & 255) != 0) return P3T_EINVAL;
    p3t_ctx *ctx = new (std::nothrow) p3t_ctx();
    if (!ctx) return P3T_ENOMEM;
    memset(ctx, 0, sizeof(*ctx));
    ctx->device = device;
    ctx->stream = reinterpret_cast<cudaStream_t>(cuda_stream);
    ctx->max_n = max_n;
    ctx->key_bits = key_bits;
    ctx->max_level = key_bits == 63 ? 21 : 10;
    ctx->nbr_capacity = nbr_capacity;
    ctx->nleaf = 16;
    ctx->ngroup = 64;
    ctx->merge_levels = 3;          // the Peano-Hilbert default (Morton: 1); see p3t_set_key_curve
    ctx->key_curve = 1;
    ctx->cells_dirty = true;
    ctx->herm_cluster_max = 4096;
    ctx->shard_rank = 0;
    ctx->shard_world = 1;
    ctx->herm_a0_bh = -1.0;
    ctx->max_refits = 0;
    ctx->stray_dist = 0.5f;
    ctx->max_stray_fraction = 0.02f;
    cudaError_t e = cudaSetDevice(device);
    cudaDeviceProp prop;
    if (e == cudaSuccess) e = cudaGetDeviceProperties(&prop, device);
    if (e != cudaSuccess) {
        delete ctx;
        return P3T_ECUDA;
    }
    ctx->sm_count = prop.multiProcessorCount;
    if (ctx->sm_count > 160) { delete ctx; return P3T_EINVAL; }
    size_t need = p3t_layout(ctx->ws, static_cast<char *>(workspace), max_n, key_bits, nbr_capacity, 160);
    if (workspace_bytes < need) {
        delete ctx;
        return P3T_ENOMEM;
    }
    ctx->base = static_cast<char *>(workspace);
    if (cudaMemsetAsync(ctx->ws.order_meta, 0, 4 * sizeof(u32), ctx->stream) != cudaSuccess) { delete ctx; return P3T_ECUDA; }
    if (cudaMemsetAsync(ctx->ws.counters, 0, CNT_WORDS * sizeof(u64), ctx->stream) != cudaSuccess) { delete ctx; return P3T_ECUDA; }
    {   // state tables of the Peano-Hilbert keys, derived on the host from the plain transform
        static u32 tab[P3T_HILBERT_TAB_WORDS];
        static bool have = false, good = false;
        if (!have) { good = p3t_hilbert_tables(tab); have = true; }
        if (!good || cudaMemcpyAsync(ctx->ws.hilbert_tab, tab, sizeof(tab), cudaMemcpyHostToDevice, ctx->stream) != cudaSuccess ||
            cudaStreamSynchronize(ctx->stream) != cudaSuccess) { delete ctx; return P3T_ECUDA; }
    }
    if (cudaMemsetAsync(ctx->ws.body_class, 0, max_n * sizeof(u32), ctx->stream) != cudaSuccess) { delete ctx; return P3T_ECUDA; }   // no history: one class, Morton order
    for (int i = 0; i < 14; ++i) {
        if (cudaEventCreate(&ctx->ev[i]) != cudaSuccess) { delete ctx; return P3T_ECUDA; }
    }
    // side stream of the Hermite part (small and mid-size clusters run beside the grid kernel of the large ones)
    if (cudaStreamCreateWithFlags(&ctx->side_stream, cudaStreamNonBlocking) != cudaSuccess ||
        cudaEventCreateWithFlags(&ctx->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&ctx->ev_join, cudaEventDisableTiming) != cudaSuccess) { delete ctx; return P3T_ECUDA; }
    *out = ctx;
    return P3T_OK;
}

extern "C" p3t_status p3t_destroy(p3t_ctx *ctx)
{
    if (!ctx) return P3T_EINVAL;
    cudaStreamSynchronize(ctx->stream);
    for (int i = 0; i < 14; ++i)
        if (ctx->ev[i]) cudaEventDestroy(ctx->ev[i]);
    if (ctx->side_stream) { cudaStreamSynchronize(ctx->side_stream); cudaStreamDestroy(ctx->side_stream); }
    if (ctx->ev_fork) cudaEventDestroy(ctx->ev_fork);
    if (ctx->ev_join) cudaEventDestroy(ctx->ev_join);
    delete ctx;
    return P3T_OK;
}

extern "C" const char *p3t_last_error(const p3t_ctx *ctx) { return ctx ? ctx->err : "null context"; }

// ------------------------------------------------------------------------------------------------
// parameters
// ------------------------------------------------------------------------------------------------
// W(y; gamma) of Eq. 16-17 as coefficients of y^k and y ln y; the denominator of Eq. 17 is taken
// as (gamma-1)^7 (reading A1).
void p3t_fill_cutoff(CutoffSet &c, float r_in, float r_out)   // (also used by static_direct.cu)
{
    double g = (double)r_in / (double)r_out;
    double g2 = g * g, g3 = g2 * g, g4 = g2 * g2, g5 = g4 * g, g6 = g3 * g3, g7 = g6 * g;
    double D = pow(g - 1.0, 7);
    c.gamma = g;
    c.inv_rout = 1.0 / (double)r_out;
    c.inv_1mg = 1.0 / (1.0 - g);
    c.wc[7] = (-10.0 / 3.0) / D;
    c.wc[6] = 14.0 * (g + 1.0) / D;
    c.wc[5] = -21.0 * (g2 + 3.0 * g + 1.0) / D;
    c.wc[4] = (35.0 / 3.0) * (g3 + 9.0 * g2 + 9.0 * g + 1.0) / D;
    c.wc[3] = -70.0 * (g3 + 3.0 * g2 + g) / D;
    c.wc[2] = 210.0 * (g3 + g2) / D;
    c.wc[0] = (g7 - 7.0 * g6 + 21.0 * g5 - 35.0 * g4) / D;
    c.wl = -140.0 * g3 / D;
    double G1 = c.wc[7] + c.wc[6] + c.wc[5] + c.wc[4] + c.wc[3] + c.wc[2] + c.wc[0];   // ln 1 = 0
    c.wc[1] = 1.0 - G1;
    double glog = g > 0.0 ? 60.0 * g3 * log(g) : 0.0;
    c.cin = 7.0 * (g6 - 9.0 * g5 + 45.0 * g4 - glog - 45.0 * g2 + 9.0 * g - 1.0) / (3.0 * D);
}

// the per-kind numbers of P3TParams from the context's two parameter sets (kind 1 = kind 0 while no classes are set)
static void p3t_refresh_class_params(p3t_ctx *ctx)
{
    P3TParams &p = ctx->prm;
    p.classes = ctx->cls_n ? 1 : 0;
    const float r_in1 = p.classes ? ctx->r_in_bf : ctx->r_in, r_out1 = p.classes ? ctx->r_out_bf : ctx->r_out,
                h1 = p.classes ? ctx->r_search_bf : ctx->r_search;
    p.rout2_k[0] = p.rout2; p.h2_k[0] = p.h2;
    p.rout2_k[1] = r_out1 * r_out1; p.h2_k[1] = h1 * h1;
    p.h_bf = fmaxf(ctx->r_search, h1);
    const float hn = p.h_bf * (1.f + 1e-5f);
    p.hnear2_bf = hn * hn;
    p.eps2_bb_d = (double)ctx->eps_bb * (double)ctx->eps_bb;
    if (r_out1 > 0.f) p3t_fill_cutoff(p.cs[1], r_in1, r_out1);
}

extern "C" p3t_status p3t_set_params(p3t_ctx *ctx, float eps, float theta, float r_in, float r_out, float r_search)
{
    if (!ctx) return P3T_EINVAL;
    if (!(eps >= 0.f) || !(theta >= 0.f) || !isfinite(eps) || !isfinite(theta) || !isfinite(r_search) ||
        !(r_in >= 0.f) || !(r_in < r_out) || !(r_out <= r_search))
        return p3t_fail(ctx, P3T_EINVAL, "need eps >= 0, theta >= 0, 0 <= r_in < r_out <= r_search, all finite");
    ctx->eps = eps; ctx->theta = theta; ctx->r_in = r_in; ctx->r_out = r_out; ctx->r_search = r_search;
    P3TParams &p = ctx->prm;
    p.eps2 = eps * eps;
    p.eps2_d = (double)eps * (double)eps;
    p.theta = theta;
    p.r_in = r_in; p.r_out = r_out; p.h = r_search;
    p.rout2 = r_out * r_out;
    p.h2 = r_search * r_search;
    {   // bodies whose distance to the group's box is below this go to the K/W + neighbour-test path
        float hn = r_search * (1.f + 1e-5f);
        p.hnear2 = hn * hn;
    }
    p3t_fill_cutoff(p.cs[0], r_in, r_out);
    p3t_refresh_class_params(ctx);
    ctx->have_params = true;
    ctx->built = false;        // theta and h enter the per-cell acceptance radius
    ctx->evaluated = false;
    return P3T_OK;
}

// Per-pair-class cutoffs (section 3.2.2.1)
extern "C" p3t_status p3t_set_pair_classes(p3t_ctx *ctx, size_t n, const uint8_t *cls, int on_device, float r_in_bf, float r_out_bf,
                                           float r_search_bf, float eps_bb)
{
    if (!ctx) return P3T_EINVAL;
    ctx->built = false;
    ctx->evaluated = false;
    ctx->topo_valid = false;          // the classes are gathered into Morton order by a build
    if (!cls) {                       // back to one kind of pair
        ctx->cls_n = 0;
        p3t_refresh_class_params(ctx);
        return P3T_OK;
    }
    if (n == 0 || n > ctx->max_n) return p3t_fail(ctx, P3T_EINVAL, "n must be in 1..max_n");
    if (!(r_in_bf >= 0.f) || !(r_in_bf < r_out_bf) || !(r_out_bf <= r_search_bf) || !isfinite(r_search_bf) || !(eps_bb >= 0.f) || !isfinite(eps_bb))
        return p3t_fail(ctx, P3T_EINVAL, "need 0 <= r_in_bf < r_out_bf <= r_search_bf and eps_bb >= 0, all finite");
    P3T_CUDA(ctx, cudaSetDevice(ctx->device));
    if (!on_device)
        for (size_t i = 0; i < n; ++i)
            if (cls[i] > 1) return p3t_fail(ctx, P3T_EINVAL, "classes must be 0 (field star) or 1 (black hole)");
    // (device input: values are reduced to their lowest bit when they are gathered)
    P3T_CUDA(ctx, cudaMemcpyAsync(ctx->ws.cls_user, cls, n, on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, ctx->stream));
    if (!on_device) P3T_CUDA(ctx, cudaStreamSynchronize(ctx->stream));    // the caller's array may be pageable and short-lived
    ctx->cls_n = n;
    ctx->r_in_bf = r_in_bf; ctx->r_out_bf = r_out_bf; ctx->r_search_bf = r_search_bf; ctx->eps_bb = eps_bb;
    p3t_refresh_class_params(ctx);
    return P3T_OK;
}

extern "C" p3t_status p3t_set_tree_params(p3t_ctx *ctx, int nleaf, int ngroup)
{
    if (!ctx) return P3T_EINVAL;
    if (nleaf < 1 || nleaf > 32 || (ngroup != 32 && ngroup != 64))
        return p3t_fail(ctx, P3T_EINVAL, "need 1 <= nleaf <= 32 and ngroup in {32, 64}");
    ctx->nleaf = nleaf;
    ctx->ngroup = ngroup;
    ctx->built = false;
    ctx->evaluated = false;
    ctx->topo_valid = false;
    return P3T_OK;
}

// undocumented tuning knob used by bench.py sweeps: levels above the natural group level whose
// boundaries an i-group may straddle (0 = groups are single octree cells)
extern "C" p3t_status p3t_set_group_merge_levels(p3t_ctx *ctx, int levels)
{
    if (!ctx || levels < 0 || (levels > 4 && levels != 32)) return P3T_EINVAL;
    ctx->merge_levels = levels;
    ctx->merge_user_set = true;
    ctx->built = false;
    ctx->evaluated = false;
    ctx->topo_valid = false;
    return P3T_OK;
}

extern "C" p3t_status p3t_set_key_curve(p3t_ctx *ctx, int curve)
{
    if (!ctx || curve < 0 || curve > 1) return P3T_EINVAL;
    ctx->key_curve = curve;
    if (!ctx->merge_user_set) ctx->merge_levels = curve ? 3 : 1;   // measured optimum of either order
    ctx->built = false;
    ctx->evaluated = false;
    ctx->topo_valid = false;
    return P3T_OK;
}

extern "C" p3t_status p3t_set_sort_passes(p3t_ctx *ctx, int passes)
{
    if (!ctx || passes < 0 || passes > 8) return P3T_EINVAL;
    ctx->sort_passes_user = passes;
    ctx->built = false;
    ctx->evaluated = false;
    ctx->topo_valid = false;
    return P3T_OK;
}

extern "C" p3t_status p3t_hilbert_state_tables(uint32_t *tab, size_t words)
{
    if (!tab || words < P3T_HILBERT_TAB_WORDS) return P3T_EINVAL;
    return p3t_hilbert_tables(tab) ? P3T_OK : P3T_ECUDA;
}

extern "C" p3t_status p3t_set_shard(p3t_ctx *ctx, int rank, int world)
{
    if (!ctx || world < 1 || rank < 0 || rank >= world) return P3T_EINVAL;
    ctx->shard_rank = rank;
    ctx->shard_world = world;
    ctx->evaluated = false;
    ctx->shard_classes_fresh = false;
    return P3T_OK;
}

extern "C" p3t_status p3t_get_shard_record(p3t_ctx *ctx, float *rec)
{
    if (!ctx) return P3T_EINVAL;
    if (!rec) return p3t_fail(ctx, P3T_EINVAL, "null rec");
    if (!ctx->evaluated) return p3t_fail(ctx, P3T_ESTATE, "p3t_get_shard_record before an eval call");
    P3T_CUDA(ctx, cudaSetDevice(ctx->device));
    return p3t_stage_shard_record(ctx, rec);
}

extern "C" p3t_status p3t_put_shard_classes(p3t_ctx *ctx, const float *rec)
{
    if (!ctx) return P3T_EINVAL;
    if (!rec) return p3t_fail(ctx, P3T_EINVAL, "null rec");
    if (!ctx->evaluated) return p3t_fail(ctx, P3T_ESTATE, "p3t_put_shard_classes before an eval call");
    P3T_CUDA(ctx, cudaSetDevice(ctx->device));
    p3t_status st = p3t_stage_shard_classes(ctx, rec);
    if (st == P3T_OK) ctx->shard_classes_fresh = true;
    return st;
}

extern "C" p3t_status p3t_set_hermite_class_params(p3t_ctx *ctx, double eta_bh, double eta_s_bh, double a0_bh)
{
    if (!ctx) return P3T_EINVAL;
    if (!std::isfinite(eta_bh) || !std::isfinite(eta_s_bh) || !std::isfinite(a0_bh)) return p3t_fail(ctx, P3T_EINVAL, "non-finite value");
    ctx->herm_eta_bh = eta_bh; ctx->herm_eta_s_bh = eta_s_bh; ctx->herm_a0_bh = a0_bh;
    return P3T_OK;
}

extern "C" p3t_status p3t_set_hermite_cluster_max(p3t_ctx *ctx, int max_members)
{
    if (!ctx) return P3T_EINVAL;
    if (max_members < 64 || max_members > (1 << 20)) return p3t_fail(ctx, P3T_EINVAL, "max_members must be in 64..1048576");
    ctx->herm_cluster_max = max_members;
    return P3T_OK;
}

extern "C" p3t_status p3t_set_walk_mode(p3t_ctx *ctx, int mode)
{
    if (!ctx || mode < 0 || mode > 4) return P3T_EINVAL;
    ctx->walk_mode = mode;
    ctx->evaluated = false;
    return P3T_OK;
}

// ------------------------------------------------------------------------------------------------
// load / build / eval
// ------------------------------------------------------------------------------------------------
// Host-side finiteness check of the input (an exponent of all ones marks inf/nan): a branch-free OR over the
// words, which the host compiler vectorises, split over a few threads for large inputs -- a scalar isfinite()
// loop cost 2.5 ms per 1M particles, a quarter of the GPU time of the whole evaluation.
static bool host_all_finite(const float *p, size_t count)
{
    auto scan = [](const float *q, size_t m) {
        const uint32_t *w = reinterpret_cast<const uint32_t *>(q);
        uint32_t bad = 0;
        for (size_t i = 0; i < m; ++i) bad |= ((w[i] & 0x7f800000u) == 0x7f800000u) ? 1u : 0u;
        return bad == 0;
    };
    const size_t hw = std::thread::hardware_concurrency();
    const size_t nthr = count >= (size_t(1) << 18) ? (hw >= 16 ? 16 : hw >= 8 ? 8 : 4) : 1;
    if (nthr == 1) return scan(p, count);
    std::vector<char> ok(nthr, 1);
    std::vector<std::thread> th;
    const size_t per = (count + nthr - 1) / nthr;
    for (size_t t = 0; t < nthr; ++t) {
        const size_t b = t * per, e = b + per < count ? b + per : count;
        if (b >= e) break;
        th.emplace_back([&, t, b, e] { ok[t] = scan(p + b, e - b) ? 1 : 0; });
    }
    for (auto &x : th) x.join();
    for (char c : ok) if (!c) return false;
    return true;
}

extern "C" p3t_status p3t_load_particles(p3t_ctx *ctx, size_t n, const float *mass, const float *pos, int on_device)
{
    if (!ctx) return P3T_EINVAL;
    if (!mass || !pos) return p3t_fail(ctx, P3T_EINVAL, "null mass/pos");
    if (n == 0 || n > ctx->max_n) return p3t_fail(ctx, P3T_EINVAL, "n must be in 1..max_n");
    P3T_CUDA(ctx, cudaSetDevice(ctx->device));
    const float *d_mass = mass, *d_pos = pos;
    ctx->loaded = false;
    ctx->built = false;
    ctx->evaluated = false;
    if (!on_device) {
        P3T_CUDA(ctx, cudaMemcpyAsync(ctx->ws.in_mass, mass, n * sizeof(float), cudaMemcpyHostToDevice, ctx->stream));
        P3T_CUDA(ctx, cudaMemcpyAsync(ctx->ws.in_pos, pos, 3 * n * sizeof(float), cudaMemcpyHostToDevice, ctx->stream));
        d_mass = ctx->ws.in_mass;
        d_pos = ctx->ws.in_pos;
    }
    ctx->n = n;
    P3T_CUDA(ctx, cudaEventRecord(ctx->ev[9], ctx->stream));
    p3t_status st = p3t_stage_pack(ctx, d_mass, d_pos);
    if (st != P3T_OK) return st;
    P3T_CUDA(ctx, cudaEventRecord(ctx->ev[10], ctx->stream));
    // host input: the error is due from THIS call (include/p3t.h).  The pack kernel has tested every value on the device
    // copy; waiting for its verdict costs the copy time the caller would wait for anyway, where a pass of the host cores
    // over the arrays took 0.8 ms per 1M particles with the device idle behind it.
    if (!on_device) {
        u64 bad = 0;
        P3T_CUDA(ctx, cudaMemcpyAsync(&bad, ctx->ws.counters + CNT_NONFINITE, sizeof(u64), cudaMemcpyDeviceToHost, ctx->stream));
        P3T_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
        if (bad) return p3t_fail(ctx, P3T_EINVAL, "non-finite mass or position");
    }
    ctx->ev_pack = true;
    ctx->loaded = true;
    return P3T_OK;
}

extern "C" p3t_status p3t_build_tree(p3t_ctx *ctx)
{
    if (!ctx) return P3T_EINVAL;
    if (!ctx->loaded) return p3t_fail(ctx, P3T_ESTATE, "p3t_build_tree before p3t_load_particles");
    if (!ctx->have_params) return p3t_fail(ctx, P3T_ESTATE, "p3t_build_tree before p3t_set_params");
    if (ctx->cls_n && ctx->cls_n != ctx->n) return p3t_fail(ctx, P3T_ESTATE, "the classes of p3t_set_pair_classes were given for another particle count");
    P3T_CUDA(ctx, cudaSetDevice(ctx->device));
    ctx->built = false;
    ctx->evaluated = false;
    ctx->topo_valid = false;
    p3t_status st;
    P3T_CUDA(ctx, cudaEventRecord(ctx->ev[0], ctx->stream));
    if ((st = p3t_stage_sort(ctx)) != P3T_OK) return st;
    P3T_CUDA(ctx, cudaEventRecord(ctx->ev[1], ctx->stream));
    if ((st = p3t_stage_build(ctx)) != P3T_OK) return st;
    P3T_CUDA(ctx, cudaEventRecord(ctx->ev[2], ctx->stream));
    if ((st = p3t_stage_moments(ctx)) != P3T_OK) return st;
    P3T_CUDA(ctx, cudaEventRecord(ctx->ev[3], ctx->stream));
    ctx->ev_build = true;
    ctx->built = true;
    ctx->topo_valid = true;
    ctx->topo_n = ctx->n;
    ctx->refits = 0;
    ctx->last_rebuilt = true;
    ctx->last_stray = 0;
    return P3T_OK;
}

static p3t_status sync_and_check(p3t_ctx *ctx);

// Tree reuse between soft steps (first half, cost per soft step L193, Eq. 28)
extern "C" p3t_status p3t_set_tree_reuse(p3t_ctx *ctx, int max_refits, float stray_dist, float max_stray_fraction)
{
    if (!ctx) return P3T_EINVAL;
    if (max_refits < 0 || !(stray_dist >= 0.f) || !(max_stray_fraction >= 0.f) || !isfinite(stray_dist) || !isfinite(max_stray_fraction))
        return p3t_fail(ctx, P3T_EINVAL, "need max_refits >= 0, stray_dist >= 0, max_stray_fraction >= 0");
    ctx->max_refits = max_refits;
    ctx->stray_dist = stray_dist;
    ctx->max_stray_fraction = max_stray_fraction;
    return P3T_OK;
}

extern "C" p3t_status p3t_refit_tree(p3t_ctx *ctx)
{
    if (!ctx) return P3T_EINVAL;
    if (!ctx->loaded) return p3t_fail(ctx, P3T_ESTATE, "p3t_refit_tree before p3t_load_particles");
    if (!ctx->have_params) return p3t_fail(ctx, P3T_ESTATE, "p3t_refit_tree before p3t_set_params");
    // no tree of these particles to reuse, or enough refits in a row: a full build
    if (!ctx->topo_valid || ctx->topo_n != ctx->n || ctx->refits >= ctx->max_refits) return p3t_build_tree(ctx);
    if (ctx->cls_n && ctx->cls_n != ctx->n) return p3t_fail(ctx, P3T_ESTATE, "the classes of p3t_set_pair_classes were given for another particle count");
    P3T_CUDA(ctx, cudaSetDevice(ctx->device));
    ctx->built = false;
    ctx->evaluated = false;
    p3t_status st;
    P3T_CUDA(ctx, cudaEventRecord(ctx->ev[0], ctx->stream));
    if ((st = p3t_stage_refit_begin(ctx)) != P3T_OK) return st;
    // the stray count decides between finishing the refit and rebuilding: one small copy and a stream synchronisation
    // (the leaf moments are already enqueued behind the gather, so the device does not idle while the host decides)
    if ((st = sync_and_check(ctx)) != P3T_OK) return st;
    ctx->last_stray = ctx->h_counters[CNT_STRAY];
    if ((double)ctx->last_stray > (double)ctx->max_stray_fraction * (double)ctx->n) return p3t_build_tree(ctx);
    P3T_CUDA(ctx, cudaEventRecord(ctx->ev[1], ctx->stream));
    P3T_CUDA(ctx, cudaEventRecord(ctx->ev[2], ctx->stream));
    if ((st = p3t_stage_refit_finish(ctx)) != P3T_OK) return st;
    P3T_CUDA(ctx, cudaEventRecord(ctx->ev[3], ctx->stream));
    ctx->ev_build = true;
    ctx->built = true;
    ctx->refits += 1;
    ctx->last_rebuilt = false;
    return P3T_OK;
}

extern "C" p3t_status p3t_eval_soft(p3t_ctx *ctx)
{
    if (!ctx) return P3T_EINVAL;
    if (!ctx->built) return p3t_fail(ctx, P3T_ESTATE, "p3t_eval_soft needs a tree built for the current particles and parameters");
    P3T_CUDA(ctx, cudaSetDevice(ctx->device));
    ctx->evaluated = false;
    p3t_status st;
    P3T_CUDA(ctx, cudaEventRecord(ctx->ev[4], ctx->stream));
    if ((st = p3t_stage_walk(ctx)) != P3T_OK) return st;
    P3T_CUDA(ctx, cudaEventRecord(ctx->ev[5], ctx->stream));
    if ((st = p3t_stage_neighbours(ctx)) != P3T_OK) return st;
    P3T_CUDA(ctx, cudaEventRecord(ctx->ev[6], ctx->stream));
    ctx->ev_eval = true;
    ctx->evaluated = true;
    ctx->lists_complete = ctx->shard_world == 1;   // a shard holds the lists of its own groups only: not symmetric
    return P3T_OK;
}

extern "C" p3t_status p3t_eval_direct(p3t_ctx *ctx, const uint32_t *i_subset, size_t n_subset, int on_device)
{
    if (!ctx) return P3T_EINVAL;
    if (!ctx->loaded) return p3t_fail(ctx, P3T_ESTATE, "p3t_eval_direct before p3t_load_particles");
    if (!ctx->have_params) return p3t_fail(ctx, P3T_ESTATE, "p3t_eval_direct before p3t_set_params");
    if (ctx->cls_n && ctx->cls_n != ctx->n) return p3t_fail(ctx, P3T_ESTATE, "the classes of p3t_set_pair_classes were given for another particle count");
    if (i_subset && (n_subset == 0 || n_subset > ctx->n)) return p3t_fail(ctx, P3T_EINVAL, "bad subset size");
    P3T_CUDA(ctx, cudaSetDevice(ctx->device));
    const u32 *d_subset = i_subset;
    if (i_subset && !on_device) {
        for (size_t k = 0; k < n_subset; ++k)
            if (i_subset[k] >= ctx->n) return p3t_fail(ctx, P3T_EINVAL, "subset index out of range");
        P3T_CUDA(ctx, cudaMemcpyAsync(ctx->ws.subset, i_subset, n_subset * sizeof(u32), cudaMemcpyHostToDevice, ctx->stream));
        d_subset = ctx->ws.subset;
    }
    ctx->evaluated = false;
    p3t_status st;
    P3T_CUDA(ctx, cudaEventRecord(ctx->ev[4], ctx->stream));
    if ((st = p3t_stage_direct(ctx, d_subset, i_subset ? n_subset : ctx->n)) != P3T_OK) return st;
    P3T_CUDA(ctx, cudaEventRecord(ctx->ev[5], ctx->stream));
    if ((st = p3t_stage_neighbours(ctx)) != P3T_OK) return st;
    P3T_CUDA(ctx, cudaEventRecord(ctx->ev[6], ctx->stream));
    ctx->ev_eval = true;
    ctx->evaluated = true;
    ctx->lists_complete = i_subset == nullptr;     // a subset leaves the other particles' lists empty
    return P3T_OK;
}

// NEXT row: hard acceleration, jerk and potential from the neighbour lists
extern "C" p3t_status p3t_eval_hard(p3t_ctx *ctx, const float *vel, double *acc, double *jerk, double *pot, int on_device)
{
    if (!ctx) return P3T_EINVAL;
    if (!vel) return p3t_fail(ctx, P3T_EINVAL, "null vel");
    if (!ctx->evaluated) return p3t_fail(ctx, P3T_ESTATE, "p3t_eval_hard needs the neighbour lists of an eval call");
    P3T_CUDA(ctx, cudaSetDevice(ctx->device));
    const size_t n = ctx->n;
    const float *d_vel = vel;
    double *d_acc = acc, *d_jerk = jerk, *d_pot = pot;
    if (!on_device) {
        if (!host_all_finite(vel, 3 * n)) return p3t_fail(ctx, P3T_EINVAL, "non-finite velocity");
        P3T_CUDA(ctx, cudaMemcpyAsync(ctx->ws.in_pos, vel, 3 * n * sizeof(float), cudaMemcpyHostToDevice, ctx->stream));
        d_vel = ctx->ws.in_pos;
        d_acc = acc ? ctx->ws.hard_out : nullptr;
        d_jerk = jerk ? ctx->ws.hard_out + 3 * n : nullptr;
        d_pot = pot ? ctx->ws.hard_out + 6 * n : nullptr;
    }
    P3T_CUDA(ctx, cudaEventRecord(ctx->ev[7], ctx->stream));
    p3t_status st = p3t_stage_hard(ctx, d_vel, d_acc, d_jerk, d_pot);
    if (st != P3T_OK) return st;
    P3T_CUDA(ctx, cudaEventRecord(ctx->ev[8], ctx->stream));
    ctx->ev_hard = true;
    if (on_device) {
        ctx->hard_unchecked = true;   // a capacity overflow (nothing computed) surfaces at the next synchronising call
        return P3T_OK;
    }
    if (acc) P3T_CUDA(ctx, cudaMemcpyAsync(acc, d_acc, 3 * n * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    if (jerk) P3T_CUDA(ctx, cudaMemcpyAsync(jerk, d_jerk, 3 * n * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    if (pot) P3T_CUDA(ctx, cudaMemcpyAsync(pot, d_pot, n * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    st = sync_and_check(ctx);
    if (st != P3T_OK) return st;
    if (ctx->h_counters[CNT_PAIRS] > ctx->nbr_capacity)
        return p3t_fail(ctx, P3T_ECAPACITY, "neighbour lists exceed the context's nbr_capacity: no hard force was computed");
    return P3T_OK;
}

// NEXT row: one soft step under H_hard, and the whole step of the scheme
static p3t_status hermite_args_ok(p3t_ctx *ctx, double dt_soft, int log2_div, double eta, double eta_s, double a0, long long max_blocks)
{
    if (!(dt_soft > 0.0) || !std::isfinite(dt_soft)) return p3t_fail(ctx, P3T_EINVAL, "dt_soft must be positive and finite");
    if (log2_div < 0 || log2_div > 30) return p3t_fail(ctx, P3T_EINVAL, "log2_div must be in 0..30");
    if (!(eta > 0.0) || !(eta_s > 0.0) || !std::isfinite(eta) || !std::isfinite(eta_s)) return p3t_fail(ctx, P3T_EINVAL, "eta, eta_s must be positive");
    if (!(a0 >= 0.0) || !std::isfinite(a0)) return p3t_fail(ctx, P3T_EINVAL, "a0 must be >= 0");
    if (max_blocks < 1) return p3t_fail(ctx, P3T_EINVAL, "max_blocks must be >= 1");
    return P3T_OK;
}

// device part shared by p3t_hermite_step and p3t_step; fills info after a synchronisation
static p3t_status hermite_on_device(p3t_ctx *ctx, double *d_pos, double *d_vel, double dt_soft, int log2_div, double eta,
                                    double eta_s, double a0, long long max_blocks, p3t_hermite_info *info)
{
    p3t_status st = sync_and_check(ctx);                  // the lists must be complete and must have fitted
    if (st != P3T_OK) return st;
    if (ctx->h_counters[CNT_PAIRS] > ctx->nbr_capacity)
        return p3t_fail(ctx, P3T_ECAPACITY, "neighbour lists exceed the context's nbr_capacity: nothing was integrated");
    u64 h_ctl[16] = {0};
    P3T_CUDA(ctx, cudaEventRecord(ctx->ev[11], ctx->stream));
    st = p3t_stage_hermite(ctx, d_pos, d_vel, dt_soft, log2_div, eta, eta_s, a0, max_blocks, h_ctl);
    if (st != P3T_OK) return st;
    P3T_CUDA(ctx, cudaEventRecord(ctx->ev[12], ctx->stream));
    P3T_CUDA(ctx, cudaMemcpyAsync(h_ctl, ctx->ws.herm_ctl, sizeof(h_ctl), cudaMemcpyDeviceToHost, ctx->stream));
    P3T_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    if (info) {
        info->n_nonisolated = h_ctl[0];
        info->n_blocks = h_ctl[4];
        info->n_steps = h_ctl[5];
        info->floor_hits = h_ctl[6];
        info->n_components = h_ctl[11];
        info->max_component = h_ctl[12];
        info->ms = 0.f;
        cudaEventElapsedTime(&info->ms, ctx->ev[11], ctx->ev[12]);
    }
    if (h_ctl[7] == 3) return p3t_fail(ctx, P3T_EINVAL, "Hermite part: non-finite force (coincident particles with eps = 0?); pos, vel are unusable");
    if (h_ctl[7] == 2) return p3t_fail(ctx, P3T_ESTATE, "Hermite part: the neighbour lists are not symmetric; pos, vel are unusable");
    if (h_ctl[7]) return p3t_fail(ctx, P3T_ELIMIT, "Hermite part: more than max_blocks block steps (a0 = 0 lets Eq. 18 collapse at the cutoff radius); pos, vel are mid-step");
    return P3T_OK;
}

extern "C" p3t_status p3t_hermite_step(p3t_ctx *ctx, double *pos, double *vel, double dt_soft, int log2_div, double eta,
                                       double eta_s, double a0, long long max_blocks, int on_device, p3t_hermite_info *info)
{
    if (!ctx) return P3T_EINVAL;
    if (!pos || !vel) return p3t_fail(ctx, P3T_EINVAL, "null pos/vel");
    if (!ctx->evaluated) return p3t_fail(ctx, P3T_ESTATE, "p3t_hermite_step needs the neighbour lists of an eval call");
    if (!ctx->lists_complete)
        return p3t_fail(ctx, P3T_ESTATE, "p3t_hermite_step needs the lists of ALL particles: the last evaluation was sharded or a subset");
    p3t_status st = hermite_args_ok(ctx, dt_soft, log2_div, eta, eta_s, a0, max_blocks);
    if (st != P3T_OK) return st;
    P3T_CUDA(ctx, cudaSetDevice(ctx->device));
    const size_t n = ctx->n;
    double *d_pos = pos, *d_vel = vel;
    if (!on_device) {
        d_pos = ctx->ws.hard_out;
        d_vel = ctx->ws.hard_out + 3 * n;
        P3T_CUDA(ctx, cudaMemcpyAsync(d_pos, pos, 3 * n * sizeof(double), cudaMemcpyHostToDevice, ctx->stream));
        P3T_CUDA(ctx, cudaMemcpyAsync(d_vel, vel, 3 * n * sizeof(double), cudaMemcpyHostToDevice, ctx->stream));
    }
    st = hermite_on_device(ctx, d_pos, d_vel, dt_soft, log2_div, eta, eta_s, a0, max_blocks, info);
    if (st != P3T_OK) return st;
    if (!on_device) {
        P3T_CUDA(ctx, cudaMemcpyAsync(pos, d_pos, 3 * n * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
        P3T_CUDA(ctx, cudaMemcpyAsync(vel, d_vel, 3 * n * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
        P3T_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    }
    return P3T_OK;
}

extern "C" p3t_status p3t_step(p3t_ctx *ctx, const float *mass, double *pos, double *vel, double dt_soft, int log2_div,
                               double eta, double eta_s, double a0, long long max_blocks, int on_device, p3t_hermite_info *info)
{
    if (!ctx) return P3T_EINVAL;
    if (!mass || !pos || !vel) return p3t_fail(ctx, P3T_EINVAL, "null mass/pos/vel");
    if (!ctx->evaluated) return p3t_fail(ctx, P3T_ESTATE, "p3t_step needs the soft force and lists of an eval call at the current positions");
    if (!ctx->lists_complete || ctx->shard_world > 1)
        return p3t_fail(ctx, P3T_ESTATE, "p3t_step needs the soft force and lists of ALL particles: not available on a sharded context or after a subset evaluation");
    p3t_status st = hermite_args_ok(ctx, dt_soft, log2_div, eta, eta_s, a0, max_blocks);
    if (st != P3T_OK) return st;
    P3T_CUDA(ctx, cudaSetDevice(ctx->device));
    const size_t n = ctx->n;
    double *d_pos = pos, *d_vel = vel;
    const float *d_mass = mass;
    if (!on_device) {
        d_pos = ctx->ws.hard_out;
        d_vel = ctx->ws.hard_out + 3 * n;
        d_mass = ctx->ws.in_mass;
        P3T_CUDA(ctx, cudaMemcpyAsync(d_pos, pos, 3 * n * sizeof(double), cudaMemcpyHostToDevice, ctx->stream));
        P3T_CUDA(ctx, cudaMemcpyAsync(d_vel, vel, 3 * n * sizeof(double), cudaMemcpyHostToDevice, ctx->stream));
        P3T_CUDA(ctx, cudaMemcpyAsync(ctx->ws.in_mass, mass, n * sizeof(float), cudaMemcpyHostToDevice, ctx->stream));
    }
    if ((st = p3t_stage_kick(ctx, d_vel, 0.5 * dt_soft)) != P3T_OK) return st;                 // step 2
    st = hermite_on_device(ctx, d_pos, d_vel, dt_soft, log2_div, eta, eta_s, a0, max_blocks, info);   // step 3
    if (st != P3T_OK) return st;
    if ((st = p3t_stage_narrow(ctx, d_pos, ctx->ws.in_pos)) != P3T_OK) return st;              // step 4: soft force at t + dt
    if ((st = p3t_load_particles(ctx, n, d_mass, ctx->ws.in_pos, 1)) != P3T_OK) return st;
    if ((st = p3t_refit_tree(ctx)) != P3T_OK) return st;      // a full build unless p3t_set_tree_reuse allows refits
    if ((st = p3t_eval_soft(ctx)) != P3T_OK) return st;
    if ((st = p3t_stage_kick(ctx, d_vel, 0.5 * dt_soft)) != P3T_OK) return st;
    if (!on_device) {
        P3T_CUDA(ctx, cudaMemcpyAsync(pos, d_pos, 3 * n * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
        P3T_CUDA(ctx, cudaMemcpyAsync(vel, d_vel, 3 * n * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
        return sync_and_check(ctx);
    }
    return P3T_OK;
}

// ------------------------------------------------------------------------------------------------
// synchronisation and deferred errors
// ------------------------------------------------------------------------------------------------
static p3t_status sync_and_check(p3t_ctx *ctx)
{
    P3T_CUDA(ctx, cudaSetDevice(ctx->device));
    P3T_CUDA(ctx, cudaMemcpyAsync(ctx->h_counters, ctx->ws.counters, sizeof(ctx->h_counters), cudaMemcpyDeviceToHost, ctx->stream));
    P3T_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    if (ctx->h_counters[CNT_NONFINITE]) return p3t_fail(ctx, P3T_EINVAL, "non-finite mass or position in the device input");
    u64 f = ctx->h_counters[CNT_ERR_BUILD] | ctx->h_counters[CNT_ERR_EVAL];
    if (ctx->h_counters[CNT_ERR_BUILD]) { ctx->cells_dirty = true; ctx->topo_valid = false; }
    // radix plan of the next build (sort.cu): the last build sorted the upper key bits only and met a long run of keys
    // equal on them (sorted all the same, by the slow path) -> eight more bits from now on
    if (ctx->sort_adapted_build != ctx->build_count) {
        ctx->sort_adapted_build = ctx->build_count;
        if (ctx->sort_passes_used < (3 * ctx->max_level + 7) / 8 && ctx->h_counters[CNT_SORT_MAXRUN] > 24 && ctx->sort_extra_bits < 48)
            ctx->sort_extra_bits += 8;
    }
    if (f & ERR_CELL_CAPACITY) return p3t_fail(ctx, P3T_ENOMEM, "octree cell capacity (3 n + 1024) exceeded");
    if (f & ERR_STACK_OVERFLOW) return p3t_fail(ctx, P3T_ENOMEM, "tree-walk stack overflow");
    if (ctx->hard_unchecked) {
        ctx->hard_unchecked = false;
        if (ctx->h_counters[CNT_PAIRS] > ctx->nbr_capacity)
            return p3t_fail(ctx, P3T_ECAPACITY, "neighbour lists exceed the context's nbr_capacity: the last p3t_eval_hard computed nothing");
    }
    return P3T_OK;
}

extern "C" p3t_status p3t_synchronize(p3t_ctx *ctx)
{
    if (!ctx) return P3T_EINVAL;
    return sync_and_check(ctx);
}

// ------------------------------------------------------------------------------------------------
// fetch
// ------------------------------------------------------------------------------------------------
extern "C" p3t_status p3t_get_acc_pot(p3t_ctx *ctx, float *acc, float *pot, int on_device)
{
    if (!ctx) return P3T_EINVAL;
    if (!ctx->evaluated) return p3t_fail(ctx, P3T_ESTATE, "p3t_get_acc_pot before an eval call");
    P3T_CUDA(ctx, cudaSetDevice(ctx->device));
    size_t n = ctx->n;
    if (on_device) return p3t_stage_unpack(ctx, acc, pot);
    // host destination: unpack into the (now free) input staging arrays, then copy out.  Accelerations and potentials are
    // final when the walk stage ends (event 5 of the last evaluation); the neighbour stage behind it on the context's
    // stream touches neither them nor the staging arrays, and nothing that does can have been enqueued since (any such
    // call clears `evaluated`).  So unpack and copies go to the side stream behind that event and run beside the
    // neighbour stage; the call returns when both streams are done.
    cudaStream_t side = ctx->side_stream;
    P3T_CUDA(ctx, cudaStreamWaitEvent(side, ctx->ev[5], 0));
    p3t_status st = p3t_stage_unpack(ctx, acc ? ctx->ws.in_pos : nullptr, pot ? ctx->ws.in_mass : nullptr, side);
    if (st != P3T_OK) return st;
    if (acc) P3T_CUDA(ctx, cudaMemcpyAsync(acc, ctx->ws.in_pos, 3 * n * sizeof(float), cudaMemcpyDeviceToHost, side));
    if (pot) P3T_CUDA(ctx, cudaMemcpyAsync(pot, ctx->ws.in_mass, n * sizeof(float), cudaMemcpyDeviceToHost, side));
    P3T_CUDA(ctx, cudaStreamSynchronize(side));
    return sync_and_check(ctx);
}

extern "C" p3t_status p3t_get_neighbour_counts(p3t_ctx *ctx, uint32_t *count, uint64_t *total, int on_device)
{
    if (!ctx) return P3T_EINVAL;
    if (!ctx->evaluated) return p3t_fail(ctx, P3T_ESTATE, "p3t_get_neighbour_counts before an eval call");
    P3T_CUDA(ctx, cudaSetDevice(ctx->device));
    if (count)
        P3T_CUDA(ctx, cudaMemcpyAsync(count, ctx->ws.nbr_count, ctx->n * sizeof(u32),
                                      on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, ctx->stream));
    if (total || !on_device) {
        p3t_status st = sync_and_check(ctx);
        if (st != P3T_OK) return st;
        if (total) *total = ctx->h_counters[CNT_PAIRS];
    }
    return P3T_OK;
}

extern "C" p3t_status p3t_get_neighbours(p3t_ctx *ctx, uint64_t *offset, uint32_t *nbr, size_t capacity, int on_device)
{
    if (!ctx) return P3T_EINVAL;
    if (!ctx->evaluated) return p3t_fail(ctx, P3T_ESTATE, "p3t_get_neighbours before an eval call");
    if (!offset) return p3t_fail(ctx, P3T_EINVAL, "null offset");
    P3T_CUDA(ctx, cudaSetDevice(ctx->device));
    cudaMemcpyKind kind = on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
    P3T_CUDA(ctx, cudaMemcpyAsync(offset, ctx->ws.nbr_offset, (ctx->n + 1) * sizeof(u64), kind, ctx->stream));
    p3t_status st = sync_and_check(ctx);
    if (st != P3T_OK) return st;
    u64 total = ctx->h_counters[CNT_PAIRS];
    if (total > ctx->nbr_capacity) return p3t_fail(ctx, P3T_ECAPACITY, "neighbour lists exceed the context's nbr_capacity");
    if (total > capacity) return p3t_fail(ctx, P3T_ECAPACITY, "neighbour lists exceed the caller's buffer");
    if (total && !nbr) return p3t_fail(ctx, P3T_EINVAL, "null nbr");
    if (total) {
        P3T_CUDA(ctx, cudaMemcpyAsync(nbr, ctx->ws.nbr, total * sizeof(u32), kind, ctx->stream));
        P3T_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    }
    return P3T_OK;
}

extern "C" p3t_status p3t_get_stats(p3t_ctx *ctx, p3t_stats *out)
{
    if (!ctx || !out) return P3T_EINVAL;
    p3t_status st = sync_and_check(ctx);
    memset(out, 0, sizeof(*out));
    const u64 *c = ctx->h_counters;
    out->n = ctx->n;
    out->n_pp = c[CNT_NPP]; out->n_pc = c[CNT_NPC]; out->n_near = c[CNT_NNEAR];
    out->n_neighbours = c[CNT_PAIRS];
    out->n_cells = (u32)c[CNT_NCELLS]; out->n_leaves = (u32)c[CNT_NLEAVES]; out->n_groups = (u32)c[CNT_NGROUPS];
    out->depth = (u32)c[CNT_DEPTH]; out->max_list = (u32)c[CNT_MAXLIST];
    out->sort_passes = (u32)ctx->sort_passes_used;
    out->sort_max_run = ctx->sort_passes_used < (3 * ctx->max_level + 7) / 8 ? (u32)c[CNT_SORT_MAXRUN] : 0u;
    if (ctx->ev_build) {
        cudaEventElapsedTime(&out->ms_sort, ctx->ev[0], ctx->ev[1]);
        cudaEventElapsedTime(&out->ms_build, ctx->ev[1], ctx->ev[2]);
        cudaEventElapsedTime(&out->ms_moments, ctx->ev[2], ctx->ev[3]);
    }
    if (ctx->ev_eval) {
        cudaEventElapsedTime(&out->ms_walk, ctx->ev[4], ctx->ev[5]);
        cudaEventElapsedTime(&out->ms_nbr, ctx->ev[5], ctx->ev[6]);
    }
    if (ctx->ev_hard) cudaEventElapsedTime(&out->ms_hard, ctx->ev[7], ctx->ev[8]);
    if (ctx->ev_pack) cudaEventElapsedTime(&out->ms_pack, ctx->ev[9], ctx->ev[10]);
    out->walk_parts = (u32)ctx->walk_parts_used;
    out->tree_refits = (u32)ctx->refits;
    out->n_stray = (u32)(ctx->last_rebuilt ? 0 : ctx->last_stray);
    return st;
}

// ------------------------------------------------------------------------------------------------
// inspection
// ------------------------------------------------------------------------------------------------
static p3t_status array_desc(p3t_ctx *ctx, p3t_array which, const void **ptr, size_t *count, size_t *elem)
{
    Workspace &w = ctx->ws;
    size_t nc = (size_t)ctx->h_counters[CNT_NCELLS], ng = (size_t)ctx->h_counters[CNT_NGROUPS], n = ctx->n;
    switch (which) {
    case P3T_ARR_ROOT_CUBE:   *ptr = w.cube; *count = 4; *elem = 4; break;
    case P3T_ARR_KEYS:        *ptr = w.keys[ctx->cur]; *count = n; *elem = 8; break;
    case P3T_ARR_SORTED_IDX:  *ptr = w.idx[ctx->cur]; *count = n; *elem = 4; break;
    case P3T_ARR_BODIES:      *ptr = w.body; *count = n; *elem = 16; break;
    case P3T_ARR_CELL_MAC:    *ptr = w.cell_mac; *count = nc; *elem = 16; break;
    case P3T_ARR_CELL_MOM0:   *ptr = w.cell_mom0; *count = nc; *elem = 16; break;
    case P3T_ARR_CELL_MOM1:   *ptr = w.cell_mom1; *count = nc; *elem = 16; break;
    case P3T_ARR_CELL_META:   *ptr = w.cell_meta; *count = nc; *elem = 8; break;
    case P3T_ARR_CELL_LEVEL:  *ptr = w.cell_level; *count = nc; *elem = 1; break;
    case P3T_ARR_CELL_START:  *ptr = w.cell_start; *count = nc; *elem = 4; break;
    case P3T_ARR_CELL_PARENT: *ptr = w.cell_parent; *count = nc; *elem = 4; break;
    case P3T_ARR_GROUP_START: *ptr = w.group_start; *count = ng + 1; *elem = 4; break;
    case P3T_ARR_CELL_BMIN:   *ptr = w.cell_bmin; *count = nc; *elem = 16; break;
    case P3T_ARR_CELL_BMAX:   *ptr = w.cell_bmax; *count = nc; *elem = 16; break;
    case P3T_ARR_GROUP_STATS: *ptr = w.group_stats; *count = ng; *elem = 16; break;
    case P3T_ARR_GROUP_ORDER: *ptr = w.group_order; *count = ng; *elem = 4; break;
    default: return p3t_fail(ctx, P3T_EINVAL, "unknown array id");
    }
    return P3T_OK;
}

extern "C" p3t_status p3t_array_info(p3t_ctx *ctx, p3t_array which, size_t *count, size_t *elem_bytes)
{
    if (!ctx || !count || !elem_bytes) return P3T_EINVAL;
    if (!ctx->built) return p3t_fail(ctx, P3T_ESTATE, "p3t_array_info before p3t_build_tree");
    p3t_status st = sync_and_check(ctx);
    if (st != P3T_OK) return st;
    const void *p;
    return array_desc(ctx, which, &p, count, elem_bytes);
}

extern "C" p3t_status p3t_copy_array(p3t_ctx *ctx, p3t_array which, void *dst, size_t dst_bytes, int on_device)
{
    if (!ctx || !dst) return P3T_EINVAL;
    if (!ctx->built) return p3t_fail(ctx, P3T_ESTATE, "p3t_copy_array before p3t_build_tree");
    p3t_status st = sync_and_check(ctx);
    if (st != P3T_OK) return st;
    const void *p;
    size_t count, elem;
    if ((st = array_desc(ctx, which, &p, &count, &elem)) != P3T_OK) return st;
    if (dst_bytes < count * elem) return p3t_fail(ctx, P3T_ECAPACITY, "destination too small");
    if (count)
        P3T_CUDA(ctx, cudaMemcpyAsync(dst, p, count * elem, on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, ctx->stream));
    P3T_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return P3T_OK;
}
