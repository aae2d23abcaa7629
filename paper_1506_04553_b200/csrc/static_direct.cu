// static_direct.cu -- p3t_direct_static: the brute-force soft force of direct.cu (Eq. 6, 8 of PAPER.md, K of Eq. 12, W of
// Eq. 16-17, neighbour rule s_ij < h) for callers that cannot allocate: no context, no workspace, no cudaMalloc.  The
// kernel's scratch -- the bodies packed as (x, y, z, m) and a header of counters -- lives in a file-scope device array of
// fixed size that every GPU loading the library holds until exit.  Not on the timed hot path; the existing entry
// points are untouched.
#include "p3t_internal.cuh"
#include <math.h>

#define SD_THREADS 128
#define SD_HEADER_WORDS 32                       // u64 words in front of the bodies (256 B): [0] neighbour entries, [1] non-finite inputs
#define SD_MAX_DEVICES 64

// ---- the scratch: header + P3T_STATIC_MAX_N packed bodies (1 MiB + 256 B per device) ---------------------------------
// In HOST code this name is only a stand-in for the symbol; its device address comes from cudaGetSymbolAddress (below).
static __device__ __align__(256) unsigned char g_sd_scratch[SD_HEADER_WORDS * sizeof(u64) + (size_t)P3T_STATIC_MAX_N * sizeof(float4)];

static unsigned char *g_sd_ptr[SD_MAX_DEVICES];   // device address of the scratch per device, set once with that device current
static char g_sd_err[256] = "";

static p3t_status sd_fail(p3t_status st, const char *msg)
{
    snprintf(g_sd_err, sizeof(g_sd_err), "%s", msg);
    return st;
}
static p3t_status sd_cuda(cudaError_t e, const char *what)
{
    if (e == cudaSuccess) return P3T_OK;
    snprintf(g_sd_err, sizeof(g_sd_err), "p3t_direct_static: %s failed: %s", what, cudaGetErrorString(e));
    return P3T_ECUDA;
}

extern "C" const char *p3t_direct_static_last_error(void) { return g_sd_err; }

// ---- kernels ---------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) sd_pack_kernel(const float *__restrict__ mass, const float *__restrict__ pos, u32 n,
                                                      float4 *__restrict__ body, u64 *hdr)
{
    const u32 i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float m = mass[i], x = pos[3 * i], y = pos[3 * i + 1], z = pos[3 * i + 2];
    if (!(isfinite(m) && isfinite(x) && isfinite(y) && isfinite(z))) atomicAdd(reinterpret_cast<unsigned long long *>(&hdr[1]), 1ull);
    body[i] = make_float4(x, y, z, m);
}

// direct_kernel of direct.cu without pair classes and without the pair buffer: one target per thread, sources staged
// through shared memory in tiles of 128, fp32 pair arithmetic, one fp64 add per tile; outputs in the caller's layout
__global__ void __launch_bounds__(SD_THREADS) sd_direct_kernel(const float4 *__restrict__ body, u32 n, CutoffSet cs, float eps2,
                                                               float rout2, float h2, float *__restrict__ acc,
                                                               float *__restrict__ pot, u32 *__restrict__ nbr_count, u64 *hdr)
{
    __shared__ float4 s_b[SD_THREADS];
    const u32 i = blockIdx.x * SD_THREADS + threadIdx.x;
    const bool active = i < n;
    const float4 bi = body[active ? i : 0u];
    double ax = 0.0, ay = 0.0, az = 0.0, ph = 0.0;
    u32 cnt = 0;
    for (u32 j0 = 0; j0 < n; j0 += SD_THREADS) {
        const u32 jl = j0 + threadIdx.x;
        s_b[threadIdx.x] = jl < n ? body[jl] : make_float4(0.f, 0.f, 0.f, 0.f);
        __syncthreads();
        const u32 lim = min((u32)SD_THREADS, n - j0);
        float fx = 0.f, fy = 0.f, fz = 0.f, fp = 0.f;
        if (active) {
            for (u32 jj = 0; jj < lim; ++jj) {
                if (j0 + jj == i) continue;                       // j != i by index (reading A13)
                const float4 bj = s_b[jj];
                const float dx = bj.x - bi.x, dy = bj.y - bi.y, dz = bj.z - bi.z;
                const float s2 = fmaf(dx, dx, fmaf(dy, dy, fmaf(dz, dz, eps2)));
                const float rinv = rsqrtf(s2);
                const float mrinv = bj.w * rinv;
                float mr3 = mrinv * (rinv * rinv);
                float K = 1.f, W = 1.f;
                if (s2 < h2) {
                    if (s2 < rout2) p3t_pair_weights(cs, s2, K, W);
                    ++cnt;
                }
                mr3 *= K;
                fx = fmaf(mr3, dx, fx); fy = fmaf(mr3, dy, fy); fz = fmaf(mr3, dz, fz);
                fp = fmaf(W, mrinv, fp);
            }
        }
        ax += (double)fx; ay += (double)fy; az += (double)fz; ph += (double)fp;
        __syncthreads();
    }
    if (active) {
        acc[3 * i] = (float)ax; acc[3 * i + 1] = (float)ay; acc[3 * i + 2] = (float)az;
        pot[i] = (float)(-ph);
        if (nbr_count) nbr_count[i] = cnt;
        if (cnt) atomicAdd(reinterpret_cast<unsigned long long *>(&hdr[0]), (unsigned long long)cnt);
    }
}

__global__ void sd_info_kernel(const u64 *__restrict__ hdr, u64 *__restrict__ info)
{
    info[0] = hdr[0];
    info[1] = hdr[1];
}

// ---- the entry point -------------------------------------------------------------------------------------------------
extern "C" p3t_status p3t_direct_static(int device, void *cuda_stream, size_t n, const float *mass, const float *pos, float eps,
                                        float r_in, float r_out, float r_search, float *acc, float *pot, uint32_t *nbr_count,
                                        uint64_t *info)
{
    if (device < 0 || device >= SD_MAX_DEVICES) return sd_fail(P3T_EINVAL, "p3t_direct_static: device must be in 0..63");
    if (!mass || !pos || !acc || !pot) return sd_fail(P3T_EINVAL, "p3t_direct_static: mass, pos, acc and pot must be device pointers");
    if (n == 0) return sd_fail(P3T_EINVAL, "p3t_direct_static: n must be at least 1");
    if (n > (size_t)P3T_STATIC_MAX_N) {
        snprintf(g_sd_err, sizeof(g_sd_err), "p3t_direct_static: n = %zu exceeds P3T_STATIC_MAX_N = %d, the size of the library's static scratch "
                 "(use a context and p3t_eval_direct / p3t_eval_soft for more)", n, P3T_STATIC_MAX_N);
        return P3T_ECAPACITY;
    }
    if (!(eps >= 0.f) || !isfinite(eps) || !isfinite(r_search) || !(r_in >= 0.f) || !(r_in < r_out) || !(r_out <= r_search))
        return sd_fail(P3T_EINVAL, "p3t_direct_static: need eps >= 0 and 0 <= r_in < r_out <= r_search, all finite");
    int prev = -1;
    p3t_status st = sd_cuda(cudaGetDevice(&prev), "cudaGetDevice");
    if (st != P3T_OK) return st;
    if (prev != device && (st = sd_cuda(cudaSetDevice(device), "cudaSetDevice")) != P3T_OK) return st;
    // set-up, once per device, with that device current: the device address of the scratch array
    if (!g_sd_ptr[device]) {
        unsigned char *p = nullptr;
        st = sd_cuda(cudaGetSymbolAddress((void **)&p, g_sd_scratch), "cudaGetSymbolAddress");
        if (st == P3T_OK && !p) st = sd_fail(P3T_ECUDA, "p3t_direct_static: cudaGetSymbolAddress returned a null address");
        if (st != P3T_OK) {
            if (prev != device) cudaSetDevice(prev);
            return st;
        }
        g_sd_ptr[device] = p;
    }
    u64 *hdr = reinterpret_cast<u64 *>(g_sd_ptr[device]);
    float4 *body = reinterpret_cast<float4 *>(g_sd_ptr[device] + SD_HEADER_WORDS * sizeof(u64));
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    CutoffSet cs;
    p3t_fill_cutoff(cs, r_in, r_out);
    // the array keeps the last call's contents: the counters must start at zero (the bodies are overwritten up to n and
    // never read beyond)
    st = sd_cuda(cudaMemsetAsync(hdr, 0, SD_HEADER_WORDS * sizeof(u64), s), "cudaMemsetAsync");
    if (st == P3T_OK) {
        sd_pack_kernel<<<div_up(n, 256), 256, 0, s>>>(mass, pos, (u32)n, body, hdr);
        sd_direct_kernel<<<div_up(n, SD_THREADS), SD_THREADS, 0, s>>>(body, (u32)n, cs, eps * eps, r_out * r_out, r_search * r_search, acc, pot,
                                                                      nbr_count, hdr);
        if (info) sd_info_kernel<<<1, 1, 0, s>>>(hdr, reinterpret_cast<u64 *>(info));
        st = sd_cuda(cudaGetLastError(), "kernel launch");
    }
    if (prev != device) cudaSetDevice(prev);
    return st;
}
