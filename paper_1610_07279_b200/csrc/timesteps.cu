// T1 block time-step levels and T2 ordered active-set compaction (R6).
// dt_i = eta sqrt(eps/|a_i|) floored to a power of two: with q = dt^4 = (eta^4 eps^2)/|a|^2 the exponent of dt is
// floor(ilogb(q)/4), read from the float's exponent field -- no transcendental, so it is bit-exact.
#include "gothic_ctx.cuh"

namespace {

constexpr int TPB = 256;
constexpr int ITEMS = 8;                 // flags per thread in the compaction passes
constexpr int TILE = TPB * ITEMS;

__device__ __forceinline__ int dt_exponent(float4 a, float c)
{
    const float a2 = fmaf(a.z, a.z, fmaf(a.y, a.y, __fmul_rn(a.x, a.x)));
    if (!(a2 > 0.0f)) return 127;
    const float q = __fdiv_rn(c, a2);
    const uint32_t u = __float_as_uint(q);
    const int ex = (int)((u >> 23) & 0xffu);
    const uint32_t man = u & 0x7fffffu;
    if (ex == 0xff) return 127;              // inf / nan
    int e;
    if (ex) e = ex - 127;
    else if (man) e = (31 - __clz(man)) - 149; // subnormal
    else return -38;                          // q == 0
    return e >> 2;                            // floor(e / 4) (arithmetic shift)
}

__global__ void k_ts_init(int32_t *tmp) { tmp[0] = 0x7fffffff; tmp[1] = 0; }

__global__ void __launch_bounds__(TPB) k_dt_exponent(const float4 *__restrict__ acc, uint32_t n, float c, int8_t *__restrict__ ex, int32_t *tmp)
{
    int emin = 0x7fffffff;
    for (uint32_t i = blockIdx.x * TPB + threadIdx.x; i < n; i += gridDim.x * TPB) {
        const int e = dt_exponent(__ldg(acc + i), c);
        ex[i] = (int8_t)e;
        emin = min(emin, e);
    }
    emin = __reduce_min_sync(0xffffffffu, emin);
    if (lane_id() == 0) atomicMin(tmp, emin);
}

__global__ void __launch_bounds__(TPB) k_levels(uint32_t n, int max_levels, uint8_t *__restrict__ level, int32_t *tmp)
{
    const int emin = tmp[0];
    int lmax = 0;
    for (uint32_t i = blockIdx.x * TPB + threadIdx.x; i < n; i += gridDim.x * TPB) {
        const int l = min((int)((int8_t)level[i]) - emin, max_levels - 1);
        level[i] = (uint8_t)l;
        lmax = max(lmax, l);
    }
    lmax = __reduce_max_sync(0xffffffffu, lmax);
    if (lane_id() == 0) atomicMax(tmp + 1, lmax);
}

__global__ void k_ts_report(const int32_t *tmp, int32_t *out) { out[0] = tmp[0]; out[1] = tmp[1] + 1; }

// ---- ordered compaction: per-tile counts -> scan -> scatter --------------------------------------------
__device__ __forceinline__ uint32_t tile_flags(const uint8_t *__restrict__ level, uint32_t n, uint32_t base, int ctz)
{
    // 8 consecutive levels per thread (one 8-byte load when fully in range)
    uint32_t f = 0;
    if (base + ITEMS <= n && (reinterpret_cast<uintptr_t>(level) & 7u) == 0) {
        const uint2 v = *reinterpret_cast<const uint2 *>(level + base);
#pragma unroll
        for (int k = 0; k < 4; k++) {
            f |= ((int)((v.x >> (8 * k)) & 0xffu) <= ctz) ? (1u << k) : 0u;
            f |= ((int)((v.y >> (8 * k)) & 0xffu) <= ctz) ? (1u << (4 + k)) : 0u;
        }
    } else {
        for (int k = 0; k < ITEMS; k++)
            if (base + k < n && (int)level[base + k] <= ctz) f |= 1u << k;
    }
    return f;
}

__global__ void __launch_bounds__(TPB) k_active_count(const uint8_t *__restrict__ level, uint32_t n, int ctz, uint32_t *__restrict__ tile_cnt)
{
    __shared__ uint32_t tot;
    if (threadIdx.x == 0) tot = 0;
    __syncthreads();
    const uint32_t base = blockIdx.x * TILE + threadIdx.x * ITEMS;
    uint32_t c = __popc(tile_flags(level, n, base, ctz));
    c = __reduce_add_sync(0xffffffffu, c);
    if (lane_id() == 0 && c) atomicAdd(&tot, c);
    __syncthreads();
    if (threadIdx.x == 0) tile_cnt[blockIdx.x] = tot;
}

__global__ void __launch_bounds__(1024) k_active_scan(uint32_t *__restrict__ tile_cnt, uint32_t ntiles, uint32_t *__restrict__ n_active)
{
    __shared__ uint32_t wexc[32];
    __shared__ uint32_t chunk_total;
    uint32_t carry = 0;   // same value in every thread
    for (uint32_t b0 = 0; b0 < ntiles; b0 += 1024) {
        const uint32_t i = b0 + threadIdx.x;
        const uint32_t v = i < ntiles ? tile_cnt[i] : 0u;
        uint32_t x = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t y = __shfl_up_sync(0xffffffffu, x, o);
            if ((int)lane_id() >= o) x += y;
        }
        if (lane_id() == 31) wexc[threadIdx.x >> 5] = x;
        __syncthreads();
        if (threadIdx.x < 32) {
            const uint32_t s = wexc[threadIdx.x];
            uint32_t t = s;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t y = __shfl_up_sync(0xffffffffu, t, o);
                if ((int)lane_id() >= o) t += y;
            }
            wexc[threadIdx.x] = t - s;
            if (threadIdx.x == 31) chunk_total = t;
        }
        __syncthreads();
        if (i < ntiles) tile_cnt[i] = carry + wexc[threadIdx.x >> 5] + x - v;
        carry += chunk_total;
        __syncthreads();
    }
    if (threadIdx.x == 0) *n_active = carry;
}

__global__ void __launch_bounds__(TPB) k_active_scatter(const uint8_t *__restrict__ level, uint32_t n, int ctz,
                                                         const uint32_t *__restrict__ tile_ofs, uint32_t *__restrict__ active)
{
    __shared__ uint32_t wsum[TPB / 32];
    const uint32_t base = blockIdx.x * TILE + threadIdx.x * ITEMS;
    const uint32_t f = tile_flags(level, n, base, ctz);
    const uint32_t c = __popc(f);
    uint32_t x = c;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t y = __shfl_up_sync(0xffffffffu, x, o);
        if ((int)lane_id() >= o) x += y;
    }
    if (lane_id() == 31) wsum[threadIdx.x >> 5] = x;
    __syncthreads();
    uint32_t pre = tile_ofs[blockIdx.x];
    for (int w = 0; w < (int)(threadIdx.x >> 5); w++) pre += wsum[w];
    uint32_t o = pre + x - c;
#pragma unroll
    for (int k = 0; k < ITEMS; k++)
        if (f & (1u << k)) active[o++] = base + k;
}

} // namespace

int gothic_stage_timesteps(gothic_ctx *c, const float4 *acc_pot, uint32_t n, float cconst, int max_levels,
                           uint32_t substep, uint8_t *level, uint32_t *active, uint32_t *n_active_dev,
                           int32_t *emin_nlev_dev, cudaStream_t s)
{
    int grid = (int)((n + TPB - 1) / TPB);
    if (grid > c->num_sms * 16) grid = c->num_sms * 16;
    if (acc_pot) {
        k_ts_init<<<1, 1, 0, s>>>(c->ts_tmp);
        GOTHIC_LAUNCH_OK(c);
        k_dt_exponent<<<grid, TPB, 0, s>>>(acc_pot, n, cconst, reinterpret_cast<int8_t *>(level), c->ts_tmp);
        GOTHIC_LAUNCH_OK(c);
        k_levels<<<grid, TPB, 0, s>>>(n, max_levels, level, c->ts_tmp);
        GOTHIC_LAUNCH_OK(c);
        if (emin_nlev_dev) {
            k_ts_report<<<1, 1, 0, s>>>(c->ts_tmp, emin_nlev_dev);
            GOTHIC_LAUNCH_OK(c);
        }
    }
    if (active && n_active_dev) {
        const int ctz = __builtin_ctz(substep);
        const uint32_t ntiles = (n + TILE - 1) / TILE;
        k_active_count<<<ntiles, TPB, 0, s>>>(level, n, ctz, c->scan_tmp);
        GOTHIC_LAUNCH_OK(c);
        k_active_scan<<<1, 1024, 0, s>>>(c->scan_tmp, ntiles, n_active_dev);
        GOTHIC_LAUNCH_OK(c);
        k_active_scatter<<<ntiles, TPB, 0, s>>>(level, n, ctz, c->scan_tmp, active);
        GOTHIC_LAUNCH_OK(c);
    }
    return GOTHIC_OK;
}

// ---- gothic_active_list_static: T2 without a context and without any allocation (include/gothic.h) ------------------------
// For hosts that cannot call cudaMalloc once they are running (all device memory already in their own arrays or pool, or a step
// loop that must not take cudaMalloc's device-wide synchronisation).  The only scratch T2 needs, the per-tile counts, lives in
// the library image instead of a gothic_ctx: 32768 words = 128 KiB per GPU that loads the library, for as long as the process
// lives.  The kernels are the three of gothic_stage_timesteps above, unchanged.
#include <mutex>

static_assert(GOTHIC_STATIC_ACTIVE_MAX_N % TILE == 0, "whole tiles");
static __device__ __align__(256) uint32_t g_static_tile_cnt[GOTHIC_STATIC_ACTIVE_MAX_N / TILE];

namespace {
constexpr int STATIC_MAX_DEVICES = 64;
std::mutex g_static_mutex;
// Device address of g_static_tile_cnt on each device, filled by the first call made with that device current.  In host code the
// name g_static_tile_cnt is only a handle for the runtime, never a pointer a kernel may be given.
uint32_t *g_static_tile_cnt_addr[STATIC_MAX_DEVICES];
}

extern "C" int gothic_active_list_static(const uint8_t *level, uint32_t n, uint32_t substep, uint32_t *active,
                                         uint32_t *n_active_dev, void *stream)
{
    if (!level || !active || !n_active_dev || n == 0 || substep == 0) return GOTHIC_ERR_ARG;
    if (n > GOTHIC_STATIC_ACTIVE_MAX_N) return GOTHIC_ERR_TOO_LARGE;
    int device = -1;
    if (cudaGetDevice(&device) != cudaSuccess) return GOTHIC_ERR_CUDA;
    if (device < 0 || device >= STATIC_MAX_DEVICES) return GOTHIC_ERR_ARG;
    uint32_t *tile_cnt;
    {
        std::lock_guard<std::mutex> lock(g_static_mutex);
        tile_cnt = g_static_tile_cnt_addr[device];
        if (!tile_cnt) {                       // set-up, once per device, with that device current
            void *p = nullptr;
            if (cudaGetSymbolAddress(&p, g_static_tile_cnt) != cudaSuccess || !p) return GOTHIC_ERR_CUDA;
            tile_cnt = g_static_tile_cnt_addr[device] = static_cast<uint32_t *>(p);
        }
    }
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const int ctz = __builtin_ctz(substep);
    const uint32_t ntiles = (n + TILE - 1) / TILE;
    // no word of tile_cnt needs to be zero on entry: k_active_count stores (not adds) one count per tile, the scan reads only those
    k_active_count<<<ntiles, TPB, 0, s>>>(level, n, ctz, tile_cnt);
    if (cudaGetLastError() != cudaSuccess) return GOTHIC_ERR_CUDA;
    k_active_scan<<<1, 1024, 0, s>>>(tile_cnt, ntiles, n_active_dev);
    if (cudaGetLastError() != cudaSuccess) return GOTHIC_ERR_CUDA;
    k_active_scatter<<<ntiles, TPB, 0, s>>>(level, n, ctz, tile_cnt, active);
    if (cudaGetLastError() != cudaSuccess) return GOTHIC_ERR_CUDA;
    return GOTHIC_OK;
}
