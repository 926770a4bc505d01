// B1 root box, B2 space-filling-curve keys, B4 gather into sorted order.
// PAPER.md:54 ("the GPU generates the Peano-Hilbert key for all N-body particles"), App. A Listings 1 and 3.
#include "gothic_ctx.cuh"

namespace {

__device__ __forceinline__ uint32_t f2ord(float f)
{
    uint32_t u = __float_as_uint(f);
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float ord2f(uint32_t u)
{
    return __uint_as_float((u & 0x80000000u) ? (u & 0x7fffffffu) : ~u);
}

__global__ void k_bbox_init(uint32_t *bits)
{
    if (threadIdx.x < 3) bits[threadIdx.x] = 0xFFFFFFFFu;      // minima
    else if (threadIdx.x < 6) bits[threadIdx.x] = 0u;          // maxima
}

// B1: per-axis min/max.  Grid-stride, float4 loads, warp shuffle + one atomic per warp per bound.
__global__ void __launch_bounds__(256) k_bbox(const float4 *__restrict__ pos, uint32_t n, uint32_t *bits)
{
    float lo[3] = {INFINITY, INFINITY, INFINITY}, hi[3] = {-INFINITY, -INFINITY, -INFINITY};
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const float4 p = __ldg(pos + i);
        lo[0] = fminf(lo[0], p.x); hi[0] = fmaxf(hi[0], p.x);
        lo[1] = fminf(lo[1], p.y); hi[1] = fmaxf(hi[1], p.y);
        lo[2] = fminf(lo[2], p.z); hi[2] = fmaxf(hi[2], p.z);
    }
#pragma unroll
    for (int k = 0; k < 3; k++) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            lo[k] = fminf(lo[k], __shfl_xor_sync(0xffffffffu, lo[k], o));
            hi[k] = fmaxf(hi[k], __shfl_xor_sync(0xffffffffu, hi[k], o));
        }
    }
    if (lane_id() == 0) {
#pragma unroll
        for (int k = 0; k < 3; k++) {
            atomicMin(bits + k, f2ord(lo[k]));
            atomicMax(bits + 3 + k, f2ord(hi[k]));
        }
    }
}

// Root cube (R1): anchor = minima; side = smallest power of two strictly greater than the extent.
__global__ void k_box_finish(const uint32_t *bits, float *box)
{
    const float x0 = ord2f(bits[0]), y0 = ord2f(bits[1]), z0 = ord2f(bits[2]);
    const float ex = __fsub_rn(ord2f(bits[3]), x0), ey = __fsub_rn(ord2f(bits[4]), y0), ez = __fsub_rn(ord2f(bits[5]), z0);
    const float ext = fmaxf(ex, fmaxf(ey, ez));
    float side = 1.0f;
    if (ext > 0.0f) {
        int e;
        (void)frexpf(ext, &e);
        side = ldexpf(1.0f, e);
    }
    box[0] = x0; box[1] = y0; box[2] = z0; box[3] = side;
    box[4] = __fdiv_rn(2097152.0f, side);   // 2^21 / side: exact power of two
}

__device__ __forceinline__ uint32_t cell_coord(float x, float x0, float scale)
{
    const float f = floorf(__fmul_rn(__fsub_rn(x, x0), scale));
    if (!(f > 0.0f)) return 0u;
    if (f >= 2097151.0f) return 2097151u;
    return (uint32_t)f;
}

// Listing 1 on 32-bit coordinate registers: per level, read one bit of each coordinate,
// conditionally invert the coordinates (masks 0 / ~0), emit the 3-bit digit, then rotate or swap axes.
__device__ __forceinline__ uint64_t peano_hilbert_63(uint32_t px, uint32_t py, uint32_t pz)
{
    uint64_t key = 0;
#pragma unroll
    for (int lev = GOTHIC_NLEV - 1; lev >= 0; lev--) {
        const uint32_t xb = (px >> lev) & 1u, yb = (py >> lev) & 1u, zb = (pz >> lev) & 1u;
        const uint32_t ny = yb ^ 1u, nz = zb ^ 1u;
        px ^= 0u - (xb & (ny | zb));
        py ^= 0u - ((xb & (yb | zb)) | (yb & nz));
        pz ^= 0u - ((xb & ny & nz) | (yb & nz));
        const uint32_t digit = (xb << 2) | ((xb ^ yb) << 1) | (xb ^ zb ^ yb);
        key = (key << 3) | digit;
        if (zb) { const uint32_t t = px; px = py; py = pz; pz = t; }
        else if (ny) { const uint32_t t = px; px = pz; pz = t; }
    }
    return key;
}

// Listing 3: spread 21 bits to every third bit by multiply-and-mask.
__device__ __forceinline__ uint64_t spread3(uint32_t v)
{
    uint64_t w = v;
    w = (w | (w << 32)) & 0x7fff00000000ffffull;
    w = (w | (w << 16)) & 0x00ff0000ff0000ffull;
    w = (w | (w << 8)) & 0x700f00f00f00f00full;
    w = (w | (w << 4)) & 0x30c30c30c30c30c3ull;
    w = (w | (w << 2)) & 0x1249249249249249ull;
    return w;
}

// B2: one thread per particle.  16 B in, 8 B out.
__global__ void __launch_bounds__(256) k_keys(const float4 *__restrict__ pos, uint32_t n, const float *__restrict__ box,
                                              int key_kind, uint64_t *__restrict__ key)
{
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float x0 = box[0], y0 = box[1], z0 = box[2], scale = box[4];
    const float4 p = __ldg(pos + i);
    const uint32_t ix = cell_coord(p.x, x0, scale), iy = cell_coord(p.y, y0, scale), iz = cell_coord(p.z, z0, scale);
    key[i] = key_kind == GOTHIC_KEY_PEANO_HILBERT ? peano_hilbert_63(ix, iy, iz)
                                                  : ((spread3(ix) << 2) | (spread3(iy) << 1) | spread3(iz));
}

// B4: pos_sorted[s] = pos[perm[s]]
__global__ void __launch_bounds__(256) k_gather(const float4 *__restrict__ pos, const uint32_t *__restrict__ perm, uint32_t n,
                                                float4 *__restrict__ out)
{
    const uint32_t s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s < n) out[s] = __ldg(pos + __ldg(perm + s));
}

} // namespace

int gothic_stage_keys(gothic_ctx *c, const float4 *pos_m, uint32_t n, int key_kind, cudaStream_t s)
{
    k_bbox_init<<<1, 32, 0, s>>>(c->bbox_bits);
    GOTHIC_LAUNCH_OK(c);
    int grid = (int)((n + 255u) / 256u);
    if (grid > c->num_sms * 8) grid = c->num_sms * 8;
    k_bbox<<<grid, 256, 0, s>>>(pos_m, n, c->bbox_bits);
    GOTHIC_LAUNCH_OK(c);
    k_box_finish<<<1, 1, 0, s>>>(c->bbox_bits, c->box);
    GOTHIC_LAUNCH_OK(c);
    c->cur = 0;
    k_keys<<<(n + 255u) / 256u, 256, 0, s>>>(pos_m, n, c->box, key_kind, c->key[0]);   // perm starts as the identity, generated by the first sort pass
    GOTHIC_LAUNCH_OK(c);
    return GOTHIC_OK;
}

int gothic_stage_gather(gothic_ctx *c, const float4 *pos_m, uint32_t n, cudaStream_t s)
{
    k_gather<<<(n + 255u) / 256u, 256, 0, s>>>(pos_m, c->idx[c->cur], n, c->pos_sorted);
    GOTHIC_LAUNCH_OK(c);
    return GOTHIC_OK;
}
