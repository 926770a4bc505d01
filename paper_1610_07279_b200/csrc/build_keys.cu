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

// Listing 1 as a finite-state machine.  What the listing does to the coordinates below the current level is always a signed
// permutation of the axes (conditional inversions, then a rotation or a swap): 48 possible states at most.  One table entry
// per (state, octant of the ORIGINAL coordinates) gives the 3-bit key digit and the next state, so a level costs one
// shared-memory lookup instead of ~20 bit operations.  The table is generated on the host by running the listing's own
// level step (hilbert_level_step below) on every reachable state; the bit-exactness tests against the oracle's keys
// check the result.
constexpr int PH_STATES_MAX = 48;
__constant__ uint16_t c_ph_table[PH_STATES_MAX * 8];      // one level:  digit | next_state << 3
__device__ uint16_t g_ph_table2[PH_STATES_MAX * 64];      // two levels: 6 key bits | next_state << 6, indexed by state * 64 + two octants

struct PhState { int perm[3]; int flip[3]; };             // current axis a = original axis perm[a], inverted if flip[a]

// one level of Listing 1 on the CURRENT coordinates' bits: digit, inversion flags, axis map
inline void hilbert_level_step(int xb, int yb, int zb, int &digit, int f[3], int sigma[3])
{
    const int ny = yb ^ 1, nz = zb ^ 1;
    f[0] = xb & (ny | zb);
    f[1] = (xb & (yb | zb)) | (yb & nz);
    f[2] = (xb & ny & nz) | (yb & nz);
    digit = (xb << 2) | ((xb ^ yb) << 1) | (xb ^ zb ^ yb);
    if (zb) { sigma[0] = 1; sigma[1] = 2; sigma[2] = 0; }    // (x, y, z) <- (y, z, x)
    else if (ny) { sigma[0] = 2; sigma[1] = 1; sigma[2] = 0; } // x <-> z
    else { sigma[0] = 0; sigma[1] = 1; sigma[2] = 2; }
}

void build_ph_table(uint16_t *table)
{
    PhState st[PH_STATES_MAX];
    int n_st = 1;
    st[0] = PhState{{0, 1, 2}, {0, 0, 0}};
    for (int s = 0; s < n_st; s++) {
        for (int oct = 0; oct < 8; oct++) {
            const int ob[3] = {(oct >> 2) & 1, (oct >> 1) & 1, oct & 1};                     // original x, y, z bits
            const int cb[3] = {ob[st[s].perm[0]] ^ st[s].flip[0], ob[st[s].perm[1]] ^ st[s].flip[1], ob[st[s].perm[2]] ^ st[s].flip[2]};
            int digit, f[3], sigma[3];
            hilbert_level_step(cb[0], cb[1], cb[2], digit, f, sigma);
            PhState nx;
            for (int a = 0; a < 3; a++) { nx.perm[a] = st[s].perm[sigma[a]]; nx.flip[a] = st[s].flip[sigma[a]] ^ f[sigma[a]]; }
            int id = -1;
            for (int t = 0; t < n_st; t++) {
                bool same = true;
                for (int a = 0; a < 3; a++) same = same && st[t].perm[a] == nx.perm[a] && st[t].flip[a] == nx.flip[a];
                if (same) { id = t; break; }
            }
            if (id < 0) { id = n_st; st[n_st++] = nx; }
            table[s * 8 + oct] = (uint16_t)(digit | (id << 3));
        }
    }
    for (int i = n_st * 8; i < PH_STATES_MAX * 8; i++) table[i] = 0;
}

// 21 Morton bits (seven octants, most significant first) through the state machine: three double steps and a single one
__device__ __forceinline__ uint32_t ph_chunk(uint32_t m21, uint32_t &state, const uint16_t *tab1, const uint16_t *tab2)
{
    uint32_t out = 0;
#pragma unroll
    for (int j = 6; j >= 2; j -= 2) {                    // octants j and j - 1
        const uint32_t v = tab2[state * 64u + ((m21 >> (3 * (j - 1))) & 63u)];
        out = (out << 6) | (v & 63u);
        state = v >> 6;
    }
    const uint32_t v = tab1[state * 8u + (m21 & 7u)];
    out = (out << 3) | (v & 7u);
    state = v >> 3;
    return out;
}

// B2: one thread per particle.  16 B in, 8 B out.
__global__ void __launch_bounds__(256) k_keys(const float4 *__restrict__ pos, uint32_t n, const float *__restrict__ box,
                                              int key_kind, uint64_t *__restrict__ key)
{
    __shared__ uint16_t s_tab[PH_STATES_MAX * 8];
    __shared__ uint16_t s_tab2[PH_STATES_MAX * 64];
    if (key_kind == GOTHIC_KEY_PEANO_HILBERT) {
        for (int t = threadIdx.x; t < PH_STATES_MAX * 8; t += blockDim.x) s_tab[t] = c_ph_table[t];
        for (int t = threadIdx.x; t < PH_STATES_MAX * 32; t += blockDim.x)
            reinterpret_cast<uint32_t *>(s_tab2)[t] = reinterpret_cast<const uint32_t *>(g_ph_table2)[t];
    }
    __syncthreads();
    const float x0 = box[0], y0 = box[1], z0 = box[2], scale = box[4];
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {      // tables loaded once per CTA
        const float4 p = __ldg(pos + i);
        const uint32_t ix = cell_coord(p.x, x0, scale), iy = cell_coord(p.y, y0, scale), iz = cell_coord(p.z, z0, scale);
        const uint64_t m = (spread3(ix) << 2) | (spread3(iy) << 1) | spread3(iz);          // Listing 3
        if (key_kind == GOTHIC_KEY_MORTON) { key[i] = m; continue; }
        uint32_t state = 0;
        const uint64_t k2 = ph_chunk((uint32_t)(m >> 42) & 0x1fffffu, state, s_tab, s_tab2);
        const uint64_t k1 = ph_chunk((uint32_t)(m >> 21) & 0x1fffffu, state, s_tab, s_tab2);
        const uint64_t k0 = ph_chunk((uint32_t)m & 0x1fffffu, state, s_tab, s_tab2);
        key[i] = (k2 << 42) | (k1 << 21) | k0;
    }
}

// B4: pos_sorted[s] = pos[perm[s]]
__global__ void __launch_bounds__(256) k_gather(const float4 *__restrict__ pos, const uint32_t *__restrict__ perm, uint32_t n,
                                                float4 *__restrict__ out)
{
    const uint32_t s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s < n) out[s] = __ldg(pos + __ldg(perm + s));
}

} // namespace

// the state table of the Peano-Hilbert machine -> constant memory of the current device (called by gothic_create)
int gothic_keys_config(gothic_ctx *c)
{
    static uint16_t table[PH_STATES_MAX * 8], table2[PH_STATES_MAX * 64];
    build_ph_table(table);
    for (int s = 0; s < PH_STATES_MAX; s++)          // two levels at once: high octant, then low octant from the state it leads to
        for (int o = 0; o < 64; o++) {
            const uint16_t a = table[s * 8 + (o >> 3)], b = table[(a >> 3) * 8 + (o & 7)];
            table2[s * 64 + o] = (uint16_t)((((a & 7) << 3) | (b & 7)) | ((b >> 3) << 6));
        }
    GOTHIC_CUDA_OK(c, cudaMemcpyToSymbol(c_ph_table, table, sizeof(table)));
    GOTHIC_CUDA_OK(c, cudaMemcpyToSymbol(g_ph_table2, table2, sizeof(table2)));
    return GOTHIC_OK;
}

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
    k_keys<<<grid, 256, 0, s>>>(pos_m, n, c->box, key_kind, c->key[0]);   // perm starts as the identity, generated by the first sort pass
    GOTHIC_LAUNCH_OK(c);
    return GOTHIC_OK;
}

int gothic_stage_gather(gothic_ctx *c, const float4 *pos_m, uint32_t n, cudaStream_t s)
{
    k_gather<<<(n + 255u) / 256u, 256, 0, s>>>(pos_m, c->idx[c->cur], n, c->pos_sorted);
    GOTHIC_LAUNCH_OK(c);
    return GOTHIC_OK;
}
