// B6: pseudo j-particle moments (Fig. 1; the paper's calcMAC, Table 2):
// m_J = total mass, r_J = centre of mass, b_J = radius of the sphere about r_J that contains all the cell's
// particles (exact maximum, R9).  Recomputed every step, so it is a separate entry point.
//
// Mass and first moment go bottom-up (leaves from particles, internal nodes from their <= 8 contiguous
// children, one launch per level from the deepest).  The radius needs every particle against every ancestor's
// centre: one thread per leaf climbs the parent chain and raises b_J^2 with an integer atomicMax on the float
// bits (non-negative floats order like unsigned ints), skipping the atomic when the stored value is already larger.
#include "gothic_ctx.cuh"

namespace {

constexpr int TPB = 256;

__device__ __forceinline__ void store_com(uint32_t J, float4 ms, float4 *__restrict__ node_msum, float4 *__restrict__ node_com,
                                          uint32_t *__restrict__ node_b2bits)
{
    node_msum[J] = ms;
    node_com[J] = make_float4(__fdiv_rn(ms.x, ms.w), __fdiv_rn(ms.y, ms.w), __fdiv_rn(ms.z, ms.w), ms.w);
    node_b2bits[J] = 0u;
}

__global__ void __launch_bounds__(TPB) k_leaf_moments(uint32_t n_nodes, const float4 *__restrict__ pos, const uint32_t *__restrict__ node_head,
                                                       const uint32_t *__restrict__ node_num, const uint32_t *__restrict__ node_child,
                                                       float4 *__restrict__ node_msum, float4 *__restrict__ node_com, uint32_t *__restrict__ node_b2bits)
{
    const uint32_t J = blockIdx.x * TPB + threadIdx.x;
    if (J >= n_nodes || node_child[J] != GOTHIC_LEAF) return;
    const uint32_t h = node_head[J], c = node_num[J];
    if (c == 1) {   // a single-particle node IS the particle (bitwise), b_J = 0
        const float4 p = __ldg(pos + h);
        node_msum[J] = make_float4(p.w * p.x, p.w * p.y, p.w * p.z, p.w);
        node_com[J] = p;
        node_b2bits[J] = 0u;
        return;
    }
    float4 ms = make_float4(0.f, 0.f, 0.f, 0.f);
    for (uint32_t j = h; j < h + c; j++) {
        const float4 p = __ldg(pos + j);
        ms.x = fmaf(p.w, p.x, ms.x); ms.y = fmaf(p.w, p.y, ms.y); ms.z = fmaf(p.w, p.z, ms.z); ms.w += p.w;
    }
    store_com(J, ms, node_msum, node_com, node_b2bits);
}

__global__ void __launch_bounds__(TPB) k_internal_moments(uint32_t first, uint32_t count, const uint32_t *__restrict__ node_child,
                                                           const uint8_t *__restrict__ node_nchild, float4 *__restrict__ node_msum,
                                                           float4 *__restrict__ node_com, uint32_t *__restrict__ node_b2bits)
{
    const uint32_t t = blockIdx.x * TPB + threadIdx.x;
    if (t >= count) return;
    const uint32_t J = first + t, c = node_child[J];
    if (c == GOTHIC_LEAF) return;
    const uint32_t nc = node_nchild[J];
    float4 ms = node_msum[c];
    for (uint32_t k = 1; k < nc; k++) {
        const float4 q = node_msum[c + k];
        ms.x += q.x; ms.y += q.y; ms.z += q.z; ms.w += q.w;
    }
    store_com(J, ms, node_msum, node_com, node_b2bits);
}

__global__ void __launch_bounds__(TPB) k_node_radius(uint32_t n_nodes, const float4 *__restrict__ pos, const uint32_t *__restrict__ node_head,
                                                      const uint32_t *__restrict__ node_num, const uint32_t *__restrict__ node_child,
                                                      const uint32_t *__restrict__ node_parent, const float4 *__restrict__ node_com,
                                                      uint32_t *__restrict__ node_b2bits)
{
    const uint32_t J = blockIdx.x * TPB + threadIdx.x;
    if (J >= n_nodes || node_child[J] != GOTHIC_LEAF) return;
    const uint32_t h = node_head[J], c = node_num[J];
    for (uint32_t A = J; A != GOTHIC_LEAF; A = node_parent[A]) {
        const float4 cm = node_com[A];
        float d2max = 0.0f;
        for (uint32_t j = h; j < h + c; j++) {
            const float4 p = __ldg(pos + j);
            const float dx = __fsub_rn(p.x, cm.x), dy = __fsub_rn(p.y, cm.y), dz = __fsub_rn(p.z, cm.z);
            d2max = fmaxf(d2max, fmaf(dz, dz, fmaf(dy, dy, __fmul_rn(dx, dx))));
        }
        const uint32_t bits = __float_as_uint(d2max);
        if (bits > *(volatile uint32_t *)(node_b2bits + A)) atomicMax(node_b2bits + A, bits);
    }
}

__global__ void __launch_bounds__(TPB) k_pack_nodes(uint32_t n_nodes, const uint32_t *__restrict__ node_head, const uint32_t *__restrict__ node_num,
                                                     const uint32_t *__restrict__ node_child, const uint8_t *__restrict__ node_nchild,
                                                     const float4 *__restrict__ node_com, const uint32_t *__restrict__ node_b2bits,
                                                     float *__restrict__ node_b, NodeRec *__restrict__ rec, uint32_t root_item)
{
    const uint32_t J = blockIdx.x * TPB + threadIdx.x;
    if (J >= n_nodes) return;
    const float4 cm = node_com[J];
    const float b = __fsqrt_rn(__uint_as_float(node_b2bits[J]));
    node_b[J] = b;
    NodeRec r;
    r.x = cm.x; r.y = cm.y; r.z = cm.z; r.m = cm.w;
    r.mb2 = __fmul_rn(__fmul_rn(cm.w, b), b);
    r.b = b;
    const uint32_t c = node_child[J];
    if (c == GOTHIC_LEAF) { r.w0 = node_head[J]; r.w1 = 0x80000000u | node_num[J]; }
    else { r.w0 = root_item + 2u * c; r.w1 = node_nchild[J]; }
    rec[J] = r;
}

} // namespace

int gothic_stage_moments(gothic_ctx *c, cudaStream_t s)
{
    const uint32_t m = c->n_nodes;
    const uint32_t grid = (m + TPB - 1) / TPB;
    k_leaf_moments<<<grid, TPB, 0, s>>>(m, c->pos_sorted, c->node_head, c->node_num, c->node_child, c->node_msum, c->node_com, c->node_b2bits);
    GOTHIC_LAUNCH_OK(c);
    for (int L = (int)c->n_levels_tree - 2; L >= 0; L--) {
        const uint32_t first = c->h_level_ofs[L], count = c->h_level_ofs[L + 1] - first;
        if (!count) continue;
        k_internal_moments<<<(count + TPB - 1) / TPB, TPB, 0, s>>>(first, count, c->node_child, c->node_nchild, c->node_msum, c->node_com, c->node_b2bits);
        GOTHIC_LAUNCH_OK(c);
    }
    k_node_radius<<<grid, TPB, 0, s>>>(m, c->pos_sorted, c->node_head, c->node_num, c->node_child, c->node_parent, c->node_com, c->node_b2bits);
    GOTHIC_LAUNCH_OK(c);
    k_pack_nodes<<<grid, TPB, 0, s>>>(m, c->node_head, c->node_num, c->node_child, c->node_nchild, c->node_com, c->node_b2bits, c->node_b, c->node_rec, c->n_max);
    GOTHIC_LAUNCH_OK(c);
    return GOTHIC_OK;
}
