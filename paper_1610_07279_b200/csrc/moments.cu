// B6: pseudo j-particle moments (Fig. 1; the paper's calcMAC, Table 2):
// m_J = total mass, r_J = centre of mass, b_J = radius of the sphere about r_J that contains all the cell's
// particles (exact maximum, R9).  Recomputed every step, so it is a separate entry point.
//
// Mass and first moment go bottom-up (leaves from particles, internal nodes from their <= 8 contiguous
// children, one launch per level from the deepest).  The radius needs every particle against every ancestor's
// centre: one thread per PARTICLE (position in registers, read once) climbs from its leaf to the root; a level costs
// one 16-byte load (r_J and the parent id share a record).  Consecutive sorted particles share their ancestors, so the
// lanes of a warp form contiguous segments with the same node: the segment maximum is taken with shuffles (one
// REDUX when the whole warp sits in one node, the usual case above the lowest levels) and only the first lane of a
// segment raises b_J^2 with an integer atomicMax on the float bits (non-negative floats order like unsigned ints),
// skipped when the stored value is already larger.
#include "gothic_ctx.cuh"

namespace {

constexpr int TPB = 256;

__device__ __forceinline__ void store_com(uint32_t J, float4 ms, float4 com, float4 *__restrict__ node_msum, float4 *__restrict__ node_com,
                                          uint32_t *__restrict__ node_b2bits, const uint32_t *__restrict__ node_parent, float4 *__restrict__ node_up,
                                          uint32_t b2bits = 0u)
{
    node_msum[J] = ms;
    node_com[J] = com;
    node_b2bits[J] = b2bits;
    node_up[J] = make_float4(com.x, com.y, com.z, __uint_as_float(node_parent[J]));
}
__device__ __forceinline__ float4 com_of(float4 ms)
{
    return make_float4(__fdiv_rn(ms.x, ms.w), __fdiv_rn(ms.y, ms.w), __fdiv_rn(ms.z, ms.w), ms.w);
}

__global__ void __launch_bounds__(TPB) k_leaf_moments(uint32_t n_nodes, const float4 *__restrict__ pos, const uint32_t *__restrict__ node_head,
                                                       const uint32_t *__restrict__ node_num, const uint32_t *__restrict__ node_child,
                                                       float4 *__restrict__ node_msum, float4 *__restrict__ node_com, uint32_t *__restrict__ node_b2bits,
                                                       const uint32_t *__restrict__ node_parent, float4 *__restrict__ node_up, float *__restrict__ node_B2)
{
    const uint32_t J = blockIdx.x * TPB + threadIdx.x;
    if (J >= n_nodes || node_child[J] != GOTHIC_LEAF) return;
    const uint32_t h = node_head[J], c = node_num[J];
    if (c == 1) {   // a single-particle node IS the particle (bitwise), b_J = 0
        const float4 p = __ldg(pos + h);
        store_com(J, make_float4(p.w * p.x, p.w * p.y, p.w * p.z, p.w), p, node_msum, node_com, node_b2bits, node_parent, node_up);
        if (node_B2) node_B2[J] = 0.0f;
        return;
    }
    float4 ms = make_float4(0.f, 0.f, 0.f, 0.f);
    for (uint32_t j = h; j < h + c; j++) {
        const float4 p = __ldg(pos + j);
        ms.x = fmaf(p.w, p.x, ms.x); ms.y = fmaf(p.w, p.y, ms.y); ms.z = fmaf(p.w, p.z, ms.z); ms.w += p.w;
    }
    const float4 cm = com_of(ms);
    // the leaf's own radius (exact maximum, same arithmetic as k_node_radius): the radius climb then starts at the leaf's parent and
    // is spared its most fragmented level
    float b2 = 0.0f;
    for (uint32_t j = h; j < h + c; j++) {
        const float4 p = __ldg(pos + j);
        const float dx = __fsub_rn(p.x, cm.x), dy = __fsub_rn(p.y, cm.y), dz = __fsub_rn(p.z, cm.z);
        b2 = fmaxf(b2, fmaf(dz, dz, fmaf(dy, dy, __fmul_rn(dx, dx))));
    }
    store_com(J, ms, cm, node_msum, node_com, node_b2bits, node_parent, node_up, __float_as_uint(b2));
    if (!node_B2) return;
    float B2 = 0.0f;                                     // eq. 4 about the stored centre
    for (uint32_t j = h; j < h + c; j++) {
        const float4 p = __ldg(pos + j);
        const float dx = p.x - cm.x, dy = p.y - cm.y, dz = p.z - cm.z;
        B2 = fmaf(p.w, fmaf(dz, dz, fmaf(dy, dy, dx * dx)), B2);
    }
    node_B2[J] = B2;
}

// m_J, r_J (and B_2) of one internal node from its children, which the level below has finished
__device__ __forceinline__ void internal_moment_of(uint32_t J, const uint32_t *__restrict__ node_child, const uint8_t *__restrict__ node_nchild,
                                                   float4 *node_msum, float4 *node_com, uint32_t *node_b2bits,
                                                   const uint32_t *__restrict__ node_parent, float4 *node_up, float *node_B2)
{
    const uint32_t c = node_child[J];
    if (c == GOTHIC_LEAF) return;
    const uint32_t nc = node_nchild[J];
    float4 ms = node_msum[c];
    for (uint32_t k = 1; k < nc; k++) {
        const float4 q = node_msum[c + k];
        ms.x += q.x; ms.y += q.y; ms.z += q.z; ms.w += q.w;
    }
    const float4 cm = com_of(ms);
    store_com(J, ms, cm, node_msum, node_com, node_b2bits, node_parent, node_up);
    if (!node_B2) return;
    float B2 = 0.0f;                                     // parallel-axis theorem over the children: B2_c + m_c |r_c - r_J|^2
    for (uint32_t k = 0; k < nc; k++) {
        const float4 q = node_com[c + k];
        const float dx = q.x - cm.x, dy = q.y - cm.y, dz = q.z - cm.z;
        B2 += fmaf(q.w, fmaf(dz, dz, fmaf(dy, dy, dx * dx)), node_B2[c + k]);
    }
    node_B2[J] = B2;
}

__global__ void __launch_bounds__(TPB) k_internal_moments(uint32_t first, uint32_t count, const uint32_t *__restrict__ node_child,
                                                           const uint8_t *__restrict__ node_nchild, float4 *node_msum,
                                                           float4 *node_com, uint32_t *node_b2bits,
                                                           const uint32_t *__restrict__ node_parent, float4 *node_up, float *node_B2)
{
    const uint32_t t = blockIdx.x * TPB + threadIdx.x;
    if (t >= count) return;
    internal_moment_of(first + t, node_child, node_nchild, node_msum, node_com, node_b2bits, node_parent, node_up, node_B2);
}

// A run of consecutive SMALL levels (the top of the tree, and its sparse deepest levels) in one launch: one CTA sweeps level l_from, then
// l_from - 1, ... down to l_to, a block barrier between levels (the children of a level were written by this CTA one barrier earlier).
// Same per-node arithmetic as k_internal_moments, so the moments do not change by a bit; it only saves the launches.
constexpr int SMALL_TPB = 1024;
constexpr uint32_t SMALL_LEVEL_MAX = 8192;      // nodes: at most 8 per thread and level
__global__ void __launch_bounds__(SMALL_TPB) k_internal_moments_small(const uint32_t *__restrict__ level_ofs, int l_from, int l_to,
                                                                       const uint32_t *__restrict__ node_child, const uint8_t *__restrict__ node_nchild,
                                                                       float4 *node_msum, float4 *node_com, uint32_t *node_b2bits,
                                                                       const uint32_t *__restrict__ node_parent, float4 *node_up, float *node_B2)
{
    for (int L = l_from; L >= l_to; L--) {
        const uint32_t first = level_ofs[L], count = level_ofs[L + 1] - first;
        for (uint32_t t = threadIdx.x; t < count; t += SMALL_TPB)
            internal_moment_of(first + t, node_child, node_nchild, node_msum, node_com, node_b2bits, node_parent, node_up, node_B2);
        __syncthreads();
    }
}

// Persistent warps, each sweeping a contiguous range of sorted particles 32 at a time.  Lane L of a warp remembers the
// node the warp was last in at level L: id, particle range, centre and the running maximum.  While a chunk lies inside
// the remembered range of a level, that level needs no memory access at all (centre broadcast by shuffle, one REDUX);
// only the lowest levels, where the chunk straddles several nodes, climb parent links from the leaves.  A remembered
// maximum is written out (guarded atomicMax) when the warp moves on to another node of that level or finishes, so the
// upper levels, which every particle contributes to, cost a few thousand atomics in total.
__global__ void __launch_bounds__(TPB) k_node_radius(uint32_t n, uint32_t per_warp, const float4 *__restrict__ pos,
                                                      const uint32_t *__restrict__ leaf_of, const uint8_t *__restrict__ leaf_level,
                                                      const uint32_t *__restrict__ node_head, const uint32_t *__restrict__ node_num,
                                                      const float4 *__restrict__ node_up, uint32_t *__restrict__ node_b2bits)
{
    const uint32_t lane = lane_id();
    const uint32_t gw = (blockIdx.x * TPB + threadIdx.x) >> 5;
    const uint64_t r0 = (uint64_t)gw * per_warp;
    if (r0 >= n) return;
    const uint32_t r1 = (uint32_t)min((uint64_t)n, r0 + per_warp);
    // lane L: level L
    uint32_t m_node = GOTHIC_LEAF, m_head = 0u, m_end = 0u, m_max = 0u;
    float m_x = 0.f, m_y = 0.f, m_z = 0.f;
    // the next chunk's particle, leaf, leaf level (its own array: no dependent load) are requested one chunk ahead, and the
    // leaf's own record as soon as its id is there
    float4 p_nx = make_float4(0.f, 0.f, 0.f, 0.f), u_nx = make_float4(0.f, 0.f, 0.f, 0.f);
    uint32_t A_nx = GOTHIC_LEAF;
    int lev_nx = -1;
    if ((uint32_t)r0 + lane < r1) {
        p_nx = __ldg(pos + (uint32_t)r0 + lane); A_nx = __ldg(leaf_of + (uint32_t)r0 + lane); lev_nx = (int)(int8_t)__ldg(leaf_level + (uint32_t)r0 + lane);
        if (A_nx != GOTHIC_LEAF) u_nx = node_up[A_nx];
    }
    for (uint32_t s0 = (uint32_t)r0; s0 < r1; s0 += 32u) {
        const uint32_t s = s0 + lane;
        const bool act = s < r1;
        const float4 p = p_nx, u_leaf = u_nx;
        uint32_t A = A_nx;
        int lev = lev_nx;
        p_nx = make_float4(0.f, 0.f, 0.f, 0.f); A_nx = GOTHIC_LEAF; lev_nx = -1;
        if (s + 32u < r1) { p_nx = __ldg(pos + s + 32u); A_nx = __ldg(leaf_of + s + 32u); lev_nx = (int)(int8_t)__ldg(leaf_level + s + 32u); }
        // ---- top-down over the levels whose remembered node contains the whole chunk (nested, so levels 0 .. Lf-1) ----
        const uint32_t in_mask = __ballot_sync(0xffffffffu, m_node != GOTHIC_LEAF && s0 >= m_head && min(s0 + 32u, r1) <= m_end);
        const int Lf = __ffs(~in_mask) - 1;
        for (int L = 0; L < Lf; L++) {
            const float cx = __shfl_sync(0xffffffffu, m_x, L), cy = __shfl_sync(0xffffffffu, m_y, L), cz = __shfl_sync(0xffffffffu, m_z, L);
            const float dx = __fsub_rn(p.x, cx), dy = __fsub_rn(p.y, cy), dz = __fsub_rn(p.z, cz);
            const uint32_t bits = act ? __float_as_uint(fmaf(dz, dz, fmaf(dy, dy, __fmul_rn(dx, dx)))) : 0u;
            const uint32_t mx = __reduce_max_sync(0xffffffffu, bits);
            if ((int)lane == L) m_max = max(m_max, mx);
        }
        // ---- bottom-up from the deepest leaf of the chunk to level Lf: a lane joins when the walk reaches its leaf's
        //      level, so that the lanes that sit in the same node are neighbours; the record of the next level is
        //      requested before the reduction of this one ----
        int L = __reduce_max_sync(0xffffffffu, lev);
        if (A_nx != GOTHIC_LEAF) u_nx = node_up[A_nx];          // the next chunk's leaf records, used one iteration from now
        float4 u = u_leaf;                                      // a lane's first record is its leaf's, already here
        for (; L >= Lf; L--) {
            const bool on = lev == L;
            const uint32_t node = on ? A : GOTHIC_LEAF;
            const float cx = u.x, cy = u.y, cz = u.z;
            uint32_t bits = 0u;
            if (on) {
                const float dx = __fsub_rn(p.x, cx), dy = __fsub_rn(p.y, cy), dz = __fsub_rn(p.z, cz);
                bits = __float_as_uint(fmaf(dz, dz, fmaf(dy, dy, __fmul_rn(dx, dx))));
                A = __float_as_uint(u.w);
                lev = L - 1;
            }
            if (on && L > Lf) u = node_up[A];                    // the parent's record; lanes that join later still hold their leaf's
            int all_same = 0;
            __match_all_sync(0xffffffffu, node, &all_same);
            if (all_same) {                                                  // whole chunk in one node: remember it
                bits = __reduce_max_sync(0xffffffffu, bits);
                if ((int)lane == L) {
                    if (m_node == node) m_max = max(m_max, bits);
                    else {
                        if (m_node != GOTHIC_LEAF && m_max > __ldcg(node_b2bits + m_node)) atomicMax(node_b2bits + m_node, m_max);
                        m_node = node; m_max = bits;
                        m_head = node_head[node]; m_end = m_head + node_num[node];
                        m_x = cx; m_y = cy; m_z = cz;
                    }
                }
            } else {                                                         // contiguous segments of equal node
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const uint32_t b2 = __shfl_down_sync(0xffffffffu, bits, o);
                    const uint32_t n2 = __shfl_down_sync(0xffffffffu, node, o);
                    if (lane + o < 32u && n2 == node) bits = max(bits, b2);
                }
                const uint32_t nprev = __shfl_up_sync(0xffffffffu, node, 1);
                if (on && (lane == 0 || nprev != node)) atomicMax(node_b2bits + node, bits);      // low levels: distinct addresses, no guard
            }
        }
    }
    if (m_node != GOTHIC_LEAF && m_max > __ldcg(node_b2bits + m_node)) atomicMax(node_b2bits + m_node, m_max);
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

// NodeRec::mb2 <- m b^2 (acceleration MAC, eq. 5) or 3 B_2 (multipole MAC, eq. 3): one 4-byte store per node
__global__ void __launch_bounds__(TPB) k_rec_slot4(uint32_t n_nodes, int multipole, const float4 *__restrict__ node_com, const float *__restrict__ node_b,
                                                    const float *__restrict__ node_B2, NodeRec *__restrict__ rec)
{
    const uint32_t J = blockIdx.x * TPB + threadIdx.x;
    if (J >= n_nodes) return;
    if (multipole) rec[J].mb2 = __fmul_rn(3.0f, node_B2[J]);
    else { const float b = node_b[J]; rec[J].mb2 = __fmul_rn(__fmul_rn(node_com[J].w, b), b); }
}

} // namespace

// B_2 (eq. 4) is only computed once somebody has asked for it (multipole MAC or tree view); from then on every moments pass of
// this context carries it along.
int gothic_stage_need_b2(gothic_ctx *c, cudaStream_t s)
{
    if (c->b2_enabled) return GOTHIC_OK;
    c->b2_enabled = true;
    return gothic_stage_moments(c, s);
}

int gothic_stage_rec_slot4(gothic_ctx *c, int mac_kind, cudaStream_t s)
{
    const int want = mac_kind == GOTHIC_MAC_MULTIPOLE ? GOTHIC_MAC_MULTIPOLE : GOTHIC_MAC_ACCELERATION;
    if (mac_kind == GOTHIC_MAC_OPENING_ANGLE || c->rec_slot4 == want) return GOTHIC_OK;     // eq. 2 reads b_J only
    if (want == GOTHIC_MAC_MULTIPOLE) {
        const int rc = gothic_stage_need_b2(c, s);
        if (rc != GOTHIC_OK) return rc;
    }
    k_rec_slot4<<<(c->n_nodes + TPB - 1) / TPB, TPB, 0, s>>>(c->n_nodes, want == GOTHIC_MAC_MULTIPOLE, c->node_com, c->node_b, c->node_B2, c->node_rec);
    GOTHIC_LAUNCH_OK(c);
    c->rec_slot4 = want;
    return GOTHIC_OK;
}

int gothic_stage_moments(gothic_ctx *c, cudaStream_t s)
{
    const uint32_t m = c->n_nodes;
    const uint32_t grid = (m + TPB - 1) / TPB;
    k_leaf_moments<<<grid, TPB, 0, s>>>(m, c->pos_sorted, c->node_head, c->node_num, c->node_child, c->node_msum, c->node_com, c->node_b2bits, c->node_parent, c->node_up, c->b2_enabled ? c->node_B2 : nullptr);
    GOTHIC_LAUNCH_OK(c);
    for (int L = (int)c->n_levels_tree - 2; L >= 0;) {
        const uint32_t first = c->h_level_ofs[L], count = c->h_level_ofs[L + 1] - first;
        if (!count) { L--; continue; }
        if (count <= SMALL_LEVEL_MAX) {           // this level and the small ones right above it: one CTA, one launch
            int l_to = L;
            while (l_to > 0 && c->h_level_ofs[l_to] - c->h_level_ofs[l_to - 1] <= SMALL_LEVEL_MAX) l_to--;
            k_internal_moments_small<<<1, SMALL_TPB, 0, s>>>(c->level_ofs, L, l_to, c->node_child, c->node_nchild, c->node_msum, c->node_com, c->node_b2bits,
                                                             c->node_parent, c->node_up, c->b2_enabled ? c->node_B2 : nullptr);
            GOTHIC_LAUNCH_OK(c);
            L = l_to - 1;
            continue;
        }
        k_internal_moments<<<(count + TPB - 1) / TPB, TPB, 0, s>>>(first, count, c->node_child, c->node_nchild, c->node_msum, c->node_com, c->node_b2bits, c->node_parent, c->node_up, c->b2_enabled ? c->node_B2 : nullptr);
        GOTHIC_LAUNCH_OK(c);
        L--;
    }
    {
        if (c->radius_blocks_per_sm < 1) {
            int q = 0;
            if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&q, k_node_radius, TPB, 0) != cudaSuccess || q < 1) q = 1;
            c->radius_blocks_per_sm = q;
        }
        const int per_sm = c->radius_blocks_per_sm;
        const uint32_t blocks = (uint32_t)(c->num_sms * per_sm), warps = blocks * (TPB / 32);     // one resident wave
        const uint32_t per_warp = (((c->n + warps - 1) / warps + 31u) / 32u) * 32u;
        k_node_radius<<<blocks, TPB, 0, s>>>(c->n, per_warp, c->pos_sorted, c->leaf_of, c->leaf_level, c->node_head, c->node_num, c->node_up, c->node_b2bits);
    }
    GOTHIC_LAUNCH_OK(c);
    k_pack_nodes<<<grid, TPB, 0, s>>>(m, c->node_head, c->node_num, c->node_child, c->node_nchild, c->node_com, c->node_b2bits, c->node_b, c->node_rec, c->n_max);
    GOTHIC_LAUNCH_OK(c);
    c->rec_slot4 = GOTHIC_MAC_ACCELERATION;
    return GOTHIC_OK;
}
