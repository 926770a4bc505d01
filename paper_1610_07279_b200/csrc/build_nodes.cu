// B5: canonical oct-tree (node ranges + links) from the sorted keys, all levels at once.
//
// PAPER.md:58 builds the tree breadth-first, one level per grid-wide barrier (Xiao & Feng lock-free barrier,
// PAPER.md:60).  On B200 that chain of <= 21 dependent grid syncs is replaced by a formulation in which every
// level is independent, so the whole topology comes out of two streaming passes over the keys:
//
//   delta(p)  = number of leading octal digits shared by key[p-1] and key[p]   (delta(0) = delta(n) = -1)
//   D(p)      = deepest level at which the run of equal-prefix keys containing p holds more than n_leaf
//               particles = max over windows [i, i+n_leaf] containing p of shared_digits(key[i], key[i+n_leaf])
//   p STARTS a node at every level L in [delta(p)+1, min(D(p)+1, 21)]
//   p ENDS   a node at every level L in [delta(p+1)+1, min(D(p)+1, 21)]
//   (both ranges are what k_node_events stores per key, four bytes; k_emit_nodes reads them back instead of the keys)
//
// (a level-L run is a node iff its parent run has more than n_leaf particles, and run sizes shrink monotonically
// with depth).  The k-th start and the k-th end of a level belong to the same node; node id = level offset +
// rank, which is exactly breadth-first order with ascending head inside a level, so children are contiguous.
// Pass 1 counts start/end events per (block, level); a small scan turns them into offsets; pass 2 emits.
#include "gothic_ctx.cuh"

namespace {

constexpr int TPB = 256;
constexpr int NW = TPB / 32;
constexpr int IPT = 8;                                   // keys per thread in the two event passes
constexpr int TILE = TPB * IPT;                          // keys per CTA (2048): key p of a tile sits in row q = (p - base) / TPB
constexpr int NROW = IPT * NW;                           // (row, warp) pairs of a tile, in key order

constexpr int KEYS_SM = TILE + 2 * GOTHIC_MAX_NLEAF;    // keys base - H .. base + TILE + H
constexpr int WIN_SM = TILE + GOTHIC_MAX_NLEAF;         // window values of positions base - H .. base + TILE

// The four event levels of one key in one word: bytes (s_lo, s_hi, e_lo, e_hi); an empty range has lo > hi.
__device__ __forceinline__ uint32_t pack_events(int s_lo, int s_hi, int e_lo, int e_hi)
{
    return (uint32_t)s_lo | ((uint32_t)s_hi << 8) | ((uint32_t)e_lo << 16) | ((uint32_t)e_hi << 24);
}
struct Events { int s_lo, s_hi, e_lo, e_hi; };
__device__ __forceinline__ Events unpack_events(uint32_t w)
{
    Events ev = {(int)(w & 255u), (int)((w >> 8) & 255u), (int)((w >> 16) & 255u), (int)(w >> 24)};
    return ev;
}

// levels at which any lane of the warp has an event: [lo, hi] (empty if lo > hi)
__device__ __forceinline__ void warp_level_range(const Events &ev, int &lo, int &hi)
{
    const bool any_s = ev.s_lo <= ev.s_hi, any_e = ev.e_lo <= ev.e_hi;
    int l = GOTHIC_NLEVP1, h = -1;
    if (any_s) { l = min(l, ev.s_lo); h = max(h, ev.s_hi); }
    if (any_e) { l = min(l, ev.e_lo); h = max(h, ev.e_hi); }
    lo = __reduce_min_sync(0xffffffffu, l);
    hi = __reduce_max_sync(0xffffffffu, h);
}

// Pass 1: the events of every key, computed once and kept as one word per key, and their counts per (tile, level).
// D(p) is a sliding-window maximum of w(i) = shared_digits(key[i], key[i + H]) over i in [p - H, p]: every w is computed once, then
// the window maxima of widths 2, 4, 8, ... are built by doubling in shared memory.
// blk_cnt layout: [kind(0 = start, 1 = end)][level][ntile]
__global__ void __launch_bounds__(TPB) k_node_events(const uint64_t *__restrict__ key, uint32_t n, int H, uint32_t *__restrict__ events,
                                                      uint32_t *__restrict__ blk_cnt, uint32_t ntile)
{
    __shared__ uint64_t sk[KEYS_SM];
    __shared__ int8_t sw[2][WIN_SM];
    __shared__ uint32_t tot[2][GOTHIC_NLEVP1];
    if (threadIdx.x < 2 * GOTHIC_NLEVP1) (&tot[0][0])[threadIdx.x] = 0;
    const long long base = (long long)blockIdx.x * TILE;
    for (int t = threadIdx.x; t < TILE + 2 * H; t += TPB) {
        const long long g = base - H + t;
        sk[t] = (g >= 0 && g < (long long)n) ? __ldg(key + g) : 0ull;
    }
    __syncthreads();
    const int len = TILE + H;
    for (int t = threadIdx.x; t < len; t += TPB) {
        const long long i = base - H + t;
        sw[0][t] = (i >= 0 && i + H < (long long)n) ? (int8_t)shared_digits(sk[t], sk[t + H]) : (int8_t)-1;
    }
    __syncthreads();
    const int W = H + 1;                                            // window width
    int8_t *cur = sw[0], *nxt = sw[1];
    int k = 1;
    while (2 * k <= W) {
        for (int t = threadIdx.x; t < len; t += TPB) nxt[t] = t + k < len ? max(cur[t], cur[t + k]) : cur[t];
        __syncthreads();
        int8_t *tmp = cur; cur = nxt; nxt = tmp;
        k *= 2;
    }
    // cur[t] = max of w over slots [t, t + k); the window of key base + j is slots [j, j + W)
#pragma unroll
    for (int q = 0; q < IPT; q++) {
        const int j = q * TPB + threadIdx.x;
        const long long p = base + j;
        Events ev = {1, 0, 1, 0};
        if (p < (long long)n) {
            const int D = max((int)cur[j], (int)cur[j + W - k]);
            const uint64_t kp = sk[H + j];
            const int dprev = p == 0 ? -1 : shared_digits(sk[H + j - 1], kp);
            const int dnext = p == (long long)n - 1 ? -1 : shared_digits(kp, sk[H + j + 1]);
            const int top = min(D + 1, GOTHIC_NLEV);
            ev.s_lo = dprev + 1; ev.s_hi = top; ev.e_lo = dnext + 1; ev.e_hi = top;
            events[p] = pack_events(ev.s_lo, ev.s_hi, ev.e_lo, ev.e_hi);
        }
        int Llo, Lhi;
        warp_level_range(ev, Llo, Lhi);
        for (int L = Llo; L <= Lhi; L++) {
            const uint32_t bs = __ballot_sync(0xffffffffu, ev.s_lo <= L && L <= ev.s_hi);
            const uint32_t be = __ballot_sync(0xffffffffu, ev.e_lo <= L && L <= ev.e_hi);
            if (lane_id() == 0) {
                if (bs) atomicAdd(&tot[0][L], __popc(bs));
                if (be) atomicAdd(&tot[1][L], __popc(be));
            }
        }
    }
    __syncthreads();
    if (threadIdx.x < 2 * GOTHIC_NLEVP1)
        blk_cnt[(size_t)threadIdx.x * ntile + blockIdx.x] = (&tot[0][0])[threadIdx.x];
}

// One block per (kind, level): exclusive scan over blocks in place; totals of the start rows -> level_cnt.
// 1024 threads x 8 consecutive counts per step.
constexpr int SCAN_TPB = 1024, SCAN_IPT = 8;
__global__ void __launch_bounds__(SCAN_TPB) k_scan_blocks(uint32_t *__restrict__ blk_cnt, uint32_t nblk, uint32_t *__restrict__ level_cnt)
{
    __shared__ uint32_t wsum[SCAN_TPB / 32];
    __shared__ uint32_t carry_s;
    uint32_t *row = blk_cnt + (size_t)blockIdx.x * nblk;
    if (threadIdx.x == 0) carry_s = 0;
    __syncthreads();
    for (uint32_t b0 = 0; b0 < nblk; b0 += SCAN_TPB * SCAN_IPT) {
        const uint32_t i0 = b0 + threadIdx.x * SCAN_IPT;
        uint32_t v[SCAN_IPT], mine = 0;
#pragma unroll
        for (int k = 0; k < SCAN_IPT; k++) { v[k] = i0 + k < nblk ? row[i0 + k] : 0u; mine += v[k]; }
        uint32_t x = mine;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t y = __shfl_up_sync(0xffffffffu, x, o);
            if ((int)lane_id() >= o) x += y;
        }
        if (lane_id() == 31) wsum[threadIdx.x >> 5] = x;
        __syncthreads();
        uint32_t wpre = 0, total = 0;
#pragma unroll
        for (int w = 0; w < SCAN_TPB / 32; w++) {
            const uint32_t s = wsum[w];
            if (w < (int)(threadIdx.x >> 5)) wpre += s;
            total += s;
        }
        uint32_t run = carry_s + wpre + x - mine;
#pragma unroll
        for (int k = 0; k < SCAN_IPT; k++) { if (i0 + k < nblk) row[i0 + k] = run; run += v[k]; }
        __syncthreads();
        if (threadIdx.x == 0) carry_s += total;
        __syncthreads();
    }
    if (threadIdx.x == 0 && blockIdx.x < GOTHIC_NLEVP1) level_cnt[blockIdx.x] = carry_s;
}

// level offsets, node count, capacity check.  flags[0] = overflow, flags[2] = n_nodes
__global__ void k_level_offsets(const uint32_t *level_cnt, uint32_t *level_ofs, uint32_t *flags, uint32_t node_max)
{
    unsigned long long acc = 0;
    for (int L = 0; L < GOTHIC_NLEVP1; L++) {
        level_ofs[L] = (uint32_t)min(acc, 0xFFFFFFFFull);
        acc += level_cnt[L];
    }
    level_ofs[GOTHIC_NLEVP1] = (uint32_t)min(acc, 0xFFFFFFFFull);
    flags[2] = (uint32_t)min(acc, 0xFFFFFFFFull);
    if (acc > node_max) flags[0] = 1u;
}

// Pass 2: node ids from the scanned counts, node arrays written.  Reads the event words of pass 1 (4 bytes per key), not the keys.
__global__ void __launch_bounds__(TPB) k_emit_nodes(const uint32_t *__restrict__ events, uint32_t n,
                                                     const uint32_t *__restrict__ blk_cnt, uint32_t ntile,
                                                     const uint32_t *__restrict__ level_ofs, const uint32_t *__restrict__ flags,
                                                     uint32_t *__restrict__ node_head, uint8_t *__restrict__ node_level,
                                                     uint32_t *__restrict__ node_child, uint32_t *__restrict__ node_end,
                                                     uint32_t *__restrict__ node_last)
{
    __shared__ uint32_t wcnt[2][GOTHIC_NLEVP1][NROW];   // counts per (row, warp) in key order -> exclusive prefix + tile base + level offset
    if (flags[0] | flags[3]) return;      // pool overflow, or keys the fast sort left unordered (end counts may then exceed start counts: ids past n_nodes)
    for (int t = threadIdx.x; t < 2 * GOTHIC_NLEVP1 * NROW; t += TPB) (&wcnt[0][0][0])[t] = 0u;
    const uint32_t base = blockIdx.x * (uint32_t)TILE;
    const int warp = threadIdx.x >> 5;
    Events ev[IPT];
#pragma unroll
    for (int q = 0; q < IPT; q++) {
        const uint32_t p = base + q * TPB + threadIdx.x;
        ev[q] = unpack_events(p < n ? __ldg(events + p) : pack_events(1, 0, 1, 0));
    }
    __syncthreads();
#pragma unroll
    for (int q = 0; q < IPT; q++) {
        int Llo, Lhi;
        warp_level_range(ev[q], Llo, Lhi);
        for (int L = Llo; L <= Lhi; L++) {
            const uint32_t bs = __ballot_sync(0xffffffffu, ev[q].s_lo <= L && L <= ev[q].s_hi);
            const uint32_t be = __ballot_sync(0xffffffffu, ev[q].e_lo <= L && L <= ev[q].e_hi);
            if (lane_id() == 0) { wcnt[0][L][q * NW + warp] = __popc(bs); wcnt[1][L][q * NW + warp] = __popc(be); }
        }
    }
    __syncthreads();
    if (threadIdx.x < 2 * GOTHIC_NLEVP1) {
        const int kind = threadIdx.x / GOTHIC_NLEVP1, L = threadIdx.x % GOTHIC_NLEVP1;
        uint32_t run = level_ofs[L] + blk_cnt[(size_t)threadIdx.x * ntile + blockIdx.x];
        for (int w = 0; w < NROW; w++) { const uint32_t c = wcnt[kind][L][w]; wcnt[kind][L][w] = run; run += c; }
    }
    __syncthreads();
    const uint32_t lt = (1u << lane_id()) - 1u;
#pragma unroll
    for (int q = 0; q < IPT; q++) {
        const uint32_t p = base + q * TPB + threadIdx.x;
        int Llo, Lhi;
        warp_level_range(ev[q], Llo, Lhi);
        uint32_t sid_below = GOTHIC_LEAF, eid_below = GOTHIC_LEAF;   // ids of this key's events one level deeper
        for (int L = Lhi; L >= Llo; L--) {
            const bool fs = ev[q].s_lo <= L && L <= ev[q].s_hi, fe = ev[q].e_lo <= L && L <= ev[q].e_hi;
            const uint32_t bs = __ballot_sync(0xffffffffu, fs);
            const uint32_t be = __ballot_sync(0xffffffffu, fe);
            if (fs) {
                const uint32_t id = wcnt[0][L][q * NW + warp] + __popc(bs & lt);
                node_head[id] = p;
                node_level[id] = (uint8_t)L;
                node_child[id] = (L + 1 <= ev[q].s_hi) ? sid_below : GOTHIC_LEAF;
                sid_below = id;
            }
            if (fe) {
                const uint32_t id = wcnt[1][L][q * NW + warp] + __popc(be & lt);
                node_end[id] = p + 1;
                node_last[id] = (L + 1 <= ev[q].e_hi) ? eid_below : GOTHIC_LEAF;
                eid_below = id;
            }
        }
    }
}

__global__ void __launch_bounds__(TPB) k_finish_nodes(uint32_t n_nodes, const uint32_t *__restrict__ node_head,
                                                       const uint32_t *__restrict__ node_end, const uint32_t *__restrict__ node_child,
                                                       const uint32_t *__restrict__ node_last, uint32_t *__restrict__ node_num,
                                                       uint8_t *__restrict__ node_nchild, uint32_t *__restrict__ node_parent)
{
    const uint32_t J = blockIdx.x * TPB + threadIdx.x;
    if (J >= n_nodes) return;
    const uint32_t h = node_head[J], num = node_end[J] - h;
    node_num[J] = num;
    const uint32_t c = node_child[J];
    uint32_t nc = 0;
    if (c != GOTHIC_LEAF) {
        nc = node_last[J] - c + 1u;
        for (uint32_t k = 0; k < nc; k++) node_parent[c + k] = J;
    }
    node_nchild[J] = (uint8_t)nc;
    if (J == 0) node_parent[0] = GOTHIC_LEAF;
}

// leaf_of / leaf_level of a particle: the PARENT of its leaf and that parent's level, which is where the radius climb of moments.cu starts
// (a leaf's own radius comes out of k_leaf_moments).  After k_finish_nodes, which writes the parent links.
__global__ void __launch_bounds__(TPB) k_leaf_links(uint32_t n_nodes, const uint32_t *__restrict__ node_head, const uint32_t *__restrict__ node_num,
                                                     const uint32_t *__restrict__ node_child, const uint32_t *__restrict__ node_parent,
                                                     const uint8_t *__restrict__ node_level, uint32_t *__restrict__ leaf_of, uint8_t *__restrict__ leaf_level)
{
    const uint32_t J = blockIdx.x * TPB + threadIdx.x;
    if (J >= n_nodes || node_child[J] != GOTHIC_LEAF) return;
    const uint32_t h = node_head[J], num = node_num[J], P = node_parent[J];
    const uint8_t lv = P == GOTHIC_LEAF ? (uint8_t)0xFFu : node_level[P];       // the tree is one leaf: nothing to climb
    for (uint32_t i = 0; i < num; i++) { leaf_of[h + i] = P; leaf_level[h + i] = lv; }
}

} // namespace

int gothic_stage_nodes(gothic_ctx *c, uint32_t n, int n_leaf, cudaStream_t s)
{
    const uint32_t nblk = (n + TILE - 1) / TILE;
    const uint64_t *key = c->key[c->cur];
    uint32_t *events = c->leaf_of;          // one word per key between the two passes; k_finish_nodes then overwrites it with the leaf ids
    // only the build's own overflow flag: flags[1] (the walk's stack overflow) stays set until gothic_check reads it, flags[2] is rewritten below
    GOTHIC_CUDA_OK(c, cudaMemsetAsync(c->flags, 0, sizeof(uint32_t), s));
    k_node_events<<<nblk, TPB, 0, s>>>(key, n, n_leaf, events, c->blk_cnt, nblk);
    GOTHIC_LAUNCH_OK(c);
    k_scan_blocks<<<2 * GOTHIC_NLEVP1, SCAN_TPB, 0, s>>>(c->blk_cnt, nblk, c->level_cnt);
    GOTHIC_LAUNCH_OK(c);
    k_level_offsets<<<1, 1, 0, s>>>(c->level_cnt, c->level_ofs, c->flags, c->node_max);
    GOTHIC_LAUNCH_OK(c);
    k_emit_nodes<<<nblk, TPB, 0, s>>>(events, n, c->blk_cnt, nblk, c->level_ofs, c->flags, c->node_head, c->node_level,
                                      c->node_child, c->node_end, c->node_last);
    GOTHIC_LAUNCH_OK(c);
    // the one host read of the build: node count + level offsets (sizes the remaining launches)
    uint32_t h_flags[4];
    GOTHIC_CUDA_OK(c, cudaMemcpyAsync(c->h_level_ofs, c->level_ofs, (GOTHIC_NLEVP1 + 1) * sizeof(uint32_t), cudaMemcpyDeviceToHost, s));
    GOTHIC_CUDA_OK(c, cudaMemcpyAsync(h_flags, c->flags, sizeof(h_flags), cudaMemcpyDeviceToHost, s));
    GOTHIC_CUDA_OK(c, cudaStreamSynchronize(s));
    if (h_flags[3]) {       // the keys are not fully sorted: nothing above can be trusted (sort_pairs.cu, gothic_build_tree repeats the build)
        GOTHIC_CUDA_OK(c, cudaMemsetAsync(c->flags + 3, 0, sizeof(uint32_t), s));
        GOTHIC_CUDA_OK(c, cudaMemsetAsync(c->flags, 0, sizeof(uint32_t), s));
        return GOTHIC_RETRY_FULL_SORT;
    }
    if (h_flags[0]) return GOTHIC_ERR_CAPACITY;
    c->n_nodes = h_flags[2];
    c->n_levels_tree = 0;
    for (int L = 0; L < GOTHIC_NLEVP1; L++)
        if (c->h_level_ofs[L + 1] > c->h_level_ofs[L]) c->n_levels_tree = L + 1;
    k_finish_nodes<<<(c->n_nodes + TPB - 1) / TPB, TPB, 0, s>>>(c->n_nodes, c->node_head, c->node_end, c->node_child, c->node_last,
                                                                c->node_num, c->node_nchild, c->node_parent);
    GOTHIC_LAUNCH_OK(c);
    k_leaf_links<<<(c->n_nodes + TPB - 1) / TPB, TPB, 0, s>>>(c->n_nodes, c->node_head, c->node_num, c->node_child, c->node_parent, c->node_level,
                                                              c->leaf_of, c->leaf_level);
    GOTHIC_LAUNCH_OK(c);
    return GOTHIC_OK;
}
