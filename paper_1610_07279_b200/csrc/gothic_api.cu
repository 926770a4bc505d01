// C-ABI entry points of libgothic_b200 (include/gothic.h).  Host logic only: argument checks, buffer
// ownership, stage sequencing.  Every step of the path runs in the kernels of the other translation units.
#include "gothic_ctx.cuh"
#include <new>
#include <string.h>

namespace {

template <typename T>
cudaError_t dev_alloc(T **p, size_t count)
{
    return cudaMalloc(reinterpret_cast<void **>(p), count * sizeof(T));
}

void free_all(gothic_ctx *c)
{
    void *ptrs[] = {c->key[0], c->key[1], c->idx[0], c->idx[1], c->items, c->box, c->bbox_bits,
                    c->node_head, c->node_num, c->node_child, c->node_parent, c->node_end, c->node_last,
                    c->node_level, c->node_nchild, c->node_com, c->node_msum, c->node_b, c->node_B2, c->node_b2bits, c->node_up, c->leaf_of, c->leaf_level,
                    c->level_ofs, c->level_cnt, c->blk_cnt, c->flags, c->sort_tmp, c->grp_mask, c->grp_list, c->grp_cnt,
                    c->stack, c->ts_tmp, c->scan_tmp, c->h2d_pos, c->h2d_aold, c->d_aold_sorted, c->d_acc,
                    c->h2d_acc, c->d_level, c->d_active, c->d_cycle_info, c->d_count};
    gothic_live_free(c);
    for (void *p : ptrs)
        if (p) cudaFree(p);
    if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
    if (c->copy_done) cudaEventDestroy(c->copy_done);
}

__global__ void k_gather_f32(const float *__restrict__ src, const uint32_t *__restrict__ perm, uint32_t n, float *__restrict__ dst)
{
    const uint32_t s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s < n) dst[s] = __ldg(src + __ldg(perm + s));
}

// sorted <- original: acc_sorted[s] = acc_orig[perm[s]], amag[s] = |a|
__global__ void k_gather_acc(const float4 *__restrict__ src, const uint32_t *__restrict__ perm, uint32_t n, float4 *__restrict__ dst,
                             float *__restrict__ amag)
{
    const uint32_t s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    const float4 a = __ldg(src + __ldg(perm + s));
    dst[s] = a;
    amag[s] = __fsqrt_rn(fmaf(a.z, a.z, fmaf(a.y, a.y, a.x * a.x)));
}

// original <- sorted: acc_orig[perm[s]] = acc_sorted[s], level_orig[perm[s]] = level_sorted[s]
__global__ void k_scatter_result(const float4 *__restrict__ acc_sorted, const uint8_t *__restrict__ level_sorted,
                                 const uint32_t *__restrict__ perm, uint32_t n, float4 *__restrict__ acc_orig, uint8_t *__restrict__ level_orig)
{
    const uint32_t s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    const uint32_t o = __ldg(perm + s);
    acc_orig[o] = acc_sorted[s];
    level_orig[o] = level_sorted[s];
}

} // namespace

extern "C" {

const char *gothic_strerror(int code)
{
    switch (code) {
    case GOTHIC_OK: return "ok";
    case GOTHIC_ERR_ARG: return "invalid argument";
    case GOTHIC_ERR_STATE: return "tree not built";
    case GOTHIC_ERR_CAPACITY: return "node pool or traversal stack capacity exceeded";
    case GOTHIC_ERR_CUDA: return "CUDA runtime error";
    case GOTHIC_ERR_UNIMPLEMENTED: return "not implemented";
    case GOTHIC_ERR_TOO_LARGE: return "n exceeds GOTHIC_STATIC_ACTIVE_MAX_N (the fixed scratch of gothic_active_list_static)";
    default: return "unknown error";
    }
}

const char *gothic_last_cuda_error(gothic_ctx *ctx)
{
    return ctx ? cudaGetErrorString(ctx->last_err) : "no context";
}

int gothic_create(gothic_ctx **out, uint32_t n_max, uint32_t node_max, int group_size, size_t scratch_bytes)
{
    if (!out || n_max == 0 || n_max > (1u << 30)) return GOTHIC_ERR_ARG;   // the sort's look-back words carry 30-bit prefixes
    if (group_size == 0) group_size = 32;
    if (group_size != 8 && group_size != 16 && group_size != 32) return GOTHIC_ERR_ARG;
    if (node_max == 0) {
        const unsigned long long d = 2ull * n_max + 64ull;
        node_max = d >= (1ull << 28) ? (1u << 28) - 1u : (uint32_t)d;
    }
    if (node_max >= (1u << 28)) return GOTHIC_ERR_ARG;
    gothic_ctx *c = new (std::nothrow) gothic_ctx;
    if (!c) return GOTHIC_ERR_ARG;
    memset(c, 0, sizeof(*c));
    c->n_max = n_max;
    c->node_max = node_max;
    c->group_size = group_size;
    c->last_err = cudaSuccess;
    *out = c;
    cudaError_t e = cudaGetDevice(&c->device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&c->num_sms, cudaDevAttrMultiProcessorCount, c->device);
    if (e != cudaSuccess) { c->last_err = e; delete c; *out = nullptr; return GOTHIC_ERR_CUDA; }
    if ((e = gothic_walk_config(c)) != cudaSuccess || (e = gothic_sort_config()) != cudaSuccess) { c->last_err = e; delete c; *out = nullptr; return GOTHIC_ERR_CUDA; }
    if (gothic_keys_config(c) != GOTHIC_OK) { delete c; *out = nullptr; return GOTHIC_ERR_CUDA; }
    c->stack_cap = 8192;   // u32 words of global spill area per resident warp (4096 families)
    if (scratch_bytes) {
        const size_t per = scratch_bytes / ((size_t)c->walk_warps * sizeof(uint32_t));
        if (per < 512) { delete c; *out = nullptr; return GOTHIC_ERR_ARG; }
        c->stack_cap = (uint32_t)(per > (1u << 20) ? (1u << 20) : per);
    }
    c->nblk_max = (n_max + 255u) / 256u;
    c->sort_tmp_bytes = gothic_sort_scratch_bytes(n_max);
    const size_t n_groups = ((size_t)n_max + group_size - 1) / group_size;
    const size_t n = n_max, m = node_max;
#define A(expr) if (e == cudaSuccess) e = (expr)
    A(dev_alloc(&c->key[0], n)); A(dev_alloc(&c->key[1], n));
    A(dev_alloc(&c->idx[0], n)); A(dev_alloc(&c->idx[1], n));
    A(dev_alloc(&c->items, n + 2 * m));   // sorted particles, then the node records (walk.cu: one item space)
    A(dev_alloc(&c->box, 8)); A(dev_alloc(&c->bbox_bits, 8));
    A(dev_alloc(&c->node_head, m)); A(dev_alloc(&c->node_num, m)); A(dev_alloc(&c->node_child, m));
    A(dev_alloc(&c->node_parent, m)); A(dev_alloc(&c->node_end, m)); A(dev_alloc(&c->node_last, m));
    A(dev_alloc(&c->node_level, m)); A(dev_alloc(&c->node_nchild, m));
    A(dev_alloc(&c->node_com, m)); A(dev_alloc(&c->node_msum, m)); A(dev_alloc(&c->node_b, m));
    A(dev_alloc(&c->node_b2bits, m)); A(dev_alloc(&c->node_B2, m)); A(dev_alloc(&c->node_up, m)); A(dev_alloc(&c->leaf_of, n)); A(dev_alloc(&c->leaf_level, n));
    A(dev_alloc(&c->level_ofs, GOTHIC_NLEVP1 + 2)); A(dev_alloc(&c->level_cnt, GOTHIC_NLEVP1 + 2));
    A(dev_alloc(&c->blk_cnt, (size_t)2 * GOTHIC_NLEVP1 * c->nblk_max));
    A(dev_alloc(&c->flags, 4));
    A(cudaMalloc(&c->sort_tmp, c->sort_tmp_bytes));
    A(dev_alloc(&c->grp_mask, n_groups)); A(dev_alloc(&c->grp_list, n_groups)); A(dev_alloc(&c->grp_cnt, 4));
    A(dev_alloc(&c->stack, (size_t)c->walk_warps * c->stack_cap));
    A(dev_alloc(&c->ts_tmp, 4)); A(dev_alloc(&c->scan_tmp, (n + 2047) / 2048 + 1));
    A(cudaMemset(c->flags, 0, 4 * sizeof(uint32_t)));
#undef A
    if (e == cudaSuccess) {
        c->pos_sorted = c->items;
        c->node_rec = reinterpret_cast<NodeRec *>(c->items + n);
    }
    if (e != cudaSuccess) {
        c->last_err = e;
        free_all(c);
        delete c;
        *out = nullptr;
        return GOTHIC_ERR_CUDA;
    }
    return GOTHIC_OK;
}

void gothic_destroy(gothic_ctx *ctx)
{
    if (!ctx) return;
    free_all(ctx);
    delete ctx;
}

int gothic_set_ball(gothic_ctx *ctx, int ball_kind)
{
    if (!ctx || (ball_kind < GOTHIC_BALL_GEO || ball_kind > GOTHIC_BALL_SEB)) return GOTHIC_ERR_ARG;
    ctx->ball_kind = ball_kind;
    return GOTHIC_OK;
}

unsigned long long gothic_launch_count(gothic_ctx *ctx) { return ctx ? ctx->launches : 0ull; }

int gothic_build_tree(gothic_ctx *c, const float *pos_m, uint32_t n, int key_kind, int n_leaf, void *stream)
{
    if (!c || !pos_m || n == 0 || n > c->n_max) return GOTHIC_ERR_ARG;
    if (key_kind != GOTHIC_KEY_PEANO_HILBERT && key_kind != GOTHIC_KEY_MORTON) return GOTHIC_ERR_ARG;
    if (n_leaf == 0) n_leaf = 16;
    if (n_leaf < 1 || n_leaf > GOTHIC_MAX_NLEAF) return GOTHIC_ERR_ARG;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const float4 *pos = reinterpret_cast<const float4 *>(pos_m);
    c->built = false;
    c->n = n;
    c->n_leaf = n_leaf;
    int rc;
    for (int full = 0; full < 2; full++) {      // second round only if the five-pass sort met a long unordered run (sort_pairs.cu)
        if ((rc = gothic_stage_keys(c, pos, n, key_kind, s)) != GOTHIC_OK) return rc;
        if ((rc = gothic_stage_sort(c, n, full != 0, s)) != GOTHIC_OK) return rc;
        if ((rc = gothic_stage_gather(c, pos, n, s)) != GOTHIC_OK) return rc;
        if ((rc = gothic_stage_nodes(c, n, n_leaf, s)) != GOTHIC_RETRY_FULL_SORT) break;
    }
    if (rc != GOTHIC_OK) return rc == GOTHIC_RETRY_FULL_SORT ? GOTHIC_ERR_STATE : rc;
    if ((rc = gothic_stage_moments(c, s)) != GOTHIC_OK) return rc;
    c->built = true;
    c->tree_gen++;
    return GOTHIC_OK;
}

int gothic_update_moments(gothic_ctx *c, const float *pos_m_sorted, void *stream)
{
    if (!c) return GOTHIC_ERR_ARG;
    if (!c->built) return GOTHIC_ERR_STATE;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    if (pos_m_sorted && pos_m_sorted != reinterpret_cast<const float *>(c->pos_sorted))
        GOTHIC_CUDA_OK(c, cudaMemcpyAsync(c->pos_sorted, pos_m_sorted, (size_t)c->n * sizeof(float4), cudaMemcpyDeviceToDevice, s));
    return gothic_stage_moments(c, s);
}

int gothic_walk_tree(gothic_ctx *c, const uint32_t *active, uint32_t n_active, const uint32_t *n_active_dev,
                     float eps, int mac_kind, float mac_param, float r_crit, const float *aold,
                     float *acc_pot, float *amag_out, unsigned long long *n_interactions, void *stream)
{
    if (!c || !acc_pot || !(eps > 0.0f) || !(mac_param >= 0.0f) || !(r_crit >= 0.0f)) return GOTHIC_ERR_ARG;
    if (mac_kind != GOTHIC_MAC_ACCELERATION && mac_kind != GOTHIC_MAC_OPENING_ANGLE && mac_kind != GOTHIC_MAC_MULTIPOLE) return GOTHIC_ERR_ARG;
    if (mac_kind == GOTHIC_MAC_ACCELERATION && !aold) return GOTHIC_ERR_ARG;
    if (!c->built) return GOTHIC_ERR_STATE;
    if (active && !n_active_dev && n_active > c->n) return GOTHIC_ERR_ARG;
    if (active && !n_active_dev && n_active == 0) return GOTHIC_OK;
    return gothic_stage_walk(c, active, n_active, n_active_dev, eps, mac_kind, mac_param, r_crit, aold,
                             reinterpret_cast<float4 *>(acc_pot), amag_out, n_interactions, static_cast<cudaStream_t>(stream));
}

int gothic_set_timesteps(gothic_ctx *c, const float *acc_pot, uint32_t n, float eps, float eta, int max_levels,
                         uint32_t substep, uint8_t *level, uint32_t *active, uint32_t *n_active_dev,
                         int32_t *emin_nlev_dev, void *stream)
{
    if (!c || !level || n == 0 || n > c->n_max) return GOTHIC_ERR_ARG;
    if (max_levels < 1 || max_levels > 32 || substep == 0) return GOTHIC_ERR_ARG;
    if ((active == nullptr) != (n_active_dev == nullptr)) return GOTHIC_ERR_ARG;
    if (acc_pot && (!(eps > 0.0f) || !(eta > 0.0f))) return GOTHIC_ERR_ARG;
    // c = (float)(eta^4 eps^2), formed once in double then rounded (R6)
    const double e4 = (double)eta * (double)eta * (double)eta * (double)eta;
    const float cconst = (float)(e4 * (double)eps * (double)eps);
    return gothic_stage_timesteps(c, reinterpret_cast<const float4 *>(acc_pot), n, cconst, max_levels, substep, level, active,
                                  n_active_dev, emin_nlev_dev, static_cast<cudaStream_t>(stream));
}

int gothic_check(gothic_ctx *c, void *stream)
{
    if (!c) return GOTHIC_ERR_ARG;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    uint32_t h[4];
    GOTHIC_CUDA_OK(c, cudaMemcpyAsync(h, c->flags, sizeof(h), cudaMemcpyDeviceToHost, s));
    GOTHIC_CUDA_OK(c, cudaStreamSynchronize(s));
    if (h[0] || h[1]) {
        const uint32_t zero[2] = {0u, 0u};
        cudaMemcpyAsync(c->flags, zero, sizeof(zero), cudaMemcpyHostToDevice, s);
        cudaStreamSynchronize(s);
        return GOTHIC_ERR_CAPACITY;
    }
    return GOTHIC_OK;
}

int gothic_get_tree_view(gothic_ctx *c, gothic_tree_view *out, void *stream)
{
    if (!c || !out) return GOTHIC_ERR_ARG;
    if (!c->built) return GOTHIC_ERR_STATE;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    {
        const int rcb = gothic_stage_need_b2(c, s);      // the view exposes B_2 (eq. 4)
        if (rcb != GOTHIC_OK) return rcb;
    }
    float hbox[8];
    GOTHIC_CUDA_OK(c, cudaMemcpyAsync(hbox, c->box, sizeof(hbox), cudaMemcpyDeviceToHost, s));
    const int rc = gothic_check(c, stream);
    if (rc != GOTHIC_OK) return rc;
    out->n = c->n;
    out->n_nodes = c->n_nodes;
    out->n_levels_tree = c->n_levels_tree;
    out->group_size = (uint32_t)c->group_size;
    for (int k = 0; k < 4; k++) out->box[k] = hbox[k];
    out->key = c->key[c->cur];
    out->perm = c->idx[c->cur];
    out->pos_m_sorted = reinterpret_cast<const float *>(c->pos_sorted);
    out->node_head = c->node_head; out->node_num = c->node_num; out->node_child = c->node_child;
    out->node_level = c->node_level; out->node_nchild = c->node_nchild;
    out->level_ofs = c->level_ofs;
    out->node_com = reinterpret_cast<const float *>(c->node_com);
    out->node_b = c->node_b;
    out->node_b2 = c->node_B2;
    return GOTHIC_OK;
}

int gothic_gravity_host(gothic_ctx *c, const float *pos_m_host, uint32_t n, int key_kind, int n_leaf,
                        float eps, int mac_kind, float mac_param, float r_crit, const float *aold_host,
                        float *acc_pot_host, uint32_t *perm_host, void *stream)
{
    if (!c || !pos_m_host || !acc_pot_host || n == 0 || n > c->n_max) return GOTHIC_ERR_ARG;
    if (mac_kind == GOTHIC_MAC_ACCELERATION && !aold_host) return GOTHIC_ERR_ARG;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    if (!c->h2d_pos) {
        cudaError_t e = dev_alloc(&c->h2d_pos, c->n_max);
        if (e == cudaSuccess) e = dev_alloc(&c->h2d_aold, c->n_max);
        if (e == cudaSuccess) e = dev_alloc(&c->d_aold_sorted, c->n_max);
        if (e == cudaSuccess) e = dev_alloc(&c->d_acc, c->n_max);
        if (e != cudaSuccess) { c->last_err = e; return GOTHIC_ERR_CUDA; }
    }
    GOTHIC_CUDA_OK(c, cudaMemcpyAsync(c->h2d_pos, pos_m_host, (size_t)n * sizeof(float4), cudaMemcpyHostToDevice, s));
    if (aold_host)
        GOTHIC_CUDA_OK(c, cudaMemcpyAsync(c->h2d_aold, aold_host, (size_t)n * sizeof(float), cudaMemcpyHostToDevice, s));
    int rc = gothic_build_tree(c, reinterpret_cast<const float *>(c->h2d_pos), n, key_kind, n_leaf, stream);
    if (rc != GOTHIC_OK) return rc;
    if (aold_host) {
        k_gather_f32<<<(n + 255u) / 256u, 256, 0, s>>>(c->h2d_aold, c->idx[c->cur], n, c->d_aold_sorted);
        GOTHIC_LAUNCH_OK(c);
    }
    rc = gothic_walk_tree(c, nullptr, 0, nullptr, eps, mac_kind, mac_param, r_crit, aold_host ? c->d_aold_sorted : nullptr,
                          reinterpret_cast<float *>(c->d_acc), nullptr, nullptr, stream);
    if (rc != GOTHIC_OK) return rc;
    GOTHIC_CUDA_OK(c, cudaMemcpyAsync(acc_pot_host, c->d_acc, (size_t)n * sizeof(float4), cudaMemcpyDeviceToHost, s));
    if (perm_host)
        GOTHIC_CUDA_OK(c, cudaMemcpyAsync(perm_host, c->idx[c->cur], (size_t)n * sizeof(uint32_t), cudaMemcpyDeviceToHost, s));
    return gothic_check(c, stream);
}

int gothic_block_cycle_host(gothic_ctx *c, const float *pos_m_host, const float *acc_prev_host, uint32_t n, int key_kind, int n_leaf,
                            float eps, float eta, int max_levels, float delta_acc, float r_crit, float *acc_pot_host, uint8_t *level_host,
                            int32_t *info_host, unsigned long long *n_interactions_host, void *stream)
{
    if (!c || !pos_m_host || !acc_prev_host || !acc_pot_host || n == 0 || n > c->n_max) return GOTHIC_ERR_ARG;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    if (!c->h2d_pos) {
        cudaError_t e = dev_alloc(&c->h2d_pos, c->n_max);
        if (e == cudaSuccess) e = dev_alloc(&c->h2d_aold, c->n_max);
        if (e == cudaSuccess) e = dev_alloc(&c->d_aold_sorted, c->n_max);
        if (e == cudaSuccess) e = dev_alloc(&c->d_acc, c->n_max);
        if (e != cudaSuccess) { c->last_err = e; return GOTHIC_ERR_CUDA; }
    }
    if (!c->h2d_acc) {
        cudaError_t e = dev_alloc(&c->h2d_acc, c->n_max);
        if (e == cudaSuccess) e = dev_alloc(&c->d_level, 2 * (size_t)c->n_max);
        if (e == cudaSuccess) e = dev_alloc(&c->d_active, c->n_max);
        if (e == cudaSuccess) e = dev_alloc(&c->d_cycle_info, 4);
        if (e == cudaSuccess) e = dev_alloc(&c->d_count, 1);
        if (e != cudaSuccess) { c->last_err = e; return GOTHIC_ERR_CUDA; }
    }
    const size_t b4 = (size_t)n * sizeof(float4);
    if (!c->copy_stream) {
        GOTHIC_CUDA_OK(c, cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking));
        GOTHIC_CUDA_OK(c, cudaEventCreateWithFlags(&c->copy_done, cudaEventDisableTiming));
    }
    // the build needs only the positions: the previous accelerations travel on a second queue while the tree is built
    GOTHIC_CUDA_OK(c, cudaMemcpyAsync(c->h2d_pos, pos_m_host, b4, cudaMemcpyHostToDevice, s));
    GOTHIC_CUDA_OK(c, cudaEventRecord(c->copy_done, s));
    GOTHIC_CUDA_OK(c, cudaStreamWaitEvent(c->copy_stream, c->copy_done, 0));     // after the positions (one H2D engine) and after earlier work on s
    GOTHIC_CUDA_OK(c, cudaMemcpyAsync(c->h2d_acc, acc_prev_host, b4, cudaMemcpyHostToDevice, c->copy_stream));
    GOTHIC_CUDA_OK(c, cudaEventRecord(c->copy_done, c->copy_stream));
    int rc = gothic_build_tree(c, reinterpret_cast<const float *>(c->h2d_pos), n, key_kind, n_leaf, stream);
    if (rc != GOTHIC_OK) { cudaStreamSynchronize(c->copy_stream); return rc; }      // the caller's buffer is still being read
    GOTHIC_CUDA_OK(c, cudaStreamWaitEvent(s, c->copy_done, 0));
    const uint32_t grid = (n + 255u) / 256u;
    float *amag = c->d_aold_sorted;
    uint8_t *level = c->d_level, *level_orig = c->d_level + c->n_max;
    uint32_t *n_active_dev = reinterpret_cast<uint32_t *>(c->d_cycle_info) + 2;
    k_gather_acc<<<grid, 256, 0, s>>>(c->h2d_acc, c->idx[c->cur], n, c->d_acc, amag);
    GOTHIC_LAUNCH_OK(c);
    rc = gothic_set_timesteps(c, reinterpret_cast<const float *>(c->d_acc), n, eps, eta, max_levels, 1u, level, nullptr, nullptr,
                              c->d_cycle_info, stream);
    if (rc != GOTHIC_OK) return rc;
    int32_t emin_nlev[2];
    GOTHIC_CUDA_OK(c, cudaMemcpyAsync(emin_nlev, c->d_cycle_info, sizeof(emin_nlev), cudaMemcpyDeviceToHost, s));
    GOTHIC_CUDA_OK(c, cudaStreamSynchronize(s));
    const int n_levels = emin_nlev[1];
    if (n_levels < 1 || n_levels > max_levels) return GOTHIC_ERR_STATE;
    const uint32_t n_sub = 1u << (n_levels - 1);
    if (n_interactions_host) GOTHIC_CUDA_OK(c, cudaMemsetAsync(c->d_count, 0, sizeof(unsigned long long), s));
    for (uint32_t sub = 1; sub <= n_sub; sub++) {
        rc = gothic_set_timesteps(c, nullptr, n, eps, eta, max_levels, sub, level, c->d_active, n_active_dev, nullptr, stream);
        if (rc != GOTHIC_OK) return rc;
        rc = gothic_update_moments(c, nullptr, stream);   // the paper recomputes the pseudo j-particles every step
        if (rc != GOTHIC_OK) return rc;
        rc = gothic_walk_tree(c, c->d_active, 0, n_active_dev, eps, GOTHIC_MAC_ACCELERATION, delta_acc, r_crit, amag,
                              reinterpret_cast<float *>(c->d_acc), amag, n_interactions_host ? c->d_count : nullptr, stream);
        if (rc != GOTHIC_OK) return rc;
    }
    k_scatter_result<<<grid, 256, 0, s>>>(c->d_acc, level, c->idx[c->cur], n, c->h2d_acc, level_orig);
    GOTHIC_LAUNCH_OK(c);
    GOTHIC_CUDA_OK(c, cudaMemcpyAsync(acc_pot_host, c->h2d_acc, b4, cudaMemcpyDeviceToHost, s));
    if (level_host) GOTHIC_CUDA_OK(c, cudaMemcpyAsync(level_host, level_orig, n, cudaMemcpyDeviceToHost, s));
    if (n_interactions_host)
        GOTHIC_CUDA_OK(c, cudaMemcpyAsync(n_interactions_host, c->d_count, sizeof(unsigned long long), cudaMemcpyDeviceToHost, s));
    if (info_host) { info_host[0] = emin_nlev[0]; info_host[1] = n_levels; info_host[2] = (int32_t)n_sub; info_host[3] = 0; }
    return gothic_check(c, stream);
}

} // extern "C"
