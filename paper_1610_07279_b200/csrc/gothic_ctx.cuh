// Internal context + helpers shared by the CUDA translation units of libgothic_b200 (sm_100a only).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include "../../include/gothic.h"

#define GOTHIC_NLEV 21          // 21 bits per axis -> 63-bit key (R1)
#define GOTHIC_NLEVP1 22        // tree levels 0..21
#define GOTHIC_LEAF 0xFFFFFFFFu
#define GOTHIC_MAX_NLEAF 64

// 32-byte node record read by the walk: one sector per MAC test.  Sorted particles and node records share one
// array of 16-byte items (particle s = item s, node J = items n_max + 2J and n_max + 2J + 1), and (w0, w1) is the
// FAMILY the walk pushes when it opens the node: first item, count | particles << 31.
struct __align__(16) NodeRec {
    float x, y, z, m;   // r_J, m_J
    float mb2;          // (m_J * b_J) * b_J (eq. 5 right-hand side, G = 1); 3 B_2 while the multipole MAC is in use (eq. 3)
    float b;            // b_J
    uint32_t w0;        // internal: item of the first child's record (n_max + 2 * child) | leaf: head (sorted index of first particle)
    uint32_t w1;        // internal: number of children                                    | leaf: 0x80000000 | num
};

struct gothic_ctx {
    uint32_t n_max, node_max;
    int group_size;
    int ball_kind;         // enclosing ball of the pseudo i-particle: GOTHIC_BALL_GEO (default) or GOTHIC_BALL_EBS
    int n_leaf;
    int device;
    int num_sms;
    int radius_blocks_per_sm;   // resident CTAs of k_node_radius per SM, asked of the runtime once (0 = not yet)
    // state of the last build
    uint32_t n;
    uint32_t n_nodes;
    uint32_t n_levels_tree;
    uint32_t h_level_ofs[GOTHIC_NLEVP1 + 1];
    bool built;
    unsigned long long tree_gen;   // number of successful gothic_build_tree calls: lets gothic_live_step see a build that was not its own
    unsigned long long launches;
    cudaError_t last_err;
    // device buffers
    uint64_t *key[2];      // double buffer for the sort
    uint32_t *idx[2];
    int cur;               // which half holds the sorted result
    float4 *items;         // [n_max + 2 * node_max]: one allocation, item space of the walk
    float4 *pos_sorted;    // = items
    float *box;            // [8]: xmin, ymin, zmin, side, scale, -, -, -
    uint32_t *bbox_bits;   // [6] ordered-int min/max accumulators
    // nodes
    uint32_t *node_head, *node_num, *node_child, *node_parent, *node_end, *node_last;
    uint8_t *node_level, *node_nchild;
    float4 *node_com, *node_msum;
    float4 *node_up;       // (r_J, parent id as bits): one 16-byte load per level of the radius climb
    uint32_t *leaf_of;     // [n_max] leaf node of every sorted particle
    uint8_t *leaf_level;   // [n_max] and its level
    float *node_b;
    float *node_B2;        // eq. 4: sum_j m_j |r_j - r_J|^2 (multipole MAC)
    bool b2_enabled;       // the moments passes of this context also compute B_2
    int rec_slot4;         // what NodeRec::mb2 holds now: GOTHIC_MAC_ACCELERATION -> m b^2, GOTHIC_MAC_MULTIPOLE -> 3 B_2
    uint32_t *node_b2bits;
    NodeRec *node_rec;     // = items + n_max
    uint32_t *level_ofs;   // [23]
    uint32_t *level_cnt;   // [22]
    uint32_t *blk_cnt;     // [2][22][nblk_max] per-block start/end event counts
    uint32_t nblk_max;
    uint32_t *flags;       // [4]: 0 = capacity overflow (nodes), 1 = stack overflow, 2 = n_nodes, 3 = the fast sort needs the full passes
    // sort scratch
    void *sort_tmp;
    size_t sort_tmp_bytes;
    // walk
    uint32_t *grp_mask;    // [ceil(n_max/G)]
    uint32_t *grp_list;    // [ceil(n_max/G)]
    uint32_t *grp_cnt;     // [4]: 0 = number of non-empty groups, 1 = work counter
    uint32_t *stack;       // per-warp global spill areas of the traversal stacks
    uint32_t stack_cap;    // u32 words per warp (2 per family)
    uint32_t walk_warps;   // resident warps of the persistent walk grid
    // time steps
    int32_t *ts_tmp;       // [4]: emin, lmax
    uint32_t *scan_tmp;    // block counts for ordered compaction
    // host staging for gothic_gravity_host
    float4 *h2d_pos; float *h2d_aold; float *d_aold_sorted; float4 *d_acc;
    cudaStream_t copy_stream; cudaEvent_t copy_done;   // second copy queue of gothic_block_cycle_host (overlaps H2D with the build)
    // extra staging for gothic_block_cycle_host
    float4 *h2d_acc; uint8_t *d_level; uint32_t *d_active; int32_t *d_cycle_info; unsigned long long *d_count;
    struct gothic_live *live;   // state of gothic_live_* (integrate.cu), NULL until gothic_live_init
};
void gothic_live_free(gothic_ctx *c);

#define GOTHIC_CUDA_OK(ctx, expr)                                   \
    do {                                                            \
        cudaError_t _e = (expr);                                    \
        if (_e != cudaSuccess) { (ctx)->last_err = _e; return GOTHIC_ERR_CUDA; } \
    } while (0)

#define GOTHIC_LAUNCH_OK(ctx)                                       \
    do {                                                            \
        (ctx)->launches++;                                          \
        cudaError_t _e = cudaGetLastError();                        \
        if (_e != cudaSuccess) { (ctx)->last_err = _e; return GOTHIC_ERR_CUDA; } \
    } while (0)

// ---- stage entry points (each in its own .cu) --------------------------------------------------------
int gothic_stage_keys(gothic_ctx *c, const float4 *pos_m, uint32_t n, int key_kind, cudaStream_t s);
int gothic_stage_sort(gothic_ctx *c, uint32_t n, bool full, cudaStream_t s);   // full = all 8 digit passes (the retry of gothic_build_tree)
#define GOTHIC_RETRY_FULL_SORT 1     // internal return of gothic_stage_nodes: the fast sort left a long run unordered (flags[3])
size_t gothic_sort_scratch_bytes(uint32_t n_max);
int gothic_keys_config(gothic_ctx *c);     // uploads the Peano-Hilbert state table (called by gothic_create)
cudaError_t gothic_sort_config();         // per-device function attributes of the sort kernels (called by gothic_create)
int gothic_stage_gather(gothic_ctx *c, const float4 *pos_m, uint32_t n, cudaStream_t s);
int gothic_stage_nodes(gothic_ctx *c, uint32_t n, int n_leaf, cudaStream_t s);
int gothic_stage_moments(gothic_ctx *c, cudaStream_t s);
int gothic_stage_need_b2(gothic_ctx *c, cudaStream_t s);   // computes B_2 now if this context has not been asked for it before
int gothic_stage_rec_slot4(gothic_ctx *c, int mac_kind, cudaStream_t s);   // switches NodeRec::mb2 between m b^2 and 3 B_2
int gothic_stage_walk(gothic_ctx *c, const uint32_t *active, uint32_t n_active, const uint32_t *n_active_dev,
                      float eps, int mac_kind, float mac_param, float r_crit, const float *aold, float4 *acc_pot,
                      float *amag_out, unsigned long long *n_inter, cudaStream_t s);
int gothic_stage_timesteps(gothic_ctx *c, const float4 *acc_pot, uint32_t n, float cconst, int max_levels,
                           uint32_t substep, uint8_t *level, uint32_t *active, uint32_t *n_active_dev,
                           int32_t *emin_nlev_dev, cudaStream_t s);
cudaError_t gothic_walk_config(gothic_ctx *c);   // function attributes + walk_warps (needs device properties)

// ---- small device helpers -----------------------------------------------------------------------------
__device__ __forceinline__ int shared_digits(uint64_t a, uint64_t b)
{
    // number of leading octal digits (of 21) shared by two 63-bit keys
    const uint64_t x = a ^ b;
    return x == 0 ? GOTHIC_NLEV : (__clzll((long long)x) - 1) / 3;
}
__device__ __forceinline__ uint32_t lane_id() { return threadIdx.x & 31u; }
