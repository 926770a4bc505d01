// Orbit integration under block time steps (eq. 15-17; NEXT row f1): prediction of all j-particles to the
// current time and correction of the active i-particles, with the level migration of DESIGN.md R15.  Both kernels are pure
// streaming passes (HBM bound): predict reads 52 B and writes 16 B per particle; correct touches only the active rows.
// Arithmetic order is part of the contract (bit-exact against the oracle): one fmaf per component, as written.
// gothic_live_* (below) strings them together with the build / moments / active-list / walk stages into the paper's per-step loop with
// moving particles: host sequencing only, the state rows stay on the device in tree order.
#include "gothic_ctx.cuh"
#include <math.h>
#include <new>
#include <string.h>

namespace {

constexpr int TPB = 256;

// same arithmetic as timesteps.cu (R6): exponent of dt = floor(ilogb(c / |a|^2) / 4)
__device__ __forceinline__ int dt_exponent(float4 a, float c)
{
    const float a2 = fmaf(a.z, a.z, fmaf(a.y, a.y, __fmul_rn(a.x, a.x)));
    if (!(a2 > 0.0f)) return 127;
    const float q = __fdiv_rn(c, a2);
    const uint32_t u = __float_as_uint(q);
    const int ex = (int)((u >> 23) & 0xffu);
    const uint32_t man = u & 0x7fffffu;
    if (ex == 0xff) return 127;
    int e;
    if (ex) e = ex - 127;
    else if (man) e = (31 - __clz(man)) - 149;
    else return -38;
    return e >> 2;
}

__global__ void __launch_bounds__(TPB) k_predict(const float4 *__restrict__ pos, const float4 *__restrict__ vel, const float4 *__restrict__ acc,
                                                 const uint32_t *__restrict__ t_last, uint32_t t_now, float dt_unit, uint32_t n,
                                                 float4 *__restrict__ pos_pred)
{
    const uint32_t j = blockIdx.x * TPB + threadIdx.x;
    if (j >= n) return;
    const float4 r = __ldg(pos + j), v = __ldg(vel + j), a = __ldg(acc + j);
    const float dt = __fmul_rn((float)(t_now - __ldg(t_last + j)), dt_unit);
    const float h = __fmul_rn(0.5f, dt);
    const float vx = fmaf(h, a.x, v.x), vy = fmaf(h, a.y, v.y), vz = fmaf(h, a.z, v.z);      // eq. 15
    pos_pred[j] = make_float4(fmaf(dt, vx, r.x), fmaf(dt, vy, r.y), fmaf(dt, vz, r.z), r.w);  // eq. 16
}

__global__ void __launch_bounds__(TPB) k_correct(const uint32_t *__restrict__ active, uint32_t n_active, const uint32_t *__restrict__ n_active_dev,
                                                 const float4 *__restrict__ pos_pred, const float4 *__restrict__ acc_new, uint32_t t_now,
                                                 float dt_unit, float4 *__restrict__ pos, float4 *__restrict__ vel, float4 *__restrict__ acc,
                                                 uint32_t *__restrict__ t_last, uint8_t *__restrict__ level, float c, int e_min, int max_levels)
{
    const uint32_t na = n_active_dev ? *n_active_dev : n_active;
    for (uint32_t q = blockIdx.x * TPB + threadIdx.x; q < na; q += gridDim.x * TPB) {
        const uint32_t i = active ? __ldg(active + q) : q;
        const float4 v = vel[i], a0 = acc[i], a1 = __ldg(acc_new + i);
        const float dt = __fmul_rn((float)(t_now - t_last[i]), dt_unit);
        const float h = __fmul_rn(0.5f, dt);
        const float vx = fmaf(h, a1.x, fmaf(h, a0.x, v.x));                                    // eq. 15 then eq. 17
        const float vy = fmaf(h, a1.y, fmaf(h, a0.y, v.y));
        const float vz = fmaf(h, a1.z, fmaf(h, a0.z, v.z));
        vel[i] = make_float4(vx, vy, vz, v.w);
        pos[i] = __ldg(pos_pred + i);
        acc[i] = a1;
        t_last[i] = t_now;
        if (level) {                                                                           // reading R15
            int want = dt_exponent(a1, c) - e_min;
            want = max(0, min(want, max_levels - 1));
            const int cur = level[i];
            if (want < cur) level[i] = (uint8_t)want;
            else if (want > cur && (t_now & ((2u << cur) - 1u)) == 0u) level[i] = (uint8_t)(cur + 1);
        }
    }
}

// state rows into the order of a new build: row s of the new order is row perm[s] of the old one
__global__ void __launch_bounds__(TPB) k_permute_state(const uint32_t *__restrict__ perm, uint32_t n, const float4 *__restrict__ pos0,
                                                       const float4 *__restrict__ vel0, const float4 *__restrict__ acc0, const float *__restrict__ amag0,
                                                       const uint32_t *__restrict__ tl0, const uint8_t *__restrict__ lev0, const uint32_t *__restrict__ orig0,
                                                       float4 *__restrict__ pos1, float4 *__restrict__ vel1, float4 *__restrict__ acc1, float *__restrict__ amag1,
                                                       uint32_t *__restrict__ tl1, uint8_t *__restrict__ lev1, uint32_t *__restrict__ orig1)
{
    const uint32_t s = blockIdx.x * TPB + threadIdx.x;
    if (s >= n) return;
    const uint32_t o = __ldg(perm + s);
    pos1[s] = __ldg(pos0 + o); vel1[s] = __ldg(vel0 + o); acc1[s] = __ldg(acc0 + o); amag1[s] = __ldg(amag0 + o);
    tl1[s] = __ldg(tl0 + o); lev1[s] = __ldg(lev0 + o); orig1[s] = orig0 ? __ldg(orig0 + o) : o;
}

__global__ void __launch_bounds__(TPB) k_gather_vel(const uint32_t *__restrict__ perm, uint32_t n, const float4 *__restrict__ vel0, float4 *__restrict__ vel1)
{
    const uint32_t s = blockIdx.x * TPB + threadIdx.x;
    if (s < n) vel1[s] = __ldg(vel0 + __ldg(perm + s));
}

} // namespace

// Device state of gothic_live_*: two copies of every row array (a rebuild writes the re-ordered rows into the other copy).
struct gothic_live {
    uint32_t n;
    int cur;                                  // which copy is the state
    float4 *pos[2], *vel[2], *acc[2];
    float *amag[2];
    uint32_t *t_last[2], *orig[2];
    uint8_t *level[2];
    float4 *pred, *acc_new;                   // predicted positions (rebuild steps only) and the walk's output
    uint32_t *active, *n_active;
    int32_t *info_dev;                        // {e_min, n_levels}
    uint32_t t_now, n_sub, steps_since_rebuild;
    unsigned long long steps;
    int e_min, n_levels;
    int key_kind, n_leaf, max_levels;
    float eps, eta;
    cudaEvent_t ev[3];                        // recorded by every step: start, after the tree stage, after the walk (gothic_live_timing)
    bool timed;                               // the last step recorded all three
    bool ready;                               // set at the end of gothic_live_init, cleared by any stage that fails: the rows may then be half-way through a step
    unsigned long long tree_gen;              // c->tree_gen after the live run's own last build
};

void gothic_live_free(gothic_ctx *c)
{
    gothic_live *L = c->live;
    if (!L) return;
    for (int k = 0; k < 2; k++) {
        void *ptrs[] = {L->pos[k], L->vel[k], L->acc[k], L->amag[k], L->t_last[k], L->orig[k], L->level[k]};
        for (void *p : ptrs)
            if (p) cudaFree(p);
    }
    void *ptrs[] = {L->pred, L->acc_new, L->active, L->n_active, L->info_dev};
    for (void *p : ptrs)
        if (p) cudaFree(p);
    for (cudaEvent_t e : L->ev)
        if (e) cudaEventDestroy(e);
    delete L;
    c->live = nullptr;
}

namespace {

float timestep_constant(float eps, float eta)      // c = (float)(eta^4 eps^2), formed once in double then rounded (R6)
{
    const double e4 = (double)eta * (double)eta * (double)eta * (double)eta;
    return (float)(e4 * (double)eps * (double)eps);
}

// levels from the current accelerations and the cycle clock back to zero; one small read-back
int live_new_cycle(gothic_ctx *c, gothic_live *L, cudaStream_t s)
{
    const int k = L->cur;
    int rc = gothic_stage_timesteps(c, L->acc[k], L->n, timestep_constant(L->eps, L->eta), L->max_levels, 1u, L->level[k], nullptr, nullptr, L->info_dev, s);
    if (rc != GOTHIC_OK) return rc;
    GOTHIC_CUDA_OK(c, cudaMemsetAsync(L->t_last[k], 0, (size_t)L->n * sizeof(uint32_t), s));
    int32_t h[2];
    GOTHIC_CUDA_OK(c, cudaMemcpyAsync(h, L->info_dev, sizeof(h), cudaMemcpyDeviceToHost, s));
    GOTHIC_CUDA_OK(c, cudaStreamSynchronize(s));
    if (h[1] < 1 || h[1] > L->max_levels) return GOTHIC_ERR_STATE;
    L->e_min = h[0];
    L->n_levels = h[1];
    L->n_sub = 1u << (h[1] - 1);
    L->t_now = 0;
    return GOTHIC_OK;
}

// the stages of one block step; the clock and the step count are committed only after the last launch has been accepted
int live_step_stages(gothic_ctx *c, gothic_live *L, float delta_acc, float r_crit, int rebuild, unsigned long long *n_interactions, void *stream)
{
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const uint32_t n = L->n, grid = (n + TPB - 1) / TPB;
    const float dt_unit = ldexpf(1.0f, L->e_min);
    int rc;
    const uint32_t t_next = L->t_now + 1u;
    int k = L->cur;
    L->timed = false;
    GOTHIC_CUDA_OK(c, cudaEventRecord(L->ev[0], s));
    if (rebuild) {
        // predicted positions in the old order -> new tree (whose gathered copy is the prediction in the new order) -> rows re-ordered
        k_predict<<<grid, TPB, 0, s>>>(L->pos[k], L->vel[k], L->acc[k], L->t_last[k], t_next, dt_unit, n, L->pred);
        GOTHIC_LAUNCH_OK(c);
        if ((rc = gothic_build_tree(c, reinterpret_cast<const float *>(L->pred), n, L->key_kind, L->n_leaf, stream)) != GOTHIC_OK) return rc;
        L->tree_gen = c->tree_gen;
        k_permute_state<<<grid, TPB, 0, s>>>(c->idx[c->cur], n, L->pos[k], L->vel[k], L->acc[k], L->amag[k], L->t_last[k], L->level[k], L->orig[k],
                                              L->pos[k ^ 1], L->vel[k ^ 1], L->acc[k ^ 1], L->amag[k ^ 1], L->t_last[k ^ 1], L->level[k ^ 1], L->orig[k ^ 1]);
        GOTHIC_LAUNCH_OK(c);
        k = L->cur = k ^ 1;
        L->steps_since_rebuild = 0;
    } else {
        // the prediction goes straight into the tree's particle array; links stay, moments are recomputed
        k_predict<<<grid, TPB, 0, s>>>(L->pos[k], L->vel[k], L->acc[k], L->t_last[k], t_next, dt_unit, n, c->pos_sorted);
        GOTHIC_LAUNCH_OK(c);
        if ((rc = gothic_stage_moments(c, s)) != GOTHIC_OK) return rc;
        L->steps_since_rebuild += 1u;
    }
    GOTHIC_CUDA_OK(c, cudaEventRecord(L->ev[1], s));
    const float cconst = timestep_constant(L->eps, L->eta);
    if ((rc = gothic_stage_timesteps(c, nullptr, n, cconst, L->max_levels, t_next, L->level[k], L->active, L->n_active, nullptr, s)) != GOTHIC_OK) return rc;
    if ((rc = gothic_stage_walk(c, L->active, 0, L->n_active, L->eps, GOTHIC_MAC_ACCELERATION, delta_acc, r_crit, L->amag[k], L->acc_new, L->amag[k],
                                n_interactions, s)) != GOTHIC_OK) return rc;
    GOTHIC_CUDA_OK(c, cudaEventRecord(L->ev[2], s));
    L->timed = true;
    int cgrid = (int)grid;
    if (cgrid > c->num_sms * 16) cgrid = c->num_sms * 16;
    k_correct<<<cgrid, TPB, 0, s>>>(L->active, 0, L->n_active, c->pos_sorted, L->acc_new, t_next, dt_unit, L->pos[k], L->vel[k], L->acc[k], L->t_last[k],
                                    L->level[k], cconst, L->e_min, L->max_levels);
    GOTHIC_LAUNCH_OK(c);
    L->t_now = t_next;
    L->steps += 1ull;
    if (t_next == L->n_sub) return live_new_cycle(c, L, s);      // everybody synchronised: fresh levels, clock back to zero
    return GOTHIC_OK;
}

} // namespace

extern "C" {

int gothic_predict(gothic_ctx *c, const float *pos_m, const float *vel, const float *acc_pot, const uint32_t *t_last,
                   uint32_t t_now, float dt_unit, uint32_t n, float *pos_pred, void *stream)
{
    if (!c || !pos_m || !vel || !acc_pot || !t_last || !pos_pred || n == 0 || n > c->n_max || !(dt_unit > 0.0f)) return GOTHIC_ERR_ARG;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    k_predict<<<(n + TPB - 1) / TPB, TPB, 0, s>>>(reinterpret_cast<const float4 *>(pos_m), reinterpret_cast<const float4 *>(vel),
                                                  reinterpret_cast<const float4 *>(acc_pot), t_last, t_now, dt_unit, n,
                                                  reinterpret_cast<float4 *>(pos_pred));
    GOTHIC_LAUNCH_OK(c);
    return GOTHIC_OK;
}

int gothic_correct(gothic_ctx *c, const uint32_t *active, uint32_t n_active, const uint32_t *n_active_dev, uint32_t n,
                   const float *pos_pred, const float *acc_new, uint32_t t_now, float dt_unit, float *pos_m, float *vel,
                   float *acc_pot, uint32_t *t_last, uint8_t *level, float eps, float eta, int e_min, int max_levels, void *stream)
{
    if (!c || !pos_pred || !acc_new || !pos_m || !vel || !acc_pot || !t_last || n == 0 || n > c->n_max || !(dt_unit > 0.0f)) return GOTHIC_ERR_ARG;
    if (acc_new == acc_pot) return GOTHIC_ERR_ARG;
    if (!active) { n_active = n; n_active_dev = nullptr; }
    else if (!n_active_dev && n_active > n) return GOTHIC_ERR_ARG;
    if (level && (!(eps > 0.0f) || !(eta > 0.0f) || max_levels < 1 || max_levels > 32)) return GOTHIC_ERR_ARG;
    if (active && !n_active_dev && n_active == 0) return GOTHIC_OK;
    const double e4 = (double)eta * (double)eta * (double)eta * (double)eta;
    const float cconst = level ? (float)(e4 * (double)eps * (double)eps) : 0.0f;
    const uint32_t bound = n_active_dev ? n : n_active;
    int grid = (int)((bound + TPB - 1) / TPB);
    if (grid > c->num_sms * 16) grid = c->num_sms * 16;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    k_correct<<<grid, TPB, 0, s>>>(active, n_active, n_active_dev, reinterpret_cast<const float4 *>(pos_pred),
                                   reinterpret_cast<const float4 *>(acc_new), t_now, dt_unit, reinterpret_cast<float4 *>(pos_m),
                                   reinterpret_cast<float4 *>(vel), reinterpret_cast<float4 *>(acc_pot), t_last, level, cconst, e_min, max_levels);
    GOTHIC_LAUNCH_OK(c);
    return GOTHIC_OK;
}

int gothic_live_init(gothic_ctx *c, const float *pos_m, const float *vel, uint32_t n, int key_kind, int n_leaf, float eps, float eta,
                     int max_levels, float theta_boot, void *stream)
{
    if (!c || !pos_m || !vel || n == 0 || n > c->n_max || !(eps > 0.0f) || !(eta > 0.0f) || max_levels < 1 || max_levels > 32 || !(theta_boot >= 0.0f))
        return GOTHIC_ERR_ARG;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    gothic_live_free(c);
    gothic_live *L = new (std::nothrow) gothic_live;
    if (!L) return GOTHIC_ERR_ARG;
    memset(L, 0, sizeof(*L));
    c->live = L;
    L->n = n; L->key_kind = key_kind; L->n_leaf = n_leaf; L->max_levels = max_levels; L->eps = eps; L->eta = eta;
    cudaError_t e = cudaSuccess;
#define A(p, T, count) if (e == cudaSuccess) e = cudaMalloc(reinterpret_cast<void **>(&(p)), (size_t)(count) * sizeof(T))
    for (int k = 0; k < 2; k++) {
        A(L->pos[k], float4, n); A(L->vel[k], float4, n); A(L->acc[k], float4, n); A(L->amag[k], float, n);
        A(L->t_last[k], uint32_t, n); A(L->orig[k], uint32_t, n); A(L->level[k], uint8_t, n);
    }
    A(L->pred, float4, n); A(L->acc_new, float4, n); A(L->active, uint32_t, n); A(L->n_active, uint32_t, 1); A(L->info_dev, int32_t, 2);
#undef A
    for (int k = 0; k < 3; k++)
        if (e == cudaSuccess) e = cudaEventCreate(&L->ev[k]);
    if (e != cudaSuccess) { c->last_err = e; gothic_live_free(c); return GOTHIC_ERR_CUDA; }
    int rc = gothic_build_tree(c, pos_m, n, key_kind, n_leaf, stream);
    if (rc != GOTHIC_OK) return rc;
    const uint32_t grid = (n + TPB - 1) / TPB;
    // rows in tree order: positions are the build's gathered copy, velocities follow the permutation, orig = perm
    GOTHIC_CUDA_OK(c, cudaMemcpyAsync(L->pos[0], c->pos_sorted, (size_t)n * sizeof(float4), cudaMemcpyDeviceToDevice, s));
    GOTHIC_CUDA_OK(c, cudaMemcpyAsync(L->orig[0], c->idx[c->cur], (size_t)n * sizeof(uint32_t), cudaMemcpyDeviceToDevice, s));
    k_gather_vel<<<grid, TPB, 0, s>>>(c->idx[c->cur], n, reinterpret_cast<const float4 *>(vel), L->vel[0]);
    GOTHIC_LAUNCH_OK(c);
    rc = gothic_stage_walk(c, nullptr, 0, nullptr, eps, GOTHIC_MAC_OPENING_ANGLE, theta_boot, INFINITY, nullptr, L->acc[0], L->amag[0], nullptr, s);
    if (rc != GOTHIC_OK) return rc;
    L->cur = 0;
    L->steps = 0;
    L->steps_since_rebuild = 0;
    if ((rc = live_new_cycle(c, L, s)) != GOTHIC_OK) return rc;
    if ((rc = gothic_check(c, stream)) != GOTHIC_OK) return rc;
    L->tree_gen = c->tree_gen;
    L->ready = true;
    return GOTHIC_OK;
}

int gothic_live_step(gothic_ctx *c, float delta_acc, float r_crit, int rebuild, unsigned long long *n_interactions, void *stream)
{
    if (!c || !(delta_acc >= 0.0f) || !(r_crit >= 0.0f)) return GOTHIC_ERR_ARG;
    gothic_live *L = c->live;
    // not after a failed gothic_live_init / gothic_live_step, and not after somebody else's build on this context (gothic_build_tree,
    // gothic_gravity_host, gothic_block_cycle_host): the rows would no longer belong to the tree, even with the same n
    if (!L || !L->ready || !c->built || c->n != L->n || c->tree_gen != L->tree_gen) return GOTHIC_ERR_STATE;
    const int rc = live_step_stages(c, L, delta_acc, r_crit, rebuild, n_interactions, stream);
    if (rc != GOTHIC_OK) L->ready = false;       // gothic_live_init starts over
    return rc;
}

int gothic_live_timing(gothic_ctx *c, float *ms_host, uint32_t *n_active_host)
{
    if (!c || !ms_host) return GOTHIC_ERR_ARG;
    gothic_live *L = c->live;
    if (!L || !L->ready || !L->timed) return GOTHIC_ERR_STATE;
    GOTHIC_CUDA_OK(c, cudaEventSynchronize(L->ev[2]));
    GOTHIC_CUDA_OK(c, cudaEventElapsedTime(ms_host + 0, L->ev[0], L->ev[1]));
    GOTHIC_CUDA_OK(c, cudaEventElapsedTime(ms_host + 1, L->ev[1], L->ev[2]));
    if (n_active_host) GOTHIC_CUDA_OK(c, cudaMemcpy(n_active_host, L->n_active, sizeof(uint32_t), cudaMemcpyDeviceToHost));
    return GOTHIC_OK;
}

int gothic_live_get(gothic_ctx *c, gothic_live_state *out)
{
    if (!c || !out) return GOTHIC_ERR_ARG;
    const gothic_live *L = c->live;
    if (!L) return GOTHIC_ERR_STATE;
    const int k = L->cur;
    out->n = L->n; out->t_now = L->t_now; out->n_substeps = L->n_sub; out->e_min = L->e_min; out->n_levels = L->n_levels;
    out->steps_since_rebuild = L->steps_since_rebuild; out->steps = L->steps;
    out->pos_m = reinterpret_cast<const float *>(L->pos[k]); out->vel = reinterpret_cast<const float *>(L->vel[k]);
    out->acc_pot = reinterpret_cast<const float *>(L->acc[k]); out->amag = L->amag[k];
    out->t_last = L->t_last[k]; out->level = L->level[k]; out->orig = L->orig[k];
    out->active = L->active; out->n_active = L->n_active;
    return GOTHIC_OK;
}

} // extern "C"
