// Orbit integration under block time steps (eq. 15-17; NEXT row f1): prediction of all j-particles to the
// current time and correction of the active i-particles, with the level migration of DESIGN.md R15.  Both kernels are pure
// streaming passes (HBM bound): predict reads 52 B and writes 16 B per particle; correct touches only the active rows.
// Arithmetic order is part of the contract (bit-exact against the oracle): one fmaf per component, as written.
#include "gothic_ctx.cuh"

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

} // extern "C"
