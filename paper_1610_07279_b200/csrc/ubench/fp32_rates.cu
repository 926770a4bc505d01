// Micro-benchmarks of the issue / FP32-pipe / XU / LDS rates that bound the walk's flush loop (W5) on sm_100a.
// Evidence for DESIGN.md section 7 and profiles/r02_microbench.md; not part of libgothic_b200.so.
//
//   nvcc -O3 -std=c++17 -gencode arch=compute_100a,code=sm_100a -lineinfo -o fp32_rates paper_1610_07279_b200/csrc/ubench/fp32_rates.cu
//   ./fp32_rates
//
// 1. k_rate: warp-instructions per clock per SM sub-partition (SMSP) of FFMA / FFMA2 / FADD2 / FMUL2 / MUFU.RSQ with
//    different numbers of distinct register operands (16 independent chains, 64 instructions per loop trip).
// 2. k_flush: the walk's interaction loop alone (a 256-entry list in shared memory, one i-particle per lane) in the
//    packed form the walk uses (V0), scalar (V1), hybrid (V2) and two re-associations (V3, V4), at several occupancies.
// 3. k_mixed: flush warps next to warps that run a pure ALU-pipe chain (LOP3 / SHF): does work on the other pipe
//    issue for free beside the packed FP32 stream?  (It does not: see profiles/r02_microbench.md.)
#include <cstdio>
#include <cstdlib>
#include <cstdint>
#include <cuda_runtime.h>
typedef unsigned long long u64;
#define CK(x) do { cudaError_t e = (x); if (e != cudaSuccess) { printf("CUDA error %s at %d\n", cudaGetErrorString(e), __LINE__); exit(1);} } while (0)

__device__ __forceinline__ u64 pack2(float lo, float hi) { u64 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ void unpack2(u64 v, float &lo, float &hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 c) { u64 r; asm volatile("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }
__device__ __forceinline__ u64 add2(u64 a, u64 b) { u64 r; asm volatile("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ u64 mul2(u64 a, u64 b) { u64 r; asm volatile("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ float rsq(float x) { float y; asm volatile("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float ffma(float a, float b, float c) { float r; asm volatile("fma.rn.f32 %0, %1, %2, %3;" : "=f"(r) : "f"(a), "f"(b), "f"(c)); return r; }

#define ITERS 1024
// kind 0: FFMA acc[i] = a[i]*b[i]+acc[i] (3 distinct regs)   1: FFMA acc[i] = a*b[i]+acc[i]   2: FFMA acc[i]=acc[i]*a+b (chain, 1 varying)
// 3: FFMA2 3 distinct  4: FFMA2 shared a  5: FFMA2 d*d+r  6: FADD2  7: FMUL2  8: MUFU.RSQ   9: FFMA imm
template <int KIND>
__global__ void __launch_bounds__(256) k_rate(float *out, long long *cyc, float s0, float s1)
{
    float a[16], b[16], c[16];
    u64 A[16], B[16], C[16];
#pragma unroll
    for (int i = 0; i < 16; i++) {
        a[i] = s0 + i + threadIdx.x; b[i] = s1 * (i + 1); c[i] = 0.f;
        A[i] = pack2(a[i], a[i] + 1.f); B[i] = pack2(b[i], b[i] + 2.f); C[i] = pack2(0.f, 0.f);
    }
    const u64 SA = pack2(s0, s1);
    long long t0 = clock64();
#pragma unroll 1
    for (int it = 0; it < ITERS; it++) {
#pragma unroll
        for (int rep = 0; rep < 4; rep++)
#pragma unroll
        for (int i = 0; i < 16; i++) {
            if (KIND == 0) c[i] = ffma(a[i], b[i], c[i]);
            if (KIND == 1) c[i] = ffma(s0, b[i], c[i]);
            if (KIND == 2) c[i] = ffma(c[i], s0, s1);
            if (KIND == 3) C[i] = fma2(A[i], B[i], C[i]);
            if (KIND == 4) C[i] = fma2(SA, B[i], C[i]);
            if (KIND == 5) C[i] = fma2(B[i], B[i], C[i]);
            if (KIND == 6) C[i] = add2(C[i], B[i]);
            if (KIND == 7) C[i] = mul2(C[i], B[i]);
            if (KIND == 8) c[i] = rsq(c[i]);
            if (KIND == 9) c[i] = ffma(c[i], 1.0001f, 0.5f);
        }
    }
    long long t1 = clock64();
    float s = 0;
#pragma unroll
    for (int i = 0; i < 16; i++) { float lo, hi; unpack2(C[i], lo, hi); s += c[i] + lo + hi; }
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
    if (threadIdx.x == 0) cyc[blockIdx.x] = t1 - t0;
}

// ---------------- flush alone: a list of NL entries in shared memory, every lane its own i-particle ----------------
constexpr int NL = 256;
struct Acc2 { u64 ax, ay, az, pot; };
__device__ __forceinline__ u64 fma2n(u64 a, u64 b, u64 c) { u64 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }
__device__ __forceinline__ u64 add2n(u64 a, u64 b) { u64 r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ u64 mul2n(u64 a, u64 b) { u64 r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ float rsqn(float x) { float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

// V0: all packed (the walk's interact2)
__device__ __forceinline__ void interact2_v0(u64 xj, u64 yj, u64 zj, u64 mj, u64 npx, u64 npy, u64 npz, u64 eps2, Acc2 &a)
{
    const u64 dx = add2n(xj, npx), dy = add2n(yj, npy), dz = add2n(zj, npz);
    u64 r2 = fma2n(dx, dx, eps2); r2 = fma2n(dy, dy, r2); r2 = fma2n(dz, dz, r2);
    float r2a, r2b; unpack2(r2, r2a, r2b);
    const u64 u = pack2(rsqn(r2a), rsqn(r2b));
    const u64 mu = mul2n(mj, u);
    a.pot = add2n(a.pot, mu);
    const u64 f = mul2n(mu, mul2n(u, u));
    a.ax = fma2n(f, dx, a.ax); a.ay = fma2n(f, dy, a.ay); a.az = fma2n(f, dz, a.az);
}
// V1: scalar everything
__device__ __forceinline__ void interact1(float xj, float yj, float zj, float mj, float px, float py, float pz, float e2, float &ax, float &ay, float &az, float &pot)
{
    const float dx = xj - px, dy = yj - py, dz = zj - pz;
    const float r2 = fmaf(dz, dz, fmaf(dy, dy, fmaf(dx, dx, e2)));
    const float u = rsqn(r2);
    const float mu = mj * u;
    pot += mu;
    const float f = mu * (u * u);
    ax = fmaf(f, dx, ax); ay = fmaf(f, dy, ay); az = fmaf(f, dz, az);
}
// V2: hybrid: sub, r2 and mul packed; the three accumulating FMAs and the potential add scalar
__device__ __forceinline__ void interact2_v2(u64 xj, u64 yj, u64 zj, u64 mj, u64 npx, u64 npy, u64 npz, u64 eps2, float &ax, float &ay, float &az, float &pot)
{
    const u64 dx = add2n(xj, npx), dy = add2n(yj, npy), dz = add2n(zj, npz);
    u64 r2 = fma2n(dx, dx, eps2); r2 = fma2n(dy, dy, r2); r2 = fma2n(dz, dz, r2);
    float r2a, r2b; unpack2(r2, r2a, r2b);
    const u64 u = pack2(rsqn(r2a), rsqn(r2b));
    const u64 mu = mul2n(mj, u);
    const u64 f = mul2n(mu, mul2n(u, u));
    float f0, f1, d0, d1, m0, m1;
    unpack2(mu, m0, m1); pot += m0; pot += m1;
    unpack2(f, f0, f1);
    unpack2(dx, d0, d1); ax = fmaf(f0, d0, ax); ax = fmaf(f1, d1, ax);
    unpack2(dy, d0, d1); ay = fmaf(f0, d0, ay); ay = fmaf(f1, d1, ay);
    unpack2(dz, d0, d1); az = fmaf(f0, d0, az); az = fmaf(f1, d1, az);
}
// V3: packed, potential folded as fma(m, u, pot) and f = (m u) (u u) -> still 13; variant with pot via fma2 to test FADD2 vs FFMA2 port
__device__ __forceinline__ void interact2_v3(u64 xj, u64 yj, u64 zj, u64 mj, u64 npx, u64 npy, u64 npz, u64 eps2, Acc2 &a)
{
    const u64 dx = add2n(xj, npx), dy = add2n(yj, npy), dz = add2n(zj, npz);
    u64 r2 = fma2n(dx, dx, eps2); r2 = fma2n(dy, dy, r2); r2 = fma2n(dz, dz, r2);
    float r2a, r2b; unpack2(r2, r2a, r2b);
    const u64 u = pack2(rsqn(r2a), rsqn(r2b));
    a.pot = fma2n(mj, u, a.pot);
    const u64 f = mul2n(mul2n(mj, u), mul2n(u, u));
    a.ax = fma2n(f, dx, a.ax); a.ay = fma2n(f, dy, a.ay); a.az = fma2n(f, dz, a.az);
}


__device__ __forceinline__ void interact2_v4(u64 xj, u64 yj, u64 zj, u64 mj, u64 npx, u64 npy, u64 npz, u64 eps2, Acc2 &a)
{
    const u64 dx = add2n(xj, npx), dy = add2n(yj, npy), dz = add2n(zj, npz);
    u64 r2 = fma2n(dx, dx, eps2); r2 = fma2n(dy, dy, r2); r2 = fma2n(dz, dz, r2);
    float r2a, r2b; unpack2(r2, r2a, r2b);
    const u64 u = pack2(rsqn(r2a), rsqn(r2b));
    const u64 mu = mul2n(mj, u);
    a.pot = add2n(a.pot, mu);
    const u64 f = mul2n(mu, mul2n(u, u));
    asm("fma.rn.f32x2 %0, %3, %4, %0;\n\tfma.rn.f32x2 %1, %3, %5, %1;\n\tfma.rn.f32x2 %2, %3, %6, %2;" : "+l"(a.ax), "+l"(a.ay), "+l"(a.az) : "l"(f), "l"(dx), "l"(dy), "l"(dz));
}

template <int V, int MINB>
__global__ void __launch_bounds__(256, MINB) k_flush(const float4 *pts, float4 *out, int reps, float eps2, long long *cyc)
{
    __shared__ __align__(16) float sx[8][4 * NL];
    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    float *L = sx[w];
    for (int e = lane; e < NL; e += 32) {
        const float4 q = pts[(blockIdx.x * 8 + w) * NL + e];
        L[e] = q.x; L[NL + e] = q.y; L[2 * NL + e] = q.z; L[3 * NL + e] = q.w;
    }
    __syncwarp();
    const float4 pi = pts[blockIdx.x * 256 + threadIdx.x];
    const u64 npx = pack2(-pi.x, -pi.x), npy = pack2(-pi.y, -pi.y), npz = pack2(-pi.z, -pi.z), e2 = pack2(eps2, eps2);
    Acc2 a = {0, 0, 0, 0};
    float ax = 0, ay = 0, az = 0, pot = 0;
    long long t0 = clock64();
#pragma unroll 1
    for (int r = 0; r < reps; r++) {
#pragma unroll 1
        for (int blk = 0; blk < NL; blk += 32) {
#pragma unroll
            for (int c = 0; c < 8; c++) {
                const float *x0 = L + blk + 4 * c;
                if (V == 1) {
                    const float4 X = *reinterpret_cast<const float4 *>(x0), Y = *reinterpret_cast<const float4 *>(x0 + NL);
                    const float4 Z = *reinterpret_cast<const float4 *>(x0 + 2 * NL), M = *reinterpret_cast<const float4 *>(x0 + 3 * NL);
                    interact1(X.x, Y.x, Z.x, M.x, pi.x, pi.y, pi.z, eps2, ax, ay, az, pot);
                    interact1(X.y, Y.y, Z.y, M.y, pi.x, pi.y, pi.z, eps2, ax, ay, az, pot);
                    interact1(X.z, Y.z, Z.z, M.z, pi.x, pi.y, pi.z, eps2, ax, ay, az, pot);
                    interact1(X.w, Y.w, Z.w, M.w, pi.x, pi.y, pi.z, eps2, ax, ay, az, pot);
                } else {
                    const ulonglong2 X = *reinterpret_cast<const ulonglong2 *>(x0), Y = *reinterpret_cast<const ulonglong2 *>(x0 + NL);
                    const ulonglong2 Z = *reinterpret_cast<const ulonglong2 *>(x0 + 2 * NL), M = *reinterpret_cast<const ulonglong2 *>(x0 + 3 * NL);
                    if (V == 0) { interact2_v0(X.x, Y.x, Z.x, M.x, npx, npy, npz, e2, a); interact2_v0(X.y, Y.y, Z.y, M.y, npx, npy, npz, e2, a); }
                    if (V == 2) { interact2_v2(X.x, Y.x, Z.x, M.x, npx, npy, npz, e2, ax, ay, az, pot); interact2_v2(X.y, Y.y, Z.y, M.y, npx, npy, npz, e2, ax, ay, az, pot); }
                    if (V == 3) { interact2_v3(X.x, Y.x, Z.x, M.x, npx, npy, npz, e2, a); interact2_v3(X.y, Y.y, Z.y, M.y, npx, npy, npz, e2, a); }
                    if (V == 4) { interact2_v4(X.x, Y.x, Z.x, M.x, npx, npy, npz, e2, a); interact2_v4(X.y, Y.y, Z.y, M.y, npx, npy, npz, e2, a); }
                }
            }
        }
    }
    long long t1 = clock64();
    float lo, hi;
    unpack2(a.ax, lo, hi); ax += lo + hi; unpack2(a.ay, lo, hi); ay += lo + hi; unpack2(a.az, lo, hi); az += lo + hi; unpack2(a.pot, lo, hi); pot += lo + hi;
    out[blockIdx.x * 256 + threadIdx.x] = make_float4(ax, ay, az, pot);
    if (threadIdx.x == 0) cyc[blockIdx.x] = t1 - t0;
}

static float *d_out; static long long *d_cyc; static int n_sm;

// warps 0..NF-1 of each CTA flush, the others run an ALU-pipe chain (LOP3/SHF) of n_alu instructions per flush block of 32 entries
template <int NF>
__global__ void __launch_bounds__(256, 4) k_mixed(const float4 *pts, float4 *out, int reps, float eps2, int alu_on, unsigned *sink)
{
    __shared__ __align__(16) float sx[8][4 * NL];
    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (w >= NF) {
        if (!alu_on) return;
        unsigned x = threadIdx.x * 2654435761u, y = blockIdx.x + 17u, z = 0x9e3779b9u, t = lane;
#pragma unroll 1
        for (int r = 0; r < reps * 8; r++) {
#pragma unroll
            for (int k = 0; k < 64; k++) {
                asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(x) : "r"(y), "r"(z));
                asm volatile("shf.l.wrap.b32 %0, %0, %1, 7;" : "+r"(y) : "r"(x));
                asm volatile("lop3.b32 %0, %0, %1, %2, 0xe8;" : "+r"(z) : "r"(x), "r"(t));
                asm volatile("shf.r.wrap.b32 %0, %0, %1, 3;" : "+r"(t) : "r"(z));
            }
        }
        sink[blockIdx.x * 256 + threadIdx.x] = x ^ y ^ z ^ t;
        return;
    }
    float *L = sx[w];
    for (int e = lane; e < NL; e += 32) {
        const float4 q = pts[(blockIdx.x * 8 + w) * NL + e];
        L[e] = q.x; L[NL + e] = q.y; L[2 * NL + e] = q.z; L[3 * NL + e] = q.w;
    }
    __syncwarp();
    const float4 pi = pts[blockIdx.x * 256 + threadIdx.x];
    const u64 npx = pack2(-pi.x, -pi.x), npy = pack2(-pi.y, -pi.y), npz = pack2(-pi.z, -pi.z), e2 = pack2(eps2, eps2);
    Acc2 a = {0, 0, 0, 0};
#pragma unroll 1
    for (int r = 0; r < reps; r++) {
#pragma unroll 1
        for (int blk = 0; blk < NL; blk += 32) {
#pragma unroll
            for (int c = 0; c < 8; c++) {
                const float *x0 = L + blk + 4 * c;
                const ulonglong2 X = *reinterpret_cast<const ulonglong2 *>(x0), Y = *reinterpret_cast<const ulonglong2 *>(x0 + NL);
                const ulonglong2 Z = *reinterpret_cast<const ulonglong2 *>(x0 + 2 * NL), M = *reinterpret_cast<const ulonglong2 *>(x0 + 3 * NL);
                interact2_v0(X.x, Y.x, Z.x, M.x, npx, npy, npz, e2, a); interact2_v0(X.y, Y.y, Z.y, M.y, npx, npy, npz, e2, a);
            }
        }
    }
    float ax, ay, az, pot, lo, hi;
    unpack2(a.ax, lo, hi); ax = lo + hi; unpack2(a.ay, lo, hi); ay = lo + hi; unpack2(a.az, lo, hi); az = lo + hi; unpack2(a.pot, lo, hi); pot = lo + hi;
    out[blockIdx.x * 256 + threadIdx.x] = make_float4(ax, ay, az, pot);
}
template <int NF> void run_mixed(const char *name, const float4 *pts, float4 *out, int reps, int alu_on)
{
    const int grid = n_sm * 4;
    unsigned *sink; cudaMalloc(&sink, grid * 256 * 4);
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    k_mixed<NF><<<grid, 256>>>(pts, out, reps, 1e-4f, alu_on, sink);
    cudaEventRecord(e0);
    k_mixed<NF><<<grid, 256>>>(pts, out, reps, 1e-4f, alu_on, sink);
    cudaEventRecord(e1); CK(cudaDeviceSynchronize());
    float ms; cudaEventElapsedTime(&ms, e0, e1);
    const double inter = (double)grid * NF * 32 * NL * reps;
    const double alu = alu_on ? (double)grid * (8 - NF) * reps * 8.0 * 256 : 0;      // warp instructions
    printf("%-44s flush warps/SMSP %d alu warps/SMSP %d: %.2f inter/clk/SM (frac %.3f), alu %.3f warp-instr/clk/SMSP, ms %.3f\n", name, NF, alu_on ? 8 - NF : 0,
           inter / (ms * 1e-3) / n_sm / 1.965e9, inter * 24 / (ms * 1e-3) / (n_sm * 128 * 2 * 1.965e9), alu / (ms * 1e-3) / (n_sm * 4) / 1.965e9, ms);
    cudaFree(sink);
}

template <int KIND> void run_rate(const char *name, int ctas_per_sm, int ops_per_instr)
{
    const int grid = n_sm * ctas_per_sm;
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    k_rate<KIND><<<grid, 256>>>(d_out, d_cyc, 1.0f, 1e-3f);
    cudaEventRecord(e0);
    k_rate<KIND><<<grid, 256>>>(d_out, d_cyc, 1.0f, 1e-3f);
    cudaEventRecord(e1); CK(cudaDeviceSynchronize());
    float ms; cudaEventElapsedTime(&ms, e0, e1);
    long long c; cudaMemcpy(&c, d_cyc, 8, cudaMemcpyDeviceToHost);
    const double instr_per_smsp = (double)ITERS * 64 * (ctas_per_sm * 8 / 4);      // warps per SMSP x instr per warp
    (void)c;
    printf("%-34s warps/SMSP %2d  %.3f warp-instr/clk/SMSP = %.2f issue cycles per instruction (CUDA events, 1.965 GHz)  ms %.3f\n", name, ctas_per_sm * 2,
           instr_per_smsp / (ms * 1e-3 * 1.965e9), (ms * 1e-3 * 1.965e9) / instr_per_smsp, ms);
}
template <int V, int MINB> void run_flush(const char *name, const float4 *pts, float4 *out, int reps)
{
    const int grid = n_sm * MINB;
    int occ = 0; cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_flush<V, MINB>, 256, 0);
    cudaFuncAttributes fa; cudaFuncGetAttributes(&fa, k_flush<V, MINB>);
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    k_flush<V, MINB><<<grid, 256>>>(pts, out, reps, 1e-4f, d_cyc);
    cudaEventRecord(e0);
    k_flush<V, MINB><<<grid, 256>>>(pts, out, reps, 1e-4f, d_cyc);
    cudaEventRecord(e1); CK(cudaDeviceSynchronize());
    float ms; cudaEventElapsedTime(&ms, e0, e1);
    const double inter = (double)grid * 256 * NL * reps;
    printf("%-34s regs %3d occ %d CTAs/SM  %.3e inter/s  %.2f inter/clk/SM  frac of 24-flop peak %.3f  ms %.3f\n", name, fa.numRegs, occ,
           inter / (ms * 1e-3), inter / (ms * 1e-3) / n_sm / 1.965e9, inter * 24 / (ms * 1e-3) / (n_sm * 128 * 2 * 1.965e9), ms);
}

int main()
{
    cudaDeviceProp p; CK(cudaGetDeviceProperties(&p, 0)); n_sm = p.multiProcessorCount;
    int clk; cudaDeviceGetAttribute(&clk, cudaDevAttrClockRate, 0);
    printf("device %s, %d SMs, clock attr %d kHz\n", p.name, n_sm, clk);
    CK(cudaMalloc(&d_out, (size_t)n_sm * 8 * 256 * 16)); CK(cudaMalloc(&d_cyc, n_sm * 8 * 8));
    run_rate<0>("FFMA 3 distinct regs", 4, 1); run_rate<0>("FFMA 3 distinct regs", 8, 1);
    run_rate<1>("FFMA shared multiplicand", 4, 1);
    run_rate<2>("FFMA c=c*s0+s1", 4, 1);
    run_rate<9>("FFMA imm", 4, 1);
    run_rate<3>("FFMA2 3 distinct", 4, 2); run_rate<3>("FFMA2 3 distinct", 8, 2);
    run_rate<4>("FFMA2 shared a", 4, 2);
    run_rate<5>("FFMA2 b*b+c", 4, 2);
    run_rate<6>("FADD2", 4, 2);
    run_rate<7>("FMUL2", 4, 2);
    run_rate<8>("MUFU.RSQ", 4, 1);
    float4 *pts, *out;
    const size_t np = (size_t)n_sm * 8 * 8 * NL;
    CK(cudaMalloc(&pts, np * 16)); CK(cudaMalloc(&out, np * 16));
    float4 *h = (float4 *)malloc(np * 16);
    srand(1);
    for (size_t i = 0; i < np; i++) h[i] = make_float4(rand() / (float)RAND_MAX, rand() / (float)RAND_MAX, rand() / (float)RAND_MAX, 1e-3f);
    CK(cudaMemcpy(pts, h, np * 16, cudaMemcpyHostToDevice));
    const int reps = 400;
    run_flush<0, 4>("flush V0 packed (walk) 4 CTAs", pts, out, reps);
    run_flush<0, 3>("flush V0 packed 3 CTAs", pts, out, reps);
    run_flush<0, 5>("flush V0 packed 5 CTAs", pts, out, reps);
    run_flush<0, 6>("flush V0 packed 6 CTAs", pts, out, reps);
    run_flush<0, 8>("flush V0 packed 8 CTAs", pts, out, reps);
    run_flush<1, 4>("flush V1 scalar 4 CTAs", pts, out, reps);
    run_flush<1, 6>("flush V1 scalar 6 CTAs", pts, out, reps);
    run_flush<2, 4>("flush V2 hybrid 4 CTAs", pts, out, reps);
    run_flush<2, 6>("flush V2 hybrid 6 CTAs", pts, out, reps);
    run_flush<3, 4>("flush V3 packed pot-fma 4 CTAs", pts, out, reps);
    run_flush<3, 6>("flush V3 packed pot-fma 6 CTAs", pts, out, reps);
    run_flush<4, 4>("flush V4 acc-asm-block 4 CTAs", pts, out, reps);
    run_flush<4, 3>("flush V4 acc-asm-block 3 CTAs", pts, out, reps);
    run_flush<0, 2>("flush V0 packed 2 CTAs (<=128 regs)", pts, out, reps);
    run_flush<0, 1>("flush V0 packed 1 CTA (<=255 regs)", pts, out, reps);
    run_flush<3, 2>("flush V3 packed pot-fma 2 CTAs", pts, out, reps);
    run_mixed<8>("mixed: 8 flush warps/CTA", pts, out, reps, 0);
    run_mixed<6>("mixed: 6 flush, 2 idle", pts, out, reps, 0);
    run_mixed<6>("mixed: 6 flush, 2 ALU chains", pts, out, reps, 1);
    run_mixed<4>("mixed: 4 flush, 4 idle", pts, out, reps, 0);
    run_mixed<4>("mixed: 4 flush, 4 ALU chains", pts, out, reps, 1);
    return 0;
}
